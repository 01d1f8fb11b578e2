"""Builds the CPU oracle (TEST INFRASTRUCTURE) into oracle/liblbm_oracle.so.

Plain g++ -O2 -ffp-contract=off: no FMA contraction, so the oracle's integer decisions (solid
test, e_c choice) use separately rounded operations.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "lbm_oracle.cpp")
OUT = os.path.join(HERE, "liblbm_oracle.so")


def build(force: bool = False) -> str:
    deps = [SRC, os.path.join(HERE, "lbm_oracle.h")]
    if (not force and os.path.exists(OUT)
            and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in deps)):
        return OUT
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", OUT, SRC]
    subprocess.run(cmd, check=True)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
