"""Builds the C-ABI shared library (hand-written sm_100a CUDA) in-tree:
paper_2308_16597_b200/liblbm_b200.so.  nvcc cross-compiles without a GPU.

particles.cu is compiled with -fmad=false (integer-valued geometric decisions must use separately
rounded operations, see the file header); everything else keeps FMA contraction.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OUT = os.path.join(HERE, "liblbm_b200.so")
OBJ = os.path.join(HERE, "build")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")

COMMON = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
          "-Xcompiler", "-fPIC", "-Xcompiler", "-Wall", "-Xptxas", "-v"]
SOURCES = {
    "stream_collide.cu": [],
    "bounce_back.cu": [],
    "particles.cu": ["-fmad=false"],
    "lbm_capi.cu": [],
}


def _deps():
    d = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    d.append(os.path.join(HERE, "..", "include", "lbm.h"))
    d.append(os.path.abspath(__file__))
    return d


def build(force: bool = False, verbose: bool = False) -> str:
    if (not force and os.path.exists(OUT)
            and all(os.path.getmtime(OUT) >= os.path.getmtime(d) for d in _deps())):
        return OUT
    os.makedirs(OBJ, exist_ok=True)
    objs = []
    log = []
    for src, extra in SOURCES.items():
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        cmd = [NVCC, *COMMON, *extra, "-c", os.path.join(CSRC, src), "-o", o]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
        if r.returncode != 0:
            sys.stderr.write(log[-1])
            raise RuntimeError(f"nvcc failed on {src}")
        objs.append(o)
    cmd = [NVCC, "-shared", "-o", OUT, *objs]
    r = subprocess.run(cmd, capture_output=True, text=True)
    log.append("$ " + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    if r.returncode != 0:
        sys.stderr.write(log[-1])
        raise RuntimeError("link failed")
    with open(os.path.join(OBJ, "build.log"), "w") as fh:
        fh.write("\n".join(log))
    if verbose:
        print("\n".join(log))
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
