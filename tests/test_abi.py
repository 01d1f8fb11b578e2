"""The C-ABI library builds, loads, and exports every symbol include/lbm.h declares.
No compute call is made here (there is no GPU on the CPU test box)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2308_16597_b200 import build
    path = build.build()
    assert os.path.exists(path)
    from paper_2308_16597_b200 import binding
    return binding.load_library()


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_]+)\s*\(", text)))


def test_header_declares_the_north_star_calls():
    names = declared_symbols()
    for required in ("lbm_create", "lbm_add_particles", "lbm_step", "lbm_get_fields",
                     "lbm_get_particles", "lbm_get_links", "lbm_set_temperature",
                     "lbm_workspace_bytes", "lbm_destroy", "lbm_last_error"):
        assert required in names


def test_every_declared_symbol_is_exported(lib):
    for name in declared_symbols():
        assert hasattr(lib, name), f"{name} declared in include/lbm.h but not exported"


def test_params_struct_layout_and_defaults(lib):
    from paper_2308_16597_b200.binding import LbmParams
    p = LbmParams()
    lib.lbm_params_default(C.byref(p))
    assert p.nu == 0.02 and p.rho0 == 1.0 and p.rep_power == 1 and p.rep_s == 2.0
    assert p.kappa == pytest.approx(0.02 / 0.7)
    assert list(p.wall_T_type) == [0, 0, 0, 0] and p.max_particles == 0
    assert C.sizeof(LbmParams) == 152   # 8 doubles, int+pad... must match the C struct (checked below)
    # host-only call: workspace size grows with the lattice and is at least two copies of 14 planes
    p.max_particles, p.max_links_per_particle = 10, 276
    small = lib.lbm_workspace_bytes(128, 256, C.byref(p))
    big = lib.lbm_workspace_bytes(256, 256, C.byref(p))
    assert small >= 2 * 14 * 8 * 128 * 256 and big > small
    assert lib.lbm_workspace_bytes(2, 2, C.byref(p)) == 0          # too small a lattice
    p.kappa = 0.2
    assert lib.lbm_workspace_bytes(128, 128, C.byref(p)) == 0      # kappa outside the D2Q5 range


def test_profile_kernel_names(lib):
    n = lib.lbm_profile_kernels()
    names = [lib.lbm_profile_kernel_name(k).decode() for k in range(n)]
    assert names[0] == "stream_collide" and "build_links" in names and "refill" in names


def test_null_handle_is_rejected(lib):
    assert lib.lbm_step(None, 1) == -1
    assert lib.lbm_destroy(None) == 0
    out = C.c_void_p()
    from paper_2308_16597_b200.binding import LbmParams
    p = LbmParams()
    lib.lbm_params_default(C.byref(p))
    # NULL workspace: rejected before any CUDA call
    assert lib.lbm_create(64, 64, C.byref(p), None, 0, None, C.byref(out)) == -1
    assert b"workspace" in lib.lbm_last_error(None)


def test_product_does_not_touch_the_oracle():
    """The product package must not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2308_16597_b200")
    for dirpath, _, files in os.walk(pkg):
        if os.path.basename(dirpath) == "build":
            continue
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "oracle_binding" not in text and "lbm_oracle" not in text, fn
