"""lbm_get_macroscopic_static (include/lbm.h): the macroscopic read-out whose device scratch is a
file-scope static array of the library -- no cudaMalloc, the caller's workspace untouched.  Its
output must equal the existing path's (lbm_get_fields) on two calls in a row, although every call
shares the array and finds the previous call's contents in it; lattices beyond the stated maximum
are rejected with a clear error.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from parity import FIELD_TOL, rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2308_16597_b200 import binding
    binding.load_library()
    return binding


def assert_matches_existing_path(sim):
    a = sim.macroscopic_static()
    b = sim.fields()
    for k in ("rho", "ux", "uy", "T"):
        assert np.isfinite(a[k]).all(), k
        assert rel_err(a[k], b[k], None, floor=1e-6) <= FIELD_TOL, k
        assert np.array_equal(a[k], b[k]), k          # the same kernel arithmetic: the same bits
    return a


def test_static_scratch_readout_equals_get_fields_on_two_calls_in_a_row(gpu, wl):
    # a lattice with moving particles (solid nodes read the rigid-body velocity through the owner map)
    w = wl.sedimentation(300, 260, 14, seed=9, y_frac_lo=0.2, d_lo=12.0, d_hi=24.0, name="noalloc")
    big = gpu.Simulation.from_workload(w)
    big.step(40)
    first = assert_matches_existing_path(big)
    # second call, on a SMALLER lattice of another simulation: the array still holds the first
    # call's fields beyond (and under) what this call writes; none of it may show
    w2 = wl.config(0)
    small = gpu.Simulation.from_workload(w2)
    small.step(25)
    second = assert_matches_existing_path(small)
    assert second["rho"].shape == (256, 128) and first["rho"].shape == (260, 300)
    # and back to back on the first one after more steps: the workspace was left alone meanwhile
    big.step(17)
    third = assert_matches_existing_path(big)
    assert not np.array_equal(third["uy"], first["uy"])
    # stepping after the read-outs continues exactly like a simulation that was never read out
    ref = gpu.Simulation.from_workload(w)
    ref.step(40 + 17)
    pa, pb = big.particles(), ref.particles()
    for k in pa:
        assert np.array_equal(pa[k], pb[k]), k


def test_static_scratch_readout_rejects_lattices_beyond_its_maximum(gpu, wl):
    p = wl.default_params()
    ok = gpu.Simulation(1024, 1024, p)                 # exactly the maximum: 2^20 nodes
    ok.step(2)
    assert_matches_existing_path(ok)
    ok.close()
    too_big = gpu.Simulation(1025, 1024, p)
    with pytest.raises(gpu.LbmError) as e:
        too_big.macroscopic_static()
    assert e.value.code == gpu.LBM_E_CAPACITY and "LBM_STATIC_MAX_NODES" in str(e.value)
    too_big.step(1)                                    # the handle is still usable
    too_big.close()
