"""Comparison helpers of the GPU parity tests (test infrastructure; imports nothing from the
product or the oracle -- it only compares the dictionaries both bindings return).

Tolerances (BASELINE.json north_star; derivation in DESIGN.md "Parity tolerances"):
  links                      bit-exact after sorting by (pid, alpha, j, i), q compared bitwise
  f, g, rho, T, (ux,uy)      max|a-b| / max|b| <= 1e-10 on nodes that are fluid on both sides
  particle x, U (and theta, Omega)   <= 1e-9 relative to the vector's scale
"""
import numpy as np

FIELD_TOL = 1e-10
PARTICLE_TOL = 1e-9


def sorted_links(L):
    order = np.lexsort((L["i"], L["j"], L["alpha"], L["pid"]))
    return {k: np.asarray(v)[order] for k, v in L.items()}


def assert_links_equal(a, b):
    a, b = sorted_links(a), sorted_links(b)
    assert len(a["q"]) == len(b["q"]), (len(a["q"]), len(b["q"]))
    for k in ("pid", "alpha", "j", "i"):
        assert np.array_equal(a[k], b[k]), k
    # bitwise: the same separately rounded operations on both sides
    assert np.array_equal(a["q"].view(np.uint64), b["q"].view(np.uint64)), \
        float(np.abs(a["q"] - b["q"]).max())


def rel_err(a, b, mask=None, floor=0.0):
    """max|a-b| / max(max|b|, floor) over `mask` (broadcast over leading population axes)."""
    a, b = np.asarray(a), np.asarray(b)
    if mask is not None:
        a, b = a[..., mask], b[..., mask]
    if a.size == 0:
        return 0.0
    scale = max(float(np.abs(b).max()), floor)
    d = float(np.abs(a - b).max())
    return d / scale if scale > 0.0 else d


def assert_fields_close(gpu, ora, tol=FIELD_TOL, populations=True):
    """gpu, ora: dicts from Simulation.fields(populations=True) / OracleSim.fields(...)."""
    assert np.array_equal(gpu["flag"], ora["flag"]), \
        f"flag maps differ on {int((gpu['flag'] != ora['flag']).sum())} nodes"
    fluid = ora["flag"] == 0
    errs = {}
    errs["rho"] = rel_err(gpu["rho"], ora["rho"], fluid)
    errs["T"] = rel_err(gpu["T"], ora["T"], fluid, floor=1e-30)
    # velocity is a vector field: one scale for both components.  Floor 1e-6: a velocity field
    # that is pure round-off noise (|u| ~ 1e-17, e.g. pure conduction) has no scale of its own;
    # every flow of the configs has |u| >= 1e-4, so the floor never loosens a real comparison
    uscale = max(float(np.abs(ora["ux"][fluid]).max(initial=0.0)),
                 float(np.abs(ora["uy"][fluid]).max(initial=0.0)), 1e-6)
    for k in ("ux", "uy"):
        errs[k] = float(np.abs(gpu[k][fluid] - ora[k][fluid]).max(initial=0.0)) / uscale
    # solid nodes: rigid-body velocity and wall temperature
    solid = ~fluid
    if solid.any():
        for k in ("rho", "T", "ux", "uy"):
            errs[k + "_solid"] = rel_err(gpu[k], ora[k], solid, floor=1e-6)
    if populations:
        errs["f"] = rel_err(gpu["f"], ora["f"], fluid)
        errs["g"] = rel_err(gpu["g"], ora["g"], fluid, floor=1e-30)
    bad = {k: v for k, v in errs.items() if not (v <= tol)}
    assert not bad, f"field parity failed: {bad} (all: {errs})"
    return errs


def assert_particles_close(gpu, ora, r_min, tol=PARTICLE_TOL, steps=1):
    n = len(ora["x"])
    assert len(gpu["x"]) == n
    if n == 0:
        return {}
    errs = {}
    pos_scale = max(float(np.abs(ora["x"]).max()), float(np.abs(ora["y"]).max()))
    vel_scale = max(float(np.abs(ora["ux"]).max()), float(np.abs(ora["uy"]).max()), 1e-30)
    # rotation is zero up to round-off for a symmetric single particle: its natural scale is the
    # rim speed U / r, not the noise itself
    om_scale = max(float(np.abs(ora["omega"]).max()), vel_scale / r_min)
    th_scale = max(float(np.abs(ora["theta"]).max()), om_scale * max(steps, 1))
    # the hydrodynamic force is a cancelling sum of ~20 r link terms of size ~ w_i rho0 ~ 0.1; on a
    # particle at rest in fluid at rest it is pure round-off (1e-18), which has no scale of its
    # own: floor = 1e-6 r (lattice units, rho0 = 1), i.e. an absolute tolerance of 1e-15 r
    f_scale = max(float(np.abs(ora["Fx"]).max()), float(np.abs(ora["Fy"]).max()), 1e-6 * r_min)
    t_scale = max(float(np.abs(ora["Tz"]).max()), f_scale * r_min)
    for k, s in (("x", pos_scale), ("y", pos_scale), ("ux", vel_scale), ("uy", vel_scale),
                 ("omega", om_scale), ("theta", th_scale), ("Fx", f_scale), ("Fy", f_scale),
                 ("Tz", t_scale)):
        errs[k] = float(np.abs(gpu[k] - ora[k]).max()) / s
    bad = {k: v for k, v in errs.items() if not (v <= tol)}
    assert not bad, f"particle parity failed: {bad} (all: {errs})"
    return errs
