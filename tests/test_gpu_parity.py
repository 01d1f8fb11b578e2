"""GPU parity tests proper: the CUDA path (through the C ABI, via the thin binding) against the
paper-order CPU oracle on the same seeded inputs, element by element.

Sizes here are ones the oracle finishes in seconds; every lattice spans several 128-thread tiles
and has a ragged tail (nx not a multiple of 128 / 16).  Full-size cases are in
test_gpu_fullsize.py.  Tolerances: tests/parity.py.
"""
import numpy as np
import pytest

from parity import (assert_fields_close, assert_links_equal, assert_particles_close)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2308_16597_b200 import binding
    binding.load_library()   # fails loudly if the CUDA library is missing: there is no fallback
    return binding


def both(gpu, ob, w):
    return gpu.Simulation.from_workload(w), ob.OracleSim.from_workload(w)


def run_and_compare(gpu, ob, w, checkpoints, r_min=10.0, links=True):
    g, o = both(gpu, ob, w)
    if links and w.particles is not None:
        assert_links_equal(g.links(), o.links())
    assert_fields_close(g.fields(populations=True), o.fields(populations=True))
    done = 0
    out = {}
    for c in checkpoints:
        g.step(c - done)
        o.step(c - done)
        done = c
        out[c] = assert_fields_close(g.fields(populations=True), o.fields(populations=True))
        if w.particles is not None:
            out[c].update(assert_particles_close(g.particles(), o.particles(), r_min, steps=c))
    return g, o, out


# ------------------------------------------------------------------ particle-free (row a1)

def test_rayleigh_benard_small_ragged(gpu, ob, wl):
    """Config 1's set-up (bottom hot, top cold, adiabatic sides, conduction profile + seeded noise)
    on 333 x 130: three 128-wide tiles with a 77-wide tail, pitch 336 != nx."""
    nx, ny = 333, 130
    w = wl.config(1)
    rng = np.random.default_rng(11)
    j = np.arange(ny, dtype=np.float64)[:, None]
    T = (1.0 - (j + 0.5) / ny) + 1e-3 * rng.uniform(-1.0, 1.0, size=(ny, nx))
    w = wl.Workload("rb_small", nx, ny, dict(w.params, gbeta=1e-4), steps=100, parity_steps=100,
                    T_init=np.ascontiguousarray(T))
    run_and_compare(gpu, ob, w, [1, 2, 100])


def test_all_wall_types_and_body_force(gpu, ob, wl):
    """Every wall branch of the rim path: W Dirichlet 0.3, E adiabatic, S Dirichlet 1, N Dirichlet
    -0.2, plus a uniform body acceleration in both directions (Guo forcing terms of Eq. 5)."""
    p = wl.default_params()
    p.update(wall_T_type=[1, 0, 1, 1], wall_T=[0.3, 0.0, 1.0, -0.2], gbeta=2e-4, T0=0.25,
             body_ax=1e-5, body_ay=-2e-5, nu=0.05, kappa=0.03)
    rng = np.random.default_rng(5)
    T = 0.25 + 0.5 * rng.uniform(-1, 1, size=(37, 141))
    w = wl.Workload("walls", 141, 37, p, 60, 60, T_init=T)
    run_and_compare(gpu, ob, w, [1, 60])


def test_two_steps_per_pass_equals_one_step_per_pass_bitwise(gpu, wl):
    """Particle-free lattices advance two time steps per pass (shared-memory tile).
    Same arithmetic per step, so every population must equal the one-step kernel's bit for bit:
    ragged sizes (tiles of 32 x 14 with partial tiles in both directions), every wall type, a
    body force, and the periodic wrap; odd step counts leave one step to the one-step kernel."""
    rng = np.random.default_rng(17)
    cases = []
    p = wl.default_params()
    p.update(wall_T_type=[1, 0, 1, 1], wall_T=[0.3, 0.0, 1.0, -0.2], gbeta=2e-4, T0=0.25,
             body_ax=1e-5, body_ay=-2e-5, nu=0.05, kappa=0.03)
    cases.append((141, 37, p))
    cases.append((64, 28, dict(p)))                      # whole tiles exactly
    q = wl.default_params()
    q.update(periodic_x=1, body_ax=1e-6, nu=0.1, gbeta=1e-4, wall_T_type=[0, 0, 1, 1], wall_T=[0, 0, 1.0, 0.0])
    cases.append((77, 45, q))                            # periodic, nx not a multiple of 32
    cases.append((33, 15, dict(q)))
    for nx, ny, prm in cases:
        T = 0.25 + 0.5 * rng.uniform(-1, 1, size=(ny, nx))
        w = wl.Workload("two_step", nx, ny, prm, 1, 1, T_init=T)
        a = gpu.Simulation.from_workload(w)
        b = gpu.Simulation.from_workload(w)
        b.set_two_step(False)
        for n in (1, 2, 7, 40):
            a.step(n)
            b.step(n)
            fa, fb = a.fields(populations=True), b.fields(populations=True)
            for k in ("f", "g", "rho", "ux", "uy", "T"):
                assert np.array_equal(fa[k], fb[k]), (nx, ny, n, k)


def test_periodic_poiseuille(gpu, ob, wl):
    """x-periodic body-force channel (the closed-form check's set-up): wrap-around pulls."""
    p = wl.default_params()
    p.update(periodic_x=1, body_ax=1e-6, nu=0.1)
    w = wl.Workload("poiseuille", 20, 33, p, 200, 200)
    g, o, _ = run_and_compare(gpu, ob, w, [1, 200])
    # and the GPU itself against the closed form after convergence (independent of the oracle)
    g.step(40000)
    ux = g.fields()["ux"]
    jj = np.arange(33, dtype=np.float64)
    exact = 1e-6 / (2 * 0.1) * (jj + 0.5) * (33 - 0.5 - jj)
    assert np.abs(ux[:, 3] - exact).max() / exact.max() < 1e-8


def test_smallest_lattice_and_zero_steps(gpu, ob, wl):
    p = wl.default_params()
    p.update(gbeta=1e-3, wall_T_type=[0, 0, 1, 1], wall_T=[0, 0, 1.0, 0.0])
    w = wl.Workload("tiny", 4, 4, p, 10, 10)
    g, o = both(gpu, ob, w)
    g.step(0)
    o.step(0)
    assert_fields_close(g.fields(populations=True), o.fields(populations=True))
    g.step(25)
    o.step(25)
    assert_fields_close(g.fields(populations=True), o.fields(populations=True))


def test_mass_conservation_closed_box_gpu(gpu, wl):
    """Property that holds at any size: particle-free closed box conserves total mass to 1e-12."""
    w = wl.config(1)
    g = gpu.Simulation.from_workload(w)
    m0 = g.fields()["rho"].sum()
    g.step(300)
    m1 = g.fields()["rho"].sum()
    assert abs(m1 - m0) / m0 < 1e-12


# ------------------------------------------------------------------ particles (rows a2-a6)

def test_config0_single_hot_particle(gpu, ob, wl):
    """BASELINE config 0 in full: 128x256, one d=20 hot particle settling from rest.  Links
    bit-exact at step 0, fields and particle state at 100 and 1000 steps (the particle has moved
    ~20 nodes by then: thousands of cover / uncover / refill events)."""
    w = wl.config(0)
    g, o, errs = run_and_compare(gpu, ob, w, [1, 100, 1000])
    pg, po = g.particles(), o.particles()
    assert po["y"][0] < 200.0 - 5.0 and abs(pg["y"][0] - po["y"][0]) < 1e-7
    # links again after the run, on the oracle's particle state injected into fresh simulations
    assert_links_after_injection(gpu, ob, wl, w, po)


def assert_links_after_injection(gpu, ob, wl, w, po):
    parts = dict(w.particles)
    parts.update(x=po["x"], y=po["y"], ux=po["ux"], uy=po["uy"], omega=po["omega"])
    if "minor" in parts:
        parts.update(theta=po["theta"])
    w2 = wl.Workload(w.name + "_inj", w.nx, w.ny, w.params, 1, 1, particles=parts)
    try:
        g2, o2 = both(gpu, ob, w2)
    except Exception as e:   # particles that drifted into overlap are rejected by both sides
        pytest.skip(f"injected state rejected: {e}")
    assert_links_equal(g2.links(), o2.links())
    fg, fo = g2.fields(), o2.fields()
    assert np.array_equal(fg["flag"], fo["flag"])


def test_moving_rotating_particles_mixed_sizes(gpu, ob, wl):
    """Several particles of different diameters with initial velocities and spins, two of them
    within the repulsion range of each other and one next to a wall: exercises the fallback
    ladders (stencil nodes inside another particle / beyond the wall), repulsion (pair and wall),
    refill in every direction.  303 x 190 lattice (ragged)."""
    nx, ny = 303, 190
    x = np.array([40.0, 62.3, 150.5, 151.0, 250.25, 12.4, 200.0, 100.7])
    y = np.array([60.0, 61.1, 100.0, 125.5, 40.5, 150.0, 174.6, 20.9])
    d = np.array([20.0, 21.5, 24.0, 24.0, 12.0, 22.0, 24.0, 18.6])
    n = len(x)
    ux = np.array([0.01, -0.01, 0.0, 0.0, 0.02, -0.01, 0.0, 0.015])
    uy = np.array([0.0, 0.0, 0.01, -0.01, 0.02, 0.0, 0.005, -0.01])
    om = np.array([0.002, -0.003, 0.0, 0.001, -0.004, 0.002, 0.0, 0.003])
    p = wl.default_params()
    p.update(g=1.6e-4, gbeta=1e-5, wall_T_type=[1, 1, 1, 1], max_particles=n,
             max_links_per_particle=wl.max_links_for_diameter(24.0))
    parts = dict(x=x, y=y, diam=d, rho_ratio=np.linspace(1.1, 2.0, n), T_w=np.linspace(0.2, 1.0, n),
                 ux=ux, uy=uy, omega=om)
    w = wl.Workload("mixed", nx, ny, p, 150, 150, particles=parts)
    g, o, errs = run_and_compare(gpu, ob, w, [1, 2, 50, 150], r_min=6.0)
    assert_links_after_injection(gpu, ob, wl, w, o.particles())


def test_drag_on_a_moving_cylinder_matches_faxen_on_the_gpu(gpu, wl):
    """The closed form the oracle is pinned to (tests/test_oracle_particles.py), checked on the
    CUDA path directly, at two blockage ratios: Stokes drag on a cylinder moving along the
    mid-plane between two walls (Faxen)."""
    from test_oracle_particles import faxen_drag_per_length, faxen_workload
    for d, W, L in ((10.0, 40, 240), (10.0, 50, 300)):
        U, nu = 0.005, 1.0 / 6.0
        steps = int(6.0 * W * W / (np.pi ** 2 * nu))
        g = gpu.Simulation.from_workload(faxen_workload(wl, d=d, W=W, L=L, U=U, nu=nu, steps=steps))
        g.step(steps - 200)
        F = []
        for _ in range(200):
            g.step(1)
            F.append(g.particles()["Fx"][0])
        drag = -np.mean(F)
        expected = faxen_drag_per_length(nu, U, d / W)
        assert abs(drag / expected - 1.0) < 0.025, (d, W, drag, expected)


def test_terminal_velocity_matches_the_faxen_balance_on_the_gpu(gpu, wl):
    """Freely settling cylinder: net weight = Faxen drag at the terminal speed (CUDA path)."""
    from test_oracle_particles import settling_workload
    U = 0.005
    g = gpu.Simulation.from_workload(settling_workload(wl, U_target=U))
    g.step(6000)
    p = g.particles()
    assert abs(-p["uy"][0] / U - 1.0) < 0.025, p["uy"][0]
    assert abs(p["ux"][0]) < 1e-10 and abs(p["x"][0] - 19.5) < 1e-7


def test_heat_flow_from_a_hot_cylinder_matches_the_shape_factor_on_the_gpu(gpu, wl):
    """The conduction closed form the oracle is pinned to, on the CUDA path, for two geometries."""
    from test_oracle_particles import (conduction_workload, shape_factor_cylinder_between_planes,
                                       wall_heat_flow)
    for d, W, L in ((10.0, 40, 400), (8.0, 48, 400)):
        kappa = 0.1
        g = gpu.Simulation.from_workload(conduction_workload(wl, d=d, W=W, L=L, kappa=kappa, steps=12000))
        g.step(12000)
        q = wall_heat_flow(g.fields()["T"], kappa)
        expected = shape_factor_cylinder_between_planes(d, 0.5 * W) * kappa
        assert abs(q / expected - 1.0) < 0.01, (d, W, q, expected)


def test_paper_repulsion_variant(gpu, ob, wl):
    """Eq. (15) as the paper prints it: quadratic, s = 3, eps_w = 1e-3; two
    particles approaching head-on and one falling onto the bottom wall."""
    nx, ny = 160, 96
    p = wl.default_params()
    p.update(g=3e-4, gbeta=0.0, rep_s=3.0, rep_power=2, max_particles=3,
             max_links_per_particle=wl.max_links_for_diameter(20.0), wall_T_type=[1, 1, 1, 1])
    parts = dict(x=np.array([40.0, 63.5, 120.0]), y=np.array([50.0, 50.0, 12.2]),
                 diam=np.array([20.0, 20.0, 20.0]), rho_ratio=np.array([1.5, 1.5, 2.5]),
                 T_w=np.array([1.0, 0.5, 0.0]), ux=np.array([0.02, -0.02, 0.0]),
                 uy=np.array([0.0, 0.0, -0.02]), omega=np.zeros(3))
    w = wl.Workload("rep", nx, ny, p, 120, 120, particles=parts)
    run_and_compare(gpu, ob, w, [1, 120])


def test_fixed_cylinder_in_channel(gpu, ob, wl):
    """Fixed (immobile) particle in an x-periodic body-force channel: force is computed, state is
    not integrated; zero-lift symmetry holds on the GPU too."""
    nx, ny = 96, 65
    p = wl.default_params()
    p.update(periodic_x=1, body_ax=2e-6, nu=0.05, max_particles=1,
             max_links_per_particle=wl.max_links_for_diameter(16.0))
    parts = dict(x=np.array([48.0]), y=np.array([32.0]), diam=np.array([16.0]),
                 rho_ratio=np.array([1.5]), T_w=np.array([0.0]), fixed=np.array([1], dtype=np.uint8))
    w = wl.Workload("cyl", nx, ny, p, 400, 400, particles=parts)
    g, o, _ = run_and_compare(gpu, ob, w, [1, 400], r_min=8.0)
    pg = g.particles()
    assert pg["x"][0] == 48.0 and pg["y"][0] == 32.0 and pg["ux"][0] == 0.0
    assert pg["Fx"][0] > 0 and abs(pg["Fy"][0]) < 1e-10 * abs(pg["Fx"][0])


def test_small_sedimentation_many_particles(gpu, ob, wl):
    """Structure of configs 2-4 at a size the oracle does in seconds: 40 particles of seeded
    diameters in [12, 24], 2-unit gaps, 420 x 300."""
    w = wl.sedimentation(420, 300, 40, seed=7, y_frac_lo=0.0, d_lo=12.0, d_hi=24.0,
                         name="sed_small")
    g, o, _ = run_and_compare(gpu, ob, w, [1, 100], r_min=6.0)
    assert_links_after_injection(gpu, ob, wl, w, o.particles())


def test_discs_driven_into_overlap(gpu, ob, wl):
    """Degenerate case of the flag/owner bookkeeping: with a repulsion too weak to matter, fast
    particles run into each other and into a fixed one, so discs share lattice nodes for many
    steps (lowest id owns a shared node; a node uncovered by one particle while
    still inside another stays solid).  Flags, links, fields and particle states are compared
    with the oracle at several stages of the overlap: pair (0, 1) lower id arriving from the left,
    pair (2, 3) higher id running into a fixed lower id, pair (4, 5) lower id running into a fixed
    higher id, and (6, 7) overlapping and separating again in y."""
    nx, ny = 330, 150
    x = np.array([40.0, 66.0, 130.0, 156.0, 230.0, 204.0, 290.0, 290.5])
    y = np.array([40.0, 41.0, 40.5, 40.0, 40.0, 41.5, 95.0, 122.0])
    d = np.array([20.0, 20.0, 22.0, 18.0, 20.0, 24.0, 20.0, 21.0])
    ux = np.array([0.12, -0.05, 0.0, -0.15, 0.0, 0.14, 0.0, 0.0])
    uy = np.array([0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.12, -0.1])
    fixed = np.array([0, 0, 1, 0, 1, 0, 0, 0], dtype=np.uint8)
    n = len(x)
    p = wl.default_params()
    p.update(g=0.0, gbeta=1e-5, rep_s=2.0, rep_eps=1e3, rep_power=1, wall_T_type=[1, 1, 1, 1],
             max_particles=n, max_links_per_particle=wl.max_links_for_diameter(24.0))
    parts = dict(x=x, y=y, diam=d, rho_ratio=np.full(n, 8.0), T_w=np.linspace(0.3, 1.0, n),
                 ux=ux, uy=uy, omega=np.zeros(n), fixed=fixed)
    w = wl.Workload("overlap", nx, ny, p, 120, 120, particles=parts)
    g, o = both(gpu, ob, w)
    done = 0
    seen_overlap = False
    for c in (1, 30, 60, 61, 90, 120):
        g.step(c - done)
        o.step(c - done)
        done = c
        assert_fields_close(g.fields(populations=True), o.fields(populations=True))
        assert_particles_close(g.particles(), o.particles(), r_min=9.0, steps=c)
        po = o.particles()
        gap01 = np.hypot(po["x"][0] - po["x"][1], po["y"][0] - po["y"][1]) - 20.0
        seen_overlap |= gap01 < -1.0
    assert seen_overlap, "the case no longer drives the discs into overlap"


def test_large_particle_wide_zone(gpu, ob, wl):
    """A d = 70.6 particle (zone 75 nodes wide: three 32-column chunks, several rounds of the link
    builder, 12N-12 = 876 slots) next to a d = 12 one, both moving."""
    nx, ny = 200, 170
    p = wl.default_params()
    p.update(g=1e-4, gbeta=1e-5, wall_T_type=[1, 0, 1, 1], max_particles=2,
             max_links_per_particle=wl.max_links_for_diameter(70.6))
    parts = dict(x=np.array([90.3, 150.0]), y=np.array([100.2, 40.0]), diam=np.array([70.6, 12.0]),
                 rho_ratio=np.array([1.2, 1.5]), T_w=np.array([1.0, 0.4]),
                 ux=np.array([0.02, -0.01]), uy=np.array([-0.03, 0.02]), omega=np.array([1e-3, -2e-3]))
    w = wl.Workload("large", nx, ny, p, 60, 60, particles=parts)
    g, o, _ = run_and_compare(gpu, ob, w, [1, 60], r_min=6.0)
    assert_links_after_injection(gpu, ob, wl, w, o.particles())


def test_elliptical_particles(gpu, ob, wl):
    """Elliptical particles (App. A) next to
    circles: different axis ratios and orientations, spinning and translating, one hugging a wall,
    two within repulsion range of each other, one nearly a circle.  Links (ray-ellipse q) bit-exact
    at step 0 and on the injected final state; fields and particle states after 1, 2 and 120
    steps."""
    nx, ny = 330, 210
    x = np.array([60.3, 118.0, 200.5, 262.0, 150.2, 24.0, 285.0])
    y = np.array([70.7, 72.0, 150.0, 60.4, 140.9, 150.0, 170.0])
    major = np.array([40.0, 24.0, 50.0, 20.0, 30.0, 36.0, 24.0])
    minor = np.array([20.0, 12.0, 25.0, 20.0, 29.0, 14.0, 16.0])
    theta = np.radians([60.0, -20.0, 90.0, 0.0, 33.0, 90.0, 10.0])
    n = len(x)
    p = wl.default_params()
    p.update(g=1.6e-4, gbeta=1e-5, wall_T_type=[1, 1, 1, 1], max_particles=n,
             max_links_per_particle=wl.max_links_for_diameter(50.0))
    parts = dict(x=x, y=y, diam=major, minor=minor, theta=theta,
                 rho_ratio=np.linspace(1.2, 1.8, n), T_w=np.linspace(0.3, 1.0, n),
                 ux=np.array([0.01, -0.012, 0.0, 0.005, -0.01, 0.0, -0.008]),
                 uy=np.array([0.0, 0.004, -0.01, 0.01, 0.0, -0.01, 0.0]),
                 omega=np.array([2e-3, -3e-3, 1e-3, 2e-3, -1e-3, 0.0, 4e-3]))
    w = wl.Workload("ellipses", nx, ny, p, 120, 120, particles=parts)
    g, o, _ = run_and_compare(gpu, ob, w, [1, 2, 120], r_min=6.0)
    assert_links_after_injection(gpu, ob, wl, w, o.particles())
    th = g.particles()["theta"]
    assert np.abs(th - theta).max() > 0.05           # they did turn


def test_paper_table4_arrangement_small(gpu, ob, wl):
    """The paper's own benchmark set-up (Table 4: d = 40, rho-ratio 1.1, nu = 0.01,
    Pr = 5, regular lines of particles at pitch 50, Eq. 15 as printed: quadratic, s = 3) at a size
    the oracle does in seconds: 4 lines of 8 particles in 400 x 300.  With a 10-unit gap between
    neighbours every particle's interpolation stencils reach into the gap next door."""
    w = wl.paper_table4(cols=8, lines=4, ny=300, name="table4_small")
    # break the lattice symmetry a little so that the particles actually interact
    rng = np.random.default_rng(40)
    n = w.n_particles
    w.particles.update(ux=1e-3 * rng.uniform(-1, 1, n), uy=-5e-3 * rng.uniform(0, 1, n),
                       omega=1e-4 * rng.uniform(-1, 1, n))
    g, o, _ = run_and_compare(gpu, ob, w, [1, 100], r_min=20.0)
    assert_links_after_injection(gpu, ob, wl, w, o.particles())


def test_overlap_and_sequential_modes_agree_bitwise(gpu, wl):
    """The schedule with the particle update chain on its own stream, concurrent with the lattice
    kernel, must give the same bits as the strictly sequential single-stream schedule."""
    w = wl.sedimentation(300, 260, 14, seed=9, y_frac_lo=0.2, d_lo=12.0, d_hi=24.0, name="ovl")
    a = gpu.Simulation.from_workload(w)
    b = gpu.Simulation.from_workload(w)
    b.set_overlap(False)
    for n in (1, 7, 505, 12, 520):
        a.step(n)
        b.step(n)
        fa, fb = a.fields(populations=True), b.fields(populations=True)
        fluid = fa["flag"] == 0
        assert np.array_equal(fa["flag"], fb["flag"])
        for k in ("f", "g"):
            assert np.array_equal(fa[k][:, fluid], fb[k][:, fluid]), k
        pa, pb = a.particles(), b.particles()
        for k in pa:
            assert np.array_equal(pa[k], pb[k]), k


def test_chain_grid_size_does_not_change_results(gpu, wl, monkeypatch):
    """The particle chain runs as a few persistent CTAs per SM under the lattice kernel; each CTA
    then loops over many particles.  With 700 small particles and one CTA per SM (5 particles per
    CTA) the results must equal, bit for bit, those of one CTA per particle."""
    w = wl.sedimentation(900, 700, 700, seed=21, y_frac_lo=0.0, d_lo=8.0, d_hi=12.0, name="grid")
    monkeypatch.setenv("LBM_CHAIN_CTAS_PER_SM", "1")
    a = gpu.Simulation.from_workload(w)
    monkeypatch.setenv("LBM_CHAIN_CTAS_PER_SM", "0")
    b = gpu.Simulation.from_workload(w)
    monkeypatch.delenv("LBM_CHAIN_CTAS_PER_SM")
    c = gpu.Simulation.from_workload(w)          # the library's own choice
    for n in (1, 40):
        for s in (a, b, c):
            s.step(n)
        fb, pb = b.fields(populations=True), b.particles()
        fluid = fb["flag"] == 0
        for s in (a, c):
            fs, ps = s.fields(populations=True), s.particles()
            assert np.array_equal(fs["flag"], fb["flag"])
            for k in ("f", "g"):
                assert np.array_equal(fs[k][:, fluid], fb[k][:, fluid]), k
            for k in pb:
                assert np.array_equal(ps[k], pb[k]), k
        La, Lb = a.links(), b.links()
        for k in Lb:
            assert np.array_equal(np.asarray(La[k]), np.asarray(Lb[k])), k


# ------------------------------------------------------------------ boundary behaviour

def test_error_codes(gpu, wl):
    p = wl.default_params()
    p.update(max_particles=2, max_links_per_particle=wl.max_links_for_diameter(20.0))
    s = gpu.Simulation(64, 64, p)
    one = dict(diam=np.array([20.0]), rho_ratio=np.array([1.5]), T_w=np.array([1.0]))
    with pytest.raises(gpu.LbmError) as e:      # touches the wall
        s.add_particles(x=np.array([5.0]), y=np.array([30.0]), **one)
    assert e.value.code == gpu.LBM_E_ARG
    s.add_particles(x=np.array([30.0]), y=np.array([30.0]), **one)
    with pytest.raises(gpu.LbmError) as e:      # overlaps the first
        s.add_particles(x=np.array([40.0]), y=np.array([30.0]), **one)
    assert e.value.code == gpu.LBM_E_ARG
    with pytest.raises(gpu.LbmError) as e:      # diameter too large for the link capacity
        s.add_particles(x=np.array([30.0]), y=np.array([30.0]), diam=np.array([40.0]),
                        rho_ratio=np.array([1.5]), T_w=np.array([1.0]))
    assert e.value.code == gpu.LBM_E_CAPACITY
    s.step(1)
    with pytest.raises(gpu.LbmError) as e:      # no insertion mid-run
        s.add_particles(x=np.array([10.0]), y=np.array([52.0]), **one)
    assert e.value.code == gpu.LBM_E_STATE
    with pytest.raises(gpu.LbmError) as e:
        s.set_temperature(np.zeros((64, 64)))
    assert e.value.code == gpu.LBM_E_STATE
    assert len(s.particles()["x"]) == 1
    # ellipses: a turned ellipse whose bounding box leaves the cavity, one whose support-function
    # gap to a circle is negative, and a major axis too long for the link capacity
    p3 = wl.default_params()
    p3.update(max_particles=3, max_links_per_particle=wl.max_links_for_diameter(30.0))
    s3 = gpu.Simulation(96, 64, p3)
    ell = dict(rho_ratio=np.array([1.5]), T_w=np.array([1.0]))
    with pytest.raises(gpu.LbmError) as e:      # vertical 30 x 10 ellipse at y = 14: hy = 15 > 14.5
        s3.add_particles(x=np.array([40.0]), y=np.array([14.0]), diam=np.array([30.0]),
                         minor=np.array([10.0]), theta=np.array([np.pi / 2]), **ell)
    assert e.value.code == gpu.LBM_E_ARG
    s3.add_particles(x=np.array([40.0]), y=np.array([14.0]), diam=np.array([30.0]),
                     minor=np.array([10.0]), theta=np.array([0.0]), **ell)      # horizontal: fits
    with pytest.raises(gpu.LbmError) as e:      # circle of d = 20 at distance 22 along x: 15 + 10 > 22
        s3.add_particles(x=np.array([62.0]), y=np.array([14.0]), diam=np.array([20.0]), **ell)
    assert e.value.code == gpu.LBM_E_ARG
    s3.add_particles(x=np.array([40.0]), y=np.array([31.0]), diam=np.array([20.0]), **ell)   # above: 5 + 10 < 17
    with pytest.raises(gpu.LbmError) as e:
        s3.add_particles(x=np.array([70.0]), y=np.array([40.0]), diam=np.array([44.0]),
                         minor=np.array([8.0]), theta=np.array([0.0]), **ell)
    assert e.value.code == gpu.LBM_E_CAPACITY
    assert len(s3.particles()["x"]) == 2 and len(s3.links()["q"]) > 0
    # no particles at all: empty link list, empty particle arrays
    s2 = gpu.Simulation(32, 32, wl.default_params())
    assert len(s2.links()["q"]) == 0 and len(s2.particles()["x"]) == 0
    s2.step(3)
