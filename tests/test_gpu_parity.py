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
    body force, and the periodic wrap; odd step counts leave one step to the one-step kernel.
    The same for THREE steps per pass (tiles of 28 x 12 with a two-node halo, levels written back
    in place), including lattices narrower than one tile and the periodic images two columns out."""
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
    cases.append((5, 9, dict(q)))                        # narrower than the halo is wide
    cases.append((29, 13, dict(p)))
    for nx, ny, prm in cases:
        T = 0.25 + 0.5 * rng.uniform(-1, 1, size=(ny, nx))
        w = wl.Workload("two_step", nx, ny, prm, 1, 1, T_init=T)
        a = gpu.Simulation.from_workload(w)          # the library's default
        a2 = gpu.Simulation.from_workload(w)
        a2.set_two_step(2)                           # two steps per pass
        a3 = gpu.Simulation.from_workload(w)
        a3.set_two_step(3)                           # three steps per pass (then two, then one)
        a3p = gpu.Simulation.from_workload(w)
        a3p.set_two_step(3)
        if not prm.get("periodic_x"):
            a3p.set_tma(False)                       # the plain three-step kernel (a3: the TMA-fed one)
        b = gpu.Simulation.from_workload(w)
        b.set_two_step(False)
        for n in (1, 2, 3, 5, 7, 40):
            b.step(n)
            fb = b.fields(populations=True)
            for s_ in (a, a2, a3, a3p):
                s_.step(n)
                fa = s_.fields(populations=True)
                for k in ("f", "g", "rho", "ux", "uy", "T"):
                    assert np.array_equal(fa[k], fb[k]), (nx, ny, n, k)


def test_tma_fed_three_step_kernel_equals_one_step_kernel_bitwise(gpu, wl):
    """k_stream_collide_3step_tma (persistent CTAs, tile images by cp.async.bulk.tensor into a
    three-deep ring, two thread groups per CTA) against the one-step kernel, bit for bit, on
    lattices large enough that every CTA walks many tiles (the ring wraps, both groups and all
    three stages are reused: 1591, 550, 150 and 15,750 tiles on 148 SMs), with a ragged last tile column
    and row, every wall type and a body force, step counts that leave one or two steps to the two-step
    and one-step kernels (so the copies alternate under the tensor maps); and that periodic lattices
    refuse it."""
    rng = np.random.default_rng(23)
    p = wl.default_params()
    p.update(wall_T_type=[1, 0, 1, 1], wall_T=[0.3, 0.0, 1.0, -0.2], gbeta=2e-4, T0=0.25,
             body_ax=1e-5, body_ay=-2e-5, nu=0.05, kappa=0.03)
    for nx, ny, steps in ((1024, 512, (3, 31)), (601, 299, (7, 8)), (4200, 12, (3,)), (27, 1790, (9,)), (2500, 2100, (6,))):
        T = 0.25 + 0.5 * rng.uniform(-1, 1, size=(ny, nx))
        w = wl.Workload("tma", nx, ny, p, 1, 1, T_init=T)
        sims = []
        for mode in (1, 2):                          # 2: row-wise hand-over instead of group barriers
            a = gpu.Simulation.from_workload(w)
            a.set_two_step(3)
            a.set_tma(mode)
            sims.append(a)
        b = gpu.Simulation.from_workload(w)
        b.set_two_step(False)
        for n in steps:
            b.step(n)
            fb = b.fields(populations=True)
            for mode, a in enumerate(sims, 1):
                a.step(n)
                fa = a.fields(populations=True)
                for k in ("f", "g", "rho", "ux", "uy", "T"):
                    assert np.array_equal(fa[k], fb[k]), (nx, ny, n, k, mode)
    q = wl.default_params()
    q.update(periodic_x=1, body_ax=1e-6)
    s_ = gpu.Simulation.from_workload(wl.Workload("tma_periodic", 64, 32, q, 1, 1))
    with pytest.raises(Exception):
        s_.set_tma(True)
    s_.set_tma(False)


def test_tma_row_handover_repeated_runs_are_identical(gpu, wl):
    """Regression test for a rare race of the persistent kernel's row-wise hand-over (a warp several
    tiles ahead passed a `full` barrier shared by both thread groups on the parity of an earlier
    use: one run in 150-250 of config 1 over 300 steps came out corrupted).  400 runs over 150 steps
    must agree with one another bit for bit and conserve mass to 1e-12."""
    w = wl.config(1)
    first = None
    for rep in range(400):
        g = gpu.Simulation.from_workload(w)
        g.step(150)
        rho = g.fields()["rho"]
        g.close()
        assert abs(rho.sum() - rho.size) / rho.size < 1e-12, rep
        if first is None:
            first = rho
        else:
            assert np.array_equal(rho, first), rep


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


def test_coupling_closed_forms_on_the_gpu(gpu, ob, wl):
    """The closed forms that pin the rotational / geometric half of the coupling in the oracle
    (tests/test_oracle_coupling_pins.py), asserted on the CUDA path directly: circular Couette
    torque on a spinning cylinder; one-step dU = F/M, dOmega = T_z/I with M, I from quadrature
    (disc and 3 : 1 ellipse); Eq. (15) against each of the four walls; the ellipse pair gap through
    the support functions and the wall gap at the vertex of an upright ellipse."""
    import math
    import test_oracle_coupling_pins as pins

    class AsOracle:                       # the pins' set-up helpers build "ob.OracleSim"s
        OracleSim = gpu.Simulation
    # (a) Couette
    r, L, nu, rim = 9.0, 64, 1.0 / 6.0, 0.01
    g = pins.spinning_cylinder(AsOracle, wl, r, L=L, nu=nu, rim_speed=rim, steps=5000)
    P = g.particles()
    expected = -4.0 * math.pi * nu * (rim / r) * r * r / (1.0 - (r / (0.5 * L)) ** 2)
    assert -0.035 < P["Tz"][0] / expected - 1.0 < 0.005, (P["Tz"][0], expected)
    # (b) mass and inertia as the step uses them
    for a, b, theta in ((5.3, 5.3, None), (9.0, 3.0, 0.5)):
        ratio = 1.6
        Mq, Iq = pins.quadrature_mass_inertia(a, b, ratio)
        p = pins.base_params(wl, 1, 2 * a, g=0.0, gbeta=0.0, nu=0.05)
        parts = dict(x=np.array([40.3]), y=np.array([31.7]), diam=np.array([2 * a]),
                     rho_ratio=np.array([ratio]), T_w=np.array([0.0]), ux=np.array([0.02]),
                     uy=np.array([0.015]), omega=np.array([0.003]))
        if theta is not None:
            parts.update(minor=np.array([2 * b]), theta=np.array([theta]))
        s = gpu.Simulation.from_workload(wl.Workload("kick", 80, 64, p, 1, 1, particles=parts))
        s.step(5)
        dux, duy, dom, Fx, Fy, Tz = pins.one_step_increments(s)
        assert abs(Fx) > 1e-3 and abs(Tz) > 1e-4
        assert dux == pytest.approx(Fx / Mq, rel=3e-3) and duy == pytest.approx(Fy / Mq, rel=3e-3)
        assert dom == pytest.approx(Tz / Iq, rel=3e-3)
        M = ratio * math.pi * a * b
        assert dux == pytest.approx(Fx / M, rel=1e-10)
        assert dom == pytest.approx(Tz / (0.25 * M * (a * a + b * b)), rel=1e-10)
    # (c), (d): the pins themselves, run with the CUDA path standing in for the oracle
    pins.test_repulsion_from_each_of_the_four_walls_in_closed_form(AsGpu(gpu), wl)
    pins.test_pair_repulsion_of_unequal_discs_uses_the_mean_force_scale(AsGpu(gpu), wl)
    pins.test_ellipse_pair_gap_is_taken_through_the_support_functions(AsGpu(gpu), wl)
    pins.test_upright_ellipse_is_repelled_by_the_bottom_wall_at_its_vertex(AsGpu(gpu), wl)
    # Eq. (14) with a moving wall on a fixed disc (the pin's brute-force case): parity of F, T_z
    r, xc, yc, U, V, Om = 6.3, 24.3, 21.8, 0.08, -0.05, 0.012
    p = pins.base_params(wl, 1, 2 * r, g=0.0, gbeta=0.0, nu=0.02)
    parts = dict(x=np.array([xc]), y=np.array([yc]), diam=np.array([2 * r]),
                 rho_ratio=np.array([2.0]), T_w=np.array([0.0]), ux=np.array([U]),
                 uy=np.array([V]), omega=np.array([Om]), fixed=np.array([1], dtype=np.uint8))
    run_and_compare(gpu, ob, wl.Workload("arm", 48, 44, p, 61, 61, particles=parts), [61], r_min=6.3)


class AsGpu:
    """Lets a pin written against the oracle binding run against the CUDA binding: the same
    constructor and method names, `OracleSim(nx, ny, params)` included."""

    def __init__(self, gpu):
        class Sim(gpu.Simulation):
            def add_particles(self, **kw):
                super().add_particles(**{k: (None if v is None else np.asarray(v, dtype=np.uint8 if k == "fixed" else np.float64))
                                         for k, v in kw.items()})
        self.OracleSim = Sim


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


def assert_same_bits(a, b):
    fa, fb = a.fields(populations=True), b.fields(populations=True)
    fluid = fa["flag"] == 0
    assert np.array_equal(fa["flag"], fb["flag"])
    for k in ("f", "g"):
        assert np.array_equal(fa[k][:, fluid], fb[k][:, fluid]), k
    pa, pb = a.particles(), b.particles()
    for k in pa:
        assert np.array_equal(pa[k], pb[k]), k


def test_graph_replay_equals_direct_launches_bitwise(gpu, wl):
    """lbm_step replays whole periods of the schedule as CUDA graphs (8 steps per launch, then 2,
    an odd last step directly).  Every mix of those must give the bits of the direct launches, in
    the overlapped and in the sequential schedule, from either phase of the A/B swap."""
    w = wl.sedimentation(300, 260, 14, seed=9, y_frac_lo=0.2, d_lo=12.0, d_hi=24.0, name="graph")
    a = gpu.Simulation.from_workload(w)              # graphs, overlapped
    b = gpu.Simulation.from_workload(w)
    b.set_graph(False)                               # direct launches, overlapped
    c = gpu.Simulation.from_workload(w)
    c.set_overlap(False)                             # graphs, sequential
    for n in (1, 2, 7, 16, 33, 8, 101):
        counts = []
        for s in (a, b, c):
            l0 = s.kernel_launches()
            s.step(n)
            counts.append(s.kernel_launches() - l0)
        assert counts[0] == counts[1] == counts[2] > 0      # replayed kernels are counted
        assert_same_bits(a, b)
        assert_same_bits(c, b)


def test_two_step_band_equals_plain_schedule_bitwise(gpu, wl):
    """Lattices with particles advance the particle-free rows below the lowest particle two steps
    per pass (lbm_set_band; periods of four steps, the band height chosen on the device at the
    start of each period).  The arithmetic per node and step is unchanged, so every fluid
    population and particle state must equal the plain schedule's bit for bit: through graph
    replays and direct launches, overlapped and sequential, for step counts that are not multiples
    of the period, while a fast particle falls into the band's rows (the band shrinks from period
    to period) and ends up too close to the floor for any band."""
    w = wl.sedimentation(333, 420, 16, seed=5, y_frac_lo=0.55, d_lo=12.0, d_hi=22.0, name="band")
    n = w.n_particles
    uy = np.zeros(n)
    k = int(np.argmin(w.particles["y"]))
    uy[k] = -0.12                                    # one particle dives through the free rows
    w.particles.update(ux=np.zeros(n), uy=uy, omega=np.zeros(n))
    ref = gpu.Simulation.from_workload(w)
    ref.set_band(False)
    ref.set_graph(False)
    sims = [gpu.Simulation.from_workload(w) for _ in range(5)]
    for s_ in sims:
        s_.set_band(2)                               # every band, however small the lattice
    sims[1].set_graph(False)                         # direct launches (the profiling path)
    sims[2].set_overlap(False)                       # one stream
    sims[3].set_band_steps(2)                        # periods of four steps, two steps per pass
    sims[4].set_band_steps(2)                        # (the default is three: periods of six)
    sims[4].set_graph(False)
    q_seen = []
    for nst in (1, 4, 8, 3, 29, 64, 402, 7, 1500):
        ref.step(nst)
        for s_ in sims:
            s_.step(nst)
            assert_same_bits(s_, ref)
        q_seen.append(sims[0].band_rows())
        assert sims[1].band_rows() == q_seen[-1] or nst < 4
    assert ref.band_rows() == 0
    assert max(q_seen) > 150                         # a real band at the start ...
    live = [q for q in q_seen if q > 0]
    assert live == sorted(live, reverse=True) and len(set(live)) > 2   # ... that shrinks
    # a particle that starts just above the smallest band worth having and falls: the band is
    # given up (Q = 0) within a few periods and the plain schedule carries on
    # (a second, fixed disc under the lid keeps the rows above free of a band of their own)
    p = wl.default_params()
    p.update(g=1.6e-4, gbeta=1e-5, wall_T_type=[1, 1, 1, 1], max_particles=2,
             max_links_per_particle=wl.max_links_for_diameter(14.0))
    parts = dict(x=np.array([60.4, 30.0]), y=np.array([47.0, 139.0]), diam=np.array([14.0, 14.0]),
                 rho_ratio=np.array([1.5, 1.5]), T_w=np.array([1.0, 0.0]), ux=np.array([0.0, 0.0]),
                 uy=np.array([-0.05, 0.0]), omega=np.array([0.0, 0.0]),
                 fixed=np.array([0, 1], dtype=np.uint8))
    w2 = wl.Workload("band_vanishes", 120, 150, p, 1, 1, particles=parts)
    for band_steps in (3, 2):
        a, b = gpu.Simulation.from_workload(w2), gpu.Simulation.from_workload(w2)
        a.set_band(2)
        a.set_band_steps(band_steps)
        b.set_band(False)
        qs = []
        for nst in (16, 16, 24, 40, 200):         # (calls shorter than 16 steps never use the band)
            a.step(nst)
            b.step(nst)
            assert_same_bits(a, b)
            qs.append(a.band_rows())
        assert qs[0] >= 28 and qs[-1] == 0, (band_steps, qs)


def test_two_step_band_above_a_settled_suspension_equals_plain_schedule_bitwise(gpu, ob, wl):
    """The mirrored band: particles low in the cavity leave the rows under the lid free; the plan
    at the start of a call picks the larger band (here the upper one: band_rows() < 0).  Bitwise
    equality with the plain schedule (graphs / direct launches / one stream) while one particle is
    thrown upwards into the free rows (the band shrinks from the other side), a heated lid and a
    periodic case against the oracle."""
    w = wl.sedimentation(300, 400, 14, seed=8, y_frac_lo=0.0, d_lo=12.0, d_hi=20.0, name="band_up")
    n = w.n_particles
    w.particles["y"] = 0.45 * w.particles["y"] + 8.0          # squeeze into the lower half (x unchanged: no overlap)
    w.particles["y"] = np.maximum(w.particles["y"], 0.5 * w.particles["diam"] + 3.0)
    # re-space vertically so that no two discs overlap after the squeeze
    order = np.argsort(w.particles["y"])
    ys = w.particles["y"].copy()
    uy = np.zeros(n)
    k = int(np.argmax(ys))
    uy[k] = +0.10                                             # thrown upwards into the free rows
    keep = []
    for a in range(n):                                        # drop discs that would overlap another one
        ok = all(np.hypot(w.particles["x"][a] - w.particles["x"][b], ys[a] - ys[b])
                 >= 0.5 * (w.particles["diam"][a] + w.particles["diam"][b]) + 2.0 for b in keep)
        if ok:
            keep.append(a)
    keep = np.array(keep)
    assert len(keep) >= 6 and k in keep
    parts = {key: np.asarray(v)[keep] for key, v in w.particles.items()}
    parts["y"] = ys[keep]
    parts.update(ux=np.zeros(len(keep)), uy=uy[keep], omega=np.zeros(len(keep)))
    w.params["max_particles"] = len(keep)
    w = wl.Workload("band_up", w.nx, w.ny, w.params, 1, 1, particles=parts)
    ref = gpu.Simulation.from_workload(w)
    ref.set_band(False)
    ref.set_graph(False)
    sims = [gpu.Simulation.from_workload(w) for _ in range(4)]
    for s_ in sims:
        s_.set_band(2)
    sims[1].set_graph(False)
    sims[2].set_overlap(False)
    sims[3].set_band_steps(2)                                 # two steps per pass (the default is three)
    q_seen = []
    for nst in (16, 29, 64, 402, 7, 900):
        ref.step(nst)
        for s_ in sims:
            s_.step(nst)
            assert_same_bits(s_, ref)
        q_seen.append(sims[0].band_rows())
    assert all(q < 0 for q in q_seen) and 400 + min(q_seen) > 120, q_seen   # a band under the lid: rows [-Q, ny)
    assert len(set(q_seen)) > 1                               # ... that the thrown particle pushes back
    # against the oracle, with a heated lid and periodic sides
    p = wl.default_params()
    p.update(g=1.6e-4, gbeta=1e-5, body_ax=1e-6, periodic_x=1, wall_T_type=[0, 0, 1, 1],
             wall_T=[0.0, 0.0, 0.1, 0.8], max_particles=2,
             max_links_per_particle=wl.max_links_for_diameter(16.0))
    parts = dict(x=np.array([40.3, 77.0]), y=np.array([30.2, 41.0]), diam=np.array([16.0, 12.5]),
                 rho_ratio=np.array([1.5, 1.3]), T_w=np.array([1.0, 0.4]))
    w2 = wl.Workload("band_up_walls", 131, 181, p, 60, 60, particles=parts)
    g, o, _ = run_and_compare(gpu, ob, w2, [60], r_min=6.0)
    assert g.band_rows() < 0 and 181 + g.band_rows() > 100     # rows [55, 181) or so


def test_two_step_band_periodic_and_wall_types(gpu, ob, wl):
    """The band next to every kind of cavity wall (Dirichlet floor, adiabatic and periodic sides,
    body force) against the oracle."""
    for periodic in (0, 1):
        p = wl.default_params()
        p.update(g=1.6e-4, gbeta=1e-5, body_ax=1e-6, periodic_x=periodic,
                 wall_T_type=[0, 0, 1, 1], wall_T=[0.0, 0.0, 0.7, 0.1], max_particles=2,
                 max_links_per_particle=wl.max_links_for_diameter(16.0))
        parts = dict(x=np.array([40.3, 77.0]), y=np.array([150.2, 139.0]), diam=np.array([16.0, 12.5]),
                     rho_ratio=np.array([1.5, 1.3]), T_w=np.array([1.0, 0.4]))
        w = wl.Workload("band_walls", 131, 181, p, 60, 60, particles=parts)
        g, o, _ = run_and_compare(gpu, ob, w, [60], r_min=6.0)
        assert g.band_rows() > 100


def test_results_do_not_depend_on_what_the_workspace_held_before(gpu, wl, monkeypatch):
    """The caller's workspace is arbitrary memory (PyTorch hands freed blocks out again, with the
    previous simulation's populations still in them): every array the path reads must have been
    initialised by the library.  Three workspaces pre-filled with 0x00, 0xFF and 0x3F bytes (the
    last reads as large positive ints and as doubles of order 5e-4) must give identical bits."""
    import torch
    w = wl.sedimentation(260, 300, 10, seed=13, y_frac_lo=0.45, d_lo=12.0, d_hi=20.0, name="poison")
    real_empty = torch.empty
    sims = []
    for fill in (0x00, 0xFF, 0x3F):
        def filled(*a, fill=fill, **kw):
            t = real_empty(*a, **kw)
            if kw.get("dtype") == torch.uint8 and t.is_cuda:
                t.fill_(fill)
            return t
        monkeypatch.setattr(torch, "empty", filled)
        sims.append(gpu.Simulation.from_workload(w))
    monkeypatch.setattr(torch, "empty", real_empty)
    for n in (1, 8, 31):
        for s_ in sims:
            s_.step(n)
        assert_same_bits(sims[1], sims[0])
        assert_same_bits(sims[2], sims[0])
    assert sims[0].band_rows() > 50


def test_prepare_builds_the_graphs_without_stepping(gpu, wl):
    """lbm_prepare(n) plans the band and captures the graphs lbm_step(n) replays, takes no time
    step, and changes no result; set-up calls are closed afterwards."""
    w = wl.sedimentation(300, 260, 14, seed=9, y_frac_lo=0.2, d_lo=12.0, d_hi=24.0, name="prep")
    a, b = gpu.Simulation.from_workload(w), gpu.Simulation.from_workload(w)
    p0 = a.particles()
    a.prepare(20)
    p1 = a.particles()
    for k in ("x", "y", "ux", "uy", "omega", "theta"):
        assert np.array_equal(p0[k], p1[k]), k
    with pytest.raises(gpu.LbmError) as e:
        a.set_temperature(np.zeros((w.ny, w.nx)))
    assert e.value.code == gpu.LBM_E_STATE
    for n in (20, 5, 20, 33):
        a.prepare(n)
        l0 = a.kernel_launches()
        a.step(n)
        b.step(n)
        assert a.kernel_launches() - l0 > 0
        assert_same_bits(a, b)
    a.prepare(0)
    c = gpu.Simulation.from_workload(wl.config(1))       # particle-free: nothing to capture
    c.prepare(12)
    c.step(12)


def dense_pack(wl, n_side=10, d=12.0, gap=1.95, big=True):
    """A hexagonal pack of d = 12 discs at surface gap 1.95 (every disc has six neighbours just
    inside the repulsion range s = 2) next to one d = 30 disc, which makes the repulsion cells 32
    wide: the 3 x 3 cells around a disc of the pack then hold more than 40 centres."""
    pitch = d + gap
    xs, ys = [], []
    for r in range(n_side):
        for c in range(n_side):
            xs.append(20.0 + c * pitch + (0.5 * pitch if r % 2 else 0.0))
            ys.append(20.0 + r * pitch * np.sqrt(3.0) / 2.0)
    ds = [d] * len(xs)
    if big:
        xs.append(200.0)
        ys.append(60.0)
        ds.append(30.0)
    n = len(xs)
    p = wl.default_params()
    p.update(g=1.6e-4, gbeta=1e-5, wall_T_type=[1, 1, 1, 1], max_particles=n,
             max_links_per_particle=wl.max_links_for_diameter(30.0))
    parts = dict(x=np.array(xs), y=np.array(ys), diam=np.array(ds), rho_ratio=np.full(n, 1.5),
                 T_w=np.full(n, 1.0))
    return wl.Workload("dense_pack", 240, 170, p, 20, 20, particles=parts)


def test_repulsion_sum_is_order_deterministic_with_many_candidates(gpu, ob, wl):
    """More than 32 candidates in the 3 x 3 repulsion cells (the integrator's batch size): the
    contributions must still be added in ascending particle id, as the oracle does, whatever
    order the cell slots were filled in (atomicAdd order of the flag update, different from run
    to run).  20 repeated runs and both schedules give identical bits; the oracle agrees."""
    w = dense_pack(wl)
    P = w.particles
    cell = 32.0
    ci, cj = np.floor(P["x"] / cell), np.floor(P["y"] / cell)
    k = 44                                            # a disc in the middle of the pack
    cand = int(((np.abs(ci - ci[k]) <= 1) & (np.abs(cj - cj[k]) <= 1)).sum())
    assert cand >= 40, cand
    ref = gpu.Simulation.from_workload(w)
    ref.set_overlap(False)
    ref.step(20)
    pr = ref.particles()
    assert np.abs(pr["ux"]).max() > 1e-3              # the pack is really pushing itself apart
    for rep in range(20):
        s = gpu.Simulation.from_workload(w)
        if rep % 2:
            s.set_graph(False)
        s.step(20)
        ps = s.particles()
        for key in pr:
            assert np.array_equal(ps[key], pr[key]), (rep, key)
    o = ob.OracleSim.from_workload(w)
    o.step(20)
    assert_particles_close(pr, o.particles(), r_min=6.0, steps=20)
    assert_fields_close(ref.fields(populations=True), o.fields(populations=True))


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
