"""Pins the oracle's particle part: link builder (brute force, Gauss circle count, 12N-12 bound),
momentum exchange (rest state, zero lift on a symmetric fixed cylinder), repulsion and integrator
inside the full step, refill sanity.  SURVEY.md 8(c) "Pins"."""
import math

import numpy as np
import pytest

EX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
EY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])


def params(wl, n, dmax=20.0, **kw):
    p = wl.default_params()
    p.update(max_particles=n, max_links_per_particle=wl.max_links_for_diameter(dmax))
    p.update(kw)
    return p


def sorted_links(L):
    order = np.lexsort((L["i"], L["j"], L["alpha"], L["pid"]))
    return {k: v[order] for k, v in L.items()}


def numpy_links(nx, ny, xs, ys, rs):
    """Independent enumeration (numpy, no oracle code): node solid iff dx*dx+dy*dy <= r*r for the
    lowest-numbered covering particle."""
    I, J = np.meshgrid(np.arange(nx, dtype=np.float64), np.arange(ny, dtype=np.float64))
    owner = np.full((ny, nx), -1)
    for p in reversed(range(len(xs))):
        dx, dy = I - xs[p], J - ys[p]
        owner[dx * dx + dy * dy <= rs[p] * rs[p]] = p
    out = []
    for a in range(1, 9):
        for j in range(ny):
            for i in range(nx):
                if owner[j, i] >= 0:
                    continue
                bi, bj = i + EX[a], j + EY[a]
                if 0 <= bi < nx and 0 <= bj < ny and owner[bj, bi] >= 0:
                    out.append((owner[bj, bi], a, j, i))
    return owner, sorted(out)


def test_gauss_circle_and_link_count(ob, wl):
    """r = 10 centred on a node: 317 solid nodes (Gauss circle problem, N(10) = 317) and 200 links,
    84 of them along the axes (SURVEY 8(c) pin (ii), recounted here with numpy)."""
    s = ob.OracleSim(40, 40, params(wl, 1))
    s.add_particles(x=[20.0], y=[20.0], diam=[20.0], rho_ratio=[1.5], T_w=[1.0])
    assert int(s.fields()["flag"].sum()) == 317
    L = s.links()
    owner, ref = numpy_links(40, 40, [20.0], [20.0], [10.0])
    assert (owner >= 0).sum() == 317
    assert len(L["q"]) == len(ref) == 200
    assert int((L["alpha"] <= 4).sum()) == 84 and int((L["alpha"] >= 5).sum()) == 116
    for a in range(1, 5):
        assert int((L["alpha"] == a).sum()) == 21
    for a in range(5, 9):
        assert int((L["alpha"] == a).sum()) == 29
    N = int(math.floor(30.0)) - int(math.floor(10.0)) + 3
    assert N == 23 and len(L["q"]) <= 12 * N - 12 == 264


@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_zone_scan_equals_bruteforce_and_numpy(ob, wl, seed):
    """Effective-zone scan == full-lattice scan == independent numpy enumeration,
    for random real-valued centres and diameters, including particles close to the walls."""
    rng = np.random.default_rng(seed)
    nx, ny = 64, 56
    w = wl.sedimentation(nx, ny, 6, seed=100 + seed, y_frac_lo=0.0, d_lo=6.0, d_hi=13.0)
    P = w.particles
    if seed == 3:   # hug the walls: gap below one lattice spacing
        P["x"][0], P["y"][0] = 0.5 * P["diam"][0] - 0.3, 0.5 * P["diam"][0] - 0.4
        P["x"][1], P["y"][1] = nx - 0.5 - 0.5 * P["diam"][1] - 0.05, 30.2
        keep = [0, 1]
        for k in range(2, 6):
            if all(math.hypot(P["x"][k] - P["x"][m], P["y"][k] - P["y"][m]) >
                   0.5 * (P["diam"][k] + P["diam"][m]) for m in keep):
                keep.append(k)
        P = {k: v[keep] for k, v in P.items()}
    s = ob.OracleSim(nx, ny, params(wl, 6, 13.0))
    s.add_particles(**P)
    A, B = sorted_links(s.links()), sorted_links(s.links_bruteforce())
    for k in ("pid", "i", "j", "alpha"):
        assert np.array_equal(A[k], B[k])
    assert np.array_equal(A["q"], B["q"])
    owner, ref = numpy_links(nx, ny, P["x"], P["y"], 0.5 * P["diam"])
    got = sorted(zip(A["pid"].tolist(), A["alpha"].tolist(), A["j"].tolist(), A["i"].tolist()))
    assert got == [tuple(int(v) for v in r) for r in ref]
    assert np.array_equal(s.fields()["flag"], (owner >= 0).astype(np.uint8))
    # per-particle bound 12N-12 and the geometric meaning of q: x_f + q e lies on the circle
    for p in range(len(P["x"])):
        r = 0.5 * P["diam"][p]
        N = int(math.floor(P["x"][p] + r)) - int(math.floor(P["x"][p] - r)) + 3
        Ny = int(math.floor(P["y"][p] + r)) - int(math.floor(P["y"][p] - r)) + 3
        assert int((A["pid"] == p).sum()) <= 12 * max(N, Ny) - 12
    xw = A["i"] + A["q"] * EX[A["alpha"]] - P["x"][A["pid"]]
    yw = A["j"] + A["q"] * EY[A["alpha"]] - P["y"][A["pid"]]
    assert np.all((A["q"] >= 0) & (A["q"] <= 1))
    assert np.abs(np.hypot(xw, yw) - 0.5 * P["diam"][A["pid"]]).max() < 1e-12
    del rng


def test_rest_state_is_a_fixed_point_with_zero_force(ob, wl):
    """Fluid at rest, particle at rest, no gravity, T_w = T0 = wall T: nothing may change and
    the momentum-exchange force vanishes (each lattice line enters and leaves the body once)."""
    p = params(wl, 1, T0=0.5)
    p["wall_T_type"] = [1, 1, 1, 1]
    p["wall_T"] = [0.5] * 4
    s = ob.OracleSim(36, 34, p)
    s.add_particles(x=[17.3], y=[16.6], diam=[11.4], rho_ratio=[1.5], T_w=[0.5])
    s.step(25)
    F = s.fields()
    fl = F["flag"] == 0
    assert np.abs(F["rho"][fl] - 1).max() < 1e-14
    assert np.abs(F["T"][fl] - 0.5).max() < 1e-14
    assert np.abs(F["ux"]).max() < 1e-15 and np.abs(F["uy"]).max() < 1e-15
    P = s.particles()
    assert abs(P["Fx"][0]) < 1e-13 and abs(P["Fy"][0]) < 1e-13 and abs(P["Tz"][0]) < 1e-12
    assert P["x"][0] == pytest.approx(17.3, abs=1e-12) and P["y"][0] == pytest.approx(16.6, abs=1e-12)


def test_zero_lift_on_symmetric_fixed_cylinder(ob, wl):
    """Fixed cylinder centred on the centreline node row of a body-force channel (periodic_x):
    |F_y|/|F_x| < 1e-10 and T_z ~ 0 by mirror symmetry; the drag is positive (along the flow)."""
    nx, ny = 60, 41
    p = params(wl, 1, dmax=10.0, periodic_x=1, body_ax=2e-6, nu=0.1)
    s = ob.OracleSim(nx, ny, p)
    s.add_particles(x=[30.0], y=[20.0], diam=[10.0], rho_ratio=[1.5], T_w=[0.0], fixed=[1])
    s.step(1200)
    P = s.particles()
    assert P["Fx"][0] > 1e-6
    assert abs(P["Fy"][0]) / abs(P["Fx"][0]) < 1e-10
    assert abs(P["Tz"][0]) / (abs(P["Fx"][0]) * 5.0) < 1e-10
    assert P["x"][0] == 30.0 and P["ux"][0] == 0.0           # fixed
    F = s.fields()
    assert np.abs(F["ux"] - F["ux"][::-1]).max() < 1e-13      # mirror-symmetric flow
    assert np.abs(F["uy"] + F["uy"][::-1]).max() < 1e-13
    # steady momentum balance: body force on the fluid = drag on cylinder + wall friction, so the
    # drag cannot exceed the total body force
    assert P["Fx"][0] < 2e-6 * (F["flag"] == 0).sum()


def faxen_drag_per_length(mu, U, k):
    """Stokes drag per unit length on a circular cylinder moving with speed U along the mid-plane
    between two parallel walls, k = diameter / wall spacing (Faxen 1946, as quoted in Happel &
    Brenner, Low Reynolds Number Hydrodynamics, Sec. 7-8): F = 4 pi mu U / Lambda(k)."""
    lam = (math.log(1.0 / k) - 0.9157 + 1.7244 * k ** 2 - 1.7302 * k ** 4 + 2.4056 * k ** 6
           - 4.5913 * k ** 8)
    return 4.0 * math.pi * mu * U / lam


def faxen_workload(wl, d=10.0, W=40, L=240, U=0.005, nu=1.0 / 6.0, steps=6000):
    """A heavy cylinder (density ratio 1e9: its velocity stays U) moving along the mid-plane of a
    long closed cavity filled with fluid at rest (closed ends: no net flow past the cylinder, as in
    Faxen's problem).  Re = U d / nu = 0.3."""
    p = wl.default_params()
    p.update(nu=nu, kappa=0.05, g=0.0, gbeta=0.0, max_particles=1, rep_s=0.5,
             max_links_per_particle=wl.max_links_for_diameter(d))
    parts = dict(x=np.array([0.3 * L]), y=np.array([0.5 * W - 0.5]), diam=np.array([d]),
                 rho_ratio=np.array([1e9]), T_w=np.array([0.0]), ux=np.array([U]),
                 uy=np.array([0.0]), omega=np.array([0.0]))
    return wl.Workload("faxen", L, W, p, steps, steps, particles=parts)


def test_drag_on_a_moving_cylinder_between_walls_matches_faxen(ob, wl):
    """Pins the whole coupled step quantitatively -- interpolated moving-wall bounce-back (Eqs. 9,
    10), Galilean-invariant momentum exchange (Eq. 13), flag update and refill (Eq. 16) of a
    particle that really moves across the lattice -- to a textbook closed form: after the
    transient (6000 steps = 6 viscous times W^2/(pi^2 nu)) the drag, averaged over the last 200
    steps (one lattice spacing of travel), is Faxen's.  A dropped wall-velocity term, a wrong
    interpolation coefficient or a force sign or factor error moves it by far more than the 2.5 %
    allowed (measured: -0.9 % at d = 10 l.u.)."""
    d, W, U, nu = 10.0, 40, 0.005, 1.0 / 6.0
    o = ob.OracleSim.from_workload(faxen_workload(wl, d=d, W=W, U=U, nu=nu, steps=6000))
    o.step(5800)
    F = []
    for _ in range(200):
        o.step(1)
        p = o.particles()
        F.append((p["Fx"][0], p["Fy"][0], p["Tz"][0]))
    F = np.array(F)
    expected = faxen_drag_per_length(nu * 1.0, U, d / W)
    drag = -F[:, 0].mean()
    assert abs(drag / expected - 1.0) < 0.025, (drag, expected)
    assert abs(F[:, 0] + drag).max() < 0.02 * drag          # lattice-position ripple is small
    assert abs(F[:, 1]).max() < 1e-9 * drag and abs(F[:, 2]).max() < 1e-8 * drag * d   # symmetry
    assert abs(p["ux"][0] - U) < 1e-6 * U and abs(p["x"][0] - (0.3 * 240 + 6000 * U)) < 1e-4


def settling_workload(wl, d=10.0, W=40, L=240, nu=1.0 / 6.0, ratio=1.2, U_target=0.005):
    """A cylinder released from rest on the axis of a tall closed channel, with gravity chosen so
    that the balance weight - buoyancy = Faxen drag gives the terminal speed U_target."""
    lam = 4.0 * math.pi * nu * U_target / faxen_drag_per_length(nu, U_target, d / W)
    g = U_target * 4.0 * nu / ((ratio - 1.0) * (0.5 * d) ** 2 * lam)
    p = wl.default_params()
    p.update(nu=nu, kappa=0.05, g=g, gbeta=0.0, max_particles=1, rep_s=0.5,
             max_links_per_particle=wl.max_links_for_diameter(d))
    parts = dict(x=np.array([0.5 * W - 0.5]), y=np.array([0.75 * L]), diam=np.array([d]),
                 rho_ratio=np.array([ratio]), T_w=np.array([0.0]))
    return wl.Workload("settling", W, L, p, 6000, 6000, particles=parts)


def test_terminal_velocity_of_a_settling_cylinder_matches_the_faxen_balance(ob, wl):
    """The closed loop of the coupling: weight minus buoyancy (pi r^2 (rho_p - rho_f) g), the
    hydrodynamic force of Eqs. (9), (10), (13) and the integrator of Eqs. (7), (8) bring a freely
    moving cylinder to the speed at which Faxen's drag balances its net weight: within 2.5 %
    (measured +0.9 %), falling straight down the axis, not rotating."""
    U = 0.005
    o = ob.OracleSim.from_workload(settling_workload(wl, U_target=U))
    o.step(5000)
    u1 = o.particles()["uy"][0]
    o.step(1000)
    p = o.particles()
    assert abs(p["uy"][0] - u1) < 2e-3 * U                         # terminal
    assert abs(-p["uy"][0] / U - 1.0) < 0.025, p["uy"][0]
    assert abs(p["ux"][0]) < 1e-12 and abs(p["omega"][0]) < 1e-12 and abs(p["x"][0] - 19.5) < 1e-9


def conduction_workload(wl, d=10.0, W=40, L=240, kappa=0.1, steps=6000):
    """A fixed hot cylinder (T_w = 1) midway between two cold walls (T = 0) of a long cavity with
    adiabatic ends, no flow (g beta = 0): pure conduction."""
    p = wl.default_params()
    p.update(nu=0.1, kappa=kappa, g=0.0, gbeta=0.0, max_particles=1, rep_s=0.5,
             max_links_per_particle=wl.max_links_for_diameter(d),
             wall_T_type=[0, 0, 1, 1], wall_T=[0.0, 0.0, 0.0, 0.0])
    parts = dict(x=np.array([0.5 * L - 0.5]), y=np.array([0.5 * W - 0.5]), diam=np.array([d]),
                 rho_ratio=np.array([2.0]), T_w=np.array([1.0]), fixed=np.array([1], dtype=np.uint8))
    return wl.Workload("conduction", L, W, p, steps, steps, particles=parts)


def wall_heat_flow(T, kappa):
    """Heat per unit time into the two cold walls: the first node row lies half a spacing from
    the wall (T_wall = 0), rho c_p = 1."""
    return kappa * (T[0, :].sum() + T[-1, :].sum()) / 0.5


def shape_factor_cylinder_between_planes(d, z):
    """Conduction shape factor per unit length of a circular cylinder of diameter d midway between
    two parallel isothermal planes at distance z from its axis, z >> d/2 (the standard heat
    transfer table entry, e.g. Incropera & DeWitt Table 4.1): S = 2 pi / ln(8 z / (pi d))."""
    return 2.0 * math.pi / math.log(8.0 * z / (math.pi * d))


def test_heat_flow_from_a_hot_cylinder_matches_the_conduction_shape_factor(ob, wl):
    """Pins the thermal side of the fluid-particle coupling -- the curved-wall Dirichlet
    bounce-back of Eqs. (11), (12) with the D2Q5 collision (kappa) and the cold cavity walls -- to
    a closed form: in steady conduction the heat flowing into the walls is S kappa (T_w - T_c)
    with the textbook shape factor of a cylinder between two planes.  A wrong c_d coefficient, a
    missing factor in the 2 w T_w term or a wrong thermal weight changes it by tens of per cent;
    allowed 2 % (measured -0.7 % at d = 10, z = 20: the formula itself assumes z >> d/2 and the
    cavity is 24 d long)."""
    d, W, kappa = 10.0, 40, 0.1
    o = ob.OracleSim.from_workload(conduction_workload(wl, d=d, W=W, kappa=kappa, steps=6000))
    o.step(5000)
    q1 = wall_heat_flow(o.fields()["T"], kappa)
    o.step(1000)
    f = o.fields()
    q2 = wall_heat_flow(f["T"], kappa)
    assert abs(q2 - q1) < 1e-2 * q2                              # (nearly) steady
    expected = shape_factor_cylinder_between_planes(d, 0.5 * W) * kappa * 1.0
    assert abs(q2 / expected - 1.0) < 0.02, (q2, expected)
    fluid = f["flag"] == 0
    assert f["T"][fluid].max() < 1.0 and f["T"][fluid].min() > -1e-12   # maximum principle
    assert float(np.abs(f["ux"][fluid]).max()) < 1e-12            # no flow was started


def test_repulsion_and_gravity_enter_the_first_step_in_closed_form(ob, wl):
    """At t = 0 the fluid is at rest, so F_hydro = 0 and U(1) = (weight + Eq. 15)/M exactly:
    pair at gap 1.5 (s = 2, p = 1 -> a quarter of C/eps) and a particle at gap 1.5 from the bottom
    wall.  (Gaps are chosen so that fluid nodes remain between the surfaces: with none, the
    momentum-exchange sum loses the links of that side and F_hydro != 0 even at rest.)"""
    g, ratio, r = 1.6e-4, 1.5, 4.75
    p = params(wl, 3, dmax=10.0, g=g, rep_s=2.0, rep_eps=1e-3, rep_power=1)
    s = ob.OracleSim(64, 48, p)
    s.add_particles(x=[20.0, 31.0, 50.0], y=[30.0, 30.0, r + 1.0], diam=[2 * r] * 3,
                    rho_ratio=[ratio] * 3, T_w=[0.0] * 3)
    s.step(1)
    P = s.particles()
    area = math.pi * r * r
    C = area * (ratio - 1) * g
    M = ratio * area
    a_g = -(ratio - 1) * area * g / M
    a_pair = (C / 1e-3) * (2.0 - 1.5) / 2.0 / M
    assert np.allclose([P["Fx"][0], P["Fy"][0]], 0, atol=1e-13)
    assert P["ux"][0] == pytest.approx(-a_pair, rel=1e-12)
    assert P["ux"][1] == pytest.approx(+a_pair, rel=1e-12)
    assert P["uy"][0] == pytest.approx(a_g, rel=1e-10) and P["uy"][1] == pytest.approx(a_g, rel=1e-10)
    a_wall = (C / 1e-3) * (2.0 - 1.5) / 2.0 / M
    assert P["uy"][2] == pytest.approx(a_g + a_wall, rel=1e-12)
    assert P["ux"][2] == pytest.approx(0.0, abs=1e-15)
    assert P["x"][0] == pytest.approx(20.0 - 0.5 * a_pair, rel=1e-14)   # trapezoid position update
    # quadratic variant of the paper (p = 2, s = 3): quarter of C/eps at half the range
    p2 = params(wl, 2, dmax=10.0, g=g, rep_s=3.0, rep_eps=1e-3, rep_power=2)
    s2 = ob.OracleSim(64, 48, p2)
    s2.add_particles(x=[20.0, 31.0], y=[30.0, 30.0], diam=[2 * r] * 2, rho_ratio=[ratio] * 2, T_w=[0.0] * 2)
    s2.step(1)
    assert s2.particles()["ux"][1] == pytest.approx((C / 1e-3) * 0.25 / M, rel=1e-12)


def test_argument_and_state_errors(ob, wl):
    p = params(wl, 2)
    s = ob.OracleSim(64, 64, p)
    with pytest.raises(ob.OracleError) as e:
        s.add_particles(x=[5.0], y=[30.0], diam=[20.0], rho_ratio=[1.5], T_w=[1.0])   # through W wall
    assert e.value.code == -1
    with pytest.raises(ob.OracleError) as e:
        s.add_particles(x=[20.0, 30.0], y=[30.0, 30.0], diam=[20.0, 20.0], rho_ratio=[1.5] * 2, T_w=[1.0] * 2)
    assert e.value.code == -1                                                            # overlap
    with pytest.raises(ob.OracleError) as e:
        s.add_particles(x=[20.0] * 3, y=[30.0] * 3, diam=[4.0] * 3, rho_ratio=[1.5] * 3, T_w=[1.0] * 3)
    assert e.value.code == -3                                                            # capacity
    s.add_particles(x=[20.0], y=[30.0], diam=[20.0], rho_ratio=[1.5], T_w=[1.0])
    s.step(1)
    with pytest.raises(ob.OracleError) as e:
        s.add_particles(x=[45.0], y=[30.0], diam=[10.0], rho_ratio=[1.5], T_w=[1.0])
    assert e.value.code == -2
    p3 = params(wl, 1)
    p3["max_links_per_particle"] = 100
    s3 = ob.OracleSim(64, 64, p3)
    with pytest.raises(ob.OracleError) as e:
        s3.add_particles(x=[20.0], y=[30.0], diam=[20.0], rho_ratio=[1.5], T_w=[1.0])
    assert e.value.code == -3


def test_moving_particle_refill_keeps_fields_sane(ob, wl):
    """A particle launched at |U| = 0.06 crosses ~5 lattice rows in 100 steps, so many nodes are
    covered and uncovered (Eqs. 16-17).  Fields stay finite and bounded, the solid-node count stays
    that of a radius-6 disc (113 +- a few), and the hot wake stays within [T0, T_w] (+-5 %)."""
    p = params(wl, 1, dmax=12.0, g=0.0, gbeta=0.0)
    p["wall_T_type"] = [1, 1, 1, 1]
    s = ob.OracleSim(48, 64, p)
    s.add_particles(x=[24.3], y=[44.2], diam=[12.0], rho_ratio=[4.0], T_w=[1.0], ux=[0.01], uy=[-0.06],
                    omega=[0.002])
    y_prev = 44.2
    for _ in range(5):
        s.step(20)
        F = s.fields()
        fl = F["flag"] == 0
        assert np.isfinite(F["rho"]).all() and np.isfinite(F["T"]).all()
        assert np.abs(F["rho"][fl] - 1).max() < 0.08
        assert F["T"][fl].min() > -0.05 and F["T"][fl].max() < 1.05
        assert abs(int(F["flag"].sum()) - 113) <= 6
        y = s.particles()["y"][0]
        assert y < y_prev
        y_prev = y
    assert 44.2 - y_prev > 3.0
    # fluid next to the particle is dragged along: downward velocity just below it
    P = s.particles()
    j, i = int(round(P["y"][0] - 8)), int(round(P["x"][0]))
    assert s.fields()["uy"][j, i] < -0.005


def test_config0_physical_sanity(ob, wl):
    """Config 0 (single hot particle): accelerates downward, stays below the reference velocity
    U_ref = sqrt(g pi d (rho_p/rho_f - 1)/2), stays on the axis, heats the fluid."""
    w = wl.config(0)
    s = ob.OracleSim.from_workload(w)
    v = []
    for _ in range(3):
        s.step(100)
        v.append(s.particles()["uy"][0])
    Uref = math.sqrt(w.params["g"] * math.pi * 20 * 0.5 / 2)
    assert Uref == pytest.approx(0.050, abs=0.001)
    assert v[0] < 0 and v[1] < v[0] and v[2] < v[1]
    assert abs(v[2]) < Uref
    P = s.particles()
    # (64, 200) is half a spacing off the box axis x = 63.5, so a tiny lateral drift is physical
    assert abs(P["x"][0] - 64.0) < 1e-2 and abs(P["omega"][0]) < 1e-4
    F = s.fields()
    fl = F["flag"] == 0
    assert F["T"][fl].max() > 0.5 and F["T"][fl].min() > -0.02
    jc, ic = int(round(P["y"][0])), 64
    assert F["T"][jc + 13, ic] > F["T"][jc - 13, ic]                # the warm wake trails above


# ------------------------------------------------------------------ elliptical particles

def ellipse_sim(ob, wl, nx, ny, x, y, major, minor, theta, **kw):
    n = len(x)
    p = params(wl, n, dmax=float(np.max(major)), **kw)
    parts = dict(x=np.asarray(x, float), y=np.asarray(y, float), diam=np.asarray(major, float),
                 minor=np.asarray(minor, float), theta=np.asarray(theta, float),
                 rho_ratio=np.full(n, 1.5), T_w=np.full(n, 1.0))
    w = wl.Workload("ell", nx, ny, p, 1, 1, particles=parts)
    return ob.OracleSim.from_workload(w), w


def numpy_ellipse_flags(nx, ny, x, y, major, minor, theta):
    """Independent rasterisation with the documented operation order: u = dx c + dy s,
    v = dy c - dx s, (u/a)^2 + (v/b)^2 <= 1 (numpy evaluates each operation separately rounded)."""
    I, J = np.meshgrid(np.arange(nx, dtype=np.float64), np.arange(ny, dtype=np.float64))
    flag = np.zeros((ny, nx), dtype=np.uint8)
    for xc, yc, A, B, th in zip(x, y, major, minor, theta):
        a, b, c, s = 0.5 * A, 0.5 * B, math.cos(th), math.sin(th)
        dx, dy = I - xc, J - yc
        u, v = dx * c + dy * s, dy * c - dx * s
        ua, vb = u / a, v / b
        flag |= (ua * ua + vb * vb <= 1.0).astype(np.uint8)
    return flag


def test_ellipse_rasterisation_matches_numpy_and_the_area(ob, wl):
    x, y = [40.3, 110.7, 170.0], [45.6, 50.2, 48.0]
    major, minor = [50.0, 30.0, 24.0], [20.0, 29.0, 8.0]
    theta = np.radians([25.0, -70.0, 90.0])
    o, _ = ellipse_sim(ob, wl, 210, 100, x, y, major, minor, theta)
    flag = o.fields()["flag"]
    assert np.array_equal(flag, numpy_ellipse_flags(210, 100, x, y, major, minor, theta))
    # lattice points in an ellipse: area pi a b up to a perimeter-sized error
    for k in range(3):
        sub = numpy_ellipse_flags(210, 100, x[k:k + 1], y[k:k + 1], major[k:k + 1], minor[k:k + 1],
                                  theta[k:k + 1])
        area = math.pi * 0.25 * major[k] * minor[k]
        assert abs(int(sub.sum()) - area) < 0.5 * (major[k] + minor[k])


def test_ray_ellipse_q_closed_forms(ob):
    """q on the axes of an axis-aligned ellipse is the distance to the vertex; turning the ellipse
    by 90 degrees swaps the axes; a = b reduces to the circle's q."""
    a, b = 12.0, 6.0
    assert abs(ob.link_q_ellipse(-13.0, 0.0, 1, 0.0, 0.0, a, b, 1.0, 0.0) - 1.0) < 1e-12
    assert abs(ob.link_q_ellipse(-12.5, 0.0, 1, 0.0, 0.0, a, b, 1.0, 0.0) - 0.5) < 1e-12
    assert abs(ob.link_q_ellipse(0.0, 6.25, 4, 0.0, 0.0, a, b, 1.0, 0.0) - 0.25) < 1e-12
    assert abs(ob.link_q_ellipse(0.0, 12.75, 4, 0.0, 0.0, a, b, 0.0, 1.0) - 0.75) < 1e-12    # turned
    # diagonal ray towards a circle written as an ellipse: same as the circle routine
    for xf, yf, al in ((-8.0, -7.0, 5), (7.5, 7.2, 7), (-7.1, 7.9, 8)):
        qe = ob.link_q_ellipse(xf, yf, al, 0.3, -0.2, 10.0, 10.0, math.cos(0.7), math.sin(0.7))
        assert abs(qe - ob.link_q(xf, yf, al, 0.3, -0.2, 10.0)) < 1e-12
    # a general case against the parametric intersection solved with numpy
    xc, yc, th = 1.3, -0.4, 0.6
    c, s = math.cos(th), math.sin(th)
    xf, yf, al = -9.0, -8.0, 5                        # e5 = (1, 1); its neighbour is inside
    q = ob.link_q_ellipse(xf, yf, al, xc, yc, a, b, c, s)
    px, py = xf + q * 1.0 - xc, yf + q * 1.0 - yc
    u, v = px * c + py * s, py * c - px * s
    assert 0.0 < q < 1.0 and abs((u / a) ** 2 + (v / b) ** 2 - 1.0) < 1e-12


def test_ellipse_zone_scan_equals_bruteforce(ob, wl):
    x, y = [40.3, 85.0, 130.0], [45.6, 50.2, 48.0]
    major, minor = [40.0, 30.0, 24.0], [18.0, 29.5, 10.0]
    theta = np.radians([35.0, -70.0, 80.0])
    o, _ = ellipse_sim(ob, wl, 170, 100, x, y, major, minor, theta)
    A, B = sorted_links(o.links()), sorted_links(o.links_bruteforce())
    assert len(A["q"]) == len(B["q"]) > 300
    for k in A:
        assert np.array_equal(A[k], B[k]), k
    assert (A["q"] >= 0).all() and (A["q"] <= 1).all()
    # every link's solid end is inside the ellipse and its fluid end outside (numpy predicate)
    flag = numpy_ellipse_flags(170, 100, x, y, major, minor, theta)
    assert (flag[A["j"], A["i"]] == 0).all()
    assert (flag[A["j"] + EY[A["alpha"]], A["i"] + EX[A["alpha"]]] == 1).all()


def test_orientation_vector_is_advanced_by_an_exact_rotation(ob):
    """The Cayley step is a rotation by 2 atan(d/2): the vector stays on the unit circle and n
    steps compose to the angle n * 2 atan(d/2), which equals n d to O(d^3)."""
    c, s, d, n = math.cos(0.3), math.sin(0.3), 2.0e-3, 5000
    for _ in range(n):
        c, s = ob.rotate_unit(c, s, d)
    assert abs(c * c + s * s - 1.0) < 1e-15
    ang = 0.3 + n * 2.0 * math.atan(0.5 * d)
    assert abs(c - math.cos(ang)) < 1e-12 and abs(s - math.sin(ang)) < 1e-12
    assert abs(ang - (0.3 + n * d)) < n * d ** 3 / 10.0


def test_ellipse_mass_inertia_and_torque_free_spin(ob, wl):
    """An ellipse in a fluid at rest without gravity: released with a spin, its angular velocity
    decays (viscous torque opposes it) and its centre stays put by symmetry; a first step under
    gravity alone moves it by the free-fall increment of a body of area pi a b."""
    o, w = ellipse_sim(ob, wl, 120, 120, [59.5], [59.5], [40.0], [20.0], [0.4], g=0.0)
    o.step(1)
    # gravity: first-step velocity -(1 - 1/ratio) g, independent of the shape (hydro force is zero)
    p2 = params(wl, 1, dmax=40.0, g=2e-4)
    parts = dict(x=np.array([59.5]), y=np.array([59.5]), diam=np.array([40.0]), minor=np.array([20.0]),
                 theta=np.array([0.4]), rho_ratio=np.array([1.5]), T_w=np.array([0.0]))
    o2 = ob.OracleSim.from_workload(wl.Workload("e", 120, 120, p2, 1, 1, particles=parts))
    o2.step(1)
    q = o2.particles()
    assert abs(q["uy"][0] + (1.0 - 1.0 / 1.5) * 2e-4) < 1e-15 and abs(q["ux"][0]) < 1e-18
    # spin decay
    parts.update(omega=np.array([2e-3]))
    o3 = ob.OracleSim.from_workload(wl.Workload("e", 120, 120, params(wl, 1, dmax=40.0, g=0.0), 1, 1,
                                                particles=parts))
    o3.step(300)
    q = o3.particles()
    assert 0.0 < q["omega"][0] < 2e-3
    assert abs(q["x"][0] - 59.5) < 1e-6 and abs(q["y"][0] - 59.5) < 1e-6
    assert q["theta"][0] > 0.4 + 0.1
