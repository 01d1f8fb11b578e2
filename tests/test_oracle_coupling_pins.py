"""Pins for the rotational and geometric half of the fluid-particle coupling in the oracle's step:
torque and rotational wall velocity (Eqs. 9-10 wall term, 13, 14), mass and moment of inertia as
used by the in-step integrator (Eqs. 7, 8), wall repulsion on all four walls and the ellipse gaps
(Eq. 15), and the ellipse refill normal.

Every expected value here is typed from the mathematics (textbook closed forms, numerical
quadrature of a definition, or a brute-force re-evaluation of the paper's printed sums on the
oracle's OUTPUT fields), never taken from either implementation.  VERDICT r1 listed six oracle
mutations that survived the old pin suite; DESIGN.md section 2 maps each to the test below that
now fails under it.
"""
import math

import numpy as np
import pytest

EX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
EY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])
OPP = np.array([0, 3, 4, 1, 2, 7, 8, 5, 6])


def base_params(wl, n, dmax, **kw):
    p = wl.default_params()
    p.update(max_particles=n, max_links_per_particle=wl.max_links_for_diameter(dmax))
    p.update(kw)
    return p


# ------------------------------------------------------------------ (a) torque: Couette

def spinning_cylinder(ob, wl, r, L=64, nu=1.0 / 6.0, rim_speed=0.01, ratio=1e9, steps=0):
    """A cylinder spinning at Omega = rim_speed / r at the centre of a closed L x L cavity filled
    with fluid at rest; density ratio 1e9 keeps Omega constant."""
    p = base_params(wl, 1, 2 * r, nu=nu, kappa=0.05, g=0.0, gbeta=0.0, rep_s=0.5)
    c = 0.5 * L - 0.5
    parts = dict(x=np.array([c]), y=np.array([c]), diam=np.array([2.0 * r]),
                 rho_ratio=np.array([ratio]), T_w=np.array([0.0]), omega=np.array([rim_speed / r]))
    o = ob.OracleSim.from_workload(wl.Workload("spin", L, L, p, steps, steps, particles=parts))
    if steps:
        o.step(steps)
    return o


@pytest.mark.parametrize("r", [6.0, 9.0])
def test_torque_on_a_spinning_cylinder_matches_circular_couette_flow(ob, wl, r):
    """Steady torque per unit length on a cylinder of radius r rotating at Omega inside a fixed
    concentric cylinder of radius R (Taylor-Couette, any fluid mechanics text):
        T_z = -4 pi mu Omega r^2 / (1 - (r/R)^2).
    The cavity is a square of half-width R = L/2 = 32 (walls half a spacing outside the outermost
    nodes), which holds a little more fluid than the inscribed circle, so the measured magnitude
    sits a little below the concentric value: -1.1 % (r = 8, R = 40) and -1.3 % (r = 12, R = 40) were
    measured; allowed here -3.5 % .. +0.5 %.  Sensitive to: the rotational part of the wall velocity
    u_w = U + Omega x (x_w - x_c) in Eqs. (9)-(10), the sign and the arm of Eq. (14), the factor 2
    w_i rho_0 / c_s^2 of the moving-wall term -- each moves the torque by tens of per cent or flips
    its sign.  Re = Omega r^2 / nu = 0.36-0.54, Mach 0.017."""
    L, nu, rim = 64, 1.0 / 6.0, 0.01
    o = spinning_cylinder(ob, wl, r, L=L, nu=nu, rim_speed=rim, steps=4500)
    T1 = o.particles()["Tz"][0]
    o.step(500)
    P = o.particles()
    Om, R = rim / r, 0.5 * L
    expected = -4.0 * math.pi * (nu * 1.0) * Om * r * r / (1.0 - (r / R) ** 2)
    assert abs(P["Tz"][0] - T1) < 2e-3 * abs(expected)               # steady
    assert -0.035 < P["Tz"][0] / expected - 1.0 < 0.005, (P["Tz"][0], expected)
    assert abs(P["Fx"][0]) < 1e-9 * abs(expected) and abs(P["Fy"][0]) < 1e-9 * abs(expected)
    assert P["omega"][0] == pytest.approx(Om, rel=1e-6)              # heavy: still spinning at Omega
    # the fluid between the cylinders turns with the cylinder: u_theta > 0 on the +x side
    F = o.fields()
    c = int(0.5 * L)
    assert F["uy"][c, c + int(r) + 3] > 0.2 * rim and F["uy"][c, c - int(r) - 4] < -0.2 * rim


# ------------------------------------------------------------------ (b) mass and inertia in the step

def quadrature_mass_inertia(a, b, rho, n=1201):
    """M = rho * area and I = rho * int (x^2 + y^2) dA of an ellipse (a circle for a = b) by the
    midpoint rule on an n x n grid over the bounding box -- the DEFINITIONS, no closed form."""
    xs = (np.arange(n) + 0.5) / n * 2.0 * a - a
    ys = (np.arange(n) + 0.5) / n * 2.0 * b - b
    X, Y = np.meshgrid(xs, ys)
    inside = (X / a) ** 2 + (Y / b) ** 2 <= 1.0
    dA = (2.0 * a / n) * (2.0 * b / n)
    return rho * inside.sum() * dA, rho * ((X * X + Y * Y) * inside).sum() * dA


def one_step_increments(o):
    """(dUx, dUy, dOmega) of particle 0 over one step, and the hydrodynamic F, T_z that step used."""
    a = o.particles()
    o.step(1)
    b = o.particles()
    return (b["ux"][0] - a["ux"][0], b["uy"][0] - a["uy"][0], b["omega"][0] - a["omega"][0],
            b["Fx"][0], b["Fy"][0], b["Tz"][0])


def test_step_accelerates_a_disc_by_F_over_M_and_T_over_half_M_r_squared(ob, wl):
    """Eqs. (7), (8) inside the step: a disc released with translation and spin in fluid at rest
    feels a hydrodynamic force and torque after a few steps; over ONE step
        U(t+1) - U(t) = F(t)/M + gravity term,   Omega(t+1) - Omega(t) = T_z(t)/I
    with M = rho_p pi r^2 and I = M r^2 / 2 (solid disc) typed here and cross-checked against a
    numerical quadrature of rho int dA and rho int (x^2+y^2) dA."""
    r, ratio, g = 5.3, 1.7, 3e-5
    M, I = ratio * math.pi * r * r, 0.5 * ratio * math.pi * r ** 4
    Mq, Iq = quadrature_mass_inertia(r, r, ratio)
    assert abs(Mq / M - 1) < 2e-3 and abs(Iq / I - 1) < 2e-3
    p = base_params(wl, 1, 2 * r, g=g, gbeta=0.0, nu=0.05)
    parts = dict(x=np.array([30.2]), y=np.array([33.6]), diam=np.array([2 * r]),
                 rho_ratio=np.array([ratio]), T_w=np.array([0.0]), ux=np.array([0.03]),
                 uy=np.array([-0.01]), omega=np.array([0.004]))
    o = ob.OracleSim.from_workload(wl.Workload("kick", 64, 64, p, 1, 1, particles=parts))
    o.step(5)
    dux, duy, dom, Fx, Fy, Tz = one_step_increments(o)
    assert abs(Fx) > 1e-3 and abs(Tz) > 1e-3                       # real forces, not round-off
    assert dux == pytest.approx(Fx / M, rel=1e-10)
    assert duy == pytest.approx((Fy - (ratio - 1.0) * math.pi * r * r * g) / M, rel=1e-10)
    assert dom == pytest.approx(Tz / I, rel=1e-10)


def test_step_accelerates_an_ellipse_by_its_quadrature_mass_and_inertia(ob, wl):
    """The same for a 3 : 1 ellipse: M and I from the midpoint-rule quadrature of their
    definitions (to 2e-3), which fixes M = rho_p pi a b and I = M (a^2 + b^2) / 4."""
    a, b, ratio = 9.0, 3.0, 1.4
    Mq, Iq = quadrature_mass_inertia(a, b, ratio)
    p = base_params(wl, 1, 2 * a, g=0.0, gbeta=0.0, nu=0.05)
    parts = dict(x=np.array([40.3]), y=np.array([31.7]), diam=np.array([2 * a]),
                 minor=np.array([2 * b]), theta=np.array([0.5]), rho_ratio=np.array([ratio]),
                 T_w=np.array([0.0]), ux=np.array([0.02]), uy=np.array([0.015]),
                 omega=np.array([0.003]))
    o = ob.OracleSim.from_workload(wl.Workload("kick_ell", 80, 64, p, 1, 1, particles=parts))
    o.step(5)
    dux, duy, dom, Fx, Fy, Tz = one_step_increments(o)
    assert abs(Fx) > 1e-3 and abs(Tz) > 1e-3
    assert dux == pytest.approx(Fx / Mq, rel=3e-3) and duy == pytest.approx(Fy / Mq, rel=3e-3)
    assert dom == pytest.approx(Tz / Iq, rel=3e-3)
    # and exactly, with the closed forms the quadrature confirms
    M = ratio * math.pi * a * b
    assert dom == pytest.approx(Tz / (0.25 * M * (a * a + b * b)), rel=1e-10)
    assert dux == pytest.approx(Fx / M, rel=1e-10)


# ------------------------------------------------------------------ Eq. (14) arm, brute force

def brute_force_momentum_exchange(flag, f_post_t, f_pre_t1, xc, yc, r, U, V, Om):
    """Eqs. (13), (14) as printed, evaluated with plain numpy loops on OUTPUT
    fields: for every fluid node x_f and direction i with x_f + e_i solid,
        dP = f_i^+(x_f, t) (e_i - u_w) - f_ibar(x_f, t + 1) (e_ibar - u_w),
        F = sum dP,   T_z = sum (x_w - x_c) x dP,   x_w = x_f + q e_i,
    q from the circle equation |x_f + q e_i - x_c| = r, u_w = U + Omega x (x_w - x_c).
    Also returns T_z with the arm taken from the NODE x_f instead (the mistake to be excluded)."""
    ny, nx = flag.shape
    F = np.zeros(2)
    Tw = Tn = 0.0
    nlinks = 0
    for j in range(ny):
        for i in range(nx):
            if flag[j, i]:
                continue
            for a in range(1, 9):
                bi, bj = i + EX[a], j + EY[a]
                if not (0 <= bi < nx and 0 <= bj < ny) or not flag[bj, bi]:
                    continue
                ex, ey = float(EX[a]), float(EY[a])
                dx, dy = i - xc, j - yc
                A, B, Cc = ex * ex + ey * ey, 2 * (ex * dx + ey * dy), dx * dx + dy * dy - r * r
                q = (-B - math.sqrt(B * B - 4 * A * Cc)) / (2 * A)
                rx, ry = dx + q * ex, dy + q * ey
                uwx, uwy = U - Om * ry, V + Om * rx
                fi, fb = f_post_t[a, j, i], f_pre_t1[OPP[a], j, i]
                px = fi * (ex - uwx) - fb * (-ex - uwx)
                py = fi * (ey - uwy) - fb * (-ey - uwy)
                F += (px, py)
                Tw += rx * py - ry * px
                Tn += dx * py - dy * px
                nlinks += 1
    return F, Tw, Tn, nlinks


def test_in_step_force_and_torque_equal_a_brute_force_sum_with_the_wall_point_arm(ob, wl):
    """A FIXED disc (it does not move across the lattice, so no node changes sides) whose surface
    translates and spins at Mach ~ 0.1 off-centre in a small box: the F, T_z the step reports must
    equal the brute-force evaluation of Eqs. (13)-(14) on the populations before and after that
    step, with the torque arm x_w - x_c of Eq. (14).  The arm x_f - x_c differs from it at O(u^2)
    only (the part of dP parallel to e_i has no moment about the shifted point), so the flow is
    made fast enough for the two to be 1e-4 apart, and the step is held to 1e-11."""
    r, xc, yc, U, V, Om = 6.3, 24.3, 21.8, 0.08, -0.05, 0.012
    p = base_params(wl, 1, 2 * r, g=0.0, gbeta=0.0, nu=0.02)
    parts = dict(x=np.array([xc]), y=np.array([yc]), diam=np.array([2 * r]),
                 rho_ratio=np.array([2.0]), T_w=np.array([0.0]), ux=np.array([U]),
                 uy=np.array([V]), omega=np.array([Om]), fixed=np.array([1], dtype=np.uint8))
    o = ob.OracleSim.from_workload(wl.Workload("arm", 48, 44, p, 1, 1, particles=parts))
    o.step(60)
    before = o.fields(populations=True)
    o.step(1)
    f_pre_t1, _ = o.precollision()
    P = o.particles()
    assert P["x"][0] == xc and P["ux"][0] == U and P["omega"][0] == Om      # fixed shape, moving wall
    F, Tw, Tn, nlinks = brute_force_momentum_exchange(before["flag"], before["f"], f_pre_t1,
                                                      xc, yc, r, U, V, Om)
    assert nlinks == len(o.links()["q"]) > 100
    scale = abs(Tw)
    assert abs(Tw - Tn) > 1e-4 * scale                       # the test can tell the two arms apart
    assert P["Tz"][0] == pytest.approx(Tw, rel=1e-11)
    assert P["Fx"][0] == pytest.approx(F[0], rel=1e-11) and P["Fy"][0] == pytest.approx(F[1], rel=1e-11)


# ------------------------------------------------------------------ (c) Eq. (15) on all four walls

def test_repulsion_from_each_of_the_four_walls_in_closed_form(ob, wl):
    """Eq. (15) against each cavity wall, first step from rest (F_hydro = 0):
    a disc at surface gap 1.5 from a wall at -1/2 or n-1/2 (s = 2, p = 1: a quarter of C/eps_w) is
    pushed AWAY from that wall with acceleration C (s - delta) / (s eps_w M); C = pi r^2 (rho_p -
    rho_f) g."""
    g, ratio, r, nx, ny = 1.6e-4, 1.5, 4.75, 96, 80
    p = base_params(wl, 4, 10.0, g=g, rep_s=2.0, rep_eps=1e-3, rep_power=1)
    s = ob.OracleSim(nx, ny, p)
    gap = 1.5
    lo = r + gap - 0.5                                   # centre at this distance from node 0
    xs = [lo, nx - 1 - lo, 30.0, 60.0]                   # W, E, S, N
    ys = [40.0, 40.0, lo, ny - 1 - lo]
    s.add_particles(x=xs, y=ys, diam=[2 * r] * 4, rho_ratio=[ratio] * 4, T_w=[0.0] * 4)
    s.step(1)
    P = s.particles()
    area = math.pi * r * r
    C, M = area * (ratio - 1.0) * g, ratio * area
    a_g = -(ratio - 1.0) * area * g / M
    a_w = (C / 1e-3) * (2.0 - gap) / 2.0 / M
    assert a_w > 50 * abs(a_g)                           # the wall force dominates: signs are unmistakable
    expect_ux = [+a_w, -a_w, 0.0, 0.0]
    expect_uy = [a_g, a_g, a_g + a_w, a_g - a_w]
    for k in range(4):
        assert P["ux"][k] == pytest.approx(expect_ux[k], rel=1e-11, abs=1e-16), k
        assert P["uy"][k] == pytest.approx(expect_uy[k], rel=1e-11), k
    # out of range (gap > s): gravity only
    s2 = ob.OracleSim(nx, ny, p)
    far = r + 2.01 - 0.5
    s2.add_particles(x=[far, nx - 1 - far], y=[40.0, 40.0], diam=[2 * r] * 2, rho_ratio=[ratio] * 2,
                     T_w=[0.0] * 2)
    s2.step(1)
    assert np.abs(s2.particles()["ux"]).max() < 1e-15


def test_pair_repulsion_of_unequal_discs_uses_the_mean_force_scale(ob, wl):
    """Eq. (15) between two particles (reading 7: the paper defines the force scale
    C = pi r^2 (rho_p - rho_f) g for a wall only; for a pair the mean of the two is taken, so that
    the forces are equal and opposite).  Two discs of different radius AND density at surface gap
    1.2 on a horizontal line, first step from rest (F_hydro = 0): both receive
    (C_a + C_b) / 2 / eps_w * (s - delta) / s along the line of centres, away from each other, so
    their momenta change by equal and opposite amounts; gravity acts on y only."""
    g, s_rep, eps = 1.6e-4, 2.0, 1e-3
    ra, rb, qa, qb, gap = 5.0, 3.25, 1.5, 1.2, 1.2
    p = base_params(wl, 2, 2 * ra, g=g, rep_s=s_rep, rep_eps=eps, rep_power=1)
    o = ob.OracleSim(120, 90, p)
    xa = 50.0
    xb = xa + ra + rb + gap
    o.add_particles(x=[xa, xb], y=[45.0, 45.0], diam=[2 * ra, 2 * rb], rho_ratio=[qa, qb], T_w=[0.0, 0.0])
    o.step(1)
    P = o.particles()
    Aa, Ab = math.pi * ra * ra, math.pi * rb * rb
    Ca, Cb = Aa * (qa - 1.0) * g, Ab * (qb - 1.0) * g
    Ma, Mb = qa * Aa, qb * Ab
    F = 0.5 * (Ca + Cb) / eps * (s_rep - gap) / s_rep
    assert abs(Ca - Cb) > 0.3 * max(Ca, Cb)             # the two scales differ: own-C readings fail
    assert P["ux"][0] == pytest.approx(-F / Ma, rel=1e-11)
    assert P["ux"][1] == pytest.approx(+F / Mb, rel=1e-11)
    assert Ma * P["ux"][0] + Mb * P["ux"][1] == pytest.approx(0.0, abs=1e-14 * F)
    assert P["uy"][0] == pytest.approx(-(qa - 1.0) / qa * g, rel=1e-11)
    assert P["uy"][1] == pytest.approx(-(qb - 1.0) / qb * g, rel=1e-11)


# ------------------------------------------------------------------ (d) ellipse gaps

def ellipse_pair(ob, wl, theta_a, theta_b, dist, a=8.0, b=4.0, ratio=1.5, g=1.6e-4, vertical=False):
    p = base_params(wl, 2, 2 * a, g=g, rep_s=2.0, rep_eps=1e-3, rep_power=1)
    if vertical:
        x, y = [40.0, 40.0], [30.0, 30.0 + dist]
    else:
        x, y = [30.0, 30.0 + dist], [40.0, 40.0]
    parts = dict(x=np.array(x), y=np.array(y), diam=np.array([2 * a] * 2),
                 minor=np.array([2 * b] * 2), theta=np.array([theta_a, theta_b]),
                 rho_ratio=np.array([ratio] * 2), T_w=np.array([0.0] * 2))
    o = ob.OracleSim.from_workload(wl.Workload("pair", 96, 96, p, 1, 1, particles=parts))
    o.step(1)
    return o.particles()


def test_ellipse_pair_gap_is_taken_through_the_support_functions(ob, wl):
    """Two equal ellipses (a = 8, b = 4) on a line, first step from rest.  The gap along the line
    of centres is dist - (half widths along that line): 2a when both major axes lie on the line,
    2b when both are turned by 90 degrees, a + b for one of each.  Expected velocity increment:
    C (s - delta) / (s eps_w M) with C = pi a b (rho_p - rho_f) g, M = rho_p pi a b, i.e. the gap
    enters alone -- a gap computed from the largest semi-axes (dist - 2a) gives a different force
    for the turned pairs, or none at all."""
    a, b, ratio, g, s_, eps = 8.0, 4.0, 1.5, 1.6e-4, 2.0, 1e-3
    accel = lambda delta: ((ratio - 1.0) * g / eps) * (s_ - delta) / s_ / ratio   # C / (eps M) = (1 - 1/ratio) g / eps
    h = 0.5 * math.pi
    # (i) major axes on the line, gap 1.2
    P = ellipse_pair(ob, wl, 0.0, 0.0, 2 * a + 1.2)
    assert P["ux"][1] == pytest.approx(accel(1.2), rel=1e-11) and P["ux"][0] == pytest.approx(-accel(1.2), rel=1e-11)
    # (ii) both turned: half width along the line is b; gap 1.2 at distance 2b + 1.2 (where the
    # largest-semi-axis gap would be negative)
    P = ellipse_pair(ob, wl, h, h, 2 * b + 1.2)
    assert P["ux"][1] == pytest.approx(accel(1.2), rel=1e-11) and P["ux"][0] == pytest.approx(-accel(1.2), rel=1e-11)
    # (iii) one of each, gap 1.4 (gaps stay above one lattice spacing: with no fluid node between
    # the surfaces the momentum-exchange sum loses links on that side and F_hydro != 0 even at rest)
    P = ellipse_pair(ob, wl, 0.0, h, a + b + 1.4)
    assert P["ux"][1] == pytest.approx(accel(1.4), rel=1e-11)
    # (iv) the same pairs stacked vertically: the roles of the axes swap
    P = ellipse_pair(ob, wl, 0.0, 0.0, 2 * b + 1.3, vertical=True)
    a_g = -(1.0 - 1.0 / ratio) * g
    assert P["uy"][1] == pytest.approx(a_g + accel(1.3), rel=1e-11)
    assert P["uy"][0] == pytest.approx(a_g - accel(1.3), rel=1e-11)
    # (v) beyond the range along the line although the bounding circles overlap: no force
    P = ellipse_pair(ob, wl, h, h, 2 * b + 2.5)
    assert np.abs(P["ux"]).max() < 1e-15
    # every case: no force across the line
    assert abs(P["uy"][0] - a_g) < 1e-15


def test_upright_ellipse_is_repelled_by_the_bottom_wall_at_its_vertex(ob, wl):
    """An ellipse standing upright (major axis vertical) above the bottom wall: the wall gap is
    measured from its lowest point, (y_c + 1/2) - a; lying flat it is (y_c + 1/2) - b."""
    a, b, ratio, g, s_, eps = 8.0, 4.0, 1.5, 1.6e-4, 2.0, 1e-3
    a_g = -(1.0 - 1.0 / ratio) * g
    accel = lambda delta: ((ratio - 1.0) * g / eps) * (s_ - delta) / s_ / ratio
    for theta, half in ((0.5 * math.pi, a), (0.0, b)):
        p = base_params(wl, 1, 2 * a, g=g, rep_s=2.0, rep_eps=1e-3, rep_power=1)
        yc = half + 1.3 - 0.5
        parts = dict(x=np.array([40.0]), y=np.array([yc]), diam=np.array([2 * a]),
                     minor=np.array([2 * b]), theta=np.array([theta]), rho_ratio=np.array([ratio]),
                     T_w=np.array([0.0]))
        o = ob.OracleSim.from_workload(wl.Workload("wall_ell", 80, 64, p, 1, 1, particles=parts))
        o.step(1)
        P = o.particles()
        assert P["uy"][0] == pytest.approx(a_g + accel(1.3), rel=1e-10), theta
        assert abs(P["ux"][0]) < 1e-15


# ------------------------------------------------------------------ (e) ellipse refill normal

def test_ellipse_normal_is_perpendicular_to_the_boundary_tangent(ob):
    """The refill normal of an elliptical particle at a boundary point
    P(t) = R(theta) (a cos t, b sin t) must be perpendicular to the tangent
    dP/dt = R(theta) (-a sin t, b cos t) and point outwards -- for a 3 : 1 ellipse it is up to
    53 degrees away from the radial direction, and picks a different lattice direction e_c."""
    a, b, th = 15.0, 5.0, 0.4
    c, s = math.cos(th), math.sin(th)
    rot = lambda u, v: (u * c - v * s, u * s + v * c)
    worst_angle, different_ec = 0.0, 0
    for t in np.linspace(0.0, 2.0 * math.pi, 97)[:-1]:
        px, py = rot(a * math.cos(t), b * math.sin(t))
        tx, ty = rot(-a * math.sin(t), b * math.cos(t))
        nx_, ny_ = ob.ellipse_normal(px, py, a, b, c, s)
        nn, tn, pn = math.hypot(nx_, ny_), math.hypot(tx, ty), math.hypot(px, py)
        assert abs(nx_ * tx + ny_ * ty) < 1e-12 * nn * tn          # perpendicular to the tangent
        assert nx_ * px + ny_ * py > 0.0                           # outward
        ang = math.degrees(math.acos(min(1.0, (nx_ * px + ny_ * py) / (nn * pn))))
        worst_angle = max(worst_angle, ang)
        if ang > 22.5:
            assert ob.refill_direction(nx_, ny_) != ob.refill_direction(px, py) or ang < 45.0
        different_ec += ob.refill_direction(nx_, ny_) != ob.refill_direction(px, py)
    assert worst_angle > 50.0 and different_ec >= 30
    # a circle written as an ellipse: the normal is radial
    nx_, ny_ = ob.ellipse_normal(3.0, -4.0, 7.0, 7.0, c, s)
    assert abs(nx_ * (-4.0) - ny_ * 3.0) < 1e-15


def test_refilled_node_beside_a_moving_ellipse_is_extrapolated_along_the_surface_normal(ob, wl):
    """In-step use of the normal.  A slender ellipse (a = 15, b = 3, turned by 30 degrees) moves
    along its own minor axis through a fluid with a linear density stratification set up by a
    body force in x (hydrostatic: rho varies along x only, no flow).  A node it uncovers near the
    tip is refilled by extrapolating along e_c (Eq. 16): with the gradient normal the stencil
    runs along the lattice direction closest to the SURFACE normal, with a radial 'normal' along
    the one closest to the ray from the centre, and the stencil nodes the two pick differ -- the
    refilled density tells which was used."""
    a, b, th = 15.0, 3.0, math.radians(30.0)
    c, s = math.cos(th), math.sin(th)
    # move along the minor axis (-s, c) so that the trailing long side uncovers nodes
    speed = 0.12
    U, V = -speed * (-s), -speed * c
    p = base_params(wl, 1, 2 * a, g=0.0, gbeta=0.0, nu=0.1, body_ax=2e-4)
    parts = dict(x=np.array([40.2]), y=np.array([36.4]), diam=np.array([2 * a]),
                 minor=np.array([2 * b]), theta=np.array([th]), rho_ratio=np.array([1e9]),
                 T_w=np.array([0.0]), ux=np.array([U]), uy=np.array([V]))
    o = ob.OracleSim.from_workload(wl.Workload("refill_ell", 80, 72, p, 1, 1, particles=parts))
    checked = 0
    for _ in range(12):
        before = o.fields()
        pb = o.particles()
        o.step(1)
        after = o.fields()
        pa = o.particles()
        f_new, _ = o.precollision()
        born = np.argwhere((before["flag"] == 1) & (after["flag"] == 0))
        for j, i in born:
            dx, dy = i - pa["x"][0], j - pa["y"][0]
            # orientation does not change (omega = 0, heavy particle)
            u, v = dx * c + dy * s, dy * c - dx * s
            gx, gy = (u / a ** 2) * c - (v / b ** 2) * s, (u / a ** 2) * s + (v / b ** 2) * c
            k_norm = best_direction(gx, gy)
            k_rad = best_direction(dx, dy)
            if k_norm == k_rad:
                continue
            # the three stencil nodes along each candidate must be plain fluid before and after
            def stencil(k):
                pts = [(j + m * EY[k], i + m * EX[k]) for m in (1, 2, 3)]
                ok = all(0 <= jj < 72 and 0 <= ii < 80 and before["flag"][jj, ii] == 0
                         and after["flag"][jj, ii] == 0 for jj, ii in pts)
                return pts, ok
            pn, okn = stencil(k_norm)
            pr, okr = stencil(k_rad)
            if not (okn and okr):
                continue
            rho = lambda pts: [f_new[:, jj, ii].sum() for jj, ii in pts]
            rn, rr = rho(pn), rho(pr)
            exp_n = 3 * rn[0] - 3 * rn[1] + rn[2]          # Eq. (16) summed over alpha (the
            exp_r = 3 * rr[0] - 3 * rr[1] + rr[2]          # momentum constraint keeps rho)
            got = f_new[:, j, i].sum()
            if abs(exp_n - exp_r) < 1e-9:
                continue
            assert abs(got - exp_n) < 1e-13, (i, j, got, exp_n, exp_r)
            assert abs(got - exp_r) > 1e-10
            checked += 1
        del pb
    assert checked >= 3, checked


def test_newborn_node_carries_the_equilibrium_temperature_of_the_moving_wall(ob, wl):
    """Eq. (17): g_alpha(x_new) = g_alpha^eq(T_w, u_w) with the wall velocity.
    A hot disc (T_w = 0.8) moves and spins through cold fluid; on every node it uncovers the
    pre-collision temperature populations must sum to T_w and carry the heat flux
    sum e_alpha g_alpha = u_w T_w of that equilibrium, u_w = U + Omega x (x_new - x_c) at t+1."""
    r, Tw = 7.3, 0.8
    p = base_params(wl, 1, 2 * r, g=0.0, gbeta=0.0, nu=0.05)
    parts = dict(x=np.array([30.4]), y=np.array([33.7]), diam=np.array([2 * r]),
                 rho_ratio=np.array([1e9]), T_w=np.array([Tw]), ux=np.array([0.11]),
                 uy=np.array([-0.07]), omega=np.array([0.01]))
    o = ob.OracleSim.from_workload(wl.Workload("refill_T", 72, 64, p, 1, 1, particles=parts))
    checked = 0
    for _ in range(10):
        before = o.fields()
        o.step(1)
        after = o.fields()
        P = o.particles()
        _, g_new = o.precollision()
        for j, i in np.argwhere((before["flag"] == 1) & (after["flag"] == 0)):
            uwx = P["ux"][0] - P["omega"][0] * (j - P["y"][0])
            uwy = P["uy"][0] + P["omega"][0] * (i - P["x"][0])
            gq = g_new[:, j, i]
            assert gq.sum() == pytest.approx(Tw, rel=1e-13)
            assert gq[1] - gq[3] == pytest.approx(uwx * Tw, rel=1e-11)
            assert gq[2] - gq[4] == pytest.approx(uwy * Tw, rel=1e-11)
            assert abs(uwx * Tw) + abs(uwy * Tw) > 0.03               # u_w = 0 would be far off
            checked += 1
    assert checked >= 10, checked


def best_direction(nx_, ny_):
    """The lattice direction alpha in 1..8 maximising n . e_alpha / |e_alpha| (reading 9)."""
    best, bs = 1, -1e300
    for k in range(1, 9):
        sc = (nx_ * EX[k] + ny_ * EY[k]) / math.hypot(EX[k], EY[k])
        if sc > bs + 1e-15:
            best, bs = k, sc
    return best
