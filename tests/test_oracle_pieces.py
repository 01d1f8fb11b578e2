"""Pins every piece of the CPU oracle to something other than itself: closed forms, algebraic
identities of the printed equations, textbook special cases (SURVEY.md 8(c) "Pins").
The expected values below are typed from the paper's equations / the mathematics, never produced
by the oracle or by the CUDA path."""
import math

import numpy as np
import pytest

EX = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1])
EY = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1])
OPP = [0, 3, 4, 1, 2, 7, 8, 5, 6]
W9 = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
RNG = np.random.default_rng(12345)


def base_params(wl, **kw):
    p = wl.default_params()
    p.update(kw)
    return p


# ---------------- transforms ----------------
def test_M_rows_orthogonal_and_inverse(ob):
    M = np.array([ob.moments_f(np.eye(9)[i]) for i in range(9)]).T  # M[k, i]
    G = M @ M.T
    assert np.array_equal(np.diag(G), [9, 36, 36, 6, 12, 6, 12, 4, 4])  # SURVEY 8(c) pins
    assert np.count_nonzero(G - np.diag(np.diag(G))) == 0
    # conserved rows are the lattice velocities themselves
    assert np.array_equal(M[0], np.ones(9))
    assert np.array_equal(M[3], EX) and np.array_equal(M[5], EY)
    f = RNG.uniform(0.01, 1.0, 9)
    assert np.allclose(ob.from_moments_f(ob.moments_f(f)), f, rtol=0, atol=1e-15)
    assert np.allclose(ob.from_moments_f(ob.moments_f(f)), np.linalg.solve(M, M @ f), atol=1e-14)


def test_N_rows_orthogonal_and_inverse(ob):
    N = np.array([ob.moments_g(np.eye(5)[i]) for i in range(5)]).T
    G = N @ N.T
    assert np.array_equal(np.diag(G), [5, 2, 2, 20, 4])
    assert np.count_nonzero(G - np.diag(np.diag(G))) == 0
    assert np.array_equal(N[0], np.ones(5))
    assert np.array_equal(N[1], EX[:5]) and np.array_equal(N[2], EY[:5])
    g = RNG.uniform(0.01, 1.0, 5)
    assert np.allclose(ob.from_moments_g(ob.moments_g(g)), g, atol=1e-15)


# ---------------- equilibria ----------------
@pytest.mark.parametrize("rho,ux,uy", [(1.0, 0.0, 0.0), (1.03, 0.05, -0.02), (0.97, -0.08, 0.06)])
def test_feq_is_the_second_order_polynomial(ob, rho, ux, uy):
    eu = EX * ux + EY * uy
    poly = W9 * rho * (1 + 3 * eu + 4.5 * eu ** 2 - 1.5 * (ux * ux + uy * uy))
    assert np.allclose(ob.feq(rho, ux, uy), poly, rtol=0, atol=2e-16)
    m = ob.moments_f(ob.feq(rho, ux, uy))
    u2 = ux * ux + uy * uy
    meq = rho * np.array([1, -2 + 3 * u2, 1 - 3 * u2, ux, -ux, uy, -uy, ux * ux - uy * uy, ux * uy])
    assert np.allclose(m, meq, atol=1e-15)


@pytest.mark.parametrize("T,ux,uy,kappa", [(1.0, 0, 0, 0.02 / 0.7), (0.37, 0.04, -0.03, 0.0223455)])
def test_geq_closed_form(ob, T, ux, uy, kappa):
    aT = 20 * math.sqrt(3) * kappa - 4
    w = np.array([(1 - aT) / 5] + [(4 + aT) / 20] * 4)
    expect = w * T + (EX[:5] * ux + EY[:5] * uy) * T / 2
    got = ob.geq(T, ux, uy, kappa)
    assert np.allclose(got, expect, atol=1e-16)
    assert got.sum() == pytest.approx(T, abs=1e-15)
    assert (EX[:5] * got).sum() == pytest.approx(ux * T, abs=1e-16)
    assert w.sum() == pytest.approx(1.0)


def test_relaxation_rates(ob):
    nu, kappa = 0.02, 0.02 / 0.7
    S, Q, aT = ob.relaxation_rates(nu, kappa)
    snu = 1 / (3 * nu + 0.5)
    assert S[0] == S[3] == S[5] == 0.0                       # conserved moments
    assert S[7] == S[8] == pytest.approx(snu)
    assert S[1] == S[2] == pytest.approx(snu)
    assert S[4] == S[6] == pytest.approx(8 * (2 - snu) / (8 - snu))
    assert Q[0] == 0.0
    qk = 3 - math.sqrt(3)
    assert Q[1] == Q[2] == pytest.approx(qk)
    assert Q[3] == Q[4] == pytest.approx(4 * math.sqrt(3) - 6)
    # kappa = (4+a_T)/10 (1/q_kappa - 1/2)
    assert (4 + aT) / 10 * (1 / qk - 0.5) == pytest.approx(kappa, rel=1e-14)
    # the "magic" combination that puts halfway walls exactly halfway:
    # (1/s_nu - 1/2)(1/s_q - 1/2) = 3/16
    assert (1 / S[7] - 0.5) * (1 / S[4] - 0.5) == pytest.approx(3 / 16, rel=1e-14)


# ---------------- collision ----------------
def test_collision_conserves_mass_heat_and_adds_exactly_F(ob, wl):
    P = base_params(wl, nu=0.03, kappa=0.04, gbeta=2e-4, T0=0.25, body_ax=3e-5, body_ay=-1e-5)
    for _ in range(20):
        f = ob.feq(1.0, 0.0, 0.0) * RNG.uniform(0.9, 1.1, 9)
        g = RNG.uniform(0.0, 0.3, 5)
        fo, go = ob.collide_node(P, f, g)
        rho, T = f.sum(), g.sum()
        Fx = rho * P["body_ax"]
        Fy = rho * (P["body_ay"] + P["gbeta"] * (T - P["T0"]))
        assert fo.sum() == pytest.approx(rho, abs=2e-15)
        assert go.sum() == pytest.approx(T, abs=2e-15)
        assert (EX * fo).sum() - (EX * f).sum() == pytest.approx(Fx, abs=1e-15)
        assert (EY * fo).sum() - (EY * f).sum() == pytest.approx(Fy, abs=1e-15)
        r, ux, uy, TT = ob.macroscopic(P, f, g)
        assert r == pytest.approx(rho, abs=1e-15) and TT == pytest.approx(T, abs=1e-15)
        assert ux == pytest.approx(((EX * f).sum() + Fx / 2) / rho, abs=1e-16)
        assert uy == pytest.approx(((EY * f).sum() + Fy / 2) / rho, abs=1e-16)


def test_equilibrium_is_a_fixed_point_without_force(ob, wl):
    P = base_params(wl)
    f = ob.feq(1.02, 0.03, -0.04)
    g = ob.geq(0.6, 0.03 / 1.0, -0.04 / 1.0, P["kappa"])
    # velocity of f is exactly (0.03, -0.04) (no force), so g_eq must be built with it
    fo, go = ob.collide_node(P, f, g)
    assert np.allclose(fo, f, atol=1e-16)
    assert np.allclose(go, g, atol=1e-16)


def test_collision_relaxes_stress_with_s_nu_and_matches_bgk_limit(ob, wl):
    """Non-equilibrium shear moment decays by (1 - s_nu): the definition of the viscosity
    nu = (1/s_nu - 1/2)/3.  When all rates are equal MRT is BGK; here only pxy is perturbed."""
    nu = 0.07
    P = base_params(wl, nu=nu)
    f0 = ob.feq(1.0, 0.0, 0.0)
    m = ob.moments_f(f0)
    m[8] += 1e-3   # p_xy
    m[7] -= 2e-3   # p_xx
    f = ob.from_moments_f(m)
    fo, _ = ob.collide_node(P, f, ob.geq(0, 0, 0, P["kappa"]))
    mo = ob.moments_f(fo)
    snu = 1 / (3 * nu + 0.5)
    assert mo[8] == pytest.approx((1 - snu) * 1e-3, abs=1e-16)
    assert mo[7] == pytest.approx(-(1 - snu) * 2e-3, abs=1e-16)


def test_forced_collision_equals_textbook_bgk_with_guo_forcing_when_all_rates_coincide(ob, wl):
    """Pins the whole forcing vector of Eq. (5) (reading 2; the paper defers it to its
    references).  s_q = 8(2 - s)/(8 - s) equals s at s = 8 - sqrt(48), i.e. nu = (1/s - 1/2)/3 =
    0.14434; every non-conserved moment then relaxes at the same rate and the MRT collision must
    equal single-relaxation-time BGK with Guo's forcing, written out here in velocity space:
      f+ = f - s (f - f_eq(rho, u)) + (1 - s/2) w_i [3 (e_i - u) + 9 (e_i . u) e_i] . F,
      u = (sum e_i f_i + F/2) / rho,  F = rho (a_x, a_y + g beta (T - T0))."""
    s = 8.0 - math.sqrt(48.0)
    nu = (1.0 / s - 0.5) / 3.0
    P = base_params(wl, nu=nu, gbeta=3e-3, body_ax=2e-3, body_ay=-1e-3, T0=0.2)
    rng = np.random.default_rng(7)
    W = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4)
    ex = np.array([0, 1, 0, -1, 0, 1, -1, -1, 1], dtype=float)
    ey = np.array([0, 0, 1, 0, -1, 1, 1, -1, -1], dtype=float)
    for _ in range(5):
        f = ob.feq(1.0 + 0.05 * rng.standard_normal(), 0.06 * rng.standard_normal(),
                   0.06 * rng.standard_normal()) + 1e-3 * rng.standard_normal(9)
        T = 0.7 + 0.1 * rng.standard_normal()
        g = ob.geq(T, 0.0, 0.0, P["kappa"])
        fo, _ = ob.collide_node(P, f, g)
        rho = f.sum()
        Fx, Fy = rho * P["body_ax"], rho * (P["body_ay"] + P["gbeta"] * (T - P["T0"]))
        ux, uy = ((ex * f).sum() + 0.5 * Fx) / rho, ((ey * f).sum() + 0.5 * Fy) / rho
        eu = ex * ux + ey * uy
        feq = W * rho * (1.0 + 3.0 * eu + 4.5 * eu * eu - 1.5 * (ux * ux + uy * uy))
        guo = W * ((3.0 * (ex - ux) + 9.0 * eu * ex) * Fx + (3.0 * (ey - uy) + 9.0 * eu * ey) * Fy)
        expect = f - s * (f - feq) + (1.0 - 0.5 * s) * guo
        assert np.abs(fo - expect).max() < 1e-15


# ---------------- links ----------------
def test_link_q_closed_forms(ob):
    assert ob.link_q(-11.0, 0.0, 1, 0.0, 0.0, 10.0) == 1.0     # SURVEY 8(c) pin (iv)
    assert ob.link_q(-11.0, 0.0, 1, 0.0, 0.0, 10.5) == 0.5
    assert ob.link_q(0.0, 11.0, 4, 0.0, 0.0, 10.25) == 0.75
    # diagonal: from (-8,-8) along (1,1) to the circle of radius 10: (8 - t) sqrt2 = 10
    assert ob.link_q(-8.0, -8.0, 5, 0.0, 0.0, 10.0) == pytest.approx(8 - 10 / math.sqrt(2), abs=1e-14)
    # off-centre: node (2,0), direction e3 toward a circle centred (0.3, 0.4) radius 1.5:
    # (2 - t - 0.3)^2 + 0.16 = 2.25  ->  t = 1.7 - sqrt(2.09)
    assert ob.link_q(2.0, 0.0, 3, 0.3, 0.4, 1.5) == pytest.approx(1.7 - math.sqrt(2.09), abs=1e-14)
    # beyond one spacing the result is clamped to [0, 1] (definition of q)
    assert ob.link_q(3.0, 0.0, 3, 0.3, 0.4, 1.5) == 1.0


# ---------------- bounce-back, Eqs. (9)-(12) ----------------
def _coeffs_f(ob, alpha, q, nbehind):
    """Coefficients multiplying fi_0, fi_1, fi_2, fib_0, fib_1 (wall at rest)."""
    c = []
    for k in range(5):
        v = [0.0] * 5
        v[k] = 1.0
        c.append(ob.bounce_back_f(alpha, q, *v, nbehind, 1.0, 0.0, 0.0))
    return np.array(c)


@pytest.mark.parametrize("alpha", [1, 4, 5, 8])
def test_eq9_eq10_coefficients_as_printed(ob, alpha):
    q = 0.25   # Eq. (9): q(2q+1), 1-4q^2, -q(1-2q)
    assert np.allclose(_coeffs_f(ob, alpha, q, 2), [0.375, 0.75, -0.125, 0, 0], atol=1e-16)
    q = 0.75   # Eq. (10): 1/(q(2q+1)), (2q-1)/q, -(2q-1)/(2q+1) on f_ibar(x_f - e_i)
    assert np.allclose(_coeffs_f(ob, alpha, q, 2), [1 / 1.875, 0, 0, 0.5 / 0.75, -0.5 / 2.5], atol=1e-15)
    assert np.allclose(_coeffs_f(ob, alpha, q, 1), [1 / 1.875, 0, 0, 0.5 / 0.75, -0.5 / 2.5], atol=1e-15)


@pytest.mark.parametrize("nbehind", [0, 1, 2])
@pytest.mark.parametrize("q", [0.0, 0.1, 0.3, 0.5, 0.5000001, 0.7, 0.95, 1.0])
def test_bounce_back_coefficients_sum_to_one(ob, q, nbehind):
    c = _coeffs_f(ob, 3, q, nbehind)
    assert c.sum() == pytest.approx(1.0, abs=1e-14)
    # uniform fluid at rest next to a wall at rest is a fixed point
    w = 1 / 9
    assert ob.bounce_back_f(3, q, w, w, w, w, w, nbehind, 1.0, 0.0, 0.0) == pytest.approx(w, abs=1e-16)


def test_bounce_back_halfway_limit_and_ladder(ob):
    # q = 1/2 belongs to Eq. (9) and reduces to halfway bounce-back
    assert np.allclose(_coeffs_f(ob, 2, 0.5, 2), [1, 0, 0, 0, 0], atol=1e-16)
    # Eq. (10) is continuous there
    assert np.allclose(_coeffs_f(ob, 2, 0.5 + 1e-12, 2), [1, 0, 0, 0, 0], atol=1e-11)
    # ladder (DESIGN.md readings): linear Bouzidi with one node behind, halfway with none
    assert np.allclose(_coeffs_f(ob, 2, 0.25, 1), [0.5, 0.5, 0, 0, 0], atol=1e-16)
    assert np.allclose(_coeffs_f(ob, 2, 0.25, 0), [1, 0, 0, 0, 0], atol=1e-16)
    assert np.allclose(_coeffs_f(ob, 2, 0.75, 0), [1 / 1.5, 0, 0, 0.5 / 1.5, 0], atol=1e-15)


@pytest.mark.parametrize("alpha", range(1, 9))
def test_moving_wall_term(ob, alpha):
    """2 w_i rho0 (e_ibar . u_w)/c_s^2 (Eq. 9); scaled by 1/(q(2q+1)) in Eq. (10)."""
    rho0, uwx, uwy = 1.3, 0.02, -0.05
    ab = OPP[alpha]
    term = 2 * W9[alpha] * rho0 * (EX[ab] * uwx + EY[ab] * uwy) * 3
    assert ob.bounce_back_f(alpha, 0.3, 0, 0, 0, 0, 0, 2, rho0, uwx, uwy) == pytest.approx(term, abs=1e-17)
    assert ob.bounce_back_f(alpha, 0.8, 0, 0, 0, 0, 0, 2, rho0, uwx, uwy) == pytest.approx(
        term / (0.8 * 2.6), abs=1e-17)
    assert ob.bounce_back_f(alpha, 0.8, 0, 0, 0, 0, 0, 0, rho0, uwx, uwy) == pytest.approx(
        term / 1.6, abs=1e-17)


def test_thermal_bounce_back_eq11_eq12(ob):
    kappa, Tw = 0.02 / 0.7, 0.8
    aT = 20 * math.sqrt(3) * kappa - 4
    w = (4 + aT) / 20
    q = 0.25
    c2 = (2 * q - 1) / (2 * q + 1)
    c4 = 2 / (2 * q + 1)
    got = ob.bounce_back_g(1, q, 0.11, 0.13, 0.17, 1, kappa, Tw)
    assert got == pytest.approx(-0.11 + c2 * 0.13 + c2 * 0.17 + c4 * 2 * w * Tw, abs=1e-16)
    # g = w T_w everywhere reproduces w T_w for every q:  -1 + 2(2q-1)/(2q+1) + 4/(2q+1) = 1
    for q in (0.0, 0.2, 0.5, 0.9, 1.0):
        for nb in (0, 1):
            v = w * Tw
            assert ob.bounce_back_g(3, q, v, v, v, nb, kappa, Tw) == pytest.approx(v, abs=1e-16)
    # q = 1/2: anti-bounce-back  -g_i + 2 w T_w
    assert ob.bounce_back_g(2, 0.5, 0.2, 9.0, 9.0, 1, kappa, Tw) == pytest.approx(-0.2 + 2 * w * Tw, abs=1e-16)
    assert ob.bounce_back_g(2, 0.1, 0.2, 9.0, 9.0, 0, kappa, Tw) == pytest.approx(-0.2 + 2 * w * Tw, abs=1e-16)


# ---------------- momentum exchange, Eqs. (13)-(14) ----------------
def test_momentum_exchange(ob):
    # wall at rest, perfect reflection: dP = 2 f e_i
    for a in range(1, 9):
        d = ob.momentum_exchange(a, 0.1, 0.1, 0.0, 0.0, 0.0, 0.0)
        assert np.allclose(d[:2], [0.2 * EX[a], 0.2 * EY[a]], atol=1e-17)
    # Galilean-invariant form with u_w: f_i (e_i - u_w) - f_ibar (e_ibar - u_w)
    d = ob.momentum_exchange(5, 0.03, 0.02, 0.1, -0.2, 2.0, 3.0)
    px = 0.03 * (1 - 0.1) - 0.02 * (-1 - 0.1)
    py = 0.03 * (1 + 0.2) - 0.02 * (-1 + 0.2)
    assert np.allclose(d, [px, py, 2.0 * py - 3.0 * px], atol=1e-16)


# ---------------- repulsion, Eq. (15) ----------------
def test_repulsion_closed_forms(ob):
    Cf, eps, s = 0.37, 1e-3, 3.0
    assert ob.repulsion_mag(Cf, eps, s, s, 2) == 0.0
    assert ob.repulsion_mag(Cf, eps, s, 3.0001, 2) == 0.0
    assert ob.repulsion_mag(Cf, eps, s, 0.0, 2) == pytest.approx(Cf / eps, rel=1e-15)
    assert ob.repulsion_mag(Cf, eps, s, s / 2, 2) == pytest.approx(0.25 * Cf / eps, rel=1e-15)
    assert ob.repulsion_mag(Cf, eps, s, s / 2, 1) == pytest.approx(0.5 * Cf / eps, rel=1e-15)
    assert ob.repulsion_mag(Cf, eps, 2.0, 0.5, 1) == pytest.approx(0.75 * Cf / eps, rel=1e-15)


# ---------------- integrator, Eqs. (7)-(8) ----------------
def test_integrator_reproduces_free_fall_exactly(ob):
    g, ratio, r = 1.6e-4, 1.5, 10.0
    mass = ratio * math.pi * r * r
    inertia = 0.5 * mass * r * r
    F = -(ratio - 1.0) * math.pi * r * r * g
    Tz = 0.3
    s = np.array([64.0, 200.0, 0.1, 0.0, 0.0, 0.0])
    for _ in range(500):
        s = ob.integrate(s, 0.0, F, Tz, mass, inertia)
    t = 500
    acc = (1 - 1 / ratio) * g
    assert s[1] == pytest.approx(200.0 - 0.5 * acc * t * t, rel=1e-13)
    assert s[4] == pytest.approx(-acc * t, rel=1e-12)
    assert s[0] == 64.0 and s[3] == 0.0
    assert s[5] == pytest.approx(Tz / inertia * t, rel=1e-12)
    assert s[2] == pytest.approx(0.1 + 0.5 * Tz / inertia * t * t, rel=1e-12)


# ---------------- refill, Eqs. (16)-(17) ----------------
def test_refill_direction(ob):
    assert ob.refill_direction(1.0, 0.0) == 1
    assert ob.refill_direction(0.0, 2.0) == 2
    assert ob.refill_direction(-3.0, 0.0) == 3
    assert ob.refill_direction(0.0, -1.0) == 4
    assert ob.refill_direction(1.0, 1.0) == 5
    assert ob.refill_direction(-1.0, 1.0) == 6
    assert ob.refill_direction(-1.0, -1.0) == 7
    assert ob.refill_direction(1.0, -1.0) == 8
    # switch between axis and diagonal at 22.5 degrees
    t = math.tan(math.radians(22.5))
    assert ob.refill_direction(1.0, t - 1e-9) == 1
    assert ob.refill_direction(1.0, t + 1e-9) == 5
    for ang in np.linspace(0, 2 * math.pi, 97)[:-1] + 0.01:
        c = ob.refill_direction(math.cos(ang), math.sin(ang))
        ea = math.atan2(EY[c], EX[c])
        dev = abs((ang - ea + math.pi) % (2 * math.pi) - math.pi)
        assert dev <= math.radians(22.5) + 1e-9


def test_refill_quadratic_extrapolation_and_constraint(ob):
    f0 = ob.feq(1.0, 0.0, 0.0)
    # uniform state reproduced exactly (weights 3 - 3 + 1 = 1), wall at rest
    assert np.allclose(ob.refill_f(3, f0, f0, f0, 1.0, 0.0, 0.0), f0, atol=1e-16)
    # a quadratic in k is extrapolated exactly to k = 0
    a, b, c = RNG.uniform(0.05, 0.2, 9), RNG.uniform(-0.01, 0.01, 9), RNG.uniform(-1e-3, 1e-3, 9)
    fk = lambda k: a + b * k + c * k * k  # noqa: E731
    uw = (0.03, -0.02)
    out = ob.refill_f(3, fk(1), fk(2), fk(3), 1.0, *uw)
    m_out, m_a = ob.moments_f(out), ob.moments_f(a)
    rho_new = a.sum()
    assert m_out[3] == pytest.approx(rho_new * uw[0], abs=1e-15)   # momentum constrained
    assert m_out[5] == pytest.approx(rho_new * uw[1], abs=1e-15)
    keep = [0, 1, 2, 4, 6, 7, 8]                                    # every other moment untouched
    assert np.allclose(m_out[keep], m_a[keep], atol=1e-14)
    # ladder: two nodes -> linear, one node -> copy, none -> equilibrium at the wall velocity
    out2 = ob.refill_f(2, fk(1), fk(2), fk(3), 1.0, 0.0, 0.0)
    assert np.allclose(np.array(ob.moments_f(out2))[keep], np.array(ob.moments_f(2 * fk(1) - fk(2)))[keep], atol=1e-14)
    out1 = ob.refill_f(1, fk(1), fk(2), fk(3), 1.0, 0.0, 0.0)
    assert np.allclose(np.array(ob.moments_f(out1))[keep], np.array(ob.moments_f(fk(1)))[keep], atol=1e-14)
    out0 = ob.refill_f(0, fk(1), fk(2), fk(3), 1.1, *uw)
    assert np.allclose(out0, ob.feq(1.1, *uw), atol=1e-16)
