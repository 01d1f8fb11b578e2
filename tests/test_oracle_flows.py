"""Pins the oracle's lattice part (collision + streaming + cavity walls) to closed-form flows:
body-force Poiseuille (nu), linear conduction and sine-mode decay (kappa), mass conservation.
SURVEY.md 8(c) "Pins"; BASELINE.json north_star names the same checks."""
import math

import numpy as np
import pytest


def test_poiseuille_body_force_is_exact(ob, wl):
    """periodic_x, halfway bounce-back walls at y=-1/2 and ny-1/2, uniform body acceleration G:
    u_x(j) = G/(2 nu) (j+1/2)(ny-1/2-j).  With s_q = 8(2-s_nu)/(8-s_nu) the discrete solution is
    the parabola to round-off."""
    nx, ny, nu, G = 4, 15, 0.1, 1e-5
    p = wl.default_params()
    p.update(periodic_x=1, body_ax=G, nu=nu, kappa=0.05)
    s = ob.OracleSim(nx, ny, p)
    s.step(9000)
    F = s.fields()
    j = np.arange(ny)
    exact = G / (2 * nu) * (j + 0.5) * (ny - 0.5 - j)
    for col in range(nx):
        assert np.abs(F["ux"][:, col] - exact).max() / exact.max() < 1e-10
    assert np.abs(F["uy"]).max() < 1e-14
    assert np.abs(F["rho"] - 1.0).max() < 1e-12


@pytest.mark.parametrize("nu", [0.02, 0.3])
def test_poiseuille_viscosity_dependence(ob, wl, nu):
    nx, ny, G = 4, 9, 1e-7
    p = wl.default_params()
    p.update(periodic_x=1, body_ax=G, nu=nu, kappa=0.05)
    s = ob.OracleSim(nx, ny, p)
    s.step(int(45 * ny * ny / nu / 9.87) + 200)
    umax = s.fields()["ux"][ny // 2, 0]
    assert umax == pytest.approx(G / (2 * nu) * (ny / 2) ** 2, rel=1e-10)


def test_linear_conduction_profile_is_exact(ob, wl):
    """gbeta = 0, bottom wall T = 1, top wall T = 0 (anti-bounce-back, walls halfway):
    T(j) = 1 - (j+1/2)/ny to round-off."""
    nx, ny = 4, 12
    p = wl.default_params()
    p.update(kappa=0.1, nu=0.05)
    p["wall_T_type"] = [0, 0, 1, 1]
    p["wall_T"] = [0.0, 0.0, 1.0, 0.0]
    s = ob.OracleSim(nx, ny, p)
    s.step(6000)
    F = s.fields()
    exact = 1 - (np.arange(ny) + 0.5) / ny
    assert np.abs(F["T"] - exact[:, None]).max() < 1e-12
    assert np.abs(F["ux"]).max() < 1e-15 and np.abs(F["uy"]).max() < 1e-15


def test_sideways_conduction_between_dirichlet_side_walls(ob, wl):
    """Same check along x (W: T = 0.2, E: T = 0.9; S/N adiabatic) -- catches a wall-index mix-up."""
    nx, ny = 10, 4
    p = wl.default_params()
    p.update(kappa=0.12, nu=0.05)
    p["wall_T_type"] = [1, 1, 0, 0]
    p["wall_T"] = [0.2, 0.9, 0.0, 0.0]
    s = ob.OracleSim(nx, ny, p)
    s.step(5000)
    T = s.fields()["T"]
    exact = 0.2 + 0.7 * (np.arange(nx) + 0.5) / nx
    assert np.abs(T - exact[None, :]).max() < 1e-12


@pytest.mark.parametrize("kappa", [0.02 / 0.7, 0.0223455, 0.1])
def test_sine_mode_decay_gives_kappa(ob, wl, kappa):
    """Periodic-x strip with adiabatic y walls: T = 1/2 + A sin(kx) decays as exp(-kappa k^2 t)
    up to O(k^2) lattice corrections."""
    nx, ny = 96, 4
    p = wl.default_params()
    p.update(periodic_x=1, kappa=kappa, nu=0.05, T0=0.5)
    s = ob.OracleSim(nx, ny, p)
    k = 2 * math.pi / nx
    T0 = 0.5 + 0.01 * np.sin(k * np.arange(nx))[None, :] * np.ones((ny, 1))
    s.set_temperature(T0)
    s.step(50)   # let the non-hydrodynamic modes die
    a0 = 2 * (s.fields()["T"][1] * np.sin(k * np.arange(nx))).mean()
    s.step(400)
    a1 = 2 * (s.fields()["T"][1] * np.sin(k * np.arange(nx))).mean()
    kappa_eff = -math.log(a1 / a0) / (k * k * 400)
    assert kappa_eff == pytest.approx(kappa, rel=5e-3)


def test_mass_and_heat_conservation_in_a_closed_box(ob, wl):
    """Config-1 set-up at 48x40: buoyancy on, noise on the conduction profile; total mass constant
    to 1e-12 relative (streaming + halfway walls conserve it exactly; collision too)."""
    nx, ny = 48, 40
    w1 = wl.config(1)
    p = dict(w1.params)
    p["gbeta"] = 1e-4      # stronger than config 1 so the flow really moves within 300 steps
    rng = np.random.default_rng(7)
    T = (1 - (np.arange(ny)[:, None] + 0.5) / ny) + 1e-3 * rng.uniform(-1, 1, (ny, nx))
    s = ob.OracleSim(nx, ny, p)
    s.set_temperature(T)
    m0 = s.fields()["rho"].sum()
    s.step(300)
    F = s.fields()
    assert abs(F["rho"].sum() - m0) / m0 < 1e-12
    assert np.abs(F["uy"]).max() > 1e-7          # something is happening
    # adiabatic walls all round: heat is conserved too
    p2 = dict(p)
    p2["wall_T_type"] = [0, 0, 0, 0]
    s2 = ob.OracleSim(nx, ny, p2)
    s2.set_temperature(T)
    h0 = s2.fields()["T"].sum()
    s2.step(200)
    assert abs(s2.fields()["T"].sum() - h0) / h0 < 1e-12


def test_initial_state_and_readout(ob, wl):
    p = wl.default_params()
    p.update(T0=0.3, rho0=1.1)
    s = ob.OracleSim(6, 5, p)
    F = s.fields(populations=True)
    assert np.all(F["rho"] == pytest.approx(1.1)) and np.all(F["T"] == pytest.approx(0.3))
    assert np.all(F["ux"] == 0) and np.all(F["flag"] == 0)
    w = np.array([4 / 9] + [1 / 9] * 4 + [1 / 36] * 4) * 1.1
    assert np.allclose(F["f"], w[:, None, None], atol=1e-16)   # f+ of a rest equilibrium is itself
    f, g = s.precollision()
    assert np.allclose(f, w[:, None, None], atol=1e-16)
    assert np.allclose(g.sum(0), 0.3, atol=1e-16)


def test_buoyancy_direction_hot_fluid_rises(ob, wl):
    """Eq. (1b): +g beta (T - T0) along +y.  A warm blob in a cold box must acquire u_y > 0."""
    nx = ny = 24
    p = wl.default_params()
    p.update(gbeta=1e-3)
    T = np.zeros((ny, nx))
    T[10:14, 10:14] = 1.0
    s = ob.OracleSim(nx, ny, p)
    s.set_temperature(T)
    s.step(20)
    F = s.fields()
    assert F["uy"][12, 12] > 1e-4
    assert abs(F["ux"][12, 11] + F["ux"][12, 12]) < 1e-12  # left-right symmetric
