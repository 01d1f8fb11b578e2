"""Seeded synthetic inputs shared by the CUDA path and the CPU oracle.

This module holds NONE of the method's arithmetic (no collision, streaming, bounce-back, force or
integration formulas): it only produces parameters, initial temperature fields and particle
placements.  Both the CUDA binding (product) and the CPU checker used by the tests (test infrastructure,
kept outside this package) receive the same arrays, so parity is taken on identical bits.

The five workloads are `BASELINE.json` `configs[0..4]` as resolved in SURVEY.md 8(d) "Synthetic
inputs" (they stand in for the paper's own benchmark, 4,800 hot particles in a 4000^2 cavity,
PAPER.md:230-246, whose shapes the configs override).  Nothing is read from a dataset.

`lattice_units()` is the paper's unit conversion (Eqs. 2-4 and Tables 1-4, PAPER.md:51-70,
173-244), a harness helper used to choose g and pinned against the paper's printed tables.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, Optional

import numpy as np

W, E, S, N = 0, 1, 2, 3  # wall order used by wall_T_type / wall_T


def default_params() -> Dict:
    return dict(nu=0.02, kappa=0.02 / 0.7, rho0=1.0, T0=0.0, g=0.0, gbeta=0.0,
                body_ax=0.0, body_ay=0.0, periodic_x=0,
                wall_T_type=[0, 0, 0, 0], wall_T=[0.0, 0.0, 0.0, 0.0],
                rep_s=2.0, rep_eps=1e-3, rep_power=1,
                max_particles=0, max_links_per_particle=0)


def max_links_for_diameter(d_max: float) -> int:
    """Capacity 12N-12 of one particle's index-array segment for the worst-case zone length
    N = floor(d)+4 (PAPER.md:258 gives N = INT(xc+d/2) - INT(xc-d/2) + 3 <= floor(d)+4)."""
    return 12 * (int(math.floor(d_max)) + 4) - 12


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    params: Dict
    steps: int                      # run length BASELINE.json names (timing/physics, not parity)
    parity_steps: int               # horizon of the parity comparison (SURVEY 8(c) protocol)
    T_init: Optional[np.ndarray] = None      # (ny, nx) float64 or None (= T0 everywhere)
    particles: Optional[Dict[str, np.ndarray]] = None  # x, y, diam, rho_ratio, T_w
    notes: str = ""
    extra: Dict = field(default_factory=dict)

    @property
    def n_particles(self) -> int:
        return 0 if self.particles is None else int(self.particles["x"].shape[0])


def gravity_from_galileo(Ga: float, nu: float, rho_ratio: float, d: float) -> float:
    """g such that Ga = sqrt(g d^3 (rho_p/rho_f - 1))/nu (the paper's Ar)."""
    return Ga * Ga * nu * nu / ((rho_ratio - 1.0) * d ** 3)


def lattice_units(*, length_m_per_lu: float, time_s_per_ts: float, d_m: float, nu_m2s: float,
                  g_ms2: float, rho_ratio: float, alpha_m2s: Optional[float] = None,
                  beta_per_K: Optional[float] = None, dT_K: Optional[float] = None) -> Dict:
    """Physical -> lattice conversion of the paper's Tables 1-4 and the derived numbers
    Ar, Re_p, Gr_p, Pr (Eq. 4)."""
    lu, ts = length_m_per_lu, time_s_per_ts
    out = dict(d=d_m / lu, nu=nu_m2s * ts / lu ** 2, g=g_ms2 * ts ** 2 / lu)
    out["Ar"] = math.sqrt(out["g"] * out["d"] ** 3 * (rho_ratio - 1.0)) / out["nu"]
    out["Re_p"] = math.sqrt(out["g"] * math.pi * out["d"] * (rho_ratio - 1.0) / 2.0) * out["d"] / out["nu"]
    if alpha_m2s is not None:
        out["alpha"] = alpha_m2s * ts / lu ** 2
        out["Pr"] = out["nu"] / out["alpha"]
    if beta_per_K is not None and dT_K is not None:
        # temperature unit: dT_K kelvin per lattice temperature unit, so Delta_T = 1 t.u.
        out["beta"] = beta_per_K * dT_K
        out["Gr_p"] = out["g"] * out["beta"] * 1.0 * out["d"] ** 3 / out["nu"] ** 2
    return out


def mlups(mesh_size: int, steps: int, seconds: float) -> float:
    """Eq. (18): mesh size x iteration steps / (running time x 1e6)."""
    return mesh_size * steps / (seconds * 1e6)


def place_particles(rng: np.random.Generator, n: int, xlo: float, xhi: float, ylo_of_r, yhi_of_r,
                    xlo_of_r, xhi_of_r, diam_sampler, gap: float, d_max: float,
                    max_tries: int = 50_000_000):
    """Random sequential placement by rejection: draw a diameter, then a centre
    uniformly in the allowed box for that radius; accept if the surface gap to every accepted
    particle is >= `gap`.  Neighbour test through a uniform cell grid of cell size d_max+gap."""
    del xlo, xhi
    cell = d_max + gap
    grid: Dict = {}
    xs, ys, ds = [], [], []
    tries = 0
    while len(xs) < n:
        tries += 1
        if tries > max_tries:
            raise RuntimeError("particle placement did not converge")
        d = float(diam_sampler(rng))
        r = 0.5 * d
        x = float(rng.uniform(xlo_of_r(r), xhi_of_r(r)))
        y = float(rng.uniform(ylo_of_r(r), yhi_of_r(r)))
        ci, cj = int(x // cell), int(y // cell)
        ok = True
        for a in (ci - 1, ci, ci + 1):
            for b in (cj - 1, cj, cj + 1):
                for k in grid.get((a, b), ()):
                    if math.hypot(x - xs[k], y - ys[k]) < r + 0.5 * ds[k] + gap:
                        ok = False
                        break
                if not ok:
                    break
            if not ok:
                break
        if ok:
            grid.setdefault((ci, cj), []).append(len(xs))
            xs.append(x)
            ys.append(y)
            ds.append(d)
    return (np.asarray(xs, dtype=np.float64), np.asarray(ys, dtype=np.float64),
            np.asarray(ds, dtype=np.float64))


def _sediment_params(d_max: float, n_particles: int, all_walls_cold: bool) -> Dict:
    p = default_params()
    nu = 0.02
    p.update(nu=nu, kappa=nu / 0.7, rho0=1.0, T0=0.0,
             g=gravity_from_galileo(40.0, nu, 1.5, 20.0),   # = 1.6e-4 (Ga taken as Ar)
             gbeta=1e-5, rep_s=2.0, rep_eps=1e-3, rep_power=1,
             max_particles=n_particles, max_links_per_particle=max_links_for_diameter(d_max))
    if all_walls_cold:
        p["wall_T_type"] = [1, 1, 1, 1]
    else:  # config 0: adiabatic side walls, cold top and bottom
        p["wall_T_type"] = [0, 0, 1, 1]
    p["wall_T"] = [0.0, 0.0, 0.0, 0.0]
    return p


def _particle_dict(x, y, d, rho_ratio=1.5, T_w=1.0):
    n = x.shape[0]
    return dict(x=x, y=y, diam=d, rho_ratio=np.full(n, rho_ratio), T_w=np.full(n, T_w))


def sedimentation(nx: int, ny: int, n_particles: int, seed: int, y_frac_lo: float,
                  d_lo: float = 20.0, d_hi: float = 20.0, name: str = "sedimentation",
                  steps: int = 100, parity_steps: int = 100) -> Workload:
    """Generic seeded sedimentation workload with the structure of configs 2-4 (hot particles of
    density ratio 1.5 in cold fluid, gap >= 2 l.u., centres in y >= y_frac_lo*ny)."""
    rng = np.random.default_rng(seed)
    if d_lo == d_hi:
        sampler = lambda g: d_lo  # noqa: E731
    else:
        sampler = lambda g: g.uniform(d_lo, d_hi)  # noqa: E731
    x, y, d = place_particles(
        rng, n_particles, 0, nx,
        ylo_of_r=lambda r: y_frac_lo * ny + r if y_frac_lo > 0 else r + 2.0,
        yhi_of_r=lambda r: ny - r - 2.0,
        xlo_of_r=lambda r: r + 2.0, xhi_of_r=lambda r: nx - r - 2.0,
        diam_sampler=sampler, gap=2.0, d_max=d_hi)
    return Workload(name=name, nx=nx, ny=ny, params=_sediment_params(d_hi, n_particles, True),
                    steps=steps, parity_steps=parity_steps, particles=_particle_dict(x, y, d))


def paper_table4(cols: int = 80, lines: int = 60, name: str = "paper_table4_4800_particles_4000",
                 ny: Optional[int] = None) -> Workload:
    """The paper's own benchmark (Table 4): hot
    circular particles of d = 40 l.u. and rho_p/rho_f = 1.1 in `lines` lines of `cols` particles in
    the upper part of a square cavity, nu = 0.01, alpha_T = 0.002 (Pr = 5), g = 7.84e-6,
    beta = 1.2e-2 per lattice temperature unit, Delta_T = 1, all four walls cold; the paper's
    repulsion (Eq. 15: quadratic, s = 3, eps_w = 0.001).  With the defaults: 4,800 particles in
    4000 x 4000, volume fraction 37.7 %.

    Reading (the paper shows the arrangement only as a picture, Fig. 4a): uniform pitch
    nx/cols = 50 l.u. in both directions with half-pitch margins to the side walls and to the top
    wall (walls half a spacing outside the outermost nodes)."""
    pitch = 50.0
    nx = int(round(cols * pitch))
    ny = nx if ny is None else ny
    m = np.arange(cols, dtype=np.float64)
    k = np.arange(lines, dtype=np.float64)
    X, Y = np.meshgrid(-0.5 + pitch * (m + 0.5), (ny - 0.5) - pitch * (k + 0.5))
    x, y = X.ravel(), Y.ravel()
    n = x.shape[0]
    p = default_params()
    p.update(nu=0.01, kappa=0.002, rho0=1.0, T0=0.0, g=7.84e-6, gbeta=7.84e-6 * 1.2e-2,
             rep_s=3.0, rep_eps=1e-3, rep_power=2, max_particles=n,
             max_links_per_particle=max_links_for_diameter(40.0))
    p["wall_T_type"] = [1, 1, 1, 1]
    p["wall_T"] = [0.0, 0.0, 0.0, 0.0]
    parts = _particle_dict(x, y, np.full(n, 40.0), rho_ratio=1.1, T_w=1.0)
    return Workload(name=name, nx=nx, ny=ny, params=p, steps=6000, parity_steps=100,
                    particles=parts,
                    notes="paper's E4 benchmark; 1750 MLUPS on 1x A100 (Table 5, PAPER.md:273-281)")


def paper_table3(name: str = "paper_table3_129_ellipses_1000x2000") -> Workload:
    """The paper's elliptical-particle case (Table 3): 129 hot
    elliptical particles, full axes A x B = 50 x 25 l.u., rho_p/rho_f = 1.5, in a 1000 x 2000
    cavity, nu = 0.01, alpha_T = 0.002 (Pr = 5), g = 9.8e-7, beta = 8.16e-3 per lattice
    temperature unit (Gr_p = 10), all walls cold; one particle at (0.5 W, 0.75 H) and six rings
    of 6, 12, 18, 24, 31, 37 particles around it; the paper's repulsion (quadratic, s = 3).

    Readings (the paper shows the cluster only as a picture, Fig. 3a): ring k has radius 60 k l.u.
    (one major axis plus a 10-unit gap), its particles equally spaced starting on the +x axis,
    every major axis horizontal."""
    nx, ny = 1000, 2000
    cx, cy = 0.5 * nx - 0.5, 0.75 * ny - 0.5
    xs, ys = [cx], [cy]
    for k, count in enumerate((6, 12, 18, 24, 31, 37), start=1):
        ang = 2.0 * math.pi * np.arange(count) / count
        xs.extend(cx + 60.0 * k * np.cos(ang))
        ys.extend(cy + 60.0 * k * np.sin(ang))
    x, y = np.asarray(xs, dtype=np.float64), np.asarray(ys, dtype=np.float64)
    n = x.shape[0]
    p = default_params()
    p.update(nu=0.01, kappa=0.002, rho0=1.0, T0=0.0, g=9.8e-7, gbeta=9.8e-7 * 8.16e-3,
             rep_s=3.0, rep_eps=1e-3, rep_power=2, max_particles=n,
             max_links_per_particle=max_links_for_diameter(50.0))
    p["wall_T_type"] = [1, 1, 1, 1]
    p["wall_T"] = [0.0, 0.0, 0.0, 0.0]
    parts = _particle_dict(x, y, np.full(n, 50.0), rho_ratio=1.5, T_w=1.0)
    parts["minor"] = np.full(n, 25.0)
    parts["theta"] = np.zeros(n)
    return Workload(name=name, nx=nx, ny=ny, params=p, steps=100000, parity_steps=20,
                    particles=parts)


def paper_dkt(name: str = "paper_dkt_two_hot_particles_400x1200") -> Workload:
    """Appendix B of the paper (Table 6): draft-kissing-tumbling of
    two hot circular particles in cold fluid.  400 x 1200 l.u., d = 40, rho_p/rho_f = 1.01,
    nu = alpha_T = 0.01 (Pr = 1), g = 1.23e-4, beta = 1.28e-3 per lattice temperature unit
    (Gr_p = 100), all walls cold and no-slip; the lower particle at (0.5 W - 0.005 d, 0.8 H), the
    upper one at (0.5 W, 0.8 H + 2 d) (walls half a spacing outside the outermost nodes); the
    paper's repulsion (Eq. 15: quadratic, s = 3, eps_w = 0.001)."""
    nx, ny, d = 400, 1200, 40.0
    x = np.array([0.5 * nx - 0.5 - 0.005 * d, 0.5 * nx - 0.5])
    y = np.array([0.8 * ny - 0.5, 0.8 * ny - 0.5 + 2.0 * d])
    p = default_params()
    p.update(nu=0.01, kappa=0.01, rho0=1.0, T0=0.0, g=1.23e-4, gbeta=1.23e-4 * 1.28e-3,
             rep_s=3.0, rep_eps=1e-3, rep_power=2, max_particles=2,
             max_links_per_particle=max_links_for_diameter(d))
    p["wall_T_type"] = [1, 1, 1, 1]
    p["wall_T"] = [0.0, 0.0, 0.0, 0.0]
    parts = _particle_dict(x, y, np.full(2, d), rho_ratio=1.01, T_w=1.0)
    return Workload(name=name, nx=nx, ny=ny, params=p, steps=160000, parity_steps=100,
                    particles=parts, notes="index 0 = lower particle (P2 of Fig. 18), 1 = upper (P1)")


def config(k: int) -> Workload:
    """BASELINE.json configs[k], resolved as in SURVEY.md 8(d); k = 5 is the paper's own Table 4
    benchmark, which BASELINE.json's config 3 replaces for the headline."""
    if k == 5:
        return paper_table4()
    if k == 0:
        p = _sediment_params(20.0, 1, all_walls_cold=False)
        parts = _particle_dict(np.array([64.0]), np.array([200.0]), np.array([20.0]))
        return Workload("config0_single_hot_particle_128x256", 128, 256, p, steps=1000,
                        parity_steps=100, particles=parts)
    if k == 1:
        nx = ny = 1024
        Ra, Pr = 1e7, 0.7
        U = 0.1 / math.sqrt(3.0)             # fixed Mach: U = 0.1 c_s
        nu = U * ny * math.sqrt(Pr / Ra)
        p = default_params()
        p.update(nu=nu, kappa=nu / Pr, gbeta=U * U / ny, g=0.0, T0=0.0)
        p["wall_T_type"] = [0, 0, 1, 1]
        p["wall_T"] = [0.0, 0.0, 1.0, 0.0]
        rng = np.random.default_rng(1)
        j = np.arange(ny, dtype=np.float64)[:, None]
        T = (1.0 - (j + 0.5) / ny) + 1e-3 * rng.uniform(-1.0, 1.0, size=(ny, nx))
        return Workload("config1_rayleigh_benard_1024", nx, ny, p, steps=10000, parity_steps=100,
                        T_init=np.ascontiguousarray(T))
    if k == 2:
        w = sedimentation(1000, 1000, 480, seed=2, y_frac_lo=0.4,
                          name="config2_480_particles_1000", steps=5000)
        return w
    if k == 3:
        w = sedimentation(4000, 4000, 4800, seed=3, y_frac_lo=0.3,
                          name="config3_4800_particles_4000", steps=2000)
        w.extra["warmup_steps"] = 200
        return w
    if k == 4:
        w = sedimentation(8192, 8192, 20000, seed=4, y_frac_lo=0.0, d_lo=12.0, d_hi=24.0,
                          name="config4_20000_particles_8192", steps=1000, parity_steps=20)
        return w
    raise ValueError("config index must be 0..5")
