"""Pins the unit-conversion helper, Eq. (18) and the workload recipes to numbers the paper prints
(tests/golden/paper_tables.txt, each with its PAPER.md citation) and to SURVEY.md 8(d)."""
import math
import os

import numpy as np
import pytest


def _golden():
    out = {}
    path = os.path.join(os.path.dirname(__file__), "golden", "paper_tables.txt")
    for line in open(path):
        line = line.split("#")[0].strip()
        if line:
            k, v = line.split()
            out[k] = float(v)
    return out


G = _golden()


def test_table4_lattice_parameters(wl):
    u = wl.lattice_units(length_m_per_lu=G["t4_length_m_per_lu"], time_s_per_ts=G["t4_time_s_per_ts"],
                         d_m=G["t4_d_m"], nu_m2s=G["t4_nu_m2s"], g_ms2=G["t4_g_ms2"],
                         rho_ratio=G["t4_rho_ratio"], beta_per_K=G["t4_beta_perK"],
                         dT_K=G["t4_temp_K_per_tu"])
    assert u["d"] == pytest.approx(G["t4_d_lu"], rel=1e-12)
    assert u["nu"] == pytest.approx(G["t4_nu_lu"], rel=1e-12)
    assert u["g"] == pytest.approx(G["t4_g_lu"], rel=1e-3)
    assert u["beta"] == pytest.approx(G["t4_beta_lu"], rel=5e-3)
    assert u["Ar"] == pytest.approx(G["t4_Ar"], abs=0.05)
    assert u["Re_p"] == pytest.approx(G["t4_Re_p"], abs=0.05)
    assert u["Gr_p"] == pytest.approx(G["t4_Gr_p"], rel=0.01)
    # relation Re_p = sqrt(pi/2) Ar
    assert u["Re_p"] == pytest.approx(math.sqrt(math.pi / 2) * u["Ar"], rel=1e-12)
    # Pr = nu/alpha from the lattice columns of Table 4
    assert G["t4_nu_lu"] / G["t4_alpha_lu"] == pytest.approx(G["t4_Pr"])
    vf = G["t4_n_particles"] * math.pi * (G["t4_d_lu"] / 2) ** 2 / G["t4_domain_lu"] ** 2
    assert 100 * vf == pytest.approx(G["t4_volume_fraction_percent"], abs=0.05)


def test_table1_numbers(wl):
    """Table 1's lattice column follows from its unit conversion, and Re_p/Ar = sqrt(pi/2).
    The printed Ar = 9.90, Re_p = 12.41 are NOT reproduced by the printed
    rho_p = 1.1 g/cm^3 (that gives Ar = 31.3); they correspond to rho_p/rho_f = 1.01.  The paper is
    at odds with itself here (listed in DESIGN.md); only the self-consistent parts are pinned."""
    u = wl.lattice_units(length_m_per_lu=2.5e-5, time_s_per_ts=3.125e-5, d_m=1e-3, nu_m2s=1e-6,
                         g_ms2=9.8, rho_ratio=1.1)
    assert u["d"] == pytest.approx(G["t1_d_lu"], rel=1e-12)
    assert u["nu"] == pytest.approx(G["t1_nu_lu"], rel=1e-12)
    assert u["g"] == pytest.approx(G["t1_g_lu"], rel=1e-3)
    assert G["t1_Re_p"] / G["t1_Ar"] == pytest.approx(math.sqrt(math.pi / 2), rel=1e-3)
    d, nu, g = G["t1_d_lu"], G["t1_nu_lu"], G["t1_g_lu"]
    assert math.sqrt(g * d ** 3 * 0.01) / nu == pytest.approx(G["t1_Ar"], abs=0.01)
    assert 100 * 800 * math.pi * 20 ** 2 / 2000 ** 2 == pytest.approx(
        G["t1_volume_fraction_percent"], abs=0.05)
    assert wl.gravity_from_galileo(u["Ar"], nu, 1.1, d) == pytest.approx(u["g"], rel=1e-12)


def test_mlups_eq18(wl):
    assert wl.mlups(int(G["t5_mesh"]), int(G["t5_steps"]), G["t5_time_indirect_s"]) == pytest.approx(
        G["t5_mlups_indirect"], abs=2)
    assert wl.mlups(int(G["t5_mesh"]), int(G["t5_steps"]), G["t5_time_direct_s"]) == pytest.approx(
        G["t5_mlups_direct"], abs=1)


def test_slot_capacity(wl):
    assert 12 * int(G["slots_N"]) - 12 == int(G["slots_capacity"])
    assert wl.max_links_for_diameter(40.0) == 12 * 44 - 12  # worst case N = floor(d)+4
    assert wl.max_links_for_diameter(20.0) >= 264


def test_config_parameters(wl):
    w0 = wl.config(0)
    assert (w0.nx, w0.ny) == (128, 256)
    assert w0.params["g"] == pytest.approx(1.6e-4, rel=1e-12)
    assert w0.params["kappa"] == pytest.approx(0.02 / 0.7)
    assert w0.params["wall_T_type"] == [0, 0, 1, 1]
    w1 = wl.config(1)
    assert w1.params["nu"] == pytest.approx(0.0156419, rel=1e-5)
    assert w1.params["kappa"] == pytest.approx(0.0223455, rel=1e-5)
    assert w1.params["gbeta"] == pytest.approx(3.2552e-6, rel=1e-4)
    Ra = w1.params["gbeta"] * 1.0 * w1.ny ** 3 / (w1.params["nu"] * w1.params["kappa"])
    assert Ra == pytest.approx(1e7, rel=1e-9)
    assert w1.T_init.shape == (1024, 1024)
    assert abs(w1.T_init - (1 - (np.arange(1024)[:, None] + 0.5) / 1024)).max() <= 1e-3


def test_sampler_is_seeded_and_non_overlapping(wl):
    a = wl.config(2)
    b = wl.config(2)
    assert a.n_particles == 480
    for k in ("x", "y", "diam"):
        assert np.array_equal(a.particles[k], b.particles[k])
    x, y, d = a.particles["x"], a.particles["y"], a.particles["diam"]
    dist = np.hypot(x[:, None] - x[None, :], y[:, None] - y[None, :]) + np.eye(len(x)) * 1e9
    gap = dist - 0.5 * (d[:, None] + d[None, :])
    assert gap.min() >= 2.0
    assert x.min() >= 12 and x.max() <= 1000 - 12
    assert y.min() >= 0.4 * 1000 + 10 and y.max() <= 1000 - 12


def test_variable_diameter_sampler(wl):
    w = wl.sedimentation(512, 512, 80, seed=4, y_frac_lo=0.0, d_lo=12.0, d_hi=24.0)
    d = w.particles["diam"]
    assert d.min() >= 12 and d.max() <= 24 and d.std() > 1
    assert w.params["max_links_per_particle"] == 12 * 28 - 12


def test_paper_table4_workload_matches_the_printed_table(wl):
    """PAPER.md:232 and Table 4: 4,800 particles of d = 40 in 4000 x 4000, volume fraction 37.7 %,
    Ar = 22.4, Gr_p = 60, Pr = 5; 60 lines of 80 particles, none touching a wall or a neighbour."""
    import math
    import numpy as np
    w = wl.config(5)
    P, p = w.particles, w.params
    assert (w.nx, w.ny, w.n_particles) == (4000, 4000, 4800)
    assert len(np.unique(P["y"])) == 60 and len(np.unique(P["x"])) == 80
    assert round(100 * w.n_particles * math.pi * 20.0 ** 2 / (w.nx * w.ny), 1) == 37.7
    assert round(math.sqrt(p["g"] * 40.0 ** 3 * 0.1) / p["nu"], 1) == 22.4
    assert round(p["gbeta"] * 1.0 * 40.0 ** 3 / p["nu"] ** 2) == 60
    assert p["nu"] / p["kappa"] == 5.0
    assert (p["rep_power"], p["rep_s"], p["rep_eps"]) == (2, 3.0, 1e-3)
    assert P["x"].min() - 20.0 > -0.5 and P["x"].max() + 20.0 < w.nx - 0.5
    assert P["y"].max() + 20.0 < w.ny - 0.5 and P["y"].min() > 0.25 * w.ny
    assert np.diff(np.unique(P["x"])).min() == 50.0


def test_paper_dkt_workload_matches_table6(wl):
    """PAPER.md:407-430, Table 6 (values in tests/golden/paper_tables.txt): Ar = 28.0,
    Re_p = 35.09, Gr_p = 100, Pr = 1; 400 x 1200, d = 40; the lower particle 0.005 d left of the
    centreline, the upper one 2 d above it."""
    import math
    w = wl.paper_dkt()
    p, P = w.params, w.particles
    d = G["t6_d_lu"]
    assert (w.nx, w.ny) == (G["t6_domain_w_lu"], G["t6_domain_h_lu"]) and w.n_particles == 2
    assert (p["nu"], p["kappa"], p["g"]) == (G["t6_nu_lu"], G["t6_alpha_lu"], G["t6_g_lu"])
    assert abs(p["gbeta"] - G["t6_g_lu"] * G["t6_beta_lu"]) < 1e-18
    assert P["rho_ratio"][0] == G["t6_rho_ratio"] and P["diam"][0] == d
    excess = G["t6_rho_ratio"] - 1.0
    assert round(math.sqrt(p["g"] * d ** 3 * excess) / p["nu"], 0) == G["t6_Ar"]
    assert abs(math.sqrt(p["g"] * math.pi * d * excess / 2.0) * d / p["nu"] - G["t6_Re_p"]) < 0.1
    assert abs(p["gbeta"] * d ** 3 / p["nu"] ** 2 - G["t6_Gr_p"]) < 1.0     # printed to 2-3 digits
    assert p["nu"] / p["kappa"] == G["t6_Pr"]
    assert abs((P["x"][1] - P["x"][0]) - 0.005 * d) < 1e-12 and P["y"][1] - P["y"][0] == 2 * d
    assert abs(P["x"][1] - (0.5 * w.nx - 0.5)) < 1e-12 and abs(P["y"][0] - (0.8 * w.ny - 0.5)) < 1e-12


def test_paper_table3_workload_matches_the_printed_table(wl):
    """PAPER.md:206-224, Table 3: 129 ellipses of 50 x 25 l.u. in 1000 x 2000, volume fraction
    6.3 %, Re_p = 31.0, Ar = 24.7, Gr_p = 10, Pr = 5; rings of 6, 12, 18, 24, 31, 37 around one."""
    import math
    import numpy as np
    w = wl.paper_table3()
    p, P = w.params, w.particles
    A, B = G["t3_major_lu"], G["t3_minor_lu"]
    assert (w.nx, w.ny, w.n_particles) == (G["t3_domain_w_lu"], G["t3_domain_h_lu"], G["t3_n_particles"])
    assert (P["diam"] == A).all() and (P["minor"] == B).all() and (P["rho_ratio"] == G["t3_rho_ratio"]).all()
    assert (p["nu"], p["kappa"], p["g"]) == (G["t3_nu_lu"], G["t3_alpha_lu"], G["t3_g_lu"])
    frac = 100.0 * w.n_particles * math.pi * 0.25 * A * B / (w.nx * w.ny)
    assert round(frac, 1) == G["t3_volume_fraction_percent"]
    ex = G["t3_rho_ratio"] - 1.0
    assert round(math.sqrt(p["g"] * A ** 3 * ex) / p["nu"], 1) == G["t3_Ar"]
    assert round(math.sqrt(p["g"] * math.pi * A * ex / 2.0) * A / p["nu"], 1) == G["t3_Re_p"]
    assert round(p["gbeta"] * A ** 3 / p["nu"] ** 2) == G["t3_Gr_p"] and p["nu"] / p["kappa"] == G["t3_Pr"]
    # the cluster: one centre particle and rings of the printed sizes, nobody touching
    r = np.hypot(P["x"] - P["x"][0], P["y"] - P["y"][0])
    counts = [int((np.abs(r - 60.0 * k) < 1e-9).sum()) for k in range(1, 7)]
    assert counts == [6, 12, 18, 24, 31, 37] and abs(P["y"][0] - (0.75 * w.ny - 0.5)) < 1e-12
    d = np.hypot(P["x"][:, None] - P["x"][None, :], P["y"][:, None] - P["y"][None, :])
    assert d[np.triu_indices(len(r), 1)].min() > A + 3.0
