"""y-slabs (include/lbm.h "y-slabs"): a cavity cut into slabs with ghost rows,
every slab holding every particle, forces combined from the owning slab, halo rows exchanged after
every step -- here with all slabs on ONE device, through the same C-ABI calls a multi-GPU run
makes.  The decomposition must not change a single bit: own rows of every slab against the rows of
one lbm_create domain, all particle states, at several horizons, while particles cross the cuts."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2308_16597_b200 import binding
    binding.load_library()
    return binding


def assert_group_equals_domain(grp, dom):
    fa, fb = grp.fields(populations=True), dom.fields(populations=True)
    assert np.array_equal(fa["flag"], fb["flag"])
    fluid = fb["flag"] == 0
    for k in ("f", "g"):
        assert np.array_equal(fa[k][:, fluid], fb[k][:, fluid]), k
    for k in ("rho", "ux", "uy", "T"):
        assert np.array_equal(fa[k], fb[k]), k          # solid nodes too (rigid-body read-out)
    pb = dom.particles()
    for s in range(len(grp.slabs)):                     # every slab carries the same particle states
        pa = grp.particles(s)
        for k in ("x", "y", "theta", "ux", "uy", "omega"):
            assert np.array_equal(pa[k], pb[k]), (s, k)
    # the combined force every slab integrated from is the single domain's, bit for bit
    pa = grp.particles(0)
    for k in ("Fx", "Fy", "Tz"):
        assert np.array_equal(pa[k], pb[k]), k


@pytest.mark.parametrize("n_slabs,fused", [(2, True), (3, True), (2, False), (3, False)])
def test_slabs_on_one_device_equal_the_single_domain_bitwise(gpu, wl, n_slabs, fused):
    """14 particles of mixed sizes fall through the cuts of a 300 x 390 cavity (some start on a
    cut, one is thrown upwards across it): ownership changes hands, discs straddle two slabs,
    newborn nodes appear in ghost rows.  fused: the lattice kernel and the refill commit push the
    rows next to a cut into the neighbour's ghost rows themselves (lbm_slab_link_peers); otherwise
    the rows are copied after the step (lbm_slab_exchange_halos)."""
    from paper_2308_16597_b200 import slabs
    w = wl.sedimentation(300, 390, 14, seed=17, y_frac_lo=0.25, d_lo=12.0, d_hi=22.0, name="slabs")
    n = w.n_particles
    y = w.particles["y"]
    cut = (390 * 1) // n_slabs
    k = int(np.argmin(np.abs(y - cut)))
    uy = np.full(n, -0.03)
    uy[k] = +0.06 if y[k] < cut else -0.08               # crosses the cut early on
    w.particles.update(ux=np.zeros(n), uy=uy, omega=1e-3 * np.ones(n))
    grp = slabs.SlabGroup(w, n_slabs, fused_halo=fused)
    dom = gpu.Simulation.from_workload(w)
    assert grp.halo == 19
    owners0 = slabs.owner_of(dom.particles()["y"], grp.ranges)
    assert_group_equals_domain(grp, dom)
    for nst in (1, 2, 37, 160, 400):
        grp.step(nst)
        dom.step(nst)
        assert_group_equals_domain(grp, dom)
    owners1 = slabs.owner_of(dom.particles()["y"], grp.ranges)
    assert (owners0 != owners1).sum() >= 1               # a particle was handed from slab to slab
    grp.close()


def test_particle_free_slabs_with_an_initial_temperature_field(gpu, wl):
    """Rayleigh-Benard set-up (hot floor, cold lid, adiabatic sides, seeded noise) on 333 x 200 in
    four slabs of 50 rows with 8 ghost rows: every wall type next to a slab, ragged width."""
    from paper_2308_16597_b200 import slabs
    nx, ny = 333, 200
    w = wl.config(1)
    rng = np.random.default_rng(3)
    j = np.arange(ny, dtype=np.float64)[:, None]
    T = (1.0 - (j + 0.5) / ny) + 1e-3 * rng.uniform(-1.0, 1.0, size=(ny, nx))
    w = wl.Workload("rb_slabs", nx, ny, w.params, 1, 1, T_init=T)
    grp = slabs.SlabGroup(w, 4)
    dom = gpu.Simulation.from_workload(w)
    dom.set_two_step(False)
    for nst in (1, 50):
        grp.step(nst)
        dom.step(nst)
        fa, fb = grp.fields(populations=True), dom.fields(populations=True)
        for k in ("f", "g", "rho", "ux", "uy", "T"):
            assert np.array_equal(fa[k], fb[k]), k
    grp.close()


def test_config2_in_two_slabs_over_the_parity_horizon(gpu, wl):
    """BASELINE config 2 (1000^2, 480 particles) cut at row 500: bit-identical to the single domain
    over the 100-step parity horizon (which the single domain holds against the oracle,
    test_gpu_fullsize.py)."""
    from paper_2308_16597_b200 import slabs
    w = wl.config(2)
    grp = slabs.SlabGroup(w, 2)
    dom = gpu.Simulation.from_workload(w)
    grp.step(w.parity_steps)
    dom.step(w.parity_steps)
    assert_group_equals_domain(grp, dom)
    grp.close()


def test_slab_error_paths(gpu, wl):
    from paper_2308_16597_b200 import binding
    p = wl.default_params()
    p.update(max_particles=1, max_links_per_particle=wl.max_links_for_diameter(30.0))
    with pytest.raises(binding.LbmError):                 # halo below the minimum
        binding.Simulation(64, 200, p, slab=(0, 100, 3))
    with pytest.raises(binding.LbmError):                 # a slab lower than its halo
        binding.Simulation(64, 200, p, slab=(0, 10, 12))
    s = binding.Simulation(64, 200, p, slab=(100, 200, 12))
    with pytest.raises(binding.LbmError) as e:            # halo too narrow for this particle
        s.add_particles(x=np.array([30.0]), y=np.array([150.0]), diam=np.array([30.0]),
                        rho_ratio=np.array([1.5]), T_w=np.array([1.0]))
    assert e.value.code == binding.LBM_E_ARG
    with pytest.raises(binding.LbmError) as e:            # lbm_step refuses slab handles
        s.step(1)
    assert e.value.code == binding.LBM_E_STATE
    s.close()


def test_one_rank_slab_runner_equals_the_single_domain(gpu, wl):
    """SlabRank with world_size 1 (bench.py --slabs on one GPU): one slab that owns every row, no
    neighbour and no all-reduce, stepped through the slab calls -- same bits as lbm_step."""
    from paper_2308_16597_b200 import slabs
    w = wl.sedimentation(200, 240, 8, seed=23, y_frac_lo=0.3, d_lo=12.0, d_hi=18.0, name="rank1")
    sr = slabs.SlabRank(w, 0, 1, "cuda:0")
    dom = gpu.Simulation.from_workload(w)
    sr.step(150)
    dom.step(150)
    fa, fb = sr.sim.fields(populations=True), dom.fields(populations=True)
    fluid = fb["flag"] == 0
    assert np.array_equal(fa["flag"], fb["flag"])
    for k in ("f", "g"):
        assert np.array_equal(fa[k][:, fluid], fb[k][:, fluid]), k
    pa, pb = sr.sim.particles(), dom.particles()
    for k in pb:
        assert np.array_equal(pa[k], pb[k]), k
    sr.close()


def test_ellipses_across_a_cut(gpu, wl):
    """Elliptical particles (their zone, support-function repulsion and gradient refill normal use
    global coordinates too) straddling and crossing the cut of two slabs: bit-identical."""
    from paper_2308_16597_b200 import slabs
    p = wl.default_params()
    p.update(g=1.6e-4, gbeta=1e-5, wall_T_type=[1, 1, 1, 1], max_particles=4,
             max_links_per_particle=wl.max_links_for_diameter(26.0))
    parts = dict(x=np.array([50.2, 110.0, 160.5, 90.0]), y=np.array([121.0, 128.3, 112.0, 170.0]),
                 diam=np.array([26.0, 20.0, 18.0, 14.0]), minor=np.array([13.0, 12.0, 18.0, 14.0]),
                 theta=np.array([0.4, -1.1, 0.0, 0.0]), rho_ratio=np.full(4, 1.5), T_w=np.full(4, 1.0),
                 ux=np.zeros(4), uy=np.array([-0.04, -0.02, 0.05, -0.06]),
                 omega=np.array([2e-3, -1e-3, 0.0, 1e-3]))
    w = wl.Workload("ellipse_slabs", 220, 240, p, 1, 1, particles=parts)
    grp = slabs.SlabGroup(w, 2)                       # cut at row 120
    dom = gpu.Simulation.from_workload(w)
    for nst in (1, 60, 300):
        grp.step(nst)
        dom.step(nst)
        assert_group_equals_domain(grp, dom)
    grp.close()
