"""Parity of the SURVEY 8(e)/(f) rows with the CPU oracle -- replica batches and reweighting (f3), species, second pair
potential and pair-correlation estimator (f4), bead shards (e / f2) -- and of the sampling loop, the error paths and the
thermostat handling.  Needs a B200; everything goes through the C ABI."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_2404_02628_b200 import workloads as wl  # noqa: E402

RTOL = 1e-9


@pytest.fixture(scope="module")
def binding():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu-marked tests need the B200 box")
    from paper_2404_02628_b200 import binding as b

    b.load()
    return b


def relerr(a, b):
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def check_forces(F, Fo, tol):
    P = F.shape[0]
    assert relerr(F, Fo) <= tol
    assert relerr(F[0], Fo[0]) <= tol
    assert relerr(F[P - 1], Fo[P - 1]) <= tol
    if P > 2:
        assert relerr(F[1:P - 1], Fo[1:P - 1]) <= tol


def make(binding, w, thermostat=0, seed=0, **kw):
    return binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat=thermostat, seed=seed, **kw)


# ---------------------------------------------------------------------------------------------------------------
# (f3) replica batches
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", [(150, 8, 2, [1.0, 0.7, 0.3]), (333, 6, 2, [0.5, -0.3, 1.0, -0.6, 0.05]), (40, 4, 3, [0.0, 0.0])],
                         ids=["bosonic", "mixed_sign", "distinguishable"])
def test_batch_replicas_match_oracle(binding, oracle, case):
    """every replica of a batch (own xi, own positions) against the oracle: first evaluation, stale-gauge evaluation,
    and after three NVE steps"""
    N, P, d, xis = case
    B = len(xis)
    w = wl.custom(N, P, d=d, beta=2.5, g=0.2, s=0.5, xi=1.0, init="ring", sigma=1.5)
    xs, vs = zip(*[wl.make_state(w, 10 + b) for b in range(B)])
    X, V = np.stack(xs), np.stack(vs)
    sim = binding.Pimd(N, P, d, w.beta, w.omega, w.g, w.s, xis, w.dt, thermostat=0, seed=list(range(B)))
    sim.set_state(torch.from_numpy(X).cuda(), torch.from_numpy(V).cuda())

    def compare(Xc):
        F, vb, sg = sim.forces()
        Fh = F.cpu().numpy()
        for b in range(B):
            tol = RTOL if xis[b] >= 0 else RTOL * oracle.conditioning(Xc[b], w.beta, xis[b])
            Fo, vbo, sgo = oracle.forces(Xc[b], w.beta, w.omega, w.g, w.s, xis[b])
            assert sg[b] == sgo and abs(vb[b] - vbo) <= tol * abs(vbo)
            check_forces(Fh[b], Fo, tol)

    compare(X)
    compare(X)
    sim.step(3)
    compare(sim.get_state()[0].cpu().numpy())
    assert sim.get_diagnostics()["fallbacks"] == 0
    sim.close()


def test_batch_trajectories_equal_single_handles(binding):
    """a replica of a batch follows the trajectory of a handle of its own with the same xi and seed (Langevin)"""
    w = wl.WORKLOADS["cfg2"].with_(N=60, P=8)
    xis, seeds = [1.0, 0.4, 0.9], [5, 6, 7]
    xs, vs = zip(*[wl.make_state(w, s) for s in seeds])
    sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, xis, w.dt, thermostat=1, seed=seeds)
    sim.set_state(torch.from_numpy(np.stack(xs)).cuda(), torch.from_numpy(np.stack(vs)).cuda())
    sim.step(12)
    Xb, Vb = [t.cpu().numpy() for t in sim.get_state()]
    epb, evb, _ = sim.estimators()
    sim.close()
    for b in range(3):
        one = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, xis[b], w.dt, thermostat=1, seed=seeds[b])
        one.set_state(torch.from_numpy(xs[b]).cuda(), torch.from_numpy(vs[b]).cuda())
        one.step(12)
        x1, v1 = [t.cpu().numpy() for t in one.get_state()]
        ep, ev, _ = one.estimators()
        one.close()
        assert relerr(Xb[b], x1) <= 1e-12 and relerr(Vb[b], v1) <= 1e-11
        assert abs(epb[b] - ep) <= 1e-10 * abs(ep) and abs(evb[b] - ev) <= 1e-10 * abs(ev)


def test_reweight_matches_oracle(binding, oracle):
    """pimd_reweight: ln|W_obs / W_samp|, its sign, and the primitive energy at xi_obs = e_prim - eps_samp + eps_obs"""
    w = wl.custom(90, 6, d=2, beta=2.0, g=0.3, xi=0.5, init="iid", sigma=0.8)
    x, v = wl.make_state(w, 3)
    sim = make(binding, w)
    sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    sim.step(2)
    xs = sim.get_state()[0].cpu().numpy()
    ep, ev, _ = sim.estimators()
    vs, _ = oracle.vb(xs, w.beta, w.xi)
    for xo in (-0.5, 0.5, 1.0, -0.5, 0.0):       # -0.5 twice: the second call runs with the gauge of the first
        lr, sg, eo, es = sim.reweight(xo)
        vo, so = oracle.vb(xs, w.beta, xo)
        kap = oracle.conditioning(xs, w.beta, xo) if xo < 0 else 1.0
        assert sg == so
        assert abs(lr - (-w.beta * (vo - vs))) <= RTOL * kap * w.beta * abs(vo)
        epo, _, _ = oracle.estimators(xs, w.beta, w.omega, w.g, w.s, xo)
        assert abs((ep - es + eo) - epo) <= RTOL * kap * max(abs(epo), abs(eo))
    # the sampling tables are untouched: forces still those of xi = 0.5
    F = sim.get_forces().cpu().numpy()
    Fo, _, _ = oracle.forces(xs, w.beta, w.omega, w.g, w.s, w.xi)
    check_forces(F, Fo, RTOL)
    sim.close()


def test_reweighted_ensemble_energy_of_fictitious_particles(binding):
    """N = 3, P = 4, beta = 2 ideal gas sampled at xi = +0.3 in a batch of 64 replicas, reweighted to
    xi = -0.3: both estimators against the exact finite-P value 4.226559 within 3 standard errors (jackknife over
    the independent replicas)."""
    from oracle import ideal_gas

    N, P, d, beta, xi_obs, B = 3, 4, 2, 2.0, -0.3, 64
    exact = ideal_gas.exact_energy(N, beta, 1.0, d, xi_obs, P)
    w = wl.custom(N, P, d=d, beta=beta, g=0.0, xi=0.3, dt=0.02, init="iid", sigma=0.7)
    xs, vs = zip(*[wl.make_state(w, 200 + b) for b in range(B)])
    sim = binding.Pimd(N, P, d, beta, 1.0, 0.0, 0.5, [0.3] * B, w.dt, thermostat=1, seed=[900 + b for b in range(B)])
    sim.set_state(torch.from_numpy(np.stack(xs)).cuda(), torch.from_numpy(np.stack(vs)).cuda())
    sim.step(2000)
    num_p, num_v, den = np.zeros(B), np.zeros(B), np.zeros(B)
    for _ in range(1500):
        sim.step(10)
        ep, ev, _ = sim.estimators()
        lr, sg, eo, es = sim.reweight(xi_obs)
        r = sg * np.exp(lr)
        num_p += r * (ep - es + eo); num_v += r * ev; den += r
    sim.close()
    for top in (num_p, num_v):
        est = top.sum() / den.sum()
        jk = np.array([(top.sum() - top[i]) / (den.sum() - den[i]) for i in range(B)])
        se = np.sqrt((B - 1) / B * np.sum((jk - jk.mean()) ** 2))
        assert abs(est - exact) <= 3.0 * se, (est, se, exact)
        assert se < 0.01 * exact


# ---------------------------------------------------------------------------------------------------------------
# (f4) species, second pair potential, pair-correlation estimator
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("counts,xi", [([60, 40], 1.0), ([33, 1, 70], 0.6), ([50, 45], -0.4)], ids=["two", "three", "signed"])
def test_species_match_oracle(binding, oracle, counts, xi):
    N = sum(counts)
    w = wl.custom(N, 8, d=2, beta=3.0, g=0.3, s=0.5, xi=xi, init="ring", sigma=1.0)
    x, v = wl.make_state(w, 4)
    sim = make(binding, w, species=counts)
    sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    tol = RTOL if xi >= 0 else RTOL * max(oracle.conditioning(np.ascontiguousarray(x[:, :counts[0]]), w.beta, xi),
                                          oracle.conditioning(np.ascontiguousarray(x[:, counts[0]:]), w.beta, xi))
    Fo, vbo, sgo = oracle.forces_species(x, w.beta, w.omega, w.g, w.s, xi, counts)
    for _ in range(2):
        F, vb, sg = sim.forces()
        assert sg == sgo and abs(vb - vbo) <= tol * abs(vbo)
        check_forces(F.cpu().numpy(), Fo, tol)
    ep, ev, hist = sim.estimators(nbins=32, rmax=5.0)
    epo, evo, ho = oracle.estimators_species(x, w.beta, w.omega, w.g, w.s, xi, counts, nbins=32, rmax=5.0)
    assert abs(ep - epo) <= tol * max(abs(epo), 1.0) * 10 and abs(ev - evo) <= 1e-9 * max(abs(evo), 1.0)
    np.testing.assert_array_equal(hist, ho)
    sim.step(3)
    xs = sim.get_state()[0].cpu().numpy()
    F, vb, sg = sim.forces()
    Fo, vbo, sgo = oracle.forces_species(xs, w.beta, w.omega, w.g, w.s, xi, counts)
    assert sg == sgo and abs(vb - vbo) <= tol * abs(vbo)
    check_forces(F.cpu().numpy(), Fo, tol)
    sim.close()


@pytest.mark.parametrize("N,P,d", [(130, 6, 2), (130, 6, 3), (1550, 3, 2), (1517, 2, 3)], ids=["n130_d2", "n130_d3", "n1550_d2", "n1517_d3"])
def test_soft_coulomb_potential_matches_oracle(binding, oracle, N, P, d):
    """N = 130 runs k_pair<., ., 1>; from N = 1500 on the two-rows-per-lane kernel k_pair2<., ., 1> (its diagonal tiles drop
    the self term and its last super-tile is padded: N is not a multiple of 64), forces and estimator variants alike."""
    w = wl.custom(N, P, d=d, beta=2.0, g=0.4, s=0.5, xi=1.0, init="iid", sigma=1.0 if N < 1000 else 4.0)
    x, _ = wl.make_state(w, 2)
    sim = make(binding, w, pair_potential=binding.PAIR_SOFT_COULOMB)
    sim.set_state(torch.from_numpy(x).cuda())
    F, vb, sg = sim.forces()
    ep, ev, _ = sim.estimators()
    sim.close()
    oracle.set_pair_potential(1)
    try:
        Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
        epo, evo, _ = oracle.estimators(x, w.beta, w.omega, w.g, w.s, w.xi)
    finally:
        oracle.set_pair_potential(0)
    assert abs(vb - vbo) <= RTOL * abs(vbo)
    check_forces(F.cpu().numpy(), Fo, RTOL)
    assert abs(ep - epo) <= RTOL * abs(epo) and abs(ev - evo) <= RTOL * abs(evo)
    Fg, _, _ = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)      # the Gaussian gives different forces
    assert relerr(F.cpu().numpy(), Fg) > 1e-3


@pytest.mark.parametrize("case", [(100, 32, 2, 64, 6.0), (257, 5, 3, 50, 4.0), (1600, 4, 2, 128, 20.0)], ids=["cfg2", "d3", "n1600"])
def test_pair_histogram_is_the_oracles(binding, oracle, case):
    """integer work: bit-exact against the oracle's pair-distance counts"""
    N, P, d, nbins, rmax = case
    w = wl.custom(N, P, d=d, beta=3.0, g=0.5, s=0.5, xi=1.0, init="iid", sigma=1.0 if N < 1000 else 5.0)
    x, _ = wl.make_state(w, 1)
    sim = make(binding, w)
    sim.set_pair_histogram(nbins, rmax)
    sim.set_state(torch.from_numpy(x).cuda())
    sim.estimators()
    g = sim.pair_histogram()
    sim.close()
    go = oracle.pair_histogram(x, nbins, rmax)
    assert go.sum() > 0
    np.testing.assert_array_equal(g, go)


# ---------------------------------------------------------------------------------------------------------------
# (e / f2) bead shards on one GPU: world shards of one system, the all-gather a device copy
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("world,P,N", [(2, 8, 200), (4, 8, 200), (3, 8, 200), (8, 8, 200), (2, 2, 200), (3, 6, 333), (2, 5, 97)])
def test_bead_shards_match_single_gpu_and_oracle(binding, oracle, world, P, N):
    from paper_2404_02628_b200 import sharding

    w = wl.custom(N, P, d=2, beta=3.0, g=0.3, s=0.5, xi=1.0, init="ring", sigma=1.5)
    x, v = wl.make_state(w, 7)
    grp = sharding.LocalShardGroup(binding, world, w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat=1, seed=42)
    for r, sim in enumerate(grp.sims):      # the C library and the Python layout helper agree
        assert (sim.j0, sim.P_local) == sharding.shard_range(P, r, world)
        assert sim.pack_doubles == sharding.pack_doubles(w.N, w.d)
    grp.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    F, vb, sg = grp.forces()
    Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
    assert sg == sgo and abs(vb - vbo) <= RTOL * abs(vbo)
    check_forces(F.cpu().numpy(), Fo, RTOL)
    ep, ev, hist = grp.estimators(nbins=16, rmax=6.0)
    epo, evo, ho = oracle.estimators(x, w.beta, w.omega, w.g, w.s, w.xi, nbins=16, rmax=6.0)
    assert abs(ep - epo) <= RTOL * abs(epo) and abs(ev - evo) <= RTOL * abs(evo)
    np.testing.assert_array_equal(hist, ho)
    # ten Langevin steps: the noise is keyed by the global degree of freedom, so the trajectory is the single-GPU one
    one = make(binding, w, thermostat=1, seed=42)
    one.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    one.step(10)
    x1, v1 = [t.cpu().numpy() for t in one.get_state()]
    one.close()
    grp.step(10)
    xs, vs = [t.cpu().numpy() for t in grp.get_state()]
    grp.close()
    assert relerr(xs, x1) <= 1e-11 and relerr(vs, v1) <= 1e-10


# ---------------------------------------------------------------------------------------------------------------
# sampling loop, thermostat handling, error paths
# ---------------------------------------------------------------------------------------------------------------
def test_run_accumulates_what_estimators_returns(binding):
    w = wl.WORKLOADS["cfg2"].with_(N=80, P=8)
    x, v = wl.make_state(w, 3)
    a = make(binding, w, thermostat=1, seed=9)
    a.set_pair_histogram(24, 4.0)
    a.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    a.run(47, est_every=10, nbins=w.nbins, rmax=w.rmax)        # samples after steps 10, 20, 30, 40
    a.run(13, est_every=10, nbins=w.nbins, rmax=w.rmax)        # 50, 60
    n, sp, sv, hs, gs = a.read_accumulators(nbins=w.nbins, nbins_gr=24)
    assert a.get_step_count() == 60 and n == 6
    b = make(binding, w, thermostat=1, seed=9)
    b.set_pair_histogram(24, 4.0)
    b.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    ep_s = ev_s = 0.0
    hist_s, gr_s = np.zeros(w.nbins), np.zeros(24)
    for _ in range(6):
        b.step(10)
        ep, ev, hist = b.estimators(nbins=w.nbins, rmax=w.rmax)
        ep_s += ep; ev_s += ev; hist_s += hist; gr_s += b.pair_histogram()
    xa, xb = a.get_state()[0].cpu().numpy(), b.get_state()[0].cpu().numpy()
    n_after = a.read_accumulators()[0]       # the first read reset the sums
    a.close(); b.close()
    assert relerr(xa, xb) <= 1e-12
    assert abs(sp - ep_s) <= 1e-10 * abs(ep_s) and abs(sv - ev_s) <= 1e-10 * abs(ev_s)
    np.testing.assert_array_equal(hs, hist_s)
    np.testing.assert_array_equal(gs, gr_s)
    assert n_after == 0


def test_set_gamma_takes_effect_on_replayed_steps(binding):
    """pimd_set_gamma after a graph was captured: the replayed steps must use the new friction"""
    w = wl.WORKLOADS["cfg2"].with_(N=50, P=8)
    x, v = wl.make_state(w, 1)
    out = []
    for chunks in ((5, 5), (1,) * 10):
        sim = make(binding, w, thermostat=1, seed=3)
        sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        k = 0
        for n in chunks:
            if k == 5:
                sim.set_gamma(7.0)
            sim.step(n)
            k += n
        out.append([t.cpu().numpy() for t in sim.get_state()])
        sim.close()
    assert relerr(out[0][0], out[1][0]) <= 1e-12 and relerr(out[0][1], out[1][1]) <= 1e-11


@pytest.mark.timeout(240, method="thread")
def test_batch_size_limit_of_the_recursion_kernel(binding, oracle):
    """Above 128 particles every replica needs a chain CTA and at least one panel worker per direction, all co-resident:
    a B200 holds 148 / 4 = 37 such replicas.  A larger batch used to start a cooperative kernel whose chain CTAs waited
    for panels nobody computed; it is refused at creation now, and the largest batch that fits runs and is right."""
    w = wl.custom(200, 4, d=2, beta=2.0, g=0.0, xi=1.0, init="ring", sigma=1.0)
    with pytest.raises(binding.PimdError) as e:
        binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, [1.0] * 40, w.dt)
    assert e.value.code == binding.EINVAL and "replicas" in str(e.value)
    small = wl.custom(128, 4, d=2, beta=2.0, g=0.0, xi=1.0, init="ring", sigma=1.0)   # no workers needed: 74 replicas fit
    binding.Pimd(small.N, small.P, small.d, small.beta, small.omega, small.g, small.s, [1.0] * 40, small.dt).close()
    B = 37
    xis = [1.0 if b % 2 == 0 else 0.5 for b in range(B)]
    sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, xis, w.dt)
    assert sim.get_diagnostics()["workers"] >= 1
    xs = np.stack([wl.make_state(w, 100 + b)[0] for b in range(B)])
    sim.set_state(torch.from_numpy(xs).cuda())
    for _ in range(2):   # the second evaluation runs the stale-gauge kernel
        F, vb, sg = sim.forces()
    F = F.cpu().numpy()
    sim.close()
    for b in (0, 17, 36):
        Fo, vbo, sgo = oracle.forces(xs[b], w.beta, w.omega, w.g, w.s, xis[b])
        assert sg[b] == sgo and abs(vb[b] - vbo) <= RTOL * abs(vbo)
        check_forces(F[b], Fo, RTOL)


def test_error_paths(binding):
    w = wl.custom(40, 4, d=2, beta=2.0, g=0.1, xi=1.0, init="iid", sigma=0.7)
    x, _ = wl.make_state(w, 0)
    # non-finite state
    sim = make(binding, w)
    xb = x.copy(); xb[1, 3, 0] = np.nan
    sim.set_state(torch.from_numpy(xb).cuda())
    with pytest.raises(binding.PimdError) as e:
        sim.forces()
    assert e.value.code == binding.ENUMERIC
    sim.set_state(torch.from_numpy(x).cuda())       # a good state clears it
    sim.forces()
    sim.close()
    # a node of the fermionic weight: two identical rings, W_2 = (e^{-2 beta E_ring} - e^{-beta E^{[1,2]}}) / 2 = 0
    ring = np.random.default_rng(1).normal(0.0, 0.5, size=(4, 1, 2))
    sim = binding.Pimd(2, 4, 2, 2.0, 1.0, 0.0, 0.5, -1.0, 0.01, thermostat=0)
    sim.set_state(torch.from_numpy(np.ascontiguousarray(np.repeat(ring, 2, axis=1))).cuda())
    with pytest.raises(binding.PimdError) as e:
        sim.forces()
    assert e.value.code == binding.ENUMERIC and "node" in str(e.value)
    sim.close()
    # workspace too small
    sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, use_torch_workspace=False)
    need = sim._lib.pimd_workspace_bytes(sim._h)
    buf = torch.empty(need, dtype=torch.uint8, device="cuda")
    import ctypes as C
    assert sim._lib.pimd_set_workspace(sim._h, C.c_void_p(buf.data_ptr()), need - 256) == binding.ENOMEM
    assert sim._lib.pimd_set_workspace(sim._h, C.c_void_p(buf.data_ptr() + 8), need) == binding.EINVAL
    sim.close()
    # N x N output beyond N = 65535
    sim = binding.Pimd(70000, 2, 1, 2.0, 1.0, 0.0, 0.5, 1.0, 0.01, use_torch_workspace=False)
    with pytest.raises(binding.PimdError) as e:
        sim.cycle_energies(out=torch.empty(1, device="cuda", dtype=torch.float64))
    assert e.value.code == binding.EINVAL
    sim.close()
    # tables for xi = 0 are refused before any copy; a mixed batch is refused at creation
    sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, 0.0, w.dt)
    sim.set_state(torch.from_numpy(x).cuda())
    sim.forces()
    with pytest.raises(binding.PimdError):
        sim.get_tables()
    sim.close()
    with pytest.raises(binding.PimdError):
        binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, [0.0, 1.0], w.dt)
    with pytest.raises(binding.PimdError):
        make(binding, w, species=[10, 10])


def _nccl_worker(q):
    """one rank over NCCL on the one GPU there is: the real ShardedPimd path (pimd_shard_* + all_gather_into_tensor)"""
    import os

    import torch.distributed as dist

    from paper_2404_02628_b200 import binding as b, sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ.setdefault("MASTER_PORT", "29631")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        b.load()
        w = wl.custom(150, 6, d=2, beta=3.0, g=0.3, s=0.5, xi=1.0, init="ring", sigma=1.5)
        x, v = wl.make_state(w, 3)
        sh = sharding.ShardedPimd(b, w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat=1, seed=11)
        sh.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        F = sh.forces().cpu().numpy()
        vb, sg = sh.sim.shard_scalars()
        sh.step(8)
        xs, vs = [t.cpu().numpy() for t in sh.sim.get_state()]
        # a second set_state drops the cached forces: the next step() must make its own export / all-gather / forces first
        sh.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        sh.step(3)
        xs2 = sh.sim.get_state()[0].cpu().numpy()
        sh.close()
        one = b.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat=1, seed=11)
        one.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        F1, vb1, sg1 = one.forces()
        one.step(8)
        x1, v1 = [t.cpu().numpy() for t in one.get_state()]
        one.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        one.step(3)
        x2 = one.get_state()[0].cpu().numpy()
        one.close()
        q.put((relerr(F, F1.cpu().numpy()), abs(vb - vb1) / abs(vb1), sg == sg1, relerr(xs, x1), relerr(vs, v1), relerr(xs2, x2)))
    except Exception as e:  # the parent must not wait for a result that never comes
        q.put(repr(e))
        raise
    finally:
        dist.destroy_process_group()


def test_sharded_stepping_through_nccl_on_one_gpu(binding):
    """ShardedPimd as torchrun would run it, with the one rank this box has: the boundary pack goes through a real NCCL
    all_gather_into_tensor on the handle's stream between pimd_shard_begin_step and pimd_shard_end_step"""
    import torch.multiprocessing as mp

    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_nccl_worker, args=(q,))
    p.start()
    res = q.get(timeout=300)
    p.join(timeout=120)
    assert p.exitcode == 0 and not isinstance(res, str), res
    ef, ev, sg_ok, ex, evel, ex2 = res
    assert ef <= 1e-12 and ev <= 1e-13 and sg_ok and ex <= 1e-11 and evel <= 1e-10 and ex2 <= 1e-11
