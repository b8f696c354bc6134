"""Parity of the CUDA path (through the C ABI, libpimd.so) with the CPU oracle -- needs a B200.

Tolerances (BASELINE.json north_star): 1e-9 relative on V_B and on the forces (max-norm), FP64.
For xi < 0 the tolerance is scaled by the conditioning kappa = sum|terms| / |sum terms| of the
signed sums (R7), computed by the oracle (orc_conditioning) for the configuration at hand.
"""
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


def make(binding, w, thermostat=0, seed=0):
    return binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat=thermostat, seed=seed)


def gpu_forces(binding, w, x):
    sim = make(binding, w)
    sim.set_state(torch.from_numpy(x).cuda())
    f, vb, sg = sim.forces()
    out = f.cpu().numpy()
    sim.close()
    return out, vb, sg


def relerr(a, b):
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


def check_forces(F, Fo, tol):
    P = F.shape[0]
    assert relerr(F, Fo) <= tol
    # per bead class: interior, bead 1, bead P
    assert relerr(F[0], Fo[0]) <= tol
    assert relerr(F[P - 1], Fo[P - 1]) <= tol
    if P > 2:
        assert relerr(F[1:P - 1], Fo[1:P - 1]) <= tol


SMALL = [
    # name, N, P, d, beta, g, xi, init, sigma
    ("n1", 1, 4, 2, 2.0, 0.0, 1.0, "iid", 1.0),
    ("n2", 2, 2, 2, 1.5, 0.3, 1.0, "iid", 0.7),
    ("n4_cfg1", 4, 16, 2, 2.0, 0.0, 1.0, "iid", 1.0),
    ("n31", 31, 5, 2, 2.0, 0.4, 1.0, "iid", 0.6),
    ("n32", 32, 4, 2, 2.0, 0.4, 1.0, "iid", 0.6),
    ("n33", 33, 4, 2, 2.0, 0.4, 1.0, "iid", 0.6),
    ("n100_cfg2", 100, 32, 2, 3.0, 0.5, 1.0, "iid", 1.0),
    ("n130_d1", 130, 6, 1, 2.0, 0.3, 1.0, "iid", 0.8),
    ("n130_d3", 130, 6, 3, 2.0, 0.3, 1.0, "iid", 0.8),
    ("n257_half", 257, 8, 2, 3.0, 0.2, 0.5, "ring", 2.0),
    ("n300_spread", 300, 8, 2, 3.0, 0.0, 1.0, "iid", 6.0),   # beta C ~ 1e3: underflow stress (R11)
    ("n421_ring", 421, 8, 2, 3.0, 0.2, 1.0, "ring", 1.0),
]


@pytest.mark.parametrize("case", SMALL, ids=[c[0] for c in SMALL])
def test_forces_and_vb_match_oracle(binding, oracle, case):
    name, N, P, d, beta, g, xi, init, sigma = case
    w = wl.custom(N, P, d=d, beta=beta, g=g, s=0.5, xi=xi, init=init, sigma=sigma)
    for seed in (0, 1):
        x, _ = wl.make_state(w, seed)
        Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
        F, vb, sg = gpu_forces(binding, w, x)
        assert sg == sgo == 1
        assert abs(vb - vbo) <= RTOL * abs(vbo)
        check_forces(F, Fo, RTOL)


@pytest.mark.parametrize("xi", [0.0])
@pytest.mark.parametrize("N", [1, 7, 100])
def test_distinguishable_limit(binding, oracle, xi, N):
    w = wl.custom(N, 8, d=2, beta=2.0, g=0.3, s=0.5, xi=xi, init="iid", sigma=0.8)
    x, _ = wl.make_state(w, 3)
    Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
    F, vb, sg = gpu_forces(binding, w, x)
    assert sg == 1
    assert abs(vb - vbo) <= RTOL * abs(vbo)
    check_forces(F, Fo, RTOL)


@pytest.mark.parametrize("xi", [-0.3, -0.5, -1.0])
@pytest.mark.parametrize("N", [3, 40, 200])
def test_signed_fictitious_particles(binding, oracle, xi, N):
    w = wl.custom(N, 8, d=2, beta=3.0, g=0.2, s=0.5, xi=xi, init="ring", sigma=3.0)
    x, _ = wl.make_state(w, 5)
    Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
    F, vb, sg = gpu_forces(binding, w, x)
    tol = RTOL * oracle.conditioning(x, w.beta, w.xi)
    assert sg == sgo
    assert abs(vb - vbo) <= tol * abs(vbo)
    check_forces(F, Fo, tol)


def test_tables_match_oracle(binding, oracle):
    w = wl.custom(75, 6, d=2, beta=2.5, g=0.0, xi=1.0, init="ring", sigma=1.0)
    x, _ = wl.make_state(w, 2)
    vbo, sgo, fwd, bwd = oracle.vb(x, w.beta, w.xi, tables=True)
    Pr = oracle.pr_matrix(x, w.beta, w.xi)
    sim = make(binding, w)
    sim.set_state(torch.from_numpy(x).cuda())
    sim.forces(want_forces=False)
    vf, vb, pn = sim.get_tables()
    sim.close()
    np.testing.assert_allclose(vf, fwd, rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(vb[1:w.N + 2], bwd[1:w.N + 2], rtol=1e-9, atol=1e-9)
    np.testing.assert_allclose(pn[:-1], np.diagonal(Pr, 1), rtol=0, atol=1e-9)
    assert pn[-1] == 0.0


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_paper_scale_configs(binding, oracle, name):
    w = wl.WORKLOADS[name]
    x, _ = wl.make_state(w, 0)
    Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
    F, vb, sg = gpu_forces(binding, w, x)
    tol = RTOL if w.xi >= 0 else RTOL * oracle.conditioning(x, w.beta, w.xi)
    assert sg == sgo
    assert abs(vb - vbo) <= tol * abs(vbo)
    check_forces(F, Fo, tol)


def test_estimators_match_oracle(binding, oracle):
    for w in (wl.WORKLOADS["cfg2"], wl.custom(77, 6, d=3, beta=2.0, g=0.3, xi=0.5, init="iid", sigma=0.8),
              wl.custom(50, 6, d=2, beta=2.0, g=0.3, xi=0.0, init="iid", sigma=0.8)):
        x, _ = wl.make_state(w, 1)
        epo, evo, ho = oracle.estimators(x, w.beta, w.omega, w.g, w.s, w.xi, nbins=w.nbins, rmax=w.rmax)
        sim = make(binding, w)
        sim.set_state(torch.from_numpy(x).cuda())
        ep, ev, hist = sim.estimators(nbins=w.nbins, rmax=w.rmax)
        sim.close()
        assert abs(ep - epo) <= 1e-9 * max(abs(epo), 1.0)
        assert abs(ev - evo) <= 1e-9 * max(abs(evo), 1.0)
        np.testing.assert_array_equal(hist, ho)


@pytest.mark.parametrize("thermostat", [0, 1, 2])
def test_ten_steps_match_oracle(binding, oracle, thermostat):
    w = wl.WORKLOADS["cfg2"].with_(N=40, P=8)
    x, v = wl.make_state(w, 4)
    seed = 1234
    xo, vo = x.copy(), v.copy()
    Fo, _, _ = oracle.forces(xo, w.beta, w.omega, w.g, w.s, w.xi)
    nhc = np.zeros((4, x.size))
    oracle.step(xo, vo, Fo, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat, 1.0, seed, 0, 10)
    sim = make(binding, w, thermostat=thermostat, seed=seed)
    sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    sim.step(4)
    sim.step(6)
    xg, vg = sim.get_state()
    assert sim.get_step_count() == 10
    sim.close()
    assert relerr(xg.cpu().numpy(), xo) <= 1e-9
    assert relerr(vg.cpu().numpy(), vo) <= 1e-8


def test_device_exponentials_match_libm(binding):
    """The three hand-written exponentials of the hot kernels against numpy's exp (<= 4 ulp), incl. the tails."""
    rng = np.random.default_rng(11)
    x = np.concatenate([rng.uniform(-40.0, 0.0, 200000), rng.uniform(-700.0, -40.0, 50000), rng.uniform(0.0, 5.0, 20000),
                        np.array([0.0, -1e-300, -0.5 * np.log(2.0), -707.9, -709.5, -1e5, -np.inf])])
    xd = torch.from_numpy(x).cuda()
    ref = np.exp(x)
    for which in (0, 1):
        y = binding.selftest_exp(which, xd).cpu().numpy()
        live = x >= -708.0
        assert np.max(np.abs(y[live] - ref[live]) / ref[live]) <= 1e-15
        assert np.all(y[~live] == 0.0)
    r2 = -x[x <= 0.0]
    r2 = r2[np.isfinite(r2)]
    ref2 = np.exp(-r2)
    live = r2 <= 700.0
    for which in (2, 3):  # 64-entry table (recursion, force pass) and 256-entry table (pair kernel)
        y = binding.selftest_exp(which, torch.from_numpy(r2).cuda()).cpu().numpy()
        # one-FMA argument reduction: relative error grows like r2 * 1.1e-16
        assert np.max(np.abs(y[live] - ref2[live]) / ref2[live] / (1.0 + r2[live])) <= 3e-16
        assert np.all(y[~live] <= 1e-300) and np.all(y >= 0.0)


def test_chain_phase_clock(binding):
    w = wl.custom(300, 4, d=2, beta=3.0, g=0.0, xi=1.0, init="ring", sigma=2.0)
    x, v = wl.make_state(w, 0)
    sim = make(binding, w, thermostat=1)
    sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    sim.step(2)
    assert sum(sim.get_chain_phases()) == 0  # profiling off: the clock is not running
    sim.set_profiling(True)
    sim.step(3)
    ph = sim.get_chain_phases()
    sim.close()
    assert len(ph) == 16 and all(c > 0 for c in ph[:4])
    nb = (w.N + 31) // 32
    per_block = sum(ph) / (3 * nb)
    assert 1e3 < per_block < 1e5  # a 32-row block costs a few thousand SM cycles


# ------------------------------------------------------------------------------------------------------------
# BASELINE.json's full sizes, in the launch configuration bench.py times (default look-ahead, workers, streams)
# ------------------------------------------------------------------------------------------------------------
def _forces_and_tables(binding, w, x):
    sim = make(binding, w)
    sim.set_state(torch.from_numpy(x).cuda())
    f, vb, sg = sim.forces()
    vf, vbw, pn = sim.get_tables()
    F = f.cpu().numpy()
    sim.close()
    return F, vb, sg, vf, vbw, pn


def test_full_size_n10000_against_oracle(binding, oracle):
    """config 5 at N = 10000 (non-interacting): V_B and every force against the oracle, element by element."""
    w = wl.WORKLOADS["cfg5_N10000"]
    x, _ = wl.make_state(w, 0)
    Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
    F, vb, sg = gpu_forces(binding, w, x)
    assert sg == sgo == 1
    assert abs(vb - vbo) <= RTOL * abs(vbo)
    check_forces(F, Fo, RTOL)


def test_full_size_identical_rings_closed_form(binding):
    """All particles on the same ring: W_N = e^{-beta N E_ring} prod_{j<N}(1 + j xi) / N!  (DESIGN.md pins; exact
    for any N and xi), so V_B = N E_ring - (1/beta) sum_j [log(1 + j xi) - log(j + 1)].  N = 10000 and 40000."""
    for N, xi in ((10000, 1.0), (10000, 0.5), (40000, 1.0)):
        P, d, beta = 16, 2, 3.0
        rng = np.random.default_rng(5)
        ring = rng.normal(0.0, 0.3, size=(P, 1, d))
        x = np.ascontiguousarray(np.repeat(ring, N, axis=1))
        w = wl.custom(N, P, d=d, beta=beta, g=0.0, xi=xi, init="iid")
        ks = P / beta ** 2
        diffs = np.diff(np.concatenate([ring[:, 0, :], ring[:1, 0, :]]), axis=0)
        e_ring = 0.5 * ks * float(np.sum(diffs ** 2))
        j = np.arange(N, dtype=np.float64)
        vb_exact = N * e_ring - float(np.sum(np.log1p(j * xi) - np.log(j + 1.0))) / beta
        F, vb, sg = gpu_forces(binding, w, x)
        assert sg == 1
        assert abs(vb - vb_exact) <= RTOL * abs(vb_exact)
        # by symmetry every particle feels the force of one closed ring of its own beads plus the trap
        xr = ring[:, 0, :]
        f_ring = -ks * (2 * xr - np.roll(xr, 1, axis=0) - np.roll(xr, -1, axis=0)) - (w.omega ** 2 / P) * xr
        ref = np.repeat(f_ring[:, None, :], N, axis=1)
        assert relerr(F, ref) <= 1e-9


@pytest.mark.parametrize("name", ["cfg5b", "cfg5_N40000"])
def test_full_size_invariants(binding, name):
    """Properties that hold at any size (no oracle run needed): forward = backward (Eq. 6 at n = N equals Eq. 11 at
    u = 1), Pr[l -> l+1] in [0, 1] with Pr[N -> N+1] = 0, the exchange + spring forces sum to zero over all beads
    (translation invariance), Newton's third law for the pair part, and Euler's theorem for the degree-2
    homogeneous V_B."""
    w = wl.WORKLOADS[name]
    x, _ = wl.make_state(w, 0)
    F, vb, sg, vf, vbw, pn = _forces_and_tables(binding, w, x)
    assert sg == 1 and np.isfinite(vb)
    assert abs(vf[w.N] - vb) <= 1e-9 * abs(vb)
    assert abs(vbw[1] - vb) <= 1e-9 * abs(vb)          # V^{[1,N]} from the backward recursion
    # Eq. 13 is 1 - (a ratio close to 1): its absolute rounding error is that of an exponent of size ~1e4 (R13)
    assert pn[-1] == 0.0 and pn.min() >= -1e-10 and pn.max() <= 1.0 + 1e-10
    # remove the trap force; what is left is translation invariant
    Fint = F + (w.omega ** 2 / w.P) * x
    scale = np.abs(Fint).sum()
    assert np.all(np.abs(Fint.sum(axis=(0, 1))) <= 1e-11 * scale)
    if w.g == 0.0:
        # Euler: sum r . grad V_B = 2 V_spring-part; with g = 0, -sum r.F_int = 2 (V_B - (1/beta) log-term) is not closed
        # form, but the virial identity -sum r . F_int = 2 <E_c> links it to the primitive estimator
        sim = make(binding, w)
        sim.set_state(torch.from_numpy(x).cuda())
        ep, ev, _ = sim.estimators()
        sim.close()
        ec = w.P * w.d * w.N / (2.0 * w.beta) + 0.5 * (w.omega ** 2 / w.P) * float(np.sum(x * x)) - ep
        assert abs(-float(np.sum(x * Fint)) - 2.0 * ec) <= 1e-9 * abs(2.0 * ec)


def test_stale_gauge_evaluations_match_oracle(binding, oracle):
    """From the second evaluation on, the recursion runs with the previous evaluation's gauge (k_chain_spec).
    Forces after a few MD steps must still match the oracle at the positions reached -- for bosons, for signed
    weights, and when the state jumps so far in one step that the stale gauge cannot fit (fallback kernel)."""
    cases = [
        (wl.custom(333, 8, d=2, beta=3.0, g=0.2, xi=1.0, init="ring", sigma=2.0), 0.01, 1.0, 1e-9),
        (wl.custom(200, 8, d=3, beta=2.0, g=0.1, xi=0.5, init="iid", sigma=0.8), 0.01, 1.0, 1e-9),
        (wl.custom(150, 8, d=2, beta=3.0, g=0.2, xi=-0.5, init="ring", sigma=3.0), 0.01, 1.0, 1e-7),
        (wl.custom(333, 8, d=2, beta=3.0, g=0.0, xi=1.0, init="ring", sigma=2.0), 1.0, 30.0, 1e-9),  # jump: fallback
        (wl.custom(1, 4, d=2, beta=2.0, g=0.0, xi=1.0, init="iid", sigma=0.7), 0.01, 1.0, 1e-9),      # one block, one row
        (wl.custom(2, 4, d=2, beta=2.0, g=0.3, xi=1.0, init="iid", sigma=0.7), 0.01, 1.0, 1e-9),
        (wl.custom(33, 6, d=2, beta=2.0, g=0.3, xi=1.0, init="iid", sigma=0.7), 0.01, 1.0, 1e-9),     # ragged second block
        (wl.custom(64, 6, d=1, beta=2.0, g=0.3, xi=1.0, init="iid", sigma=0.7), 0.01, 1.0, 1e-9),
        (wl.custom(129, 6, d=2, beta=2.0, g=0.0, xi=-1.0, init="ring", sigma=2.0), 0.01, 1.0, 1e-7),  # fermionic weights
    ]
    for w, dt, vscale, tol in cases:
        x, v = wl.make_state(w, 9)
        sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, dt, thermostat=0, seed=1)
        sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v * vscale).cuda())
        sim.step(3)
        xg, _ = sim.get_state()
        F, vb, sg = sim.forces()       # a fourth evaluation at the same positions, again with the stale gauge
        xs = xg.cpu().numpy()
        Fo, vbo, sgo = oracle.forces(xs, w.beta, w.omega, w.g, w.s, w.xi)
        sim.close()
        if w.xi < 0:
            tol = RTOL * oracle.conditioning(xs, w.beta, w.xi)
        assert sg == sgo
        assert abs(vb - vbo) <= tol * abs(vbo)
        check_forces(F.cpu().numpy(), Fo, tol)


def test_shifted_cloud_keeps_parity(binding, oracle):
    """The helper warps of k_chain_spec expand |rho - sigma|^2 about a block-local origin; a cloud that
    sits far from the coordinate origin, with the particle index unrelated to the position, must not cost accuracy.
    First evaluation: max-plus kernel; second and third: stale-gauge kernel with the tabulated terms."""
    for d, shift in ((2, (40.0, -25.0)), (3, (-30.0, 12.5, 55.0)), (1, (80.0,))):
        w = wl.custom(300, 8, d=d, beta=2.5, omega=0.01, g=0.0, xi=1.0, init="iid", sigma=1.2)  # weak trap: spring forces set the scale
        x, _ = wl.make_state(w, 21)
        x = x + np.asarray(shift).reshape((1, 1, d))
        sim = make(binding, w)
        sim.set_state(torch.from_numpy(x).cuda(), None)
        Fo, vbo, sgo = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
        for _ in range(3):
            F, vb, sg = sim.forces()
            assert sg == sgo
            assert abs(vb - vbo) <= 1e-9 * abs(vbo)
            check_forces(F.cpu().numpy(), Fo, 1e-9)
        sim.close()


def test_forces_round_trip_and_resume(binding, oracle):
    """pimd_get_forces returns what pimd_forces computed; a second handle fed (x, v, F) through set_state +
    set_forces continues bit-identically to the first one (NVE: no noise involved), without re-evaluating."""
    w = wl.custom(97, 6, d=2, beta=2.0, g=0.3, xi=1.0, init="iid", sigma=0.8)
    x, v = wl.make_state(w, 6)
    a = make(binding, w)
    a.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    with pytest.raises(binding.PimdError):
        a.get_forces()
    F, _, _ = a.forces()
    assert torch.equal(a.get_forces(), F)
    a.step(2)
    xa, va = a.get_state()
    Fa = a.get_forces()
    b = make(binding, w)
    b.set_state(xa, va)
    b.set_forces(Fa)
    l0 = b.launch_count()
    b.step(1)
    assert b.launch_count() - l0 <= 12  # one evaluation, not two
    a.step(1)
    xb, vb_ = b.get_state()
    xa2, va2 = a.get_state()
    a.close(); b.close()
    assert relerr(xb.cpu().numpy(), xa2.cpu().numpy()) <= 1e-13
    assert relerr(vb_.cpu().numpy(), va2.cpu().numpy()) <= 1e-12


@pytest.mark.parametrize("case", [(70, 6, 2, 2.5, 1.0), (133, 5, 3, 2.0, 0.5), (45, 4, 1, 2.0, -0.4), (33, 4, 2, 2.0, 0.0)],
                         ids=["n70", "n133_d3", "n45_d1_neg", "n33_xi0"])
def test_materialised_matrices_match_oracle(binding, oracle, case):
    """pimd_cycle_energies (Eq. 7-10) and pimd_connection_probabilities (Eq. 12-14) against the oracle's
    matrices, element by element; rows and columns of Pr sum to one."""
    N, P, d, beta, xi = case
    w = wl.custom(N, P, d=d, beta=beta, g=0.0, xi=xi, init="ring", sigma=1.0)
    x, _ = wl.make_state(w, 8)
    sim = make(binding, w)
    sim.set_state(torch.from_numpy(x).cuda())
    E = sim.cycle_energies().cpu().numpy()
    Pr = sim.connection_probabilities().cpu().numpy()
    sim.close()
    Eo = oracle.cycle_energies(x, beta)
    assert np.all(np.tril(E, -1) == 0.0)
    assert np.max(np.abs(E - np.triu(Eo))) <= 1e-10 * np.max(np.abs(Eo))
    Pro = oracle.pr_matrix(x, beta, xi)
    tol = 1e-9 if xi >= 0 else 1e-9 * oracle.conditioning(x, beta, xi)
    assert np.max(np.abs(Pr - Pro)) <= tol
    np.testing.assert_allclose(Pr.sum(axis=1), 1.0, atol=10 * tol)
    np.testing.assert_allclose(Pr.sum(axis=0), 1.0, atol=10 * tol)


def test_materialised_matrices_full_size(binding):
    """N = 10000 (0.8 GB each): every row and column of Pr sums to one, Pr is zero two above the diagonal;
    E on the diagonal is the single-ring energy, E^{[u,v]} - E^{[u,v-1]} telescopes as Eq. 10 says for sampled entries."""
    w = wl.WORKLOADS["cfg5_N10000"]
    x, _ = wl.make_state(w, 0)
    sim = make(binding, w)
    sim.set_state(torch.from_numpy(x).cuda())
    Pr = sim.connection_probabilities()
    rows, cols = Pr.sum(dim=1).cpu().numpy(), Pr.sum(dim=0).cpu().numpy()
    assert np.max(np.abs(rows - 1.0)) <= 1e-9 and np.max(np.abs(cols - 1.0)) <= 1e-9
    assert float(torch.triu(Pr, 2).abs().max()) == 0.0
    del Pr
    E = sim.cycle_energies()
    sim.close()
    ks = w.P / w.beta ** 2
    ring = np.concatenate([x, x[:1]], axis=0)
    e_self = 0.5 * ks * np.sum(np.diff(ring, axis=0) ** 2, axis=(0, 2))          # every particle closed on itself
    assert np.max(np.abs(torch.diagonal(E).cpu().numpy() - e_self)) <= 1e-9 * np.max(e_self)
    rng = np.random.default_rng(2)
    for _ in range(50):
        u = int(rng.integers(0, w.N - 1)); v = int(rng.integers(u + 1, w.N))
        # Eq. 10: E^{[u,v]} = E^{[u,v-1]} - C(v-1,u) + C(v-1,v) + E_int(v) + C(v,u)
        c = lambda a, b: 0.5 * ks * float(np.sum((x[w.P - 1, a] - x[0, b]) ** 2))
        eint_v = 0.5 * ks * float(np.sum(np.diff(x[:, v], axis=0) ** 2))
        lhs = float(E[u, v])
        rhs = float(E[u, v - 1]) - c(v - 1, u) + c(v - 1, v) + eint_v + c(v, u)
        assert abs(lhs - rhs) <= 1e-9 * abs(lhs)


@pytest.mark.parametrize("xi,thermostat", [(1.0, 1), (0.0, 1), (1.0, 2), (0.0, 2)],
                         ids=["bosons_langevin", "distinguishable_langevin", "bosons_nhc", "distinguishable_nhc"])
def test_ensemble_energy_matches_exact_ideal_gas_and_oracle(binding, oracle, xi, thermostat):
    """BASELINE config 1 (N = 4, P = 16, beta = 2, non-interacting): 64 independent replicas (one batch, own seeds and
    initial states), 5e3 steps of equilibration, 3e5 sampled steps each with the estimators every 10 steps (pimd_run).
    One mean per replica, so the standard error is that of 64 independent numbers.  north_star: the primitive and the
    virial energy agree with the exact finite-P canonical value (oracle/ideal_gas.py) within 3
    standard errors -- no further slack -- and with the same run through the oracle's orc_step (smaller budget) within 3
    combined standard errors."""
    from oracle import ideal_gas

    B = 64
    w = wl.WORKLOADS["cfg1"].with_(xi=xi)
    exact = ideal_gas.exact_energy(w.N, w.beta, w.omega, w.d, xi, w.P)
    xs, vs = zip(*[wl.make_state(w, 1000 + b) for b in range(B)])
    sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, [xi] * B, w.dt, thermostat=thermostat,
                       seed=[5000 + b for b in range(B)])
    sim.set_state(torch.from_numpy(np.stack(xs)).cuda(), torch.from_numpy(np.stack(vs)).cuda())
    sim.step(5000)
    sim.run(300000, est_every=10)
    n, sp, sv, _, _ = sim.read_accumulators()
    sim.close()
    assert np.all(n == 30000)
    # the oracle on a smaller budget: 12 seeds, 2e3 + 3e4 steps
    o_p, o_v = [], []
    for k in range(12):
        x, v = wl.make_state(w, 2000 + k)
        F, _, _ = oracle.forces(x, w.beta, w.omega, w.g, w.s, xi)
        nhc = np.zeros((4, x.size))
        oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, xi, w.dt, thermostat, 1.0, 7000 + k, 0, 2000)
        a = b = 0.0
        for i in range(3000):
            oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, xi, w.dt, thermostat, 1.0, 7000 + k, 2000 + 10 * i, 10)
            ep, ev, _ = oracle.estimators(x, w.beta, w.omega, w.g, w.s, xi)
            a += ep; b += ev
        o_p.append(a / 3000); o_v.append(b / 3000)
    for sums, orc in ((sp, o_p), (sv, o_v)):
        vals = sums / n
        mean, se = vals.mean(), vals.std(ddof=1) / np.sqrt(B)
        omean, ose = np.mean(orc), np.std(orc, ddof=1) / np.sqrt(len(orc))
        assert se <= 0.005 * abs(exact), (mean, se, exact)      # the run is long enough to mean something
        assert abs(mean - exact) <= 3.0 * se, (mean, se, exact)
        assert abs(mean - omean) <= 3.0 * np.hypot(se, ose), (mean, se, omean, ose)


def test_graph_replay_matches_step_by_step(binding):
    """pimd_step(n >= 3) replays a captured CUDA graph for all but the last step; the trajectory (Langevin noise
    included: the Philox step counter lives on the device meanwhile) must be the one single-step calls produce."""
    w = wl.WORKLOADS["cfg2"].with_(N=70, P=8)
    x, v = wl.make_state(w, 12)
    out = []
    for chunks in ((25,), (1,) * 25, (3, 7, 15)):
        sim = make(binding, w, thermostat=1, seed=77)
        sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        for n in chunks:
            sim.step(n)
        assert sim.get_step_count() == 25
        xg, vg = sim.get_state()
        out.append((xg.cpu().numpy(), vg.cpu().numpy()))
        sim.close()
    for xs, vs in out[1:]:
        # identical kernels and arguments; atomics in the pair / force-pass kernels make the last bits order dependent
        assert relerr(xs, out[0][0]) <= 1e-12
        assert relerr(vs, out[0][1]) <= 1e-11


@pytest.mark.parametrize("thermostat", [1, 2], ids=["langevin", "nhc"])
def test_resume_through_the_thermostats(binding, thermostat):
    """Checkpoint / resume with a thermostat: 20 steps on one handle against 10 steps, a snapshot of
    (x, v, F, step counter, Nose-Hoover chain variables) moved into a SECOND handle, and 10 more steps there.  The Langevin
    noise is keyed by (seed, degree of freedom, step counter), so pimd_set_step_count is what lines the noise up; the chain
    variables go through pimd_get_nhc / pimd_set_nhc (after pimd_set_state, which zeroes them).  Agreement is to rounding,
    not to the bit: the second handle's first evaluation has no gauge history and the pair forces are summed with atomics
    (pimd.h says so).  Leaving the counter / the chain variables out must visibly change the trajectory."""
    w = wl.custom(97, 6, d=2, beta=2.0, g=0.3, xi=1.0, init="iid", sigma=0.8)
    x, v = wl.make_state(w, 6)
    a = make(binding, w, thermostat=thermostat, seed=21)
    a.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
    a.step(10)
    xa, va = a.get_state()
    Fa = a.get_forces()
    count = a.get_step_count()
    assert count == 10
    nhc = a.get_nhc() if thermostat == 2 else None
    a.step(10)
    x20, v20 = [t.cpu().numpy() for t in a.get_state()]
    a.close()

    def resume(full):
        b = make(binding, w, thermostat=thermostat, seed=21)
        b.set_state(xa, va)
        b.set_forces(Fa)
        if full:
            b.set_step_count(count)
            if nhc is not None:
                b.set_nhc(nhc)
        b.step(10)
        out = [t.cpu().numpy() for t in b.get_state()]
        n = b.get_step_count()
        b.close()
        return out, n

    (xb, vb_), n = resume(True)
    assert n == 20
    assert relerr(xb, x20) <= 1e-12 and relerr(vb_, v20) <= 1e-11
    (xc, vc), _ = resume(False)
    assert relerr(vc, v20) > 1e-3
