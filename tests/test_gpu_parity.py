"""Parity of the CUDA path (through the C ABI, libpimd.so) with the CPU oracle -- needs a B200.

Tolerances (BASELINE.json north_star): 1e-9 relative on V_B and on the forces (max-norm), FP64.
For xi < 0 the tolerance is scaled by the conditioning kappa = sum|terms| / |sum terms| of the
signed sums (R7); here kappa stays O(1..100) and a fixed 1e-7 bound is used.
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
    assert sg == sgo
    assert abs(vb - vbo) <= 1e-7 * abs(vbo)
    check_forces(F, Fo, 1e-7)


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
    tol = RTOL if w.xi >= 0 else 1e-7
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
    y = binding.selftest_exp(2, torch.from_numpy(r2).cuda()).cpu().numpy()
    ref2 = np.exp(-r2)
    live = r2 <= 700.0
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
    assert len(ph) == 16 and all(c > 0 for c in ph[:9])
    nb = (w.N + 31) // 32
    per_block = sum(ph[:9]) / (3 * nb)
    assert 1e3 < per_block < 1e5  # a 32-row block costs a few thousand SM cycles
