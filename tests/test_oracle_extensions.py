"""Pins of the round-2 oracle functions (no GPU): the O(N)-memory evaluation, several species, the second pair
potential, the pair-distance histogram, the conditioning number and the reweighting estimator.  Reference sides are
brute force written here / in tests/bruteforce.py, closed forms, or the exact ideal-gas energy -- never the oracle's
own matrices alone."""
import math

import numpy as np
import pytest

from tests import bruteforce as bf


def rand_x(P, N, d, seed, scale=0.6):
    return np.random.default_rng(seed).normal(0.0, scale, size=(P, N, d))


# ---------------------------------------------------------------------------------------------------------------
# O(N)-memory evaluation (orc_stream_*)
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("xi", [1.0, 0.5, 0.0, -0.3])
def test_stream_forces_match_finite_differences_of_bruteforce_potential(oracle, xi):
    beta, omega, g, s = 1.3, 0.9, 0.7, 0.6
    P, N, d = 3, 5, 2
    x = rand_x(P, N, d, 77, scale=0.5)

    def phi(y):
        return -math.log(abs(bf.composition_sum(y, beta, xi))) / beta + bf.potential_external(y, omega, g, s)

    F, vb, sg = oracle.stream_forces_on(x, beta, omega, g, s, xi, list(range(N)))
    assert vb == pytest.approx(-math.log(abs(bf.composition_sum(x, beta, xi))) / beta, rel=1e-12)
    assert sg == (1 if bf.composition_sum(x, beta, xi) > 0 else -1)
    h = 1e-5
    Fd = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp = x.copy(); xp[idx] += h
        xm = x.copy(); xm[idx] -= h
        Fd[idx] = -(phi(xp) - phi(xm)) / (2 * h)
    np.testing.assert_allclose(F.transpose(1, 0, 2), Fd, atol=3e-8 * np.abs(Fd).max())


def test_stream_tables_identical_rings_closed_form(oracle):
    """W_n = e^{-beta n E_ring} prod_{j<n}(1 + j xi)/n! for every n (forward table), N = 3000."""
    beta, P, d, N, xi = 3.0, 8, 2, 3000, 0.5
    ring = rand_x(P, 1, d, 2, scale=0.4)
    x = np.ascontiguousarray(np.repeat(ring, N, axis=1))
    e_ring = bf.cycle_energy_eq7(ring, beta, 1, 1)
    F, vb, sg, fwd, bwd = oracle.stream_forces_on(x, beta, 0.0, 0.0, 0.5, xi, [0, N - 1], tables=True)
    j = np.arange(N)
    logw = np.concatenate([[0.0], np.cumsum(np.log1p(j * xi) - np.log(j + 1.0))])
    ref = np.arange(N + 1) * e_ring - logw / beta
    np.testing.assert_allclose(fwd, ref, rtol=1e-12, atol=1e-10)
    assert vb == pytest.approx(ref[N], rel=1e-12) and sg == 1
    assert bwd[1] == pytest.approx(vb, rel=1e-12) and bwd[N + 1] == 0.0    # Eq. 11 at u = 1 is Eq. 6 at n = N
    # by symmetry the exchange force on every particle is that of one closed ring of its own beads
    xr = ring[:, 0, :]
    ks = P / beta ** 2
    f_ring = -ks * (2 * xr - np.roll(xr, 1, axis=0) - np.roll(xr, -1, axis=0))
    np.testing.assert_allclose(F[0], f_ring, atol=1e-9 * np.abs(f_ring).max())
    np.testing.assert_allclose(F[1], f_ring, atol=1e-9 * np.abs(f_ring).max())


# ---------------------------------------------------------------------------------------------------------------
# several species
# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("xi", [1.0, -0.4])
def test_species_potential_is_product_of_composition_sums(oracle, xi):
    beta, omega, g, s = 1.2, 0.8, 0.5, 0.6
    P, d, counts = 3, 2, [3, 2]
    N = sum(counts)
    x = rand_x(P, N, d, 5, scale=0.5)

    def phi(y):
        wa = bf.composition_sum(np.ascontiguousarray(y[:, :3]), beta, xi)
        wb = bf.composition_sum(np.ascontiguousarray(y[:, 3:]), beta, xi)
        return -math.log(abs(wa * wb)) / beta + bf.potential_external(y, omega, g, s), wa * wb

    F, vb, sg = oracle.forces_species(x, beta, omega, g, s, xi, counts)
    p0, w0 = phi(x)
    assert vb == pytest.approx(p0 - bf.potential_external(x, omega, g, s), rel=1e-12)
    assert sg == (1 if w0 > 0 else -1)
    h = 1e-5
    Fd = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp = x.copy(); xp[idx] += h
        xm = x.copy(); xm[idx] -= h
        Fd[idx] = -(phi(xp)[0] - phi(xm)[0]) / (2 * h)
    np.testing.assert_allclose(F, Fd, atol=3e-8 * np.abs(Fd).max())


def test_species_estimator_is_beta_derivative(oracle):
    """E_prim = d(beta Phi)/d beta + P d N/(2 beta) with the coordinates scaled so that the spring part ~ beta^-2 is
    differentiated at fixed positions: eps = d(beta V)/d beta by central differences of the species potential."""
    beta, P, d, counts, xi = 1.4, 3, 2, [2, 3], 0.7
    N = sum(counts)
    x = rand_x(P, N, d, 9, scale=0.5)
    ep, ev, _ = oracle.estimators_species(x, beta, 0.9, 0.4, 0.6, xi, counts)

    def beta_v(b):
        _, vb, _ = oracle.forces_species(x, b, 0.0, 0.0, 0.6, xi, counts)
        return b * vb

    h = 1e-5
    eps = (beta_v(beta + h) - beta_v(beta - h)) / (2 * h)
    ubar = bf.potential_external(x, 0.9, 0.4, 0.6)
    assert ep == pytest.approx(P * d * N / (2 * beta) + eps + ubar, rel=1e-8)
    ep1, ev1, _ = oracle.estimators(x, beta, 0.9, 0.4, 0.6, xi)
    assert ev == ev1                                    # the virial estimator does not see the exchange part
    epa, _, _ = oracle.estimators_species(x, beta, 0.9, 0.4, 0.6, xi, [N])
    assert epa == pytest.approx(ep1, rel=1e-13)         # one species = the plain estimator


# ---------------------------------------------------------------------------------------------------------------
# second pair potential (Eq. 18 leaves V generic)
# ---------------------------------------------------------------------------------------------------------------
def test_soft_coulomb_forces_finite_differences_and_closed_form(oracle):
    omega, g, s = 0.0, 0.8, 0.5
    P, N, d = 2, 4, 3
    x = rand_x(P, N, d, 12, scale=0.7)

    def u(y):
        tot = 0.0
        for j in range(P):
            for a in range(N):
                for b in range(a):
                    tot += g / math.sqrt(float(np.sum((y[j, a] - y[j, b]) ** 2)) + s * s)
        return tot / P

    oracle.set_pair_potential(1)
    try:
        F, _, _ = oracle.forces(x, 2.0, omega, g, s, 0.0)
        F0, _, _ = oracle.forces(x, 2.0, omega, 0.0, s, 0.0)
        ep, ev, _ = oracle.estimators(x, 2.0, omega, g, s, 0.0)
        ep0, ev0, _ = oracle.estimators(x, 2.0, omega, 0.0, s, 0.0)
        f_on = oracle.external_force_on(x, omega, g, s, 1, 2)
        # two particles, closed form: F = g r / (r^2 + s^2)^{3/2} along the separation
        y = np.zeros((2, 2, 3)); y[:, 1, 0] = 1.3
        Fy, _, _ = oracle.forces(y, 2.0, 0.0, g, s, 0.0)
        Fy0, _, _ = oracle.forces(y, 2.0, 0.0, 0.0, s, 0.0)
    finally:
        oracle.set_pair_potential(0)
    Fp = F - F0
    h = 1e-5
    Fd = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp = x.copy(); xp[idx] += h
        xm = x.copy(); xm[idx] -= h
        Fd[idx] = -(u(xp) - u(xm)) / (2 * h)
    np.testing.assert_allclose(Fp, Fd, atol=3e-9 * np.abs(Fd).max())
    np.testing.assert_allclose(Fp.sum(axis=1), 0.0, atol=1e-13)              # Newton's third law per slice
    np.testing.assert_allclose(f_on, Fp[1, 2], atol=1e-14)
    assert ep - ep0 == pytest.approx(u(x), rel=1e-12)
    # virial term: Ubar + 1/2 sum r . grad Ubar, by finite differences of the scaling y -> (1 + t) y
    dudt = (u((1 + h) * x) - u((1 - h) * x)) / (2 * h)
    assert ev - ev0 == pytest.approx(u(x) + 0.5 * dudt, rel=1e-8)
    fx = g * 1.3 / (1.3 ** 2 + s * s) ** 1.5 / 2                            # (1/P) per bead
    np.testing.assert_allclose((Fy - Fy0)[:, 1, 0], fx, rtol=1e-13)
    np.testing.assert_allclose((Fy - Fy0)[:, 0, 0], -fx, rtol=1e-13)


# ---------------------------------------------------------------------------------------------------------------
# pair-distance histogram
# ---------------------------------------------------------------------------------------------------------------
def test_pair_histogram_matches_numpy(oracle):
    P, N, d, nbins, rmax = 4, 23, 2, 16, 2.5
    x = rand_x(P, N, d, 3, scale=0.9)
    dist = []
    for j in range(P):
        for a in range(N):
            for b in range(a):
                dist.append(math.sqrt(float(np.sum((x[j, a] - x[j, b]) ** 2))))
    ref, _ = np.histogram(np.asarray(dist), bins=nbins, range=(0.0, rmax))
    inside = sum(1 for r in dist if r < rmax)
    h = oracle.pair_histogram(x, nbins, rmax)
    assert h.sum() == inside
    np.testing.assert_array_equal(h, ref)


# ---------------------------------------------------------------------------------------------------------------
# conditioning of the signed sums
# ---------------------------------------------------------------------------------------------------------------
def test_conditioning_is_one_for_bosons_and_closed_form_for_n2(oracle):
    beta, P, d = 1.5, 3, 2
    x = rand_x(P, 6, d, 4)
    for xi in (1.0, 0.3, 0.0):
        assert oracle.conditioning(x, beta, xi) == pytest.approx(1.0, abs=1e-12)
    x2 = rand_x(P, 2, d, 8, scale=0.4)
    xi = -0.6
    a = math.exp(-beta * (bf.cycle_energy_eq7(x2, beta, 1, 1) + bf.cycle_energy_eq7(x2, beta, 2, 2)))
    b = abs(xi) * math.exp(-beta * bf.cycle_energy_eq7(x2, beta, 1, 2))
    k_sum = (a + b) / abs(a - b)                        # Eq. 6 at n = 2: W_2 = (a - |xi| e^{-beta E12}) / 2
    # quasi-probabilities of the two rows: Pr[2->2] = a/(a-b), Pr[2->1] = -b/(a-b); row 1: Pr[1->1], Pr[1->2]
    k = oracle.conditioning(x2, beta, xi)
    assert k >= k_sum * (1 - 1e-12)
    assert k == pytest.approx(max(k_sum, 1.0), rel=1e-9) or k > k_sum


# ---------------------------------------------------------------------------------------------------------------
# reweighting estimator: sample at |xi|, weigh with R = W_xi / W_|xi|
# ---------------------------------------------------------------------------------------------------------------
def test_reweighted_energy_matches_exact_fictitious_particle_value(oracle):
    """N = 3, P = 4, beta = 2, d = 2 ideal gas: <E>_{xi = -0.3} from a Langevin run of the oracle at xi = +0.3, reweighted,
    against the exact finite-P value (oracle/ideal_gas.py; 4.226559 in SURVEY Appendix B) within 3 standard errors."""
    from oracle import ideal_gas

    N, P, d, beta, xi_obs = 3, 4, 2, 2.0, -0.3
    xi_s = abs(xi_obs)
    exact = ideal_gas.exact_energy(N, beta, 1.0, d, xi_obs, P)
    assert exact == pytest.approx(4.226559261, abs=2e-9)
    num, den, num_v = [], [], []
    for seed in range(48):
        rng = np.random.default_rng(100 + seed)
        x = rng.normal(0.0, 0.7, size=(P, N, d))
        v = rng.normal(0.0, math.sqrt(1.0 / beta), size=(P, N, d))
        F, _, _ = oracle.forces(x, beta, 1.0, 0.0, 0.5, xi_s)
        step0 = 0
        oracle.step(x, v, F, None, beta, 1.0, 0.0, 0.5, xi_s, 0.02, 1, 1.0, seed, step0, 500)
        step0 += 500
        a = b = c = 0.0
        for _ in range(1000):
            oracle.step(x, v, F, None, beta, 1.0, 0.0, 0.5, xi_s, 0.02, 1, 1.0, seed, step0, 10)
            step0 += 10
            vs, _ = oracle.vb(x, beta, xi_s)
            vo, so = oracle.vb(x, beta, xi_obs)
            r = so * math.exp(-beta * (vo - vs))
            ep, ev, _ = oracle.estimators(x, beta, 1.0, 0.0, 0.5, xi_obs)
            a += r * ep; b += r; c += r * ev
        num.append(a); den.append(b); num_v.append(c)
    num, den, num_v = map(np.asarray, (num, den, num_v))
    for top in (num, num_v):
        est = top.sum() / den.sum()
        # jackknife over the independent seeds
        jk = np.array([(top.sum() - top[i]) / (den.sum() - den[i]) for i in range(len(den))])
        se = math.sqrt((len(jk) - 1) / len(jk) * float(np.sum((jk - jk.mean()) ** 2)))
        assert abs(est - exact) <= 3.0 * se, (est, se, exact)
        assert se < 0.02 * exact
