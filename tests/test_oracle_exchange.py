"""Pins of the oracle's exchange potential, probabilities and forces (CPU only).

Every check compares oracle/pimd_oracle.c with something that is NOT the oracle: a brute-force
definition written in tests/bruteforce.py, a closed form, an invariant, or finite differences.
"""
import itertools
import math

import numpy as np
import pytest

from tests import bruteforce as bf

XIS = [1.0, 0.5, 0.0, -0.3]


def rand_x(P, N, d, seed, scale=0.6):
    return np.random.default_rng(seed).normal(0.0, scale, size=(P, N, d))


# ---------------------------------------------------------------- E^{[u,v]} (Eq. 7-10)
@pytest.mark.parametrize("N,P,d", [(1, 2, 1), (3, 2, 2), (6, 5, 2), (8, 4, 3)])
def test_cycle_energies_match_literal_eq7(oracle, N, P, d):
    beta = 1.7
    x = rand_x(P, N, d, 11)
    E = oracle.cycle_energies(x, beta)
    E10 = oracle.cycle_energies_eq10(x, beta)
    for u in range(1, N + 1):
        for v in range(u, N + 1):
            ref = bf.cycle_energy_eq7(x, beta, u, v)  # literal triple loop, boundary rule PAPER.md:76
            assert E[u - 1, v - 1] == pytest.approx(ref, rel=1e-13)
            assert E10[u - 1, v - 1] == pytest.approx(ref, rel=1e-12)  # the paper's iteration, Eq. 8+10
            assert oracle.cycle_energy_eq7(x, beta, u, v) == pytest.approx(ref, rel=1e-13)


def test_eint_matches_eq9(oracle):
    P, N, d, beta = 7, 5, 2, 2.3
    x = rand_x(P, N, d, 3)
    ref = 0.5 * bf.ks_of(P, beta) * np.sum((x[1:] - x[:-1]) ** 2, axis=(0, 2))
    np.testing.assert_allclose(oracle.eint(x, beta), ref, rtol=1e-14)


# ---------------------------------------------------------------- V_B (Eq. 6)
@pytest.mark.parametrize("xi", XIS)
@pytest.mark.parametrize("N,P", [(1, 3), (2, 2), (5, 3), (9, 2)])
def test_vb_equals_composition_sum(oracle, xi, N, P):
    """Eq. 6 unrolled: sum over the 2^(N-1) cuts of 1..N into runs of consecutive indices."""
    beta, d = 1.3, 2
    x = rand_x(P, N, d, 100 + N)
    vb, sign = oracle.vb(x, beta, xi)
    W = bf.composition_sum(x, beta, xi)
    assert sign == (1 if W > 0 else -1)
    assert math.exp(-beta * vb) == pytest.approx(abs(W), rel=1e-11)


@pytest.mark.parametrize("xi", XIS)
@pytest.mark.parametrize("N", [2, 3, 4, 5])
def test_relabel_average_equals_permutation_sum(oracle, xi, N):
    """Eq. 2 vs Eq. 4+6: the recursion weight averaged over all N! relabellings of the particles
    equals (1/N!) sum_p xi^{N_p} exp(-beta E_p) pointwise (reading R16)."""
    beta, P, d = 0.9, 3, 2
    x = rand_x(P, N, d, 7 * N)
    ref = bf.permutation_sum(x, beta, xi)
    acc = 0.0
    for perm in itertools.permutations(range(N)):
        vb, sign = oracle.vb(np.ascontiguousarray(x[:, list(perm), :]), beta, xi)
        acc += sign * math.exp(-beta * vb)
    acc /= math.factorial(N)
    assert acc == pytest.approx(ref, rel=2e-11)


def test_n2_closed_form(oracle):
    """N=2: e^{-beta V} = 1/2 [ e^{-beta(E11+E22)} + xi e^{-beta E12} ] (Eq. 6 with V^{[1,0]}=0)."""
    beta, P, d = 1.1, 4, 2
    x = rand_x(P, 2, d, 5)
    E11 = bf.cycle_energy_eq7(x, beta, 1, 1)
    E22 = bf.cycle_energy_eq7(x, beta, 2, 2)
    E12 = bf.cycle_energy_eq7(x, beta, 1, 2)
    for xi in XIS + [-1.0]:
        W = 0.5 * (math.exp(-beta * (E11 + E22)) + xi * math.exp(-beta * E12))
        vb, sign = oracle.vb(x, beta, xi)
        assert sign * math.exp(-beta * vb) == pytest.approx(W, rel=1e-12)


@pytest.mark.parametrize("xi,N", [(1.0, 5), (1.0, 300), (1.0, 3000), (0.5, 5), (0.5, 300), (0.5, 3000),
                                  (0.0, 5), (0.0, 300), (-0.3, 5), (-0.3, 40), (-0.45, 9), (-0.7, 12)])
def test_identical_rings_closed_form(oracle, xi, N):
    """All particles on the same ring: E^{[u,v]} = (v-u+1) E_ring, so Eq. 6 gives
    W_N = e^{-beta N E_ring} prod_{j<N} (1 + j xi) / N!   (xi=1: V_B = N E_ring).  Tests the
    stabilised log-sum-exp at scale (beta N E_ring ~ 1e4).  For xi<0 the sum cancels; the
    tolerance is scaled by the conditioning kappa = prod (1+j|xi|) / prod |1+j xi| (R7)."""
    beta, P, d = 3.0, 8, 2
    ring = rand_x(P, 1, d, 2, scale=0.4)
    x = np.ascontiguousarray(np.repeat(ring, N, axis=1))
    e_ring = bf.cycle_energy_eq7(ring, beta, 1, 1)
    log_abs, log_kappa, sgn = 0.0, 0.0, 1
    for j in range(N):
        f = 1.0 + j * xi
        assert f != 0.0, "parametrisation hits a node"
        log_abs += math.log(abs(f)) - math.log(j + 1)
        log_kappa += math.log(1.0 + j * abs(xi)) - math.log(abs(f))
        sgn *= 1 if f > 0 else -1
    vb, sign = oracle.vb(x, beta, xi)
    ref = N * e_ring - log_abs / beta
    assert sign == sgn
    assert vb == pytest.approx(ref, rel=1e-12, abs=1e-10 + 1e-15 * math.exp(log_kappa))


def test_xi0_distinguishable_closed_form(oracle):
    """xi=0 (0^0=1): V = sum_l E^{[l,l]} + (1/beta) ln N!; Pr = identity."""
    beta, P, d, N = 2.0, 6, 2, 40
    x = rand_x(P, N, d, 9)
    ref = sum(bf.cycle_energy_eq7(x, beta, l, l) for l in range(1, N + 1)) + math.lgamma(N + 1) / beta
    vb, sign = oracle.vb(x, beta, 0.0)
    assert sign == 1 and vb == pytest.approx(ref, rel=1e-13)
    np.testing.assert_allclose(oracle.pr_matrix(x, beta, 0.0), np.eye(N), atol=1e-13)


@pytest.mark.parametrize("xi", XIS)
def test_forward_equals_backward(oracle, xi):
    """Eq. 11 at u=1 must reproduce Eq. 6 at n=N -- only true with the base V^{[N+1,N]}=0 (R2)."""
    beta, P, d, N = 1.5, 4, 2, 60
    x = rand_x(P, N, d, 21, scale=0.5)
    vb, sign, fwd, bwd = oracle.vb(x, beta, xi, tables=True)
    assert fwd[0] == 0.0 and bwd[N + 1] == 0.0
    assert bwd[1] == pytest.approx(vb, rel=1e-12)
    assert fwd[N] == vb


# ---------------------------------------------------------------- Pr (Eq. 12-14)
@pytest.mark.parametrize("xi", XIS)
@pytest.mark.parametrize("N", [1, 2, 7, 50])
def test_probabilities_rows_and_columns_sum_to_one(oracle, xi, N):
    beta, P, d = 1.2, 3, 2
    x = rand_x(P, N, d, 40 + N, scale=0.5)
    Pr = oracle.pr_matrix(x, beta, xi)
    np.testing.assert_allclose(Pr.sum(axis=1), 1.0, atol=1e-11)
    np.testing.assert_allclose(Pr.sum(axis=0), 1.0, atol=1e-11)
    # Eq. 14: nothing beyond the first super-diagonal
    assert np.all(np.triu(Pr, 2) == 0.0)
    if xi >= 0:
        assert Pr.min() >= -1e-14 and Pr.max() <= 1 + 1e-14


def test_probabilities_n3_against_explicit_permutation_weights(oracle):
    """N=3, xi=1: Pr[G(3)=l'] follows from the three k-terms of Eq. 6 at n=3 directly."""
    beta, P, d = 0.8, 2, 2
    x = rand_x(P, 3, d, 77, scale=0.5)
    _, _, fwd, _ = oracle.vb(x, beta, 1.0, tables=True)
    W = [math.exp(-beta * v) for v in fwd]
    terms = [math.exp(-beta * bf.cycle_energy_eq7(x, beta, u, 3)) * W[u - 1] / 3.0 for u in (1, 2, 3)]
    Pr = oracle.pr_matrix(x, beta, 1.0)
    np.testing.assert_allclose(Pr[2], np.array(terms) / W[3], rtol=1e-12)


# ---------------------------------------------------------------- forces (Eq. 15-17)
@pytest.mark.parametrize("xi", [1.0, 0.5, 0.0, -0.3])
@pytest.mark.parametrize("N,P,d", [(1, 2, 1), (2, 2, 2), (4, 3, 2), (6, 5, 3), (12, 4, 2)])
def test_exchange_forces_match_finite_differences(oracle, xi, N, P, d):
    beta = 1.4
    x = rand_x(P, N, d, 500 + N + P, scale=0.5)
    F, vb, sign = oracle.forces(x, beta, 1.0, 0.0, 0.5, xi, include_external=False)
    h = 1e-5
    Fd = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp = x.copy(); xp[idx] += h
        xm = x.copy(); xm[idx] -= h
        Fd[idx] = -(oracle.vb(xp, beta, xi)[0] - oracle.vb(xm, beta, xi)[0]) / (2 * h)
    scale = np.abs(F).max()
    np.testing.assert_allclose(F, Fd, atol=2e-8 * scale)
    # translation invariance of V_B
    np.testing.assert_allclose(F.sum(axis=(0, 1)), 0.0, atol=1e-10 * scale)


def test_full_forces_match_finite_differences_of_bruteforce_potential(oracle):
    """-grad of (composition-sum V_B + brute-force U/P): no oracle code on the reference side."""
    beta, omega, g, s, xi = 1.3, 0.9, 0.7, 0.6, 1.0
    P, N, d = 3, 4, 2
    x = rand_x(P, N, d, 31, scale=0.5)

    def phi(y):
        return -math.log(bf.composition_sum(y, beta, xi)) / beta + bf.potential_external(y, omega, g, s)

    F, vb, _ = oracle.forces(x, beta, omega, g, s, xi)
    assert oracle.potential(x, beta, omega, g, s, xi) == pytest.approx(phi(x), rel=1e-12)
    h = 1e-5
    Fd = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp = x.copy(); xp[idx] += h
        xm = x.copy(); xm[idx] -= h
        Fd[idx] = -(phi(xp) - phi(xm)) / (2 * h)
    np.testing.assert_allclose(F, Fd, atol=2e-8 * np.abs(F).max())


def test_xi0_forces_are_independent_closed_rings(oracle):
    beta, P, N, d = 2.0, 5, 6, 2
    x = rand_x(P, N, d, 8)
    F, _, _ = oracle.forces(x, beta, 1.0, 0.0, 0.5, 0.0, include_external=False)
    ks = bf.ks_of(P, beta)
    ref = -ks * (2 * x - np.roll(x, 1, axis=0) - np.roll(x, -1, axis=0))  # closed ring per particle
    np.testing.assert_allclose(F, ref, rtol=1e-12, atol=1e-12)


def test_euler_homogeneity(oracle):
    """V_B is homogeneous of degree 2 in the coordinates: sum r . grad V_B = 2 V_B' where V_B'
    is the Pr-weighted spring energy; checked as -sum r.F = 2 * (d(beta V)/d beta identity below)."""
    beta, P, N, d, xi = 1.6, 4, 9, 2, 1.0
    x = rand_x(P, N, d, 13, scale=0.5)
    F, vb, _ = oracle.forces(x, beta, 1.0, 0.0, 0.5, xi, include_external=False)
    lam = 1.0 + 1e-6
    # homogeneity of exp(-beta V): V(lam x) at beta equals V(x) at spring constant lam^2 ks
    vb_scaled, _ = oracle.vb(lam * x, beta, xi)
    dV = (vb_scaled - oracle.vb(x / lam, beta, xi)[0]) / (lam - 1 / lam)
    assert -np.sum(x * F) == pytest.approx(dV, rel=1e-6)


# ---------------------------------------------------------------- pair / trap part
def test_pair_forces_newton_third_law_and_two_particle_closed_form(oracle):
    beta, omega, g, s = 1.0, 0.0, 0.8, 0.7
    P, N, d = 3, 5, 2
    x = rand_x(P, N, d, 17)
    F_all, _, _ = oracle.forces(x, beta, omega, g, s, 1.0)
    F_ex, _, _ = oracle.forces(x, beta, omega, g, s, 1.0, include_external=False)
    Fp = F_all - F_ex
    np.testing.assert_allclose(Fp.sum(axis=1), 0.0, atol=1e-14)  # per slice
    x2 = rand_x(2, 2, 2, 3)
    F2 = oracle.forces(x2, beta, 0.0, g, s, 1.0)[0] - oracle.forces(x2, beta, 0.0, g, s, 1.0, False)[0]
    for j in range(2):
        r = x2[j, 0] - x2[j, 1]
        f = (1.0 / 2) * (2 * g / s**2) * math.exp(-np.dot(r, r) / s**2) * r
        np.testing.assert_allclose(F2[j, 0], f, rtol=1e-13)
        np.testing.assert_allclose(F2[j, 1], -f, rtol=1e-13)
    # single-bead sampler agrees with the full routine
    Ft = oracle.forces(x, beta, 1.3, g, s, 1.0)[0] - F_ex
    for (j, l) in [(0, 0), (2, 4), (1, 2)]:
        np.testing.assert_allclose(oracle.external_force_on(x, 1.3, g, s, j, l), Ft[j, l], rtol=1e-12)


def test_g_zero_gives_trap_only(oracle):
    P, N, d = 4, 3, 3
    x = rand_x(P, N, d, 4)
    Fa = oracle.forces(x, 1.0, 1.5, 0.0, 0.5, 1.0)[0] - oracle.forces(x, 1.0, 1.5, 0.0, 0.5, 1.0, False)[0]
    np.testing.assert_allclose(Fa, -(1.5**2) * x / P, rtol=1e-12, atol=1e-13)
