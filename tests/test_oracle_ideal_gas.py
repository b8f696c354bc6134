"""Pins of oracle/ideal_gas.py (exact finite-P canonical energy of trapped ideal xi-particles)."""
import math

import numpy as np
import pytest

from oracle import ideal_gas as ig


@pytest.mark.parametrize("n,P,beta,omega", [(3, 3, 1.0, 1.0), (8, 4, 2.0, 0.7), (32, 16, 3.0, 1.0)])
def test_single_cycle_partition_function_against_determinant(n, P, beta, omega):
    """z = (P/2 pi beta)^{n/2} Int exp(-beta[1/2 k_s sum (x_{i+1}-x_i)^2 + (omega^2/2P) sum x_i^2])
    evaluated as a Gaussian integral with the explicit n x n matrix; n = kP beads, one dimension."""
    assert n % P == 0
    k = n // P
    ks = P / beta**2
    A = np.zeros((n, n))
    for i in range(n):
        A[i, i] += 2 * ks + omega**2 / P
        A[i, (i + 1) % n] -= ks
        A[(i + 1) % n, i] -= ks
    sign, logdet = np.linalg.slogdet(beta * A)
    assert sign > 0
    log_z = 0.5 * n * math.log(P / (2 * math.pi * beta)) + 0.5 * n * math.log(2 * math.pi) - 0.5 * logdet
    assert float(ig.log_z_cycle(k, beta, omega, 1, P)) == pytest.approx(log_z, rel=1e-11, abs=1e-11)


def test_single_particle_limits():
    beta, omega, d = 2.0, 1.3, 2
    # P -> infinity: textbook harmonic oscillator, E = d (omega/2) coth(beta omega/2)
    assert ig.exact_energy(1, beta, omega, d, 1.0, None) == pytest.approx(d * 0.5 * omega / math.tanh(0.5 * beta * omega))
    # finite P converges to it as 1/P^2
    e = [ig.exact_energy(1, beta, omega, d, 1.0, P) for P in (50, 100, 200)]
    inf = ig.exact_energy(1, beta, omega, d, 1.0, None)
    assert (inf - e[0]) / (inf - e[1]) == pytest.approx(4.0, rel=2e-2)
    assert (inf - e[1]) / (inf - e[2]) == pytest.approx(4.0, rel=2e-2)


@pytest.mark.parametrize("xi", [1.0, 0.5, 0.0, -0.3, -1.0])
@pytest.mark.parametrize("P", [None, 4, 16])
def test_energy_is_minus_dlnZ_dbeta(xi, P):
    N, beta, omega, d = 6, 1.5, 1.0, 2
    h = 1e-5
    lp = ig.log_Z_and_energy(N, beta + h, omega, d, xi, P)[0][N]
    lm = ig.log_Z_and_energy(N, beta - h, omega, d, xi, P)[0][N]
    assert ig.exact_energy(N, beta, omega, d, xi, P) == pytest.approx(-(lp - lm) / (2 * h),
                                                                         rel=1e-8 if xi >= 0 else 1e-6)


def test_two_bosons_closed_form():
    beta, omega, d = 1.2, 1.0, 2

    def z(b):
        return (2 * math.sinh(0.5 * b * omega)) ** (-d)

    def lnZ2(b, xi):
        return math.log(0.5 * (z(b) ** 2 + xi * z(2 * b)))

    for xi in (1.0, -1.0, 0.3):
        h = 1e-5
        ref = -(lnZ2(beta + h, xi) - lnZ2(beta - h, xi)) / (2 * h)
        assert ig.exact_energy(2, beta, omega, d, xi, None) == pytest.approx(ref, rel=1e-8)


def test_ground_state_limit():
    """T -> 0 bosons: E -> N d omega/2 (the paper's E = N for d=2)."""
    assert ig.exact_energy(50, 12.0, 1.0, 2, 1.0, None) == pytest.approx(50.0, rel=1e-4)


def test_values_listed_in_survey_appendix_b():
    """Cross-check against the values the survey computed independently."""
    assert ig.exact_energy(4, 2.0, 1.0, 2, 1.0, 16) == pytest.approx(4.453587907135, rel=1e-11)
    assert ig.exact_energy(4, 2.0, 1.0, 2, 0.0, 16) == pytest.approx(5.243793218385, rel=1e-11)
    assert ig.exact_energy(4, 2.0, 1.0, 2, -0.5, 16) == pytest.approx(6.921426682, rel=1e-9)
    assert ig.exact_energy(3, 2.0, 1.0, 2, 0.5, 4) == pytest.approx(3.524198509, rel=1e-9)
    assert ig.exact_energy(2500, 3.0, 1.0, 2, 1.0, 16) == pytest.approx(2489.206984742, rel=1e-11)
    assert ig.exact_energy(100, 3.0, 1.0, 2, 1.0, 32) == pytest.approx(100.011658, rel=1e-7)
