"""Exact canonical energy of N non-interacting xi-particles in an isotropic d-dimensional
harmonic trap AT FINITE P -- TEST INFRASTRUCTURE (pins ensemble energies; north_star:
"exact canonical energy of non-interacting bosons in a harmonic trap (partition-function
recursion)").

Derivation (hbar = m = 1).  A cycle that threads k particles is one ring polymer of
n = kP beads (Eq. 7) with spring constant k_s = P/beta^2 and the
trap entering as U/P (Eq. 4).  Per dimension its configurational integral with
the prefactor of Eq. 4 is Gaussian:

    z = (P/(2 pi beta))^{n/2} Int d^n x exp(-1/2 x^T (beta A) x),
    beta A = (P/beta) [ Lap_n + a^2 I ],   a = beta omega / P,

Lap_n the Laplacian of the n-cycle with eigenvalues 4 sin^2(pi m/n).  Hence
z = det(Lap_n + a^2)^{-1/2} and, with a = 2 sinh(theta/2),
prod_m (4 sin^2(pi m/n) + a^2) = (2 sinh(n theta/2))^2, so

    z_P(k) = [2 sinh(k P theta/2)]^{-d},   theta = 2 asinh(beta omega/(2P)),
    e_k = -d ln z_P(k)/d beta = d (k omega/2) coth(k P theta/2) / cosh(theta/2).

The recursion of Eq. 6, integrated over coordinates, is the canonical recursion
    Z_0 = 1,  Z_n = (1/n) sum_{k=1}^{n} xi^{k-1} z_P(k) Z_{n-k},
    E_n = sum_k w_k (e_k + E_{n-k}) / sum_k w_k,   w_k = xi^{k-1} z_P(k) Z_{n-k}.
P -> infinity gives the textbook z(k) = [2 sinh(k beta omega/2)]^{-d}.

Pins (tests/test_oracle_ideal_gas.py): numerical determinant of the spring+trap matrix,
N = 1 and N = 2 closed forms, -d ln Z/d beta by finite differences, the P -> infinity limit.
"""
from __future__ import annotations

import math

import numpy as np


def theta(beta: float, omega: float, P: int | None) -> float:
    if P is None:  # P -> infinity
        return float("nan")
    return 2.0 * math.asinh(beta * omega / (2.0 * P))


def log_z_cycle(k, beta, omega, d, P):
    """ln z_P(k) for k (array ok)."""
    k = np.asarray(k, dtype=np.float64)
    a = k * beta * omega if P is None else k * P * theta(beta, omega, P)  # = 2 * (argument of sinh)
    # ln(2 sinh(a/2)) = a/2 + ln(1 - e^{-a})
    return -d * (0.5 * a + np.log1p(-np.exp(-a)))


def e_cycle(k, beta, omega, d, P):
    """-d ln z_P(k) / d beta."""
    k = np.asarray(k, dtype=np.float64)
    if P is None:
        a = k * beta * omega
        return d * 0.5 * k * omega / np.tanh(0.5 * a)
    th = theta(beta, omega, P)
    return d * 0.5 * k * omega / np.tanh(0.5 * k * P * th) / math.cosh(0.5 * th)


def log_Z_and_energy(N: int, beta: float, omega: float, d: int, xi: float, P: int | None):
    """Returns (ln|Z_n|, sign Z_n, E_n) for n = 0..N."""
    ks = np.arange(1, N + 1)
    lz = log_z_cycle(ks, beta, omega, d, P)
    ek = e_cycle(ks, beta, omega, d, P)
    lam = math.log(abs(xi)) if xi != 0 else 0.0
    sx = -1.0 if xi < 0 else 1.0
    logZ = np.zeros(N + 1)
    sgZ = np.ones(N + 1)
    E = np.zeros(N + 1)
    for n in range(1, N + 1):
        kk = 1 if xi == 0 else n
        k = ks[:kk]
        t = (k - 1) * lam + lz[:kk] + logZ[n - k]
        sg = np.where((k - 1) % 2 == 1, sx, 1.0) * sgZ[n - k]
        m = t.max()
        w = sg * np.exp(t - m)
        den = w.sum()
        logZ[n] = -math.log(n) + m + math.log(abs(den))
        sgZ[n] = 1.0 if den > 0 else -1.0
        E[n] = float((w * (ek[:kk] + E[n - k])).sum() / den)
    return logZ, sgZ, E


def exact_energy(N: int, beta: float, omega: float = 1.0, d: int = 2, xi: float = 1.0, P: int | None = None) -> float:
    """<E> of the ensemble sampled by Eq. 4 at N, beta, P (P=None: P -> infinity)."""
    return float(log_Z_and_energy(N, beta, omega, d, xi, P)[2][N])
