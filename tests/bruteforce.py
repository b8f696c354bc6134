"""Brute-force definitions written out in NumPy/pure Python for tiny inputs.

These are the pins of the oracle: they restate the DEFINITIONS of the paper (Eq. 2, 4, 6, 7)
without any of the oracle's code.  x has layout [P][N][d]; particle/bead indices below are 0-based.
"""
from __future__ import annotations

import itertools
import math

import numpy as np


def ks_of(P, beta):
    # m omega_P^2 with omega_P = sqrt(P)/(beta hbar)
    return P / beta**2


def ring_energy_of_permutation(x, beta, sigma):
    """Spring energy of the ring-polymer configuration in which bead P of particle l is tied to
    bead 1 of particle sigma[l] (the kinetic action of <p{r}|e^{-beta H}|{r}>, Eq. 2 / Eq. 7)."""
    P, N, d = x.shape
    e = 0.0
    for l in range(N):
        for j in range(P):
            nxt = x[j + 1, l] if j + 1 < P else x[0, sigma[l]]
            e += float(np.sum((nxt - x[j, l]) ** 2))
    return 0.5 * ks_of(P, beta) * e


def n_cycles(sigma):
    seen = [False] * len(sigma)
    c = 0
    for i in range(len(sigma)):
        if not seen[i]:
            c += 1
            k = i
            while not seen[k]:
                seen[k] = True
                k = sigma[k]
    return c


def permutation_sum(x, beta, xi):
    """(1/N!) sum_{p in S_N} xi^{N_p} exp(-beta E_p), N_p = N - #cycles(p)  (Eq. 2)."""
    P, N, d = x.shape
    tot = 0.0
    for sigma in itertools.permutations(range(N)):
        npow = N - n_cycles(sigma)
        w = 1.0 if npow == 0 else xi**npow  # 0^0 = 1
        tot += w * math.exp(-beta * ring_energy_of_permutation(x, beta, sigma))
    return tot / math.factorial(N)


def cycle_energy_eq7(x, beta, u, v):
    """Eq. 7 literally, 1-based u <= v."""
    P, N, d = x.shape
    e = 0.0
    for l in range(u, v + 1):
        for j in range(1, P + 1):
            a = x[j - 1, l - 1]
            if j < P:
                b = x[j, l - 1]
            elif l < v:
                b = x[0, l]
            else:
                b = x[0, u - 1]
            e += float(np.sum((b - a) ** 2))
    return 0.5 * ks_of(P, beta) * e


def composition_sum(x, beta, xi):
    """Unrolled Eq. 6: W_N = sum over cuts of 1..N into runs [u,v] of consecutive indices,
    each run weighted xi^{v-u} / v * exp(-beta E^{[u,v]})."""
    P, N, d = x.shape
    E = {(u, v): cycle_energy_eq7(x, beta, u, v) for u in range(1, N + 1) for v in range(u, N + 1)}
    tot = 0.0
    for cuts in itertools.product([0, 1], repeat=N - 1):
        # cuts[i] == 1: a run ends after particle i+1
        w = 1.0
        u = 1
        for v in range(1, N + 1):
            if v == N or cuts[v - 1]:
                k = v - u
                w *= (1.0 if k == 0 else xi**k) / v * math.exp(-beta * E[(u, v)])
                u = v + 1
        tot += w
    return tot


def potential_external(x, omega, g, s):
    """U/P of Eq. 4/5/18-20 with v(r) = g exp(-r^2/s^2)."""
    P, N, d = x.shape
    u = 0.5 * omega**2 * float(np.sum(x**2))
    if g != 0.0:
        for j in range(P):
            diff = x[j][:, None, :] - x[j][None, :, :]
            r2 = np.sum(diff**2, axis=-1)
            iu = np.triu_indices(N, 1)
            u += g * float(np.sum(np.exp(-r2[iu] / s**2)))
    return u / P
