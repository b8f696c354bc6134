"""Pins of the oracle's estimators, random numbers and dynamics (CPU only)."""
import math

import numpy as np
import pytest

from oracle import ideal_gas as ig
from paper_2404_02628_b200 import workloads as wl
from tests import bruteforce as bf


def rand_x(P, N, d, seed, scale=0.6):
    return np.random.default_rng(seed).normal(0.0, scale, size=(P, N, d))


# ---------------------------------------------------------------- random numbers
def test_philox4x32_10_known_answers(oracle):
    """Known-answer vectors of Philox4x32-10 (Salmon et al. SC'11; Random123 kat_vectors)."""
    assert oracle.philox_raw(0, 0, 0) == [0x6627E8D5, 0xE169C58D, 0xBC57AC4C, 0x9B00DBD8]
    ones = 2**64 - 1
    assert oracle.philox_raw(ones, ones, ones) == [0x408F276D, 0x41C83B0E, 0xA20BC7C6, 0x6D5451FD]
    seed = (0x299F31D0 << 32) | 0xA4093822
    dof = (0x85A308D3 << 32) | 0x243F6A88
    step = (0x03707344 << 32) | 0x13198A2E
    assert oracle.philox_raw(seed, dof, step) == [0xD16CFE09, 0x94FDCCEB, 0x5001E420, 0x24126EA1]


def test_philox_normals_follow_the_documented_map(oracle):
    w = oracle.philox_raw(12345, 678, 9)
    u1 = (((w[0] << 32) | w[1]) >> 11) * 2.0**-53 + 2.0**-54
    u2 = (((w[2] << 32) | w[3]) >> 11) * 2.0**-53 + 2.0**-54
    r = math.sqrt(-2 * math.log(u1))
    z0, z1 = oracle.philox_normal(12345, 678, 9)
    assert z0 == pytest.approx(r * math.cos(2 * math.pi * u2), rel=1e-13, abs=1e-15)
    assert z1 == pytest.approx(r * math.sin(2 * math.pi * u2), rel=1e-13, abs=1e-15)
    z = np.array([oracle.philox_normal(7, i, 3) for i in range(20000)]).ravel()
    assert abs(z.mean()) < 4 / math.sqrt(z.size)
    assert z.var() == pytest.approx(1.0, abs=4 * math.sqrt(2.0 / z.size))
    assert np.mean(z**4) == pytest.approx(3.0, abs=0.2)


# ---------------------------------------------------------------- estimators
@pytest.mark.parametrize("xi", [1.0, 0.5, 0.0, -0.3])
def test_primitive_estimator_is_beta_derivative(oracle, xi):
    """E_prim - PdN/(2 beta) - Ubar = d(beta V_xi^{[1,N]})/d beta at fixed coordinates
    (E = -d ln Z/d beta applied to Eq. 4; k_s = P/beta^2 carries the beta dependence)."""
    P, N, d, beta, omega, g, s = 4, 7, 2, 1.3, 0.8, 0.6, 0.7
    x = rand_x(P, N, d, 99, scale=0.5)
    ep, ev, _ = oracle.estimators(x, beta, omega, g, s, xi)
    h = 1e-6
    fp = (beta + h) * oracle.vb(x, beta + h, xi)[0]
    fm = (beta - h) * oracle.vb(x, beta - h, xi)[0]
    ubar = bf.potential_external(x, omega, g, s)
    assert ep - P * d * N / (2 * beta) - ubar == pytest.approx((fp - fm) / (2 * h), rel=1e-7, abs=1e-7)


def test_primitive_estimator_equals_probability_weighted_springs(oracle):
    """eps^{(N)} = -( sum_l E_int^{(l)} + sum_{l,l'} Pr[G(l)=l'] C(l,l') )  (R9)."""
    P, N, d, beta = 5, 11, 2, 1.7
    x = rand_x(P, N, d, 5, scale=0.5)
    ks = bf.ks_of(P, beta)
    for xi in (1.0, 0.4, -0.3):
        ep, _, _ = oracle.estimators(x, beta, 0.0, 0.0, 0.5, xi)
        Pr = oracle.pr_matrix(x, beta, xi)
        Cm = 0.5 * ks * np.sum((x[P - 1][:, None, :] - x[0][None, :, :]) ** 2, axis=-1)
        e_c = oracle.eint(x, beta).sum() + np.sum(Pr * Cm)
        assert ep - P * d * N / (2 * beta) == pytest.approx(-e_c, rel=1e-11)


def test_virial_estimator_and_histogram(oracle):
    P, N, d, beta, omega, g, s = 3, 6, 2, 1.0, 1.1, 0.9, 0.6
    x = rand_x(P, N, d, 12, scale=0.8)
    _, ev, hist = oracle.estimators(x, beta, omega, g, s, 1.0, nbins=16, rmax=2.0)
    # E_vir = Ubar + 1/2 sum r . grad Ubar, gradient by finite differences of the brute-force Ubar
    h = 1e-6
    grad = np.zeros_like(x)
    for idx in np.ndindex(*x.shape):
        xp = x.copy(); xp[idx] += h
        xm = x.copy(); xm[idx] -= h
        grad[idx] = (bf.potential_external(xp, omega, g, s) - bf.potential_external(xm, omega, g, s)) / (2 * h)
    assert ev == pytest.approx(bf.potential_external(x, omega, g, s) + 0.5 * np.sum(x * grad), rel=1e-8)
    r = np.sqrt(np.sum(x**2, axis=-1)).ravel()
    ref, _ = np.histogram(r, bins=16, range=(0.0, 2.0))
    ref[-1] -= np.sum(r == 2.0)
    np.testing.assert_array_equal(hist, ref)


# ---------------------------------------------------------------- dynamics
def _forces(oracle, w, x):
    return oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)[0]


def test_nve_is_time_reversible_and_conserves_energy(oracle):
    w = wl.custom(N=5, P=4, d=2, beta=1.5, g=0.5, s=0.6, xi=1.0, dt=0.002, sigma=0.5)
    x0, v0 = wl.make_state(w, 1)

    def energy(x, v):
        return 0.5 * np.sum(v**2) + oracle.potential(x, w.beta, w.omega, w.g, w.s, w.xi)

    drift = []
    for dt in (0.004, 0.002):
        x, v = x0.copy(), v0.copy()
        F = _forces(oracle, w, x)
        e0 = energy(x, v)
        oracle.step(x, v, F, None, w.beta, w.omega, w.g, w.s, w.xi, dt, 0, 1.0, 0, 0, int(round(0.4 / dt)))
        drift.append(abs(energy(x, v) - e0))
        if dt == 0.002:
            v *= -1.0
            oracle.step(x, v, F, None, w.beta, w.omega, w.g, w.s, w.xi, dt, 0, 1.0, 0, 0, int(round(0.4 / dt)))
            np.testing.assert_allclose(x, x0, atol=1e-11)
            np.testing.assert_allclose(-v, v0, atol=1e-11)
    assert drift[0] < 2e-3 * abs(e0)
    assert drift[1] < 0.5 * drift[0]  # O(dt^2): halving dt must at least halve the error


def _ensemble(oracle, w, thermostat, nsteps, every, seed, gamma=1.0, nequil=2000):
    x, v = wl.make_state(w, seed)
    F = _forces(oracle, w, x)
    nhc = None
    if thermostat == 2:
        nhc = np.random.default_rng(seed + 1).normal(0.0, math.sqrt(w.P / w.beta**2), size=(4, x.size))
    nhc = oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat, gamma, seed, 0, nequil)
    ep, ev, v2 = [], [], []
    done = nequil
    while done < nequil + nsteps:
        oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat, gamma, seed, done, every)
        done += every
        a, b, _ = oracle.estimators(x, w.beta, w.omega, w.g, w.s, w.xi)
        ep.append(a); ev.append(b); v2.append(np.mean(v**2))
    return np.array(ep), np.array(ev), np.array(v2)


def _mean_se(a, nblocks=20):
    b = a[: len(a) // nblocks * nblocks].reshape(nblocks, -1).mean(axis=1)
    return b.mean(), b.std(ddof=1) / math.sqrt(nblocks)


@pytest.mark.parametrize("xi,thermostat", [(1.0, 1), (0.0, 1), (1.0, 2)])
def test_ensemble_energy_matches_exact_ideal_gas(oracle, xi, thermostat):
    """N=3, P=4, beta=2, d=2 ideal trapped xi-particles: both estimators agree with the exact
    finite-P canonical energy within 3 standard errors, and <v^2> = 1/beta (R6)."""
    w = wl.custom(N=3, P=4, d=2, beta=2.0, g=0.0, xi=xi, dt=0.05, sigma=0.7)
    ep, ev, v2 = _ensemble(oracle, w, thermostat, nsteps=120000, every=4, seed=3)
    exact = ig.exact_energy(w.N, w.beta, w.omega, w.d, xi, w.P)
    for est in (ep, ev):
        m, se = _mean_se(est)
        assert se < 0.03 * exact
        # dt = 0.05 carries an O(dt^2) integrator bias of a few 1e-3; allow it beside 3 SE
        assert abs(m - exact) < 3 * se + 0.004 * exact
    m, se = _mean_se(v2)
    assert abs(m - 1.0 / w.beta) < 3 * se + 0.004 / w.beta


def test_ensemble_primitive_equals_virial_with_interaction(oracle):
    w = wl.custom(N=3, P=4, d=2, beta=2.0, g=0.5, s=0.5, xi=1.0, dt=0.05, sigma=0.7)
    ep, ev, _ = _ensemble(oracle, w, 1, nsteps=120000, every=4, seed=11)
    m, se = _mean_se(ep - ev)
    assert abs(m) < 3 * se + 0.01
    assert _mean_se(ep)[0] > ig.exact_energy(3, 2.0, 1.0, 2, 1.0, 4)  # repulsion raises the energy


# ---------------------------------------------------------------- Nose-Hoover chain pins
def _nhc_case():
    w = wl.custom(N=4, P=4, d=2, beta=1.5, g=0.4, s=0.6, xi=1.0, dt=0.002, sigma=0.5)
    x0, v0 = wl.make_state(w, 5)
    # chain velocities of thermal size, sqrt(kT/Q) = sqrt(P)/beta, all four links excited so that every coupling acts
    nhc0 = np.random.default_rng(6).normal(0.0, math.sqrt(w.P) / w.beta, size=(4, x0.size))
    return w, x0, v0, nhc0


def test_nhc_is_time_reversible(oracle):
    """The chain update is a symmetric product of exact sub-flows, each of which commutes with (v, v_xi) -> (-v, -v_xi)
    up to inversion, so n steps, a sign flip of the particle AND the chain velocities, and n more steps must lead back to
    the start (x, -v, -v_xi) to rounding.  This pins the structure of every link: a force G_k that depended on the link it
    drives (e.g. vx[k] for vx[k-1] in G, checked by hand on a mutated copy of the oracle: the return error rises from
    3e-14 to 2e-2), an update order that is not palindromic, or unequal scaling factors on the two sides of a kick are no
    longer self-inverse under the flip and miss the start at O(dt^2) per step."""
    w, x0, v0, nhc0 = _nhc_case()
    x, v, nhc = x0.copy(), v0.copy(), nhc0.copy()
    F = _forces(oracle, w, x)
    n = 150
    oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, 2, 1.0, 0, 0, n)
    assert np.max(np.abs(x - x0)) > 1e-3  # it moved
    v *= -1.0
    nhc *= -1.0
    oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, 2, 1.0, 0, 0, n)
    np.testing.assert_allclose(x, x0, atol=1e-10)
    np.testing.assert_allclose(-v, v0, atol=1e-10)
    np.testing.assert_allclose(-nhc, nhc0, atol=1e-10)


def test_nhc_conserves_the_extended_energy(oracle):
    """Nose-Hoover chain dynamics conserve H' = 1/2 sum v^2 + Phi(x) + sum_dof sum_k (1/2 Q v_xi_k^2 + kT xi_k) with
    d xi_k/dt = v_xi_k (Martyna, Klein, Tuckerman; the paper's refs at PAPER.md:299-303).  The oracle carries only the chain
    velocities, so the thermostat positions are integrated here from the velocities it returns after every step
    (trapezoid rule, O(dt^2) like the integrator).  H' must stay put to O(dt^2) -- the drift at dt/2 is about a quarter --
    while each of its parts moves by far more.  A wrong factor in a kick (h/2), in a scaling (h/4 twice) or in the particle
    scaling (h), or a G_k built from the wrong link or with a wrong Q, breaks the cancellation between neighbouring links
    and gives an O(1) drift that does not shrink with dt (checked on mutated copies of the oracle: 0.25 -> 0.5 in the
    scaling gives a drift of 14.6, 0.5 -> 0.25 in a kick 1.2, h -> h/2 in the particle scaling 2.4, vx[k-1] -> vx[k] in G
    7.2, against 7e-5 at dt = 0.004 and 1.8e-5 at dt = 0.002 for the oracle as it stands)."""
    w, x0, v0, nhc0 = _nhc_case()
    kT, Q = 1.0 / w.beta, w.beta / w.P

    def run(dt, T=0.3):
        x, v, nhc = x0.copy(), v0.copy(), nhc0.copy()
        F = _forces(oracle, w, x)
        xi_sum = 0.0  # sum over dof and links of xi_k
        def parts():
            return (0.5 * np.sum(v**2), oracle.potential(x, w.beta, w.omega, w.g, w.s, w.xi), 0.5 * Q * np.sum(nhc**2), kT * xi_sum)
        p0 = parts()
        worst, swing = 0.0, 0.0
        for it in range(int(round(T / dt))):
            before = nhc.sum()
            oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, dt, 2, 1.0, 0, it, 1)
            xi_sum += 0.5 * dt * (before + nhc.sum())
            p = parts()
            worst = max(worst, abs(sum(p) - sum(p0)))
            swing = max(swing, max(abs(a - b) for a, b in zip(p, p0)))
        return worst, swing

    d1, swing = run(0.004)
    d2, _ = run(0.002)
    assert swing > 1.0            # energy does flow between particles, potential and chains ...
    assert d1 < 2e-3 * swing      # ... while the sum stays put
    assert d2 < 0.35 * d1         # O(dt^2)
