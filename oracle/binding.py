"""ctypes marshalling for oracle/pimd_oracle.c (TEST INFRASTRUCTURE; no arithmetic here)."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pimd_oracle.c")
_LIB = os.path.join(_HERE, "libpimd_oracle.so")
_lock = threading.Lock()
_lib = None

NHC_M = 4


class OracleError(RuntimeError):
    pass


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C11, -O2, OpenMP on the pair loop only)."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(
                ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-o", tmp, _SRC, "-lm"]
            )
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.orc_cycle_energy_eq7.restype = C.c_double
    return _lib


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _x(x):
    x = np.ascontiguousarray(x, dtype=np.float64)
    if x.ndim != 3:
        raise ValueError("x must have shape [P][N][d]")
    P, N, d = x.shape
    return x, N, P, d


def _check(rc, what):
    if rc != 0:
        raise OracleError("%s failed with code %d" % (what, rc))


def eint(x, beta):
    x, N, P, d = _x(x)
    out = np.zeros(N)
    _check(_load().orc_eint(_dp(x), N, P, d, C.c_double(beta), _dp(out)), "orc_eint")
    return out


def cycle_energy_eq7(x, beta, u, v):
    x, N, P, d = _x(x)
    return float(_load().orc_cycle_energy_eq7(_dp(x), N, P, d, C.c_double(beta), int(u), int(v)))


def cycle_energies(x, beta):
    """E[u-1, v-1] = E^{[u,v]} (upper triangle)."""
    x, N, P, d = _x(x)
    out = np.zeros((N, N))
    _check(_load().orc_cycle_energies_d(_dp(x), N, P, d, C.c_double(beta), _dp(out)), "orc_cycle_energies")
    return out


def cycle_energies_eq10(x, beta):
    x, N, P, d = _x(x)
    out = np.zeros((N, N))
    _check(_load().orc_cycle_energies_eq10(_dp(x), N, P, d, C.c_double(beta), _dp(out)), "orc_cycle_energies_eq10")
    return out


def vb(x, beta, xi, tables=False):
    """V_xi^{[1,N]} and sign; with tables=True also V^{[1,n]} (n=0..N) and V^{[u,N]} (u=1..N+1)."""
    x, N, P, d = _x(x)
    v = C.c_double()
    s = C.c_int()
    if tables:
        fwd = np.zeros(N + 1)
        bwd = np.zeros(N + 2)
        _check(_load().orc_vb(_dp(x), N, P, d, C.c_double(beta), C.c_double(xi), C.byref(v), C.byref(s),
                              _dp(fwd), _dp(bwd)), "orc_vb")
        return v.value, s.value, fwd, bwd
    _check(_load().orc_vb(_dp(x), N, P, d, C.c_double(beta), C.c_double(xi), C.byref(v), C.byref(s),
                          None, None), "orc_vb")
    return v.value, s.value


def pr_matrix(x, beta, xi):
    x, N, P, d = _x(x)
    out = np.zeros((N, N))
    _check(_load().orc_pr_matrix(_dp(x), N, P, d, C.c_double(beta), C.c_double(xi), _dp(out)), "orc_pr_matrix")
    return out


def forces(x, beta, omega, g, s, xi, include_external=True):
    """F = -grad(V_xi^{[1,N]} + U/P), V_B, sign."""
    x, N, P, d = _x(x)
    F = np.zeros_like(x)
    v = C.c_double()
    sg = C.c_int()
    _check(_load().orc_forces(_dp(x), N, P, d, C.c_double(beta), C.c_double(omega), C.c_double(g), C.c_double(s),
                              C.c_double(xi), int(bool(include_external)), _dp(F), C.byref(v), C.byref(sg)),
           "orc_forces")
    return F, v.value, sg.value


def external_force_on(x, omega, g, s, j, l):
    x, N, P, d = _x(x)
    f = np.zeros(3)
    _check(_load().orc_external_force_on(_dp(x), N, P, d, C.c_double(omega), C.c_double(g), C.c_double(s),
                                         int(j), int(l), _dp(f)), "orc_external_force_on")
    return f[:d].copy()


def potential(x, beta, omega, g, s, xi):
    x, N, P, d = _x(x)
    phi = C.c_double()
    _check(_load().orc_potential(_dp(x), N, P, d, C.c_double(beta), C.c_double(omega), C.c_double(g),
                                 C.c_double(s), C.c_double(xi), C.byref(phi)), "orc_potential")
    return phi.value


def estimators(x, beta, omega, g, s, xi, nbins=0, rmax=1.0):
    x, N, P, d = _x(x)
    ep = C.c_double()
    ev = C.c_double()
    hist = np.zeros(max(nbins, 1))
    _check(_load().orc_estimators(_dp(x), N, P, d, C.c_double(beta), C.c_double(omega), C.c_double(g),
                                  C.c_double(s), C.c_double(xi), C.byref(ep), C.byref(ev), _dp(hist), int(nbins),
                                  C.c_double(rmax)), "orc_estimators")
    return ep.value, ev.value, hist[:nbins].copy()


def philox_raw(seed, dof, step):
    out = (C.c_uint32 * 4)()
    _load().orc_philox_raw(C.c_uint64(seed), C.c_uint64(dof), C.c_uint64(step), out)
    return [int(w) for w in out]


def philox_normal(seed, dof, step):
    out = (C.c_double * 2)()
    _load().orc_philox_normal(C.c_uint64(seed), C.c_uint64(dof), C.c_uint64(step), out)
    return float(out[0]), float(out[1])


def step(x, v, F, nhc, beta, omega, g, s, xi, dt, thermostat, gamma, seed, step0, nsteps):
    """Advance (x, v, F, nhc) in place by nsteps MD steps.  F must hold forces(x) on entry."""
    assert x.flags.c_contiguous and v.flags.c_contiguous and F.flags.c_contiguous
    assert x.dtype == np.float64 and v.dtype == np.float64 and F.dtype == np.float64
    P, N, d = x.shape
    if nhc is None:
        nhc = np.zeros((NHC_M, x.size))
    assert nhc.flags.c_contiguous and nhc.shape == (NHC_M, x.size)
    _check(_load().orc_step(_dp(x), _dp(v), _dp(F), _dp(nhc), N, P, d, C.c_double(beta), C.c_double(omega),
                            C.c_double(g), C.c_double(s), C.c_double(xi), C.c_double(dt), int(thermostat),
                            C.c_double(gamma), C.c_uint64(seed), C.c_uint64(step0), int(nsteps)), "orc_step")
    return nhc


def set_pair_potential(kind):
    """0: v = g exp(-r^2/s^2) (default), 1: v = g / sqrt(r^2 + s^2).  Global switch of the oracle library."""
    _load().orc_set_pair_potential(int(kind))


def conditioning(x, beta, xi):
    """kappa = max sum|terms| / |sum terms| over the signed sums of Eq. 6, 11, 12-14 (1 for xi >= 0)."""
    x, N, P, d = _x(x)
    k = C.c_double()
    _check(_load().orc_conditioning(_dp(x), N, P, d, C.c_double(beta), C.c_double(xi), C.byref(k)), "orc_conditioning")
    return k.value


def forces_species(x, beta, omega, g, s, xi, counts):
    x, N, P, d = _x(x)
    F = np.zeros_like(x)
    v, sg = C.c_double(), C.c_int()
    cnt = (C.c_int * len(counts))(*[int(c) for c in counts])
    _check(_load().orc_forces_species(_dp(x), N, P, d, C.c_double(beta), C.c_double(omega), C.c_double(g), C.c_double(s),
                                      C.c_double(xi), len(counts), cnt, _dp(F), C.byref(v), C.byref(sg)), "orc_forces_species")
    return F, v.value, sg.value


def estimators_species(x, beta, omega, g, s, xi, counts, nbins=0, rmax=1.0):
    x, N, P, d = _x(x)
    ep, ev = C.c_double(), C.c_double()
    hist = np.zeros(max(nbins, 1))
    cnt = (C.c_int * len(counts))(*[int(c) for c in counts])
    _check(_load().orc_estimators_species(_dp(x), N, P, d, C.c_double(beta), C.c_double(omega), C.c_double(g), C.c_double(s),
                                          C.c_double(xi), len(counts), cnt, C.byref(ep), C.byref(ev), _dp(hist), int(nbins),
                                          C.c_double(rmax)), "orc_estimators_species")
    return ep.value, ev.value, hist[:nbins].copy()


def pair_histogram(x, nbins, rmax):
    x, N, P, d = _x(x)
    hist = np.zeros(max(nbins, 1))
    _check(_load().orc_pair_histogram(_dp(x), N, P, d, _dp(hist), int(nbins), C.c_double(rmax)), "orc_pair_histogram")
    return hist[:nbins].copy()


def stream_forces_on(x, beta, omega, g, s, xi, particles, tables=False):
    """O(N)-memory evaluation: total force on every bead of the listed particles [k][P][d], V_B, sign
    (and V^{[1,n]}, V^{[u,N]} with tables=True)."""
    x, N, P, d = _x(x)
    ls = np.ascontiguousarray(particles, dtype=np.int32)
    F = np.zeros((len(ls), P, d))
    v, sg = C.c_double(), C.c_int()
    fwd = np.zeros(N + 1) if tables else None
    bwd = np.zeros(N + 2) if tables else None
    _check(_load().orc_stream_forces_on(_dp(x), N, P, d, C.c_double(beta), C.c_double(omega), C.c_double(g), C.c_double(s),
                                        C.c_double(xi), ls.ctypes.data_as(C.POINTER(C.c_int)), len(ls), _dp(F), C.byref(v),
                                        C.byref(sg), _dp(fwd) if tables else None, _dp(bwd) if tables else None),
           "orc_stream_forces_on")
    if tables:
        return F, v.value, sg.value, fwd, bwd
    return F, v.value, sg.value
