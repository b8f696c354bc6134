"""Thin ctypes binding of libpimd.so (include/pimd.h).  Argument marshalling only.

PyTorch supplies device memory (tensors whose data_ptr() is handed to the library) and the CUDA
stream; every step of the hot path runs inside the library's kernels.  There is no CPU fallback:
loading fails loudly if libpimd.so is missing, and pimd_create fails without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpimd.so")

OK, EINVAL, ENOMEM, ECUDA, ENUMERIC = 0, -1, -2, -3, -4
THERMOSTAT_NVE, THERMOSTAT_LANGEVIN, THERMOSTAT_NHC = 0, 1, 2
NHC_LENGTH = 4
PROF_SLOTS = ("bead", "prep", "chain", "forcepass", "assemble", "finalize", "integrate", "combine", "pair", "chain_fallback", "emat", "prmat")

# every symbol include/pimd.h declares: (restype, argtypes)
_dp = C.POINTER(C.c_double)
_SYMBOLS = {
    "pimd_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                              C.c_double, C.c_double, C.c_double, C.c_int, C.c_uint64]),
    "pimd_destroy": (C.c_int, [C.c_void_p]),
    "pimd_set_stream": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_workspace_bytes": (C.c_size_t, [C.c_void_p]),
    "pimd_set_workspace": (C.c_int, [C.c_void_p, C.c_void_p, C.c_size_t]),
    "pimd_set_gamma": (C.c_int, [C.c_void_p, C.c_double]),
    "pimd_set_concurrency": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_get_state": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_set_state_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_get_state_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_get_step_count": (C.c_int, [C.c_void_p, C.POINTER(C.c_uint64)]),
    "pimd_set_step_count": (C.c_int, [C.c_void_p, C.c_uint64]),
    "pimd_get_nhc": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_set_nhc": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_forces": (C.c_int, [C.c_void_p, C.c_void_p, _dp, C.POINTER(C.c_int)]),
    "pimd_forces_host": (C.c_int, [C.c_void_p, C.c_void_p, _dp, C.POINTER(C.c_int)]),
    "pimd_get_forces": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_forces_host": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_set_forces": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_set_forces_host": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_tables": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_cycle_energies": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_connection_probabilities": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_step": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_estimators": (C.c_int, [C.c_void_p, _dp, _dp, C.c_void_p, C.c_int, C.c_double]),
    "pimd_launch_count": (C.c_uint64, [C.c_void_p]),
    "pimd_set_profiling": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_get_profile": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_get_chain_phases": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_selftest_exp": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_size_t]),
    "pimd_probe_fp64_peak": (C.c_int, [C.c_void_p, _dp]),
    "pimd_last_error": (C.c_char_p, [C.c_void_p]),
    "pimd_version": (C.c_char_p, []),
}
EXPORTED_SYMBOLS = tuple(_SYMBOLS)

_lib = None


class PimdError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libpimd error %d: %s" % (code, msg))
        self.code = code


def load():
    """dlopen libpimd.so and declare the prototypes.  Raises if the library is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(
                "%s is missing: build it with `python -m paper_2404_02628_b200.build` "
                "(the hot path has no CPU fallback)" % LIB_PATH)
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in _SYMBOLS.items():
            fn = getattr(lib, name)  # AttributeError if a declared symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def _ptr(t):
    """Device/host pointer of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return C.c_void_p(t.data_ptr())
    return C.c_void_p(t.ctypes.data)


class Pimd:
    """One simulation handle.  Method names mirror the C entry points (pimd_<name>)."""

    def __init__(self, N, P, d, beta, omega, g, s, xi, dt, thermostat=THERMOSTAT_LANGEVIN, seed=0,
                 stream=None, use_torch_workspace=True):
        self._lib = load()
        self._h = C.c_void_p()
        self.N, self.P, self.d = int(N), int(P), int(d)
        rc = self._lib.pimd_create(C.byref(self._h), int(N), int(P), int(d), float(beta), float(omega), float(g),
                                   float(s), float(xi), float(dt), int(thermostat), int(seed))
        if rc != OK:
            raise PimdError(rc, self._lib.pimd_last_error(None).decode())
        self._ws = None
        import torch  # device memory and streams only

        self._torch = torch
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        self._check(self._lib.pimd_set_stream(self._h, C.c_void_p(stream)))
        if use_torch_workspace:
            nbytes = self._lib.pimd_workspace_bytes(self._h)
            self._ws = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
            base = (self._ws.data_ptr() + 255) // 256 * 256
            self._check(self._lib.pimd_set_workspace(self._h, C.c_void_p(base), nbytes))

    # -- plumbing
    def _check(self, rc):
        if rc != OK:
            raise PimdError(rc, self._lib.pimd_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            self._lib.pimd_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _empty_state(self):
        return self._torch.empty((self.P, self.N, self.d), dtype=self._torch.float64, device="cuda")

    # -- C ABI mirrors
    def set_stream(self, cuda_stream):
        self._check(self._lib.pimd_set_stream(self._h, C.c_void_p(cuda_stream)))

    def set_gamma(self, gamma):
        self._check(self._lib.pimd_set_gamma(self._h, float(gamma)))

    def set_concurrency(self, on):
        self._check(self._lib.pimd_set_concurrency(self._h, int(bool(on))))

    def set_state(self, x_dev, v_dev=None):
        self._check(self._lib.pimd_set_state(self._h, _ptr(x_dev), _ptr(v_dev)))

    def get_state(self, want_v=True):
        x = self._empty_state()
        v = self._empty_state() if want_v else None
        self._check(self._lib.pimd_get_state(self._h, _ptr(x), _ptr(v)))
        return x, v

    def set_state_host(self, x_host, v_host=None):
        self._check(self._lib.pimd_set_state_host(self._h, _ptr(x_host), _ptr(v_host)))

    def get_state_host(self, x_host, v_host=None):
        self._check(self._lib.pimd_get_state_host(self._h, _ptr(x_host), _ptr(v_host)))

    def get_step_count(self):
        out = C.c_uint64()
        self._check(self._lib.pimd_get_step_count(self._h, C.byref(out)))
        return out.value

    def set_step_count(self, step):
        self._check(self._lib.pimd_set_step_count(self._h, int(step)))

    def get_nhc(self):
        t = self._torch.empty((NHC_LENGTH, self.P * self.N * self.d), dtype=self._torch.float64, device="cuda")
        self._check(self._lib.pimd_get_nhc(self._h, _ptr(t)))
        return t

    def set_nhc(self, nhc_dev):
        self._check(self._lib.pimd_set_nhc(self._h, _ptr(nhc_dev)))

    def forces(self, out=None, want_forces=True):
        """(F [P][N][d] device tensor or None, V_B, sign)."""
        f = None
        if want_forces:
            f = out if out is not None else self._empty_state()
        vb, sg = C.c_double(), C.c_int()
        self._check(self._lib.pimd_forces(self._h, _ptr(f), C.byref(vb), C.byref(sg)))
        return f, vb.value, sg.value

    def forces_host(self, f_host):
        vb, sg = C.c_double(), C.c_int()
        self._check(self._lib.pimd_forces_host(self._h, _ptr(f_host), C.byref(vb), C.byref(sg)))
        return vb.value, sg.value

    def get_forces(self, out=None):
        f = out if out is not None else self._empty_state()
        self._check(self._lib.pimd_get_forces(self._h, _ptr(f)))
        return f

    def get_forces_host(self, f_host):
        self._check(self._lib.pimd_get_forces_host(self._h, _ptr(f_host)))

    def set_forces(self, f_dev):
        self._check(self._lib.pimd_set_forces(self._h, _ptr(f_dev)))

    def set_forces_host(self, f_host):
        self._check(self._lib.pimd_set_forces_host(self._h, _ptr(f_host)))

    def get_tables(self):
        import numpy as np

        vf, vb, pn = np.zeros(self.N + 1), np.zeros(self.N + 2), np.zeros(self.N)
        self._check(self._lib.pimd_get_tables(self._h, _ptr(vf), _ptr(vb), _ptr(pn)))
        return vf, vb, pn

    def get_pnext(self):
        import numpy as np

        pn = np.zeros(self.N)
        self._check(self._lib.pimd_get_tables(self._h, None, None, _ptr(pn)))
        return pn

    def cycle_energies(self, out=None):
        """E[u, v] = E^{[u+1,v+1]} (u <= v), device tensor [N][N]."""
        e = out if out is not None else self._torch.empty((self.N, self.N), dtype=self._torch.float64, device="cuda")
        self._check(self._lib.pimd_cycle_energies(self._h, _ptr(e)))
        return e

    def connection_probabilities(self, out=None):
        """Pr[l, m] = Pr[G(l+1) = m+1], device tensor [N][N]."""
        pr = out if out is not None else self._torch.empty((self.N, self.N), dtype=self._torch.float64, device="cuda")
        self._check(self._lib.pimd_connection_probabilities(self._h, _ptr(pr)))
        return pr

    def step(self, nsteps=1):
        self._check(self._lib.pimd_step(self._h, int(nsteps)))

    def estimators(self, nbins=0, rmax=1.0):
        import numpy as np

        ep, ev = C.c_double(), C.c_double()
        hist = np.zeros(max(int(nbins), 1))
        self._check(self._lib.pimd_estimators(self._h, C.byref(ep), C.byref(ev), _ptr(hist), int(nbins), float(rmax)))
        return ep.value, ev.value, hist[: int(nbins)].copy()

    def set_profiling(self, on):
        self._check(self._lib.pimd_set_profiling(self._h, int(bool(on))))

    def get_profile(self):
        """{slot name: (total ms, launches)} since the previous call."""
        ms = (C.c_double * len(PROF_SLOTS))()
        cnt = (C.c_uint64 * len(PROF_SLOTS))()
        self._check(self._lib.pimd_get_profile(self._h, ms, cnt))
        return {name: (float(ms[i]), int(cnt[i])) for i, name in enumerate(PROF_SLOTS)}

    def get_chain_phases(self):
        """16 cycle counters of the forward chain CTA (see pimd_get_chain_phases); reset on read."""
        out = (C.c_uint64 * 16)()
        self._check(self._lib.pimd_get_chain_phases(self._h, out))
        return [int(v) for v in out]

    def launch_count(self):
        return int(self._lib.pimd_launch_count(self._h))


def probe_fp64_peak(stream=None):
    """Measured DFMA rate of the current device in TFLOP/s (2 flop per FMA)."""
    lib = load()
    out = C.c_double()
    rc = lib.pimd_probe_fp64_peak(C.c_void_p(stream or 0), C.byref(out))
    if rc != OK:
        raise PimdError(rc, lib.pimd_last_error(None).decode())
    return out.value


def selftest_exp(which, x_dev, stream=None):
    """y = the device exponential `which` (see pimd_selftest_exp) applied to the CUDA float64 tensor x_dev."""
    import torch

    lib = load()
    y = torch.empty_like(x_dev)
    rc = lib.pimd_selftest_exp(C.c_void_p(stream or 0), int(which), _ptr(x_dev), _ptr(y), x_dev.numel())
    if rc != OK:
        raise PimdError(rc, lib.pimd_last_error(None).decode())
    return y


def version():
    return load().pimd_version().decode()
