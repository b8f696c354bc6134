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
PROF_SLOTS = ("bead", "prep", "chain", "assemble", "finalize", "integrate", "combine", "pair", "emat", "prmat", "gr", "shard")
MAX_SPECIES, MAX_BINS = 4, 4096
NOALLOC_MAX_N = 16384
PROFILE_EVENTS, PROFILE_PHASES = 1, 2
PAIR_GAUSSIAN, PAIR_SOFT_COULOMB = 0, 1

# every symbol include/pimd.h declares: (restype, argtypes)
_dp = C.POINTER(C.c_double)
_SYMBOLS = {
    "pimd_create": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                              C.c_double, C.c_double, C.c_double, C.c_int, C.c_uint64]),
    "pimd_create_batch": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double,
                                    C.c_double, _dp, C.c_double, C.c_int, C.POINTER(C.c_uint64)]),
    "pimd_create_sharded": (C.c_int, [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double,
                                      C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_uint64]),
    "pimd_destroy": (C.c_int, [C.c_void_p]),
    "pimd_set_species": (C.c_int, [C.c_void_p, C.c_int, C.POINTER(C.c_int)]),
    "pimd_set_pair_potential": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_set_pair_histogram": (C.c_int, [C.c_void_p, C.c_int, C.c_double]),
    "pimd_pair_histogram": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_run": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double]),
    "pimd_read_accumulators": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int]),
    "pimd_reweight": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_shard_layout": (C.c_int, [C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_size_t)]),
    "pimd_shard_export": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_shard_forces": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_shard_begin_step": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_shard_end_step": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_shard_scalars": (C.c_int, [C.c_void_p, _dp, C.POINTER(C.c_int)]),
    "pimd_get_diagnostics": (C.c_int, [C.c_void_p, C.c_void_p]),
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
    "pimd_forces": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_forces_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_get_forces": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_forces_host": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_set_forces": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_set_forces_host": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_get_tables": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "pimd_cycle_energies": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_connection_probabilities": (C.c_int, [C.c_void_p, C.c_void_p]),
    "pimd_cycle_energies_noalloc": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_double, C.c_void_p]),
    "pimd_step": (C.c_int, [C.c_void_p, C.c_int]),
    "pimd_estimators": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double]),
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
    """One simulation handle.  Method names mirror the C entry points (pimd_<name>).

    xi / seed given as sequences make a batch of B replicas (pimd_create_batch): state and force tensors are then
    [B][P][N][d] and per-evaluation scalars come back as numpy arrays of B entries.  shard=(rank, world) makes a bead
    shard (pimd_create_sharded) holding P_local slices.  species=(n0, n1, ..) calls pimd_set_species."""

    def __init__(self, N, P, d, beta, omega, g, s, xi, dt, thermostat=THERMOSTAT_LANGEVIN, seed=0,
                 stream=None, use_torch_workspace=True, species=None, pair_potential=None, shard=None):
        self._lib = load()
        self._h = C.c_void_p()
        self.N, self.P, self.d = int(N), int(P), int(d)
        self.batched = hasattr(xi, "__len__")
        if self.batched:
            xs = [float(v) for v in xi]
            sd = [int(v) for v in seed] if hasattr(seed, "__len__") else [int(seed) + k for k in range(len(xs))]
            self.B = len(xs)
            rc = self._lib.pimd_create_batch(C.byref(self._h), self.B, int(N), int(P), int(d), float(beta), float(omega), float(g),
                                             float(s), (C.c_double * self.B)(*xs), float(dt), int(thermostat),
                                             (C.c_uint64 * self.B)(*sd))
        elif shard is not None:
            self.B = 1
            rc = self._lib.pimd_create_sharded(C.byref(self._h), int(shard[0]), int(shard[1]), int(N), int(P), int(d), float(beta),
                                               float(omega), float(g), float(s), float(xi), float(dt), int(thermostat), int(seed))
        else:
            self.B = 1
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
        if species is not None:
            cnt = [int(c) for c in species]
            self._check(self._lib.pimd_set_species(self._h, len(cnt), (C.c_int * len(cnt))(*cnt)))
        if pair_potential is not None:
            self._check(self._lib.pimd_set_pair_potential(self._h, int(pair_potential)))
        self.P_local, self.j0, self.pack_doubles = self.shard_layout()
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
        shape = (self.P_local, self.N, self.d)
        return self._torch.empty(((self.B,) + shape) if self.batched else shape, dtype=self._torch.float64, device="cuda")

    def _scalars(self, arr):
        """per-replica HOST outputs: a numpy array for a batch, a plain number otherwise"""
        return arr.copy() if self.batched else arr[0].item()

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
        shape = (NHC_LENGTH, self.P_local * self.N * self.d)
        t = self._torch.empty(((self.B,) + shape) if self.batched else shape, dtype=self._torch.float64, device="cuda")
        self._check(self._lib.pimd_get_nhc(self._h, _ptr(t)))
        return t

    def set_nhc(self, nhc_dev):
        self._check(self._lib.pimd_set_nhc(self._h, _ptr(nhc_dev)))

    def forces(self, out=None, want_forces=True):
        """(F [P][N][d] device tensor or None, V_B, sign)."""
        import numpy as np

        f = None
        if want_forces:
            f = out if out is not None else self._empty_state()
        vb, sg = np.zeros(self.B), np.zeros(self.B, dtype=np.int32)
        self._check(self._lib.pimd_forces(self._h, _ptr(f), _ptr(vb), _ptr(sg)))
        return f, self._scalars(vb), self._scalars(sg)

    def forces_host(self, f_host):
        import numpy as np

        vb, sg = np.zeros(self.B), np.zeros(self.B, dtype=np.int32)
        self._check(self._lib.pimd_forces_host(self._h, _ptr(f_host), _ptr(vb), _ptr(sg)))
        return self._scalars(vb), self._scalars(sg)

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

        ep, ev = np.zeros(self.B), np.zeros(self.B)
        hist = np.zeros((self.B, max(int(nbins), 1)))
        self._check(self._lib.pimd_estimators(self._h, _ptr(ep), _ptr(ev), _ptr(hist), int(nbins), float(rmax)))
        hist = hist[:, : int(nbins)].copy()
        return self._scalars(ep), self._scalars(ev), (hist if self.batched else hist[0])

    def run(self, nsteps, est_every=0, nbins=0, rmax=1.0):
        self._check(self._lib.pimd_run(self._h, int(nsteps), int(est_every), int(nbins), float(rmax)))

    def read_accumulators(self, nbins=0, nbins_gr=0, reset=True):
        """(number of samples, sum e_prim, sum e_vir, radial histogram sum, pair histogram sum) per replica."""
        import numpy as np

        n, sp, sv = np.zeros(self.B), np.zeros(self.B), np.zeros(self.B)
        hs, gs = np.zeros((self.B, max(int(nbins), 1))), np.zeros((self.B, max(int(nbins_gr), 1)))
        self._check(self._lib.pimd_read_accumulators(self._h, _ptr(n), _ptr(sp), _ptr(sv), _ptr(hs), int(nbins), _ptr(gs),
                                                     int(nbins_gr), int(bool(reset))))
        hs, gs = hs[:, : int(nbins)], gs[:, : int(nbins_gr)]
        if not self.batched:
            hs, gs = hs[0], gs[0]
        return self._scalars(n), self._scalars(sp), self._scalars(sv), hs.copy(), gs.copy()

    def set_pair_potential(self, kind):
        self._check(self._lib.pimd_set_pair_potential(self._h, int(kind)))

    def set_pair_histogram(self, nbins, rmax):
        self._nbins_gr = int(nbins)
        self._check(self._lib.pimd_set_pair_histogram(self._h, int(nbins), float(rmax)))

    def pair_histogram(self):
        import numpy as np

        g = np.zeros((self.B, max(getattr(self, "_nbins_gr", 0), 1)))
        self._check(self._lib.pimd_pair_histogram(self._h, _ptr(g)))
        return g.copy() if self.batched else g[0].copy()

    def reweight(self, xi_obs):
        """(ln|R|, sign, eps_obs, eps_samp) per replica for R = W_{xi_obs} / W_{xi} at the current positions."""
        import numpy as np

        xo = np.ascontiguousarray(np.broadcast_to(np.asarray(xi_obs, dtype=np.float64), (self.B,)))
        lr, sg, eo, es = np.zeros(self.B), np.zeros(self.B, dtype=np.int32), np.zeros(self.B), np.zeros(self.B)
        self._check(self._lib.pimd_reweight(self._h, _ptr(xo), _ptr(lr), _ptr(sg), _ptr(eo), _ptr(es)))
        return self._scalars(lr), self._scalars(sg), self._scalars(eo), self._scalars(es)

    # -- bead shards
    def shard_layout(self):
        j0, pl, n = C.c_int(), C.c_int(), C.c_size_t()
        self._check(self._lib.pimd_shard_layout(self._h, C.byref(j0), C.byref(pl), C.byref(n)))
        return pl.value, j0.value, n.value

    def shard_export(self, send_dev):
        self._check(self._lib.pimd_shard_export(self._h, _ptr(send_dev)))

    def shard_forces(self, gathered_dev):
        self._check(self._lib.pimd_shard_forces(self._h, _ptr(gathered_dev)))

    def shard_begin_step(self, send_dev):
        self._check(self._lib.pimd_shard_begin_step(self._h, _ptr(send_dev)))

    def shard_end_step(self, gathered_dev):
        self._check(self._lib.pimd_shard_end_step(self._h, _ptr(gathered_dev)))

    def shard_scalars(self):
        vb, sg = C.c_double(), C.c_int()
        self._check(self._lib.pimd_shard_scalars(self._h, C.byref(vb), C.byref(sg)))
        return vb.value, sg.value

    def get_diagnostics(self):
        out = (C.c_uint64 * 4)()
        self._check(self._lib.pimd_get_diagnostics(self._h, out))
        return {"fallbacks": int(out[0]), "status_seen": int(out[1]), "workers": int(out[2]), "replica_stride": int(out[3])}

    def set_profiling(self, on, phases=True):
        """off / PIMD_PROFILE_PHASES (events + the chain CTA's phase clock; default) / PIMD_PROFILE_EVENTS (phases=False:
        event pairs only, the uninstrumented kernels)"""
        self._check(self._lib.pimd_set_profiling(self._h, (PROFILE_PHASES if phases else PROFILE_EVENTS) if on else 0))

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


def cycle_energies_noalloc(x_dev, beta, out, stream=None):
    """pimd_cycle_energies_noalloc: E[u, v] = E^{[u+1,v+1]} of the positions x_dev ([P][N][d] CUDA float64 tensor) written
    into the caller's `out` ([N][N] CUDA float64 tensor).  No handle; the library allocates nothing (its O(N) tables sit
    in a fixed 512 KiB device array, N <= NOALLOC_MAX_N), and this wrapper allocates nothing either: both tensors are the
    caller's.  Asynchronous on `stream` (default: torch's current stream).  See include/pimd.h for who needs this and for
    the sharing rules (one array per GPU: do not let two calls overlap)."""
    import torch

    lib = load()
    P, N, d = x_dev.shape
    if not (x_dev.is_cuda and out.is_cuda and x_dev.is_contiguous() and out.is_contiguous()
            and x_dev.dtype == torch.float64 and out.dtype == torch.float64 and out.numel() == N * N):
        raise ValueError("cycle_energies_noalloc: contiguous CUDA float64 tensors x [P][N][d] and out [N][N] are required")
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    rc = lib.pimd_cycle_energies_noalloc(C.c_void_p(stream), _ptr(x_dev), int(N), int(P), int(d), float(beta), _ptr(out))
    if rc != OK:
        raise PimdError(rc, lib.pimd_last_error(None).decode())
    return out


def version():
    return load().pimd_version().decode()
