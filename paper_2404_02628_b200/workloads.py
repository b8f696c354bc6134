"""Seeded synthetic workloads (inputs only -- none of the method's arithmetic lives here).

These stand in for the trapped-gas simulations of arXiv 2404.02628 section IV,
whose own configurations and figure data are not available; shapes and parameters follow
BASELINE.json `configs` with the readings listed in DESIGN.md ("Input recipe", R6, R11).
Both the CUDA path and the oracle are fed the SAME arrays produced here.

Layout: x[P][N][d], v[P][N][d], float64, C-contiguous (bead-major).
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    N: int
    P: int
    d: int
    beta: float
    omega: float
    g: float
    s: float
    xi: float
    dt: float
    init: str          # "iid" (every bead coordinate i.i.d.) or "ring" (centre + compact ring)
    sigma: float       # std of the bead (iid) or of the particle centre (ring)
    nbins: int = 64
    rmax: float = 6.0

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


def _cfg5(N: int) -> Workload:
    return Workload(f"cfg5_N{N}", N, 16, 2, 3.0, 1.0, 0.0, 0.5, 1.0, 0.01, "ring", float(N) ** 0.25,
                    rmax=6.0 * float(N) ** 0.25)


WORKLOADS = {
    # BASELINE.json configs[0]: non-interacting bosons, N=4, P=16, beta=2
    "cfg1": Workload("cfg1", 4, 16, 2, 2.0, 1.0, 0.0, 0.5, 1.0, 0.01, "iid", 1.0),
    # configs[1]: weakly interacting bosons, N=100, P=32, beta=3, g=0.5, s=0.5; 64 bins on [0,6]
    "cfg2": Workload("cfg2", 100, 32, 2, 3.0, 1.0, 0.5, 0.5, 1.0, 0.01, "iid", 1.0),
    # configs[2]: the paper's headline scale, N=1600, P=32, g=0.2
    "cfg3": Workload("cfg3", 1600, 32, 2, 3.0, 1.0, 0.2, 0.5, 1.0, 0.01, "ring", 1600.0 ** 0.25, rmax=24.0),
    # configs[3]: fictitious particles, N=1000, xi=-0.5 (also -0.3, 0)
    "cfg4": Workload("cfg4", 1000, 32, 2, 3.0, 1.0, 0.2, 0.5, -0.5, 0.01, "ring", 3.0, rmax=12.0),
    # configs[4]: large-N non-interacting sweep
    "cfg5_N2500": _cfg5(2500),
    "cfg5_N10000": _cfg5(10000),
    "cfg5_N20000": _cfg5(20000),
    "cfg5_N40000": _cfg5(40000),
    # SURVEY.md 8(d) "config 5b": the N=10000 point with the pair interaction switched on,
    # because north_star states the pair-kernel target at N=10000
    "cfg5b": _cfg5(10000).with_(name="cfg5b", g=0.2),
}


def make_state(w: Workload, seed: int = 0):
    """Initial positions and velocities for workload `w` from `seed` (numpy PCG64).

    iid : every bead coordinate ~ N(0, sigma^2)                      (configs 1, 2, literal)
    ring: particle centre c_l ~ N(0, sigma^2 I), beads c_l + N(0, beta/(2P)) per coordinate
          (neighbour-bead spread of a free ring polymer; R11)
    velocities ~ N(0, 1/beta) per coordinate (unit mass, T = 1/beta; R6).
    """
    rng = np.random.default_rng(seed)
    shape = (w.P, w.N, w.d)
    if w.init == "iid":
        x = rng.normal(0.0, w.sigma, size=shape)
    elif w.init == "ring":
        c = rng.normal(0.0, w.sigma, size=(1, w.N, w.d))
        x = c + rng.normal(0.0, np.sqrt(w.beta / (2.0 * w.P)), size=shape)
    else:
        raise ValueError(w.init)
    v = rng.normal(0.0, np.sqrt(1.0 / w.beta), size=shape)
    return np.ascontiguousarray(x, dtype=np.float64), np.ascontiguousarray(v, dtype=np.float64)


def custom(N, P, d=2, beta=3.0, omega=1.0, g=0.0, s=0.5, xi=1.0, dt=0.01, init="iid", sigma=1.0, name=None):
    return Workload(name or f"custom_N{N}_P{P}_d{d}", N, P, d, beta, omega, g, s, xi, dt, init, sigma)
