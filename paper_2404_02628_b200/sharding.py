"""Bead-slice sharding across GPUs: control flow only, no arithmetic.

Rank r of `world` holds the bead slices [floor(P r / world), floor(P (r+1) / world)) of every ring polymer.  One
exchange step per MD step: the all-gather of every rank's boundary pack

    [ first local slice : N d ][ last local slice : N d ][ E_int of the springs between local slices : N ]

(2 N d + N doubles, padded to an even count; written by pimd_shard_export, consumed by pimd_shard_forces / pimd_shard_end_step).  Everything
else -- springs, trap, pair forces, integrator on the local slices, the exchange recursion redundantly on every rank --
runs inside libpimd's kernels.

    ShardedPimd      one process per GPU; the all-gather is torch.distributed (NCCL over NVLink on GPUs)
    LocalShardGroup  all shards in one process on one GPU, the all-gather is a device copy; the kernels of different
                     shards never wait on one another (they are launched one after the other on one stream)

The layout helpers are plain integer arithmetic shared with the CPU (gloo) tests.
"""
from __future__ import annotations


def shard_range(P: int, rank: int, world: int):
    """(first slice, number of slices) of `rank` -- the same formula as pimd_create_sharded."""
    if not (0 <= rank < world <= P):
        raise ValueError("need 0 <= rank < world <= P")
    j0 = P * rank // world
    return j0, P * (rank + 1) // world - j0


def pack_doubles(N: int, d: int) -> int:
    """doubles per boundary pack, padded to an even count (the packs stay 16-byte aligned in the gathered buffer)"""
    return (2 * N * d + N + 1) // 2 * 2


def pack_offsets(N: int, d: int):
    """offsets (in doubles) of the three parts of a boundary pack: first slice, last slice, partial E_int"""
    return 0, N * d, 2 * N * d


def halo_sources(rank: int, world: int):
    """(rank, part) whose pack part is this rank's lower / upper halo slice (None where the ring polymer ends):
    the slice below my first one is the LAST slice of rank-1, the slice above my last one the FIRST slice of rank+1."""
    lo = (rank - 1, "last") if rank > 0 else None
    hi = (rank + 1, "first") if rank + 1 < world else None
    return lo, hi


class ShardedPimd:
    """One bead shard per process (torchrun: one rank per GPU).  `group` is a torch.distributed process group."""

    def __init__(self, binding, N, P, d, beta, omega, g, s, xi, dt, thermostat=1, seed=0, group=None, **kw):
        import torch
        import torch.distributed as dist

        self._dist, self._torch, self.group = dist, torch, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        self.sim = binding.Pimd(N, P, d, beta, omega, g, s, xi, dt, thermostat=thermostat, seed=seed,
                                shard=(self.rank, self.world), **kw)
        self.j0, self.P_local = self.sim.j0, self.sim.P_local
        n = self.sim.pack_doubles
        self.send = torch.empty(n, dtype=torch.float64, device="cuda")
        self.gathered = torch.empty(self.world * n, dtype=torch.float64, device="cuda")
        self._have_forces = False  # the library holds forces of the current positions (set_state invalidates them)

    def set_state(self, x_global, v_global=None):
        """global [P][N][d] device tensors; the local slices are taken"""
        sl = slice(self.j0, self.j0 + self.P_local)
        self.sim.set_state(x_global[sl].contiguous(), None if v_global is None else v_global[sl].contiguous())
        self._have_forces = False

    def _all_gather(self):
        self._dist.all_gather_into_tensor(self.gathered, self.send, group=self.group)

    def forces(self):
        self.sim.shard_export(self.send)
        self._all_gather()
        self.sim.shard_forces(self.gathered)
        self._have_forces = True
        return self.sim.get_forces()

    def step(self, nsteps=1):
        if nsteps > 0 and not self._have_forces:
            self.forces()
        for _ in range(nsteps):
            self.sim.shard_begin_step(self.send)
            self._all_gather()
            self.sim.shard_end_step(self.gathered)

    def close(self):
        self.sim.close()


class LocalShardGroup:
    """`world` bead shards of one system on ONE GPU, stepped in lock step; the all-gather is a device copy."""

    def __init__(self, binding, world, N, P, d, beta, omega, g, s, xi, dt, thermostat=1, seed=0, **kw):
        import torch

        self._torch, self.world, self.P = torch, world, P
        self.sims = [binding.Pimd(N, P, d, beta, omega, g, s, xi, dt, thermostat=thermostat, seed=seed, shard=(r, world), **kw)
                     for r in range(world)]
        n = self.sims[0].pack_doubles
        self.gathered = torch.empty(world * n, dtype=torch.float64, device="cuda")
        self._n = n
        self._have_forces = False

    def set_state(self, x_global, v_global=None):
        for sim in self.sims:
            sl = slice(sim.j0, sim.j0 + sim.P_local)
            sim.set_state(x_global[sl].contiguous(), None if v_global is None else v_global[sl].contiguous())
        self._have_forces = False

    def _gather(self, export):
        for r, sim in enumerate(self.sims):
            export(sim, self.gathered[r * self._n:(r + 1) * self._n])

    def forces(self):
        """global [P][N][d] forces, V_B, sign (of rank 0; the exchange part is the same on every rank)"""
        self._gather(lambda sim, buf: sim.shard_export(buf))
        for sim in self.sims:
            sim.shard_forces(self.gathered)
        self._have_forces = True
        f = self._torch.cat([sim.get_forces() for sim in self.sims], dim=0)
        vb, sg = self.sims[0].shard_scalars()
        return f, vb, sg

    def step(self, nsteps=1):
        if nsteps > 0 and not self._have_forces:
            self.forces()
        for _ in range(nsteps):
            self._gather(lambda sim, buf: sim.shard_begin_step(buf))
            for sim in self.sims:
                sim.shard_end_step(self.gathered)

    def get_state(self):
        xs, vs = zip(*[sim.get_state() for sim in self.sims])
        return self._torch.cat(xs, dim=0), self._torch.cat(vs, dim=0)

    def estimators(self, nbins=0, rmax=1.0):
        """sum of the ranks' shares"""
        parts = [sim.estimators(nbins=nbins, rmax=rmax) for sim in self.sims]
        return sum(p[0] for p in parts), sum(p[1] for p in parts), sum(p[2] for p in parts)

    def close(self):
        for sim in self.sims:
            sim.close()
