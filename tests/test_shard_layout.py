"""Bead-slice sharding: the host-side partition / halo / pack arithmetic with two (and three) CPU processes
over gloo.  The GPU kernels cannot run here; what is checked is that the boundary packs the layout prescribes,
all-gathered exactly as sharding.ShardedPimd does it (all_gather_into_tensor of pack_doubles doubles per rank), give
every rank everything its share of the force evaluation needs -- compared against the oracle's single-rank results:
  * the halo slices are the ring neighbours' boundary slices, bead 1 / bead P arrive from rank 0 / the last rank,
  * E_int assembled from the ranks' partial sums plus the springs that cross a rank boundary equals orc_eint (Eq. 9),
  * the spring + trap + pair forces of the local slices, computed from the local slices and the halos alone, equal the
    oracle's forces on the interior beads (Eq. 17, 18) -- nothing else is needed from other ranks,
  * the local slices tile 0..P-1 without gap or overlap for any world <= P."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

torch = pytest.importorskip("torch")


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_slices_tile_the_ring_for_every_world_size():
    from paper_2404_02628_b200 import sharding

    for P in (2, 5, 8, 16, 32, 72):
        for world in range(1, P + 1):
            nxt = 0
            for r in range(world):
                j0, pl = sharding.shard_range(P, r, world)
                assert j0 == nxt and pl >= 1
                nxt = j0 + pl
            assert nxt == P
    with pytest.raises(ValueError):
        sharding.shard_range(4, 0, 5)
    assert sharding.pack_doubles(10, 3) == 70 and sharding.pack_offsets(10, 3) == (0, 30, 60)
    assert sharding.pack_doubles(37, 2) == 186          # 185 rounded up: packs stay 16-byte aligned
    assert sharding.halo_sources(0, 3) == (None, (1, "first")) and sharding.halo_sources(2, 3) == ((1, "last"), None)


def _worker(rank, world, port, out):
    import torch.distributed as dist

    import oracle
    from paper_2404_02628_b200 import sharding
    from paper_2404_02628_b200 import workloads as wl

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = wl.custom(37, 7, d=2, beta=2.0, g=0.3, s=0.5, xi=1.0, init="iid", sigma=0.8)
        x, _ = wl.make_state(w, 5)                      # the same global state on every rank; a rank keeps its slices only
        N, P, d = w.N, w.P, w.d
        ks = P / w.beta ** 2
        j0, pl = sharding.shard_range(P, rank, world)
        xl = x[j0:j0 + pl].copy()
        o_first, o_last, o_eint = sharding.pack_offsets(N, d)
        n = sharding.pack_doubles(N, d)
        # this rank's boundary pack (what k_shard_pack writes)
        send = torch.zeros(n, dtype=torch.float64)
        send[o_first:o_first + N * d] = torch.from_numpy(xl[0].reshape(-1))
        send[o_last:o_last + N * d] = torch.from_numpy(xl[-1].reshape(-1))
        send[o_eint:o_eint + N] = torch.from_numpy(0.5 * ks * np.sum(np.diff(xl, axis=0) ** 2, axis=(0, 2)))
        gathered = torch.zeros(world * n, dtype=torch.float64)
        dist.all_gather_into_tensor(gathered, send)
        g = gathered.numpy().reshape(world, n)
        part = {"first": lambda r: g[r, o_first:o_first + N * d].reshape(N, d),
                "last": lambda r: g[r, o_last:o_last + N * d].reshape(N, d)}
        ok = []
        # halos, bead 1, bead P
        lo, hi = sharding.halo_sources(rank, world)
        halo_lo = part[lo[1]](lo[0]) if lo else None
        halo_hi = part[hi[1]](hi[0]) if hi else None
        ok.append(halo_lo is None or np.array_equal(halo_lo, x[j0 - 1]))
        ok.append(halo_hi is None or np.array_equal(halo_hi, x[j0 + pl]))
        ok.append((halo_lo is None) == (j0 == 0) and (halo_hi is None) == (j0 + pl == P))
        ok.append(np.array_equal(part["first"](0), x[0]) and np.array_equal(part["last"](world - 1), x[P - 1]))
        # E_int: partial sums + the springs that cross a rank boundary (what k_shard_eint forms)
        eint = g[:, o_eint:o_eint + N].sum(axis=0)
        for r in range(world - 1):
            eint = eint + 0.5 * ks * np.sum((part["first"](r + 1) - part["last"](r)) ** 2, axis=1)
        ok.append(np.allclose(eint, oracle.eint(x, w.beta), rtol=1e-13, atol=0))
        # local forces from local slices + halos only: springs to the ring neighbours (Eq. 17), trap, pair (Eq. 18)
        ext = np.concatenate([halo_lo[None] if halo_lo is not None else np.zeros((0, N, d)), xl,
                              halo_hi[None] if halo_hi is not None else np.zeros((0, N, d))])
        off = 1 if halo_lo is not None else 0
        F = np.zeros_like(xl)
        for jl in range(pl):
            k = jl + off
            F[jl] = -(w.omega ** 2 / P) * xl[jl]
            if k > 0:
                F[jl] -= ks * (ext[k] - ext[k - 1])
            if k + 1 < ext.shape[0]:
                F[jl] -= ks * (ext[k] - ext[k + 1])
            diff = xl[jl][:, None, :] - xl[jl][None, :, :]
            e = w.g * np.exp(-np.sum(diff ** 2, axis=-1) / w.s ** 2)
            F[jl] += (2.0 / w.s ** 2 / P) * np.sum(e[:, :, None] * diff, axis=1)
        Fo, _, _ = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
        interior = [jl for jl in range(pl) if 0 < j0 + jl < P - 1]       # beads 1 and P also take the exchange forces
        ok.append(all(np.allclose(F[jl], Fo[j0 + jl], rtol=0, atol=1e-11 * np.abs(Fo).max()) for jl in interior))
        out.put((rank, j0, pl, ok))
    except Exception as e:  # a failing worker must not leave the parent waiting for its result
        out.put((rank, -1, -1, [repr(e)]))
        raise
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_boundary_packs_over_gloo(world):
    import torch.multiprocessing as mp

    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs), res
    assert sum(r[2] for r in res) == 7
    for rank, j0, pl, ok in res:
        assert j0 >= 0 and all(v is True or v == np.True_ for v in ok), (rank, ok)
