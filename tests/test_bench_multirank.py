"""The N > 1 path of bench.py is "replicas only": every rank advances its own seeded copy,
there is no data-path collective, and the only cross-rank logic is the max-over-ranks timing and the whole-job
rate.  That logic is exercised here with two CPU processes over gloo (the GPU run uses the same functions
over NCCL).  Also: the seeded workloads differ per rank and are reproducible."""
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


def _worker(rank, world, port, out):
    import torch.distributed as dist

    import bench
    from paper_2404_02628_b200 import workloads as wl

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r "took" (r + 1) seconds for 10 steps
        t = bench.max_over_ranks(float(rank + 1), world, device="cpu")
        rate = bench.whole_job_rate(10, float(rank + 1), world, device="cpu")
        x, _ = wl.make_state(wl.WORKLOADS["cfg2"], rank)
        out.put((rank, t, rate, float(x.sum())))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world_size_2():
    import torch.multiprocessing as mp

    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # both ranks see the slowest rank's time, and the whole-job rate counts both replicas
    assert [r[1] for r in res] == [2.0, 2.0]
    assert [r[2] for r in res] == [10.0, 10.0]  # 2 ranks * 10 steps / 2 s
    # replicas are different seeded copies
    assert res[0][3] != res[1][3]


def test_single_rank_needs_no_process_group():
    import bench

    assert bench.max_over_ranks(3.5, 1, device="cpu") == 3.5
    assert bench.whole_job_rate(7, 2.0, 1, device="cpu") == 3.5


def test_workloads_are_reproducible_and_seed_dependent():
    from paper_2404_02628_b200 import workloads as wl

    w = wl.WORKLOADS["cfg3"]
    x0, v0 = wl.make_state(w, 0)
    x0b, v0b = wl.make_state(w, 0)
    x1, _ = wl.make_state(w, 1)
    np.testing.assert_array_equal(x0, x0b)
    np.testing.assert_array_equal(v0, v0b)
    assert not np.array_equal(x0, x1)
    assert x0.shape == (w.P, w.N, w.d) and x0.dtype == np.float64
