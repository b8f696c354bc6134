"""pimd_cycle_energies_noalloc against the handle path pimd_cycle_energies.

Why the entry point exists: a program that has handed all of its device memory to its own allocator, that keeps several
streams busy and cannot take the device-wide stall of a cudaMalloc, or that runs where its host forbids allocation calls,
cannot create a handle (which allocates a workspace, pinned memory, streams).  For such callers the library offers one
call that only launches kernels; its O(N) tables sit in a fixed 512 KiB device array inside libpimd.so, shared by every
call on that GPU and never cleared (include/pimd.h).

What is checked here: the same positions give the same N x N matrix as the handle path, within the tolerance the matrix
test of tests/test_gpu_parity.py uses (1e-10 of the largest entry; the two paths add the bead differences of a ring in a
different order, so the last bits may differ), on two calls in a row -- the second with a smaller system, so that it runs on
top of the first call's left-overs in the shared array -- and that a system larger than the array is refused with a message
and leaves the output untouched.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
other tests.  The test does not depend on what ran before it (the first call on a device does its own set-up).
"""
import numpy as np
import pytest
import torch

from paper_2404_02628_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_2404_02628_b200 import binding as b, build

    build.build()
    b.load()
    return b


def handle_path(binding, w, x_dev):
    """E from pimd_cycle_energies: the existing path (handle, workspace, its own copies of the tables)."""
    sim = binding.Pimd(w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, thermostat=binding.THERMOSTAT_NVE, seed=1)
    try:
        sim.set_state(x_dev)
        return sim.cycle_energies()
    finally:
        sim.close()


# two calls in a row, the larger system first: several 1024-column segments with a ragged tail, then a small one that reuses
# only the head of each table
CASES = [(2500, 6, 3, 1.5), (333, 5, 2, 2.0), (77, 4, 1, 0.7)]


def test_noalloc_matches_handle_path_on_consecutive_calls(binding):
    for k, (N, P, d, beta) in enumerate(CASES):
        w = wl.custom(N, P, d=d, beta=beta, g=0.0, xi=1.0, init="ring", sigma=1.0)
        x, _ = wl.make_state(w, 40 + k)
        x_dev = torch.from_numpy(x).cuda()
        out = torch.full((N, N), float("nan"), dtype=torch.float64, device="cuda")  # caller-owned output
        ret = binding.cycle_energies_noalloc(x_dev, beta, out)
        assert ret is out
        torch.cuda.synchronize()
        ref = handle_path(binding, w, x_dev)
        E, Er = out.cpu().numpy(), ref.cpu().numpy()
        assert np.all(np.isfinite(E))
        assert np.all(np.tril(E, -1) == 0.0)
        assert np.max(np.abs(E - Er)) <= 1e-10 * np.max(np.abs(Er)), (N, P, d)


def test_noalloc_same_input_twice_is_bit_identical(binding):
    """The shared tables keep the previous call's contents; a call must not depend on them."""
    N, P, d, beta = 1200, 8, 2, 2.0
    w = wl.custom(N, P, d=d, beta=beta, g=0.0, xi=1.0, init="ring", sigma=1.0)
    x, _ = wl.make_state(w, 7)
    x_dev = torch.from_numpy(x).cuda()
    a = torch.empty((N, N), dtype=torch.float64, device="cuda")
    b = torch.empty((N, N), dtype=torch.float64, device="cuda")
    binding.cycle_energies_noalloc(x_dev, beta, a)
    # another system in between dirties the tables
    w2 = wl.custom(1500, 4, d=d, beta=1.0, g=0.0, xi=1.0, init="ring", sigma=2.0)
    x2, _ = wl.make_state(w2, 8)
    binding.cycle_energies_noalloc(torch.from_numpy(x2).cuda(), 1.0, torch.empty((1500, 1500), dtype=torch.float64, device="cuda"))
    binding.cycle_energies_noalloc(x_dev, beta, b)
    torch.cuda.synchronize()
    assert torch.equal(a, b)


def test_noalloc_refuses_sizes_beyond_the_built_in_tables(binding):
    N = binding.NOALLOC_MAX_N + 1
    x_dev = torch.zeros((2, N, 1), dtype=torch.float64, device="cuda")
    # the size check comes before anything is launched: a small sentinel buffer shows that the output is not written
    import ctypes as C

    lib = binding.load()
    out = torch.full((16,), -7.0, dtype=torch.float64, device="cuda")
    rc = lib.pimd_cycle_energies_noalloc(None, C.c_void_p(x_dev.data_ptr()), N, 2, 1, 1.0, C.c_void_p(out.data_ptr()))
    assert rc == binding.EINVAL
    msg = lib.pimd_last_error(None).decode()
    assert "PIMD_NOALLOC_MAX_N" in msg and str(binding.NOALLOC_MAX_N) in msg
    torch.cuda.synchronize()
    assert bool((out == -7.0).all())
    for bad in [dict(N=0), dict(P=1), dict(d=4), dict(beta=0.0)]:
        a = dict(N=4, P=3, d=1, beta=1.0)
        a.update(bad)
        assert lib.pimd_cycle_energies_noalloc(None, C.c_void_p(x_dev.data_ptr()), a["N"], a["P"], a["d"], a["beta"],
                                               C.c_void_p(out.data_ptr())) == binding.EINVAL
