#!/usr/bin/env python
"""Benchmark of the PIMD hot path (arXiv 2404.02628) on B200: MD steps/s and bead-pair evaluations/s.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

A "step" is one pass of the whole hot path (spring/trap/pair forces, closing springs, forward and
backward recursions, connection probabilities and exterior forces, thermostatted velocity Verlet)
over one seeded synthetic configuration of the named workload.  One JSON line is printed by rank 0.
DESIGN.md ("Measurement") states the roofline conventions used here.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "PIMD MD steps/s"
UNIT = "steps/s"
# algorithmic FP64 work of the pair kernel: 25 FP64 instructions per unordered bead pair at d = 2
# (SURVEY.md 8(d)), counted as FMA-equivalents = 2 flop each
FLOP_PER_PAIR = 50.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
# (profiles/r1_d_cfg3.md for cfg3 -- unchanged since r1_b_cfg3.md --, profiles/r1_b_cfg5b.md for cfg5b); None where no
# capture of that workload exists
NCU_TRAFFIC = {("cfg3", "pair"): 1706240 + 0, ("cfg3", "forcepass"): 291072 + 0,
               ("cfg5b", "pair"): 5186048 + 0, ("cfg5b", "forcepass"): 1768960 + 0}


def describe(w):
    return ("%s: N=%d P=%d d=%d beta=%g omega=%g g=%g s=%g xi=%g dt=%g, Langevin thermostat (gamma=1), "
            "init=%s sigma=%.3g" % (w.name, w.N, w.P, w.d, w.beta, w.omega, w.g, w.s, w.xi, w.dt, w.init, w.sigma))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [c.strip() for c in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.15 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons, "samples": len(rows),
                "power_w_max": max(float(r[2]) for r in rows)}


def max_over_ranks(value, world, device="cuda"):
    """MAX of a per-rank scalar over all ranks (the timing rule for every multi-GPU number) and the
    whole-job rate helper: works with any initialised torch.distributed backend (NCCL on GPUs; gloo
    in the CPU tests)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank, seconds_per_rank, world, device="cuda"):
    """Replicas: every rank does `units_per_rank`; value = all units / slowest rank's time."""
    return world * units_per_rank / max_over_ranks(seconds_per_rank, world, device)


def recursion_report(w, kern, phases, steps, clocks):
    """Latency figures of the N-long chain (neither roofline binds it)."""
    ch = kern.get("chain", {}).get("ms_avg")
    nb = (w.N + 31) // 32
    out = {"kernel": "k_chain_spec (forward + backward recursion with the previous step's gauge, one cooperative launch)",
           "bound": "latency",
           "ms": ch, "ns_per_row": (ch * 1e6 / w.N if ch else None), "rows_per_block": 32}
    if ch and sum(phases[:4]) > 0:
        per = [c / float(steps * nb) for c in phases[:16]]
        out["cycles_per_block"] = {"barrier_wait": per[0], "prologue": per[1], "dependent_steps_32": per[2], "epilogue": per[3],
                                   "sum": sum(per[:4]),
                                   "helpers": {"m_tile": per[4], "older_blocks": per[5], "tiles_prepared": per[8],
                                               "columns_published": per[7], "panel_fetched": per[9],
                                               "panel_reads_per_block": per[10], "tables_and_prefetch": per[15]}}
        out["floor_cycles_per_block"] = 32 * 38
        out["note"] = ("SM cycles of the forward chain CTA per 32-row block (clock64 inside k_chain_spec, the stale-gauge "
                       "kernel every timed step runs); floor = 32 x (SHFL + DFMA) from measured latencies; the block time is "
                       "set by the helper warps / the workers' panel (barrier_wait), not by the dependent steps")
    return out


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    except OSError:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0}, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------
# the oracle, timed on the host cores (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def time_oracle(w, budget_s, max_steps=None):
    import numpy as np

    import oracle
    from paper_2404_02628_b200 import workloads as wl

    oracle.build()
    x, v = wl.make_state(w, 0)
    F, _, _ = oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)
    nhc = np.zeros((4, x.size))
    t0 = time.perf_counter()
    oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, 1, 1.0, 0, 0, 1)
    t_first = time.perf_counter() - t0
    n = max(1, int(budget_s / max(t_first, 1e-6)))
    if max_steps is not None:
        n = min(n, max_steps)
    t0 = time.perf_counter()
    oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, 1, 1.0, 0, 1, n)
    dt = time.perf_counter() - t0
    return n / dt, n, dt


def cpu_baseline(w, budget_s=15.0):
    sps, n, dt = time_oracle(w, budget_s)
    return {"value": sps, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
            "sample": "%d full MD steps of %s by oracle/pimd_oracle.c (gcc -O2, OpenMP on the pair loop only) in %.1f s"
                      % (n, w.name, dt)}


def run_reference(args, w):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    budget = min(150.0, max(10.0, 0.6 * args.steps))
    sps, n, dt = time_oracle(w, budget, max_steps=args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": sps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 / sps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": describe(w), "parallelism": "host cores"},
        "cpu_baseline": {"value": sps, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                         "sample": "%d of the %d requested MD steps of %s timed in %.1f s (bounded sample)"
                                   % (n, args.steps, w.name, dt)},
        "e2e": {"value": sps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------------
def timed_steps(torch, sim, steps, flush):
    """Device time of `steps` MD steps, one event pair per step, an L2 flush between steps."""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        if flush is not None:
            flush.zero_()
        a.record()
        sim.step(1)
        b.record()
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in evs) * 1e-3


def run_ours(args, w):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2404_02628_b200 import binding, build
    from paper_2404_02628_b200 import workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the hot path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if build.needs_build():
        if rank == 0:
            build.build()
        if world > 1:
            dist.barrier()
    binding.load()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def make_sim(wk, seed):
        sim = binding.Pimd(wk.N, wk.P, wk.d, wk.beta, wk.omega, wk.g, wk.s, wk.xi, wk.dt,
                           thermostat=binding.THERMOSTAT_LANGEVIN, seed=seed)
        x, v = wl.make_state(wk, seed)
        sim.set_state(torch.from_numpy(x).cuda(), torch.from_numpy(v).cuda())
        return sim, x, v

    # replicas: every rank advances its own seeded copy of the workload
    sim, x0, v0 = make_sim(w, rank)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    sim.step(max(args.warmup, 3))
    torch.cuda.synchronize()
    sim.set_profiling(True)
    sim.get_profile()
    l0 = sim.launch_count()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t0 = time.time()
    t_dev = timed_steps(torch, sim, args.steps, flush)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    launches = sim.launch_count() - l0
    prof = sim.get_profile()
    sim.set_profiling(False)
    phases = sim.get_chain_phases()
    t_dev = max_over_ranks(t_dev, world)
    value = world * args.steps / t_dev

    # the same K steps back to back with the state left in L2 (how an MD run actually executes)
    barrier()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    sim.step(args.steps)
    b.record()
    torch.cuda.synchronize()
    resident_sps = args.steps / (a.elapsed_time(b) * 1e-3)

    # end to end through the C ABI with HOST buffers: every step uploads the full state (x, v and the forces that
    # belong to x, as a checkpointed host-resident run would), advances one MD step, and reads x, v, F back
    xh = torch.from_numpy(x0.copy()).pin_memory()
    vh = torch.from_numpy(v0.copy()).pin_memory()
    fh = torch.empty_like(xh).pin_memory()
    sim.set_state_host(xh, vh)
    sim.forces_host(fh)
    ne2e = max(3, min(args.steps, 50))

    def e2e_step():
        sim.set_state_host(xh, vh)
        sim.set_forces_host(fh)
        sim.step(1)
        sim.get_state_host(xh, vh)
        sim.get_forces_host(fh)  # synchronises

    for _ in range(2):
        e2e_step()
    barrier()
    te = time.perf_counter()
    for _ in range(ne2e):
        e2e_step()
    barrier()
    te = time.perf_counter() - te
    e2e = whole_job_rate(ne2e, te, world)
    nbytes = int(x0.nbytes + v0.nbytes + x0.nbytes)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks, peak_src = load_peaks()
    fp64_peak = binding.probe_fp64_peak()
    # the same kernels timed alone (exchange and bead parts serialised on one stream): the burst figure
    sim.set_concurrency(False)
    sim.set_profiling(True)
    sim.get_profile()
    sim.step(max(5, min(args.steps, 20)))
    iso = {k: ms / n for k, (ms, n) in sim.get_profile().items() if n}
    sim.set_profiling(False)
    sim.set_concurrency(True)
    pairs = w.P * w.N * (w.N - 1) / 2.0 if w.g != 0.0 else 0.0
    kern = {k: {"ms_avg": (ms / n if n else None), "launches": n} for k, (ms, n) in prof.items() if n}
    bead_ms = kern.get("pair", {}).get("ms_avg")
    if pairs and bead_ms:
        ach = pairs * FLOP_PER_PAIR / (bead_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "k_pair (pair forces, Newton's third law)", "achieved": ach, "peak": fp64_peak,
                    "unit": "TFLOP/s", "frac": ach / fp64_peak, "traffic": NCU_TRAFFIC.get((w.name, "pair")),
                    "traffic_note": "DRAM bytes per launch (ncu); the algorithmic inputs are L2-resident: %d B of positions" % (w.P * w.N * w.d * 8),
                    "peak_source": "FP64 FMA issue rate measured live by pimd_probe_fp64_peak (nominal 148 SM x 64 FMA/clk x "
                                   "1.965 GHz x 2 = 37.2 TFLOP/s)",
                    "convention": "50 flop (25 FP64 instructions, SURVEY.md 8(d)) per unordered bead pair, %d pairs per launch; "
                                  "the shipped kernel spends 16 FP64 instructions per pair (table-driven exp), so frac can "
                                  "exceed the FP64 pipe utilisation ncu reports" % int(pairs),
                    "timed": "inside the step, sharing the GPU with the recursion kernel on another stream",
                    "alone": {"ms": iso.get("pair"), "frac": pairs * FLOP_PER_PAIR / (iso["pair"] * 1e-3) / 1e12 / fp64_peak}}
    else:
        # non-interacting workloads: the exchange passes dominate; they recompute the closing springs
        # instead of streaming an N x N matrix, so they are ALU bound too
        fp_ms = kern.get("forcepass", {}).get("ms_avg")
        elems = float(w.N) * (w.N + 1)  # two sweeps over the lower triangle
        ach = elems * 54.0 / (fp_ms * 1e-3) / 1e12 if fp_ms else None
        roofline = {"bound": "alu", "kernel": "k_forcepass (connection probabilities)", "achieved": ach, "peak": fp64_peak,
                    "unit": "TFLOP/s", "frac": (ach / fp64_peak if ach else None), "traffic": NCU_TRAFFIC.get((w.name, "forcepass")),
                    "peak_source": "FP64 FMA issue rate measured live by pimd_probe_fp64_peak",
                    "convention": "54 flop (27 FP64 instructions) per matrix element, N(N+1) elements per launch",
                    "alone": {"ms": iso.get("forcepass"),
                              "frac": (elems * 54.0 / (iso["forcepass"] * 1e-3) / 1e12 / fp64_peak) if iso.get("forcepass") else None}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(w), "l2": "flushed between timed steps (256 MiB device write outside the events)",
                   "parallelism": "replicas x%d (one independent seeded copy per GPU, no collective on the data path)" % world},
        "clocks": clocks,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "note": "pimd_set_state_host + pimd_set_forces_host + pimd_step(1) + pimd_get_state_host + pimd_get_forces_host per "
                        "step, pinned host buffers, wall clock"},
        "gpu_launches": launches,
        "pair_forces_per_s": pairs * value,
        "steps_per_s_l2_resident": resident_sps * world,
        "kernels": kern,
        "kernels_alone_ms": iso,
        "recursion": recursion_report(w, kern, phases, args.steps, clocks),
        "roofline": roofline,
        "peaks": {"fp64_tflops_probe": fp64_peak, "hbm_gbs": peaks.get("hbm_gbs"), "source": peak_src},
    }
    sim.close()

    if world == 1 and not args.no_sweep:
        sweep = []
        for name in args.sweep.split(","):
            wk = wl.WORKLOADS[name]
            s2, _, _ = make_sim(wk, 0)
            s2.step(3)
            torch.cuda.synchronize()
            n2 = args.sweep_steps
            a.record()
            s2.step(n2)
            b.record()
            torch.cuda.synchronize()
            sps = n2 / (a.elapsed_time(b) * 1e-3)
            s2.set_profiling(True)
            s2.get_profile()
            s2.step(5)
            pr = s2.get_profile()
            pp = wk.P * wk.N * (wk.N - 1) / 2.0 if wk.g != 0.0 else 0.0
            sweep.append({"workload": name, "N": wk.N, "P": wk.P, "g": wk.g, "steps_per_s": sps, "pair_forces_per_s": pp * sps,
                          "kernels_ms": {k: ms / n for k, (ms, n) in pr.items() if n}})
            s2.close()
        line["sweep"] = sweep
    if world == 1 and not args.no_nxn:
        # the paper's N x N intermediates, materialised on request (not on the hot path): HBM-write rooflines at N = 10000
        wk = wl.WORKLOADS["cfg5_N10000"]
        s3, _, _ = make_sim(wk, 0)
        s3.forces(want_forces=False)
        buf = torch.empty((wk.N, wk.N), dtype=torch.float64, device="cuda")
        s3.set_profiling(True)
        for _ in range(2):
            s3.cycle_energies(out=buf)
            s3.connection_probabilities(out=buf)
        s3.get_profile()
        reps = 5
        for _ in range(reps):
            flush.zero_()
            s3.cycle_energies(out=buf)
            flush.zero_()
            s3.connection_probabilities(out=buf)
        pr3 = s3.get_profile()
        nbytes_nn = 8.0 * wk.N * wk.N
        line["nxn_passes"] = {"workload": "cfg5_N10000", "bound": "hbm", "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                              "bytes_per_launch": nbytes_nn, "peak_source": peak_src}
        for key, name in (("emat", "k_emat (cycle energies, Eq. 7-10)"), ("prmat", "k_prmat (connection probabilities, Eq. 12-14)")):
            ms = pr3[key][0] / max(pr3[key][1], 1)
            gbs = nbytes_nn / (ms * 1e-3) / 1e9
            line["nxn_passes"][key] = {"kernel": name, "ms": ms, "achieved": gbs, "frac": gbs / peaks.get("hbm_gbs")}
        del buf
        s3.close()
    if world == 1 and not args.no_cpu:
        line["cpu_baseline"] = cpu_baseline(w, args.cpu_seconds)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--sweep", default="cfg1,cfg2,cfg4,cfg5_N2500,cfg5_N10000,cfg5_N20000,cfg5_N40000,cfg5b")
    ap.add_argument("--sweep-steps", type=int, default=20)
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-nxn", action="store_true", help="skip the materialised N x N passes (0.8 GB at N=10000)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    from paper_2404_02628_b200 import workloads as wl

    w = wl.WORKLOADS[args.workload]
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    sys.exit(main())
