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
# (SURVEY.md 8(d)), counted as FMA-equivalents = 2 flop each; the shipped kernel
# executes 16 FP64 instructions per pair (SASS: 2 differences, 2 for r^2, 8 table exponential, 4 force FMAs)
FLOP_PER_PAIR = 50.0
FLOP_PER_PAIR_EXECUTED = 32.0
FLOP_PER_ELEMENT = 48.0   # exchange bulk: 24 FP64 instructions per lower-triangle entry and direction (fused row)


TRAFFIC_CSV = "r3_traffic.csv"
TRAFFIC_SOURCE = ("from the committed ncu --set full capture profiles/%s (command and code state in profiles/r3_traffic.md), "
                  "not measured in this run" % TRAFFIC_CSV)


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` at `workload`, from the summary of the
    `ncu --set full` capture of the shipped code state (profiles/r3_traffic.csv: workload,kernel,read,write); None if
    that capture has no such row."""
    try:
        with open(os.path.join(ROOT, "profiles", TRAFFIC_CSV)) as f:
            for line in f:
                c = [t.strip() for t in line.split(",")]
                if len(c) >= 4 and c[0] == workload and c[1] == kernel:
                    return int(float(c[2]) + float(c[3]))
    except OSError:
        pass
    return None


def exact_energy(name):
    """exact canonical energy of the non-interacting workloads at finite P (tests/golden/ideal_gas_energies.txt, written by a
    committed script from oracle/ideal_gas.py; BASELINE configs[4] "energy versus the exact ideal-Bose value"); None if the
    workload interacts or is not listed"""
    try:
        with open(os.path.join(ROOT, "tests", "golden", "ideal_gas_energies.txt")) as f:
            for ln in f:
                c = ln.split()
                if c and c[0] == name:
                    return float(c[6])
    except OSError:
        pass
    return None


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
    """(steps/s, steps, seconds) of orc_step on a bounded sample of workload w.  One call of orc_step is one complete MD
    step (force evaluation included).  At N >= 5000 a step takes tens of seconds: the sample is then that one step, started
    from zero forces instead of paying a second force evaluation for the opening half kick (timing is value-independent)."""
    import numpy as np

    import oracle
    from paper_2404_02628_b200 import workloads as wl

    oracle.build()
    x, v = wl.make_state(w, 0)
    big = w.N >= 5000
    F = np.zeros_like(x) if big else oracle.forces(x, w.beta, w.omega, w.g, w.s, w.xi)[0]
    nhc = np.zeros((4, x.size))
    t0 = time.perf_counter()
    oracle.step(x, v, F, nhc, w.beta, w.omega, w.g, w.s, w.xi, w.dt, 1, 1.0, 0, 0, 1)
    t_first = time.perf_counter() - t0
    if big or t_first >= budget_s:
        return 1.0 / t_first, 1, t_first
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
EST_EVERY = 10   # BASELINE config 3: "energy and density estimators every 10 steps", inside the timed region
REPEATS = 3      # 3 repeats, median


def timed_steps(torch, sim, steps, flush, w, est_every):
    """Device time of `steps` MD steps, one event pair per step, an L2 flush (outside the events) between steps.
    With est_every > 0 the steps whose number is a multiple of it evaluate and accumulate the estimators (pimd_run)."""
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for a, b in evs:
        if flush is not None:
            flush.zero_()
        a.record()
        if est_every:
            sim.run(1, est_every=est_every, nbins=w.nbins, rmax=w.rmax)
        else:
            sim.step(1)
        b.record()
    torch.cuda.synchronize()
    return sum(a.elapsed_time(b) for a, b in evs) * 1e-3


def median_rate(torch, sim, steps, flush, w, est_every, world=1):
    """median over REPEATS of steps / (max over ranks of the device time of `steps` flushed steps)"""
    rates = []
    for _ in range(REPEATS):
        t = max_over_ranks(timed_steps(torch, sim, steps, flush, w, est_every), world)
        rates.append(world * steps / t)
    rates.sort()
    return rates[len(rates) // 2], rates


def pair_roofline(w, kern, iso, fp64_peak):
    """ALU roofline of the pair kernel (None for g = 0) from its time inside the step (kern) and alone (iso), ms"""
    pairs = w.P * w.N * (w.N - 1) / 2.0 if w.g != 0.0 else 0.0
    if not (pairs and kern.get("pair")):
        return None
    t, ta = kern["pair"] * 1e-3, iso.get("pair", 0.0) * 1e-3
    ach = pairs * FLOP_PER_PAIR_EXECUTED / t / 1e12
    return {"bound": "alu", "kernel": "k_pair2 / k_pair (pair forces, Newton's third law)", "ms_in_step": kern["pair"],
            "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach / fp64_peak,
            "frac_executed": ach / fp64_peak,
            "frac_algorithmic": pairs * FLOP_PER_PAIR / t / 1e12 / fp64_peak,
            "traffic": ncu_traffic(w.name, "k_pair"), "traffic_source": TRAFFIC_SOURCE,
            "traffic_note": "DRAM bytes per launch (ncu); the algorithmic inputs are L2-resident: %d B of positions" % (w.P * w.N * w.d * 8),
            "peak_source": "FP64 FMA issue rate measured live by pimd_probe_fp64_peak (nominal 148 SM x 64 FMA/clk x "
                           "1.965 GHz x 2 = 37.2 TFLOP/s)",
            "convention": "frac = frac_executed: the 16 FP64 instructions (32 flop) per unordered bead pair the shipped SASS executes, "
                          "%d pairs per launch -- the figure to hold against north_star's 50 %%; frac_algorithmic counts SURVEY.md "
                          "8(d)'s 25 instructions (50 flop) per pair and over-counts the exponential (it can read above 1)" % int(pairs),
            "timed": "inside the step, sharing the GPU with the recursion kernel on another stream (event pairs only, no "
                     "instrumentation)",
            "alone": {"ms": iso.get("pair"), "frac": (pairs * FLOP_PER_PAIR_EXECUTED / ta / 1e12 / fp64_peak) if ta else None,
                      "frac_executed": (pairs * FLOP_PER_PAIR_EXECUTED / ta / 1e12 / fp64_peak) if ta else None,
                      "frac_algorithmic": (pairs * FLOP_PER_PAIR / ta / 1e12 / fp64_peak) if ta else None}}


def chain_roofline(w, kern, iso, fp64_peak, recursion):
    """The recursion kernel.  It recomputes the closing springs instead of streaming an N x N matrix, so its bulk is ALU
    work (SURVEY 8(d), row "fused / recomputed": 2 passes x N^2/2 entries x about 24 FP64 instructions), but up to
    N ~ 2e4 the kernel is bound by the latency of its N-long dependent chain: the ALU fraction is reported beside the
    latency figures (ns per row, cycles per 32-row block against the 32 x 38 cycle floor)."""
    ch_ms = kern.get("chain")
    if not ch_ms:
        return None
    elems = float(w.N) * (w.N + 1)  # both directions over the lower triangle
    ach = elems * FLOP_PER_ELEMENT / (ch_ms * 1e-3) / 1e12
    cha = iso.get("chain")
    cyc = (recursion or {}).get("cycles_per_block") or {}
    return {"bound": "latency", "kernel": "k_chain_spec (forward + backward recursion, panel workers with the force sums, force band "
                                          "and exterior forces as its tail)",
            "ms_in_step": ch_ms, "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s", "frac": ach / fp64_peak,
            "ns_per_row": ch_ms * 1e6 / w.N, "cycles_per_block": cyc.get("sum"), "floor_cycles_per_block": 32 * 38,
            "traffic": ncu_traffic(w.name, "k_chain_spec"), "traffic_source": TRAFFIC_SOURCE,
            "peak_source": "FP64 FMA issue rate measured live by pimd_probe_fp64_peak",
            "convention": "achieved / frac: 48 flop (24 FP64 instructions, SURVEY.md 8(d) fused row) per lower-triangle entry and "
                          "direction, N(N+1) entries per launch, over the kernel's time inside the step; neither roofline binds the "
                          "kernel below N ~ 2e4 -- one dependent DFMA + SHFL per row (ns_per_row; cycles_per_block from the phase "
                          "clock of a separate instrumented run, floor 32 x 38) -- the workers' bulk takes over near N = 4e4",
            "alone": {"ms": cha, "frac": (elems * FLOP_PER_ELEMENT / (cha * 1e-3) / 1e12 / fp64_peak) if cha else None}}


def rooflines_of(w, kern, iso, fp64_peak, recursion=None):
    """(roofline of the kernel that sets the step, [every hot kernel's roofline]): the dominant one is the kernel with the
    larger duration inside the step (the two run concurrently on two streams)"""
    rows = [r for r in (chain_roofline(w, kern, iso, fp64_peak, recursion), pair_roofline(w, kern, iso, fp64_peak)) if r]
    if not rows:
        return None, []
    top = max(rows, key=lambda r: r["ms_in_step"])
    for r in rows:
        r["dominant"] = r is top
    return top, rows


def kernel_profile(sim, nsteps, w, phases=True):
    """per-kernel device time (ms per launch) over nsteps steps with event pairs only (the kernels run uninstrumented), and
    -- from a second run of nsteps steps with the clock64 instrumentation armed -- the chain's phase clock and the
    instrumented chain time (an upper bound, reported separately)"""
    sim.set_profiling(True, phases=False)
    sim.get_profile()
    sim.run(nsteps, est_every=EST_EVERY, nbins=w.nbins, rmax=w.rmax)
    prof = sim.get_profile()
    ph, chain_instr = [0] * 16, None
    if phases:
        sim.set_profiling(True, phases=True)
        sim.get_chain_phases()
        sim.run(nsteps, est_every=EST_EVERY, nbins=w.nbins, rmax=w.rmax)
        p2 = sim.get_profile()
        ph = sim.get_chain_phases()
        if p2.get("chain", (0, 0))[1]:
            chain_instr = p2["chain"][0] / p2["chain"][1]
    sim.set_profiling(False)
    kern = {k: ms / n for k, (ms, n) in prof.items() if n}
    if chain_instr is not None:
        kern["chain_with_phase_clock"] = chain_instr
    return kern, {k: n for k, (ms, n) in prof.items() if n}, ph


def e2e_rate(torch, sim, x0, v0, ne2e, world, barrier):
    """end to end through the C ABI with HOST buffers: every step uploads the full state (x, v and the forces that belong
    to x, as a checkpointed host-resident run would), advances one MD step, and reads x, v, F back"""
    xh = torch.from_numpy(x0.copy()).pin_memory()
    vh = torch.from_numpy(v0.copy()).pin_memory()
    fh = torch.empty_like(xh).pin_memory()
    sim.set_state_host(xh, vh)
    sim.forces_host(fh)

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
    nbytes = int(x0.nbytes + v0.nbytes + x0.nbytes)
    return whole_job_rate(ne2e, te, world), nbytes


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

    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    W = max(args.warmup, 3)

    def measure(wk, steps, seed, full):
        """the headline protocol on workload wk: W warm-up steps; REPEATS x `steps` flushed steps from the seeded initial
        cloud; args.equil untimed steps of equilibration on the GPU; REPEATS x `steps` flushed steps from the thermalised
        state with the estimators every EST_EVERY steps inside the timed region (median of the repeats = value)"""
        sim, x0, v0 = make_sim(wk, seed)
        sim.step(W)
        torch.cuda.synchronize()
        barrier()
        v_init, _ = median_rate(torch, sim, steps, flush, wk, 0, world)
        # untimed equilibration on the GPU.  With forces -(1/P) grad U on unit-mass beads the cloud's centroid oscillates
        # in the trap at omega / sqrt(P); the friction that damps it fastest is twice that (the default gamma = 1
        # overdamps it: 1/e time gamma P / omega^2 = 32 time units at P = 32)
        sim.set_gamma(2.0 * wk.omega / np.sqrt(wk.P))
        sim.step(args.equil)
        sim.set_gamma(1.0)
        torch.cuda.synchronize()
        fb0 = sim.get_diagnostics()["fallbacks"]
        l0 = sim.launch_count()
        barrier()
        sampler = ClockSampler(local) if (rank == 0 and full) else None
        t0 = time.time()
        v_therm, reps = median_rate(torch, sim, steps, flush, wk, EST_EVERY, world)
        barrier()
        t1 = time.time()
        out = {"value": v_therm, "repeats": reps, "value_initial_cloud": v_init,
               "gpu_launches": (sim.launch_count() - l0) // REPEATS,
               "clocks": sampler.stop(t0, t1) if sampler else None}
        # the same steps back to back with the state left in L2 (how an MD run actually executes; graph replay)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        sim.run(steps, est_every=EST_EVERY, nbins=wk.nbins, rmax=wk.rmax)
        b.record()
        torch.cuda.synchronize()
        out["steps_per_s_l2_resident"] = world * steps / (a.elapsed_time(b) * 1e-3)
        nsamp, sp, sv, _, _ = sim.read_accumulators()
        out["sampled"] = {"n": float(nsamp), "e_prim_mean": float(sp / max(nsamp, 1.0)), "e_vir_mean": float(sv / max(nsamp, 1.0)),
                          "energy_exact": exact_energy(wk.name),
                          "note": "means over the few estimator samples of the timed steps (no error bar: tests/test_gpu_timed_path.py "
                                  "holds the ensemble check against energy_exact)"}
        kern, counts, phases = kernel_profile(sim, max(5, min(steps, 20)), wk)
        out["kernels_ms"] = kern
        out["recursion"] = recursion_report(wk, {"chain": {"ms_avg": kern.get("chain")}}, phases, max(5, min(steps, 20)), None)
        met, skipped = phases[11], phases[12]
        out["recursion"]["helper_batches_skipped_frac"] = (skipped / met) if met else None
        nbk = (wk.N + 31) // 32
        out["recursion"]["factorised_blocks_frac"] = phases[6] / float(max(5, min(steps, 20)) * nbk)
        out["fallbacks_in_timed_steps"] = sim.get_diagnostics()["fallbacks"] - fb0
        if full:
            # the same kernels timed alone (exchange and bead parts serialised on one stream): the burst figure
            sim.set_concurrency(False)
            iso, _, _ = kernel_profile(sim, max(5, min(steps, 20)), wk, phases=False)
            sim.set_concurrency(True)
            out["kernels_alone_ms"] = iso
            out["e2e_value"], out["e2e_bytes"] = e2e_rate(torch, sim, x0, v0, max(3, min(steps, 50)), world, barrier)
        sim.close()
        return out

    # replicas: every rank advances its own seeded copy of the workload
    m = measure(w, args.steps, rank, True)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    peaks, peak_src = load_peaks()
    fp64_peak = binding.probe_fp64_peak()
    pairs = w.P * w.N * (w.N - 1) / 2.0 if w.g != 0.0 else 0.0
    nb = m["e2e_bytes"]
    line = {
        "metric": METRIC, "value": m["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
        "ms_per_step": 1e3 * world / m["value"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": describe(w), "l2": "flushed between timed steps (256 MiB device write outside the events)",
                   "state": "thermalised on the GPU by %d untimed steps (friction 2 omega/sqrt(P), the centroid's critical damping) after the seeded initial cloud" % args.equil,
                   "estimators": "energy + radial density every %d steps inside the timed region" % EST_EVERY,
                   "protocol": "median of %d repeats of %d steps" % (REPEATS, args.steps),
                   "parallelism": "replicas x%d (one independent seeded copy per GPU, no collective on the data path)" % world},
        "clocks": m["clocks"],
        "e2e": {"value": m["e2e_value"], "unit": UNIT, "h2d_bytes_per_step": nb, "d2h_bytes_per_step": nb,
                "note": "pimd_set_state_host + pimd_set_forces_host + pimd_step(1) + pimd_get_state_host + pimd_get_forces_host per "
                        "step, pinned host buffers, wall clock"},
        "gpu_launches": m["gpu_launches"],
        "repeats": m["repeats"],
        "value_initial_cloud": m["value_initial_cloud"],
        "pair_forces_per_s": pairs * m["value"],
        "steps_per_s_l2_resident": m["steps_per_s_l2_resident"],
        "fallbacks_in_timed_steps": m["fallbacks_in_timed_steps"],
        "sampled": m["sampled"],
        "kernels_ms": m["kernels_ms"],
        "kernels_alone_ms": m["kernels_alone_ms"],
        "recursion": m["recursion"],
        "roofline": rooflines_of(w, m["kernels_ms"], m["kernels_alone_ms"], fp64_peak, m["recursion"])[0],
        "rooflines": rooflines_of(w, m["kernels_ms"], m["kernels_alone_ms"], fp64_peak, m["recursion"])[1],
        "peaks": {"fp64_tflops_probe": fp64_peak, "hbm_gbs": peaks.get("hbm_gbs"), "source": peak_src},
    }

    if world == 1 and not args.no_also:
        # north_star states its targets at N = 10000: the same objects for config 5 (N = 10000) and 5b
        also = []
        for name in args.also.split(","):
            wk = wl.WORKLOADS[name]
            r = measure(wk, args.sweep_steps, 0, True)
            pp = wk.P * wk.N * (wk.N - 1) / 2.0 if wk.g != 0.0 else 0.0
            row = {"workload": describe(wk), "value": r["value"], "unit": UNIT, "value_initial_cloud": r["value_initial_cloud"],
                   "pair_forces_per_s": pp * r["value"], "steps_per_s_l2_resident": r["steps_per_s_l2_resident"],
                   "kernels_ms": r["kernels_ms"], "kernels_alone_ms": r["kernels_alone_ms"], "recursion": r["recursion"],
                   "roofline": rooflines_of(wk, r["kernels_ms"], r["kernels_alone_ms"], fp64_peak, r["recursion"])[0],
                   "rooflines": rooflines_of(wk, r["kernels_ms"], r["kernels_alone_ms"], fp64_peak, r["recursion"])[1],
                   "e2e": {"value": r["e2e_value"], "unit": UNIT, "h2d_bytes_per_step": r["e2e_bytes"], "d2h_bytes_per_step": r["e2e_bytes"]},
                   "fallbacks_in_timed_steps": r["fallbacks_in_timed_steps"]}
            if not args.no_cpu:
                row["cpu_baseline"] = cpu_baseline(wk, 1.0)
            also.append(row)
        line["also"] = also
        for row in also:   # north_star: >= 50 % of the FP64 roofline on the pair kernel at N = 10000 -- in the step AND alone
            pr = [r for r in row["rooflines"] if r["kernel"].startswith("k_pair")]
            if pr and "cfg5b" in row["workload"]:
                line["pair_kernel_N10000"] = {"workload": "cfg5b", "frac_executed_in_step": pr[0]["frac_executed"],
                                              "frac_executed_alone": pr[0]["alone"]["frac_executed"],
                                              "ms_in_step": pr[0]["ms_in_step"], "ms_alone": pr[0]["alone"]["ms"],
                                              "peak_tflops": fp64_peak, "target": 0.5}
    if world == 1 and not args.no_sweep:
        sweep = []
        for name in args.sweep.split(","):
            wk = wl.WORKLOADS[name]
            r = measure(wk, args.sweep_steps, 0, False)
            pp = wk.P * wk.N * (wk.N - 1) / 2.0 if wk.g != 0.0 else 0.0
            sweep.append({"workload": name, "N": wk.N, "P": wk.P, "g": wk.g, "steps_per_s": r["value"],
                          "steps_per_s_initial_cloud": r["value_initial_cloud"], "steps_per_s_l2_resident": r["steps_per_s_l2_resident"],
                          "pair_forces_per_s": pp * r["value"], "kernels_ms": r["kernels_ms"],
                          "ns_per_row": r["recursion"].get("ns_per_row"),
                          "helper_batches_skipped_frac": r["recursion"].get("helper_batches_skipped_frac"),
                          "sampled": r["sampled"],
                          "fallbacks_in_timed_steps": r["fallbacks_in_timed_steps"]})
        line["sweep"] = sweep
        line["sweep_protocol"] = "as the headline: thermalised by %d steps, L2 flushed between steps, median of %d x %d steps" % (
            args.equil, REPEATS, args.sweep_steps)
    if world == 1 and not args.no_batch:
        # replica batches: B replicas of the small configurations in one set of launches
        rows = []
        for name, B in (("cfg1", 64), ("cfg2", 32), ("cfg4", 5)):
            wk = wl.WORKLOADS[name]
            xis = [wk.xi] * B if name != "cfg4" else [-0.5, -0.3, 0.3, 0.5, 1.0]
            xs, vs = zip(*[wl.make_state(wk, b) for b in range(B)])
            sb = binding.Pimd(wk.N, wk.P, wk.d, wk.beta, wk.omega, wk.g, wk.s, xis, wk.dt, thermostat=1, seed=list(range(B)))
            sb.set_state(torch.from_numpy(np.stack(xs)).cuda(), torch.from_numpy(np.stack(vs)).cuda())
            sb.step(50)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            nst = 400
            a.record()
            sb.run(nst, est_every=EST_EVERY, nbins=wk.nbins, rmax=wk.rmax)
            b.record()
            torch.cuda.synchronize()
            rows.append({"workload": name, "replicas": B, "xi": sorted(set(xis)), "batch_steps_per_s": nst / (a.elapsed_time(b) * 1e-3),
                         "replica_steps_per_s": B * nst / (a.elapsed_time(b) * 1e-3)})
            sb.close()
        line["replica_batches"] = rows
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
                              "bytes_per_launch": nbytes_nn, "peak_source": peak_src,
                              "note": "on-request write-only kernels; the hot path has no N x N pass (DESIGN.md section 6)"}
        for key, name in (("emat", "k_emat (cycle energies, Eq. 7-10)"), ("prmat", "k_prmat (connection probabilities, Eq. 12-14)")):
            ms = pr3[key][0] / max(pr3[key][1], 1)
            gbs = nbytes_nn / (ms * 1e-3) / 1e9
            dram = ncu_traffic("cfg5_N10000", "k_" + key)
            line["nxn_passes"][key] = {"kernel": name, "ms": ms, "achieved": gbs, "frac": gbs / peaks.get("hbm_gbs"),
                                       "convention": "achieved = 8 N^2 bytes written / kernel time; by_dram_bytes = the DRAM bytes ncu "
                                                     "saw inside one launch (part of the output is still in L2 when it ends) / the same time",
                                       "by_dram_bytes": ({"traffic": dram, "achieved": dram / (ms * 1e-3) / 1e9,
                                                          "frac": dram / (ms * 1e-3) / 1e9 / peaks.get("hbm_gbs"),
                                                          "traffic_source": TRAFFIC_SOURCE} if dram else None)}
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
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--equil", type=int, default=3000, help="untimed equilibration steps before the timed region")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--sweep", default="cfg1,cfg2,cfg4,cfg5_N2500,cfg5_N10000,cfg5_N20000,cfg5_N40000,cfg5b")
    ap.add_argument("--also", default="cfg5_N10000,cfg5b", help="workloads that get roofline + e2e + cpu_baseline beside the headline")
    ap.add_argument("--sweep-steps", type=int, default=20)
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-also", action="store_true")
    ap.add_argument("--no-batch", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-nxn", action="store_true", help="skip the materialised N x N passes (0.8 GB at N=10000)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    args = ap.parse_args()
    from paper_2404_02628_b200 import workloads as wl

    w = wl.WORKLOADS[args.workload]
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and world == 1 and "RANK" not in os.environ:
        # asked for N GPUs without a launcher: start one rank per GPU ourselves (the driver uses the same command line)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(29500 + os.getpid() % 1000), os.path.abspath(__file__)] + sys.argv[1:]
        return subprocess.call(cmd)
    if args.gpus != world and "RANK" in os.environ:
        raise SystemExit("--gpus %d does not match WORLD_SIZE %d" % (args.gpus, world))
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    sys.exit(main())
