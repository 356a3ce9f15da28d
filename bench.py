#!/usr/bin/env python3
"""bench.py — headline benchmark: integrand events/s (fp64) for gg -> t tbar g g on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C3] [--impl ours|reference]

One STEP = one pass of the whole hot path over one batch of 2^22 synthetic
events of BASELINE.json configs[3] (the config the metric is quoted on): mf_unweight (Philox -> VEGAS map ->
RAMBO -> cuts -> PDF -> |M|^2 -> weight -> sums -> histograms -> hit-or-miss unweighting + compaction)
followed by mf_refine_grid.  Step k is VEGAS iteration k, so the warm-up steps also adapt the grid.

Numbers on the JSON line:
  value      events/s with everything resident in HBM (CUDA events around each step on the launch stream)
  e2e        the same through the C ABI with HOST buffers: grid host->device before, result/histogram/grid/
             accepted records device->host after, inside the timed region
  roofline   bound "alu": static fp64 operation count of the matrix-element code (csrc/gen_me.py) x events
             passing the cuts / duration of the fused-pass kernel, against the FP64 peak measured on this GPU
             by mf_measure_fp64_peak
  cpu_baseline  the oracle, as it stands, on a bounded sample of the same workload (rank 0, N=1 only)
--impl reference times the oracle (this tier has no reference implementation).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "integrand events/sec (fp64) for gg->ttbar gg"      # BASELINE.json metric (C3, C4)
PROCESS_LABEL = {0: "e+e- -> mu+mu-", 1: "gg->ttbar", 2: "gg->ttbar g", 3: "gg->ttbar gg", 4: "pp->ttbar (gg + q qbar)", 5: "pp->ttbar j (gg + q qbar, q g, qbar g)", 6: "gg->ttbar ggg", 7: "pp->ttbar gg (gg + q qbar)"}


def metric_for(wl):
    """the BASELINE.json metric for the headline process; the same quantity, named after its process, for --config"""
    return METRIC if wl.process == 3 else "integrand events/sec (fp64) for " + PROCESS_LABEL[wl.process]
UNIT = "events/s"
# ---- the roofline numerator ------------------------------------------------------------------------
# achieved = (n_pass x flop per matrix element + n_events x flop per event outside it) / kernel time.
#  * cooperative / block kernels (processes 2, 3, 6): flop per matrix element = the generators' static operation count,
#    read from the generated headers at run time (FLOP_HEADERS; a DMMA.884 counts its 2 x 256 flop); the rest of the chain
#    (a1-a6, a10-a14 incl. the software sqrt / div / log / sincos sequences and the owner-side wavefunctions) is OTHER_FLOPS,
#    calibrated by ncu: executed (2 dfma + dadd + dmul) of one launch minus n_pass x the static count (FLOP_PROFILES).
#  * thread-per-event kernels (0, 1, 4), pp -> ttbar j (5), g g -> ttbar ggg (6) and pp -> ttbar gg (7, prepass + fused pass): the
#    ncu-executed TOTAL per event (per passing event for 5, 6, 7; for 6 / 7 plus their 3840 / 48 DMMA x 512 flop) is used (ME_FLOPS_MEASURED): for 0, 1, 4 the compiler
#    folds constants into the matrix element, so the static count overestimates; for 6 the generator's static count
#    (5.89 M) misses 7 % of the executed operations (sign and scale multiplications).
# tests/test_host_logic.py::test_bench_flop_constants recomputes every literal below from the committed ncu csv files.
FLOP_HEADERS = {2: ("mf_me_ttg_coop_generated.cuh", "kFlopsMe2Coop_1g"), 3: ("mf_me_ttgg_coop_generated.cuh", "kFlopsMe2Coop_2g")}
FLOP_PROFILES = {0: "profiles/r1_flops_C0.csv", 1: "profiles/r1_flops_C1.csv", 2: "profiles/r1_flops_C2.csv",
                 3: "profiles/r1_flops_C3.csv", 4: "profiles/r1_flops_C5.csv", 5: "profiles/r2_flops_C6.csv",
                 6: "profiles/r2_flops_C7.csv", 7: "profiles/r2_flops_C8.csv"}
FLOP_PROFILE_EVENTS = {0: (1_000_000, 1.0), 1: (1 << 20, 1.0), 2: (1 << 22, 0.8934), 3: (1 << 22, 0.7825), 4: (1 << 20, 1.0),
                       5: (1 << 22, 0.8945), 6: (1 << 18, 0.653), 7: (1 << 22, 0.7855)}      # events of the profiled launch, cut pass rate
FLOP_PROFILE_DMMA = {6: 3840 * 512.0, 7: 48 * 512.0}            # flop per matrix element on the tensor path (not seen by the op_dfma counter)
FLOP_PROFILE_ME = {2: 21472.0, 3: 157956.0}      # the static matrix-element count of the build that was profiled
OTHER_FLOPS = {0: 0.0, 1: 0.0, 2: 2930.0, 3: 5290.0, 4: 0.0, 5: 0.0, 6: 0.0, 7: 0.0}
ME_FLOPS_MEASURED = {0: 1232.0, 1: 3766.0, 4: 5023.0, 5: 54030.0, 6: 6.31e6, 7: 321600.0}    # 5, 6: per event PASSING the cuts
# kernels of this library launched per step (mf_unweight + mf_refine_grid): fused pass, finalize, refine; g g -> ttbar g and
# pp -> ttbar j add the record kernel of their accepted events, pp -> ttbar gg that and the quark prepass
LAUNCHES_PER_STEP = {2: 4, 5: 4, 7: 5}
# dram__bytes_read + dram__bytes_write per launch of the fused pass from an ncu capture of this very command
# (profiles/r1_coop_v4_traffic.md), keyed by (process, events per launch); None where no capture was taken
MEASURED_TRAFFIC = {(3, 1 << 22): 3.86e7}
NOMINAL_FP64 = 148 * 64 * 2 * 1.965e9   # SMs x FP64 lanes x 2 flop x max SM clock = 37.2 Tflop/s


def me_flops(process):
    import re
    if process in ME_FLOPS_MEASURED:
        return ME_FLOPS_MEASURED[process]
    csrc = os.path.join(ROOT, "paper_2106_10279_b200", "csrc")
    if process in FLOP_HEADERS:   # the cooperative / block programs are what the fused pass runs
        name = FLOP_HEADERS[process]
        txt = open(os.path.join(csrc, name[0])).read()
        return float(re.search(name[1] + r" = ([0-9.]+);", txt).group(1))
    raise KeyError(process)


def executed_flops_of_profile(path):
    """2 dfma + dadd + dmul (thread instructions, predicated on) of the ncu --csv metric log `path`"""
    import csv
    v = {"dfma": 0.0, "dadd": 0.0, "dmul": 0.0}            # summed over the profiled launches (C8: prepass + fused pass)
    for row in csv.reader(open(os.path.join(ROOT, path))):
        if len(row) > 14 and row[12].startswith("smsp__sass_thread_inst_executed_op_d"):
            v[row[12].split("_op_")[1].split("_")[0]] += float(row[14])
    return 2.0 * v["dfma"] + v["dadd"] + v["dmul"]


def config_by_name(name):
    from paper_2106_10279_b200 import workloads as W
    return {"C0": W.C0, "C1": W.C1, "C2": W.C2, "C3": W.C3, "C4": W.C4, **W.EXTRA_CONFIGS}[name]


# ---- clocks ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            for nme, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        mx = max((float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()), default=None)
        pw = max((float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()), default=None)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "power_w_max": pw,
                "reasons": sorted(reasons), "samples": len(sm)}


# ---- the oracle arm (cpu_baseline and --impl reference) ---------------------------------------------------------
_SAMPLE_WORKER = r"""
import sys, time
sys.path.insert(0, sys.argv[1])
from oracle import mfo
from paper_2106_10279_b200 import workloads as W
wl = {"C0": W.C0, "C1": W.C1, "C2": W.C2, "C3": W.C3, "C4": W.C4, **W.EXTRA_CONFIGS}[sys.argv[2]]
seconds, n_first = float(sys.argv[3]), int(sys.argv[4])
op = mfo.Process(wl, W.pdf_for(wl.process))
grid = W.uniform_grid(wl.n_dims, wl.n_bins)
t0 = time.perf_counter()
op.vegas_iterate(grid, wl.seed, 0, 0, n_first)
per = (time.perf_counter() - t0) / n_first
n = int(max(n_first, min(wl.n_events, seconds / per)))
t0 = time.perf_counter()
op.vegas_iterate(grid, wl.seed, 0, 0, n)
print(n, time.perf_counter() - t0)
"""


def oracle_sample(config, seconds=15.0, n_first=64):
    """Times the oracle, as it stands, single-threaded, on events [0, n) of iteration 0 of the config on the uniform
    grid; n is sized from a short probe so the sample takes about `seconds`.  Runs in a SUBPROCESS: the process that
    times the CUDA path never loads oracle/libmfo.so."""
    r = subprocess.run([sys.executable, "-c", _SAMPLE_WORKER, ROOT, config, str(seconds), str(n_first)],
                       stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
    if r.returncode != 0:
        raise RuntimeError("oracle sample failed: " + r.stderr[-2000:])
    n, dt = r.stdout.split()
    n, dt = int(n), float(dt)
    return n / dt, n, dt


_ALL_CORES_WORKER = r"""
import sys, time
sys.path.insert(0, sys.argv[1])
from oracle import mfo
from paper_2106_10279_b200 import workloads as W
wl = {"C0": W.C0, "C1": W.C1, "C2": W.C2, "C3": W.C3, "C4": W.C4, **W.EXTRA_CONFIGS}[sys.argv[2]]
first, n = int(sys.argv[3]), int(sys.argv[4])
op = mfo.Process(wl, W.pdf_for(wl.process))
grid = W.uniform_grid(wl.n_dims, wl.n_bins)
t0 = time.perf_counter()
op.vegas_iterate(grid, wl.seed, 0, first, n)
print(time.perf_counter() - t0)
"""


def oracle_all_cores(config, per_event_s, seconds=10.0):
    """The same single-threaded oracle as P independent processes on disjoint event-index ranges (possible because the
    RNG is counter based), P = the host's logical cores: aggregate events/s."""
    P = os.cpu_count() or 1
    n = max(16, int(seconds / per_event_s))
    t0 = time.perf_counter()
    procs = [subprocess.Popen([sys.executable, "-c", _ALL_CORES_WORKER, ROOT, config, str(i * n), str(n)],
                              stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True) for i in range(P)]
    ok = all(p.wait() == 0 for p in procs)
    dt = time.perf_counter() - t0
    return (P * n / dt, P, n, dt) if ok else None


def run_reference(args, wl):
    """--impl reference: the oracle on the host cores (one thread), each step a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import mfo
    from paper_2106_10279_b200 import workloads as W
    op = mfo.Process(wl, W.pdf_for(wl.process))
    grid = W.uniform_grid(wl.n_dims, wl.n_bins)
    n = {0: 200000, 1: 40000, 2: 4000, 3: 400, 4: 20000, 5: 2000, 6: 24, 7: 150}[wl.process]     # ~2 s per step
    times = []
    for k in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        hist, res = op.vegas_iterate(grid, wl.seed, k, 0, n)
        grid = op.refine_grid(grid, hist, W.VEGAS_ALPHA)
        if k >= args.warmup:
            times.append(time.perf_counter() - t0)
    tot = sum(times)
    val = n * len(times) / tot
    sample = "%d events/step of %s (iteration k on the oracle's own adapting grid), 1 thread" % (n, wl.name)
    print(json.dumps({"impl": "reference", "metric": metric_for(wl), "value": val, "unit": UNIT, "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / len(times),
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                      "data": "synthetic", "config": {"workload": wl.name, "events_per_step": n},
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# ---- our arm -----------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="C3")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--seed", type=int, default=None, help="Philox seed (default: the configuration's, 0)")
    ap.add_argument("--events", type=int, default=0,
                    help="events per step per GPU (default: the config's; smaller values are for ncu captures only)")
    args = ap.parse_args()
    wl = config_by_name(args.config)
    if args.events > 0:
        wl = wl.scaled(args.events)
    if args.seed is not None:
        from dataclasses import replace
        wl = replace(wl, seed=args.seed)
    if args.impl == "reference":
        return run_reference(args, wl)
    if args.warmup < 3:
        args.warmup = 3
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` on its own: start N ranks (one per GPU) under torch.distributed.run
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))

    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2106_10279_b200 import api, build, integrate
    from paper_2106_10279_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    if world != args.gpus:
        raise SystemExit("bench.py: --gpus %d but %d rank(s) were launched (WORLD_SIZE)" % (args.gpus, world))
    if local_rank >= torch.cuda.device_count():
        raise SystemExit("bench.py: rank %d has no GPU (%d visible)" % (local_rank, torch.cuda.device_count()))
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    build.build()
    proc = api.Process(wl, W.pdf_for(wl.process))
    n = wl.n_events                                   # per rank (weak scaling: shards need no exchange until
    first_event = rank * n                            # the per-iteration sums)
    stream = torch.cuda.current_stream()
    grid = proc.new_grid()
    hist, res = proc.new_hist(), proc.new_result()
    capacity = max(1 << 16, n // 64)
    records = torch.zeros(capacity * proc.record_size, dtype=torch.uint8, device="cuda")
    count = torch.zeros(1, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    state = {"k": 0, "w_max": 0.0, "pass": 0, "events": 0}

    def step(timed):
        """iteration k: mf_unweight (all of a1-a12 + a14; the first one, with no w_max yet, is mf_vegas_iterate)
        then the exchange (N>1) and mf_refine_grid (a13)"""
        k = state["k"]
        flush.fill_(k & 0xFF)                          # flush L2 between steps (outside the step's events)
        count.zero_()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        if state["w_max"] > 0.0:
            proc.unweight(grid, wl.seed, k, first_event, n, state["w_max"], records, capacity, count, hist, res)
        else:
            proc.vegas_iterate(grid, wl.seed, k, first_event, n, hist, res)
        if world > 1:
            integrate.combine_across_ranks(hist, res)
        proc.refine_grid(grid, hist, W.VEGAS_ALPHA)
        e1.record(stream)
        e1.synchronize()
        r = proc.result_to_host(res)
        state["w_max"] = max(state["w_max"], r.max_abs_w)
        state["k"] = k + 1
        if timed:
            state["pass"] += r.n_pass
            state["events"] += n * world
        return e0.elapsed_time(e1), r

    for _ in range(args.warmup):
        step(False)
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t_wall = time.perf_counter()
    ms = []
    last = None
    for _ in range(args.steps):
        t, last = step(True)
        ms.append(t)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop() if rank == 0 else None
    total_ms = torch.tensor([sum(ms)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_ms = float(total_ms.item())
    value = n * world * args.steps / (total_ms * 1e-3)

    # ---- kernel-only timing of the dominant kernel (the fused pass) for the roofline -----------------------------
    kern_ms = []
    for _ in range(3):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        count.zero_()
        flush.fill_(1)
        e0.record(stream)
        proc.unweight(grid, wl.seed, state["k"], first_event, n, state["w_max"], records, capacity, count, None, res)
        e1.record(stream)
        e1.synchronize()
        kern_ms.append(e0.elapsed_time(e1))
    r_k = proc.result_to_host(res)
    kern = sorted(kern_ms)[1]
    flops_launch = r_k.n_pass * me_flops(wl.process) + n * OTHER_FLOPS[wl.process]
    achieved = flops_launch / (kern * 1e-3) / 1e12

    # ---- end to end through the C ABI with host buffers -----------------------------------------------------------
    h_grid = grid.cpu().pin_memory()
    h_res = torch.empty(5, dtype=torch.float64).pin_memory()
    h_hist = torch.empty((proc.n_dims, proc.n_bins), dtype=torch.float64).pin_memory()
    h_count = torch.empty(1, dtype=torch.int64).pin_memory()
    h_rec = torch.empty(capacity * proc.record_size, dtype=torch.uint8).pin_memory()
    h2d = d2h = 0
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(args.steps):
        k = state["k"] + 1 + i
        grid.copy_(h_grid, non_blocking=True)
        count.zero_()
        proc.unweight(grid, wl.seed, k, first_event, n, state["w_max"], records, capacity, count, hist, res)
        if world > 1:
            integrate.combine_across_ranks(hist, res)
        proc.refine_grid(grid, hist, W.VEGAS_ALPHA)
        h_res.copy_(res, non_blocking=True)
        h_hist.copy_(hist, non_blocking=True)
        h_grid.copy_(grid, non_blocking=True)
        h_count.copy_(count, non_blocking=True)
        torch.cuda.synchronize()
        nrec = min(int(h_count.item()), capacity)
        nb = nrec * proc.record_size
        h_rec[:nb].copy_(records[:nb])
        if i == 0:
            h2d = h_grid.numel() * 8
            d2h = (h_res.numel() + h_hist.numel() + h_grid.numel() + 1) * 8 + nb
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t_e2e = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
    e2e_value = n * world * args.steps / float(t_e2e.item())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak_flops, _ = api.mf_measure_fp64_peak(1 << 17)
    peak = peak_flops / 1e12
    dmma_flops, _ = api.mf_measure_dmma_peak(1 << 14)
    out = {
        "metric": metric_for(wl), "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "ms_per_step_median": sorted(ms)[len(ms) // 2], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: BASELINE.json configs[%d], %d events/step/GPU, step = mf_unweight + mf_refine_grid"
                               % (wl.name, wl.process if args.config != "C4" else 4, n),
                   "events_per_step": n * world, "n_bins": wl.n_bins, "seed": wl.seed,
                   "l2": "256 MiB flush write between steps; the pass reads ~10 kB of tables and no per-event HBM",
                   "launch": {"blocks": proc.blocks, "threads": proc.threads}},
        "clocks": clocks, "gpu_launches": LAUNCHES_PER_STEP.get(wl.process, 3) * args.steps,
        "wall_ms_per_step_incl_flush": 1e3 * t_wall / args.steps,
        "pass_rate": state["pass"] / max(state["events"], 1),
        "me_evals_per_s": value * state["pass"] / max(state["events"], 1),
        "n_accept_last_step": last.n_accept,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
        "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                     "traffic": MEASURED_TRAFFIC.get((wl.process, n)), "traffic_source": "profiles/r1_coop_v4_traffic.md",
                     "kernel": "fused_pass_cta_kernel<true>" if wl.process == 6 else ("fused_pass_coop_kernel<%d,true>" if wl.process >= 2 else "fused_pass_kernel<%d,true>") % wl.process, "kernel_ms": kern,
                     "flops_per_me": me_flops(wl.process), "flops_per_event_outside_me": OTHER_FLOPS[wl.process],
                     "flops_source": ("static count of csrc/%s" % FLOP_HEADERS[wl.process][0] if wl.process in FLOP_HEADERS and wl.process not in ME_FLOPS_MEASURED
                                      else "ncu-executed total, " + FLOP_PROFILES[wl.process]),
                     "peak_source": "mf_measure_fp64_peak (DFMA chains) on this GPU",
                     "dmma_peak": dmma_flops / 1e12,
                     "nominal_peak": NOMINAL_FP64 / 1e12, "frac_of_nominal": achieved / (NOMINAL_FP64 / 1e12)},
    }
    if world == 1 and not args.no_cpu_baseline:
        v, ns, dt = oracle_sample(args.config)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": "events [0,%d) of iteration 0 of %s on the uniform grid, %.1f s, 1 thread of %d"
                                         % (ns, wl.name, dt, os.cpu_count())}
        allc = oracle_all_cores(args.config, dt / ns)
        if allc is not None:    # context only: the same program, one process per logical core (start-up included)
            out["cpu_baseline_all_cores"] = {"value": allc[0], "unit": UNIT, "cores": allc[1], "kind": "oracle",
                                             "sample": "%d processes x %d events, disjoint index ranges, %.1f s wall"
                                                       % (allc[1], allc[2], allc[3])}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
