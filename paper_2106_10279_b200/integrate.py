"""Integration driver over the C ABI: the VEGAS iteration loop of one configuration (SURVEY.md
§8(c) O13-O15).  Host policy only — which call runs in which iteration, when the grid is refined, which
w_max a frozen iteration uses, and how the per-iteration estimates combine.  All arithmetic on events is in
the library.

  iterations 0 .. n_adapt-1        mf_vegas_iterate, then mf_refine_grid
  iterations n_adapt .. n_it-1     frozen grid; mf_unweight if wl.unweight (w_max = largest max|w| returned by
                                   iterations n_adapt-1 .. k-1), else mf_vegas_iterate
"""
import math
from dataclasses import dataclass, field

from . import api
from . import workloads as W


@dataclass
class IterationRecord:
    iteration: int
    n_events: int
    sum_w: float
    sum_w2: float
    max_abs_w: float
    n_pass: int
    n_accept: int
    w_max_used: float = 0.0

    @property
    def integral(self):
        return self.sum_w / self.n_events

    @property
    def sigma(self):
        n = self.n_events
        var = (self.sum_w2 / n - self.integral ** 2) / (n - 1)
        return math.sqrt(max(var, 0.0))


@dataclass
class RunResult:
    iterations: list = field(default_factory=list)
    grid: object = None          # final grid (torch tensor, device)
    records: object = None       # uint8 tensor (device) or None
    n_records: int = 0           # accepted events (may exceed capacity: overflow signal)

    def combined(self):
        """I = sum(I_k/s_k^2)/sum(1/s_k^2), sigma = (sum 1/s_k^2)^-1/2, chi2/dof."""
        its = [r for r in self.iterations if r.sigma > 0]
        if not its:
            r = self.iterations[-1]
            return r.integral, r.sigma, 0.0
        sw = sum(1.0 / r.sigma ** 2 for r in its)
        mean = sum(r.integral / r.sigma ** 2 for r in its) / sw
        chi2 = sum((r.integral - mean) ** 2 / r.sigma ** 2 for r in its)
        return mean, sw ** -0.5, chi2 / max(len(its) - 1, 1)


def shard_range(n_events, rank, world):
    """Contiguous event-index range [first, first + n) of `rank` when n_events are split over `world` ranks
    (events are independent and the RNG is counter-based, so shards need no exchange
    until the per-iteration sums).  The first n_events % world ranks take one extra event."""
    base, extra = divmod(n_events, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def combine_across_ranks(hist, result, group=None):
    """The one exchange step of a sharded iteration: every rank contributes its mf_iter_result (5 x 8 bytes:
    sum_w, sum_w2, max_abs_w as fp64, n_pass, n_accept as u64) and its [D][nb] histogram; ONE all-gather of
    5 + D*nb words, then every rank adds the contributions in rank order, so all ranks hold bit-identical
    totals and refine their grids identically.  Works on CUDA tensors (NCCL) and CPU tensors (gloo).
    In place on `hist` and `result`."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    if world == 1:
        return
    buf = torch.cat([result.reshape(-1), hist.reshape(-1)]).contiguous()
    flat = torch.empty(world * buf.numel(), dtype=buf.dtype, device=buf.device)
    dist.all_gather_into_tensor(flat, buf, group=group)
    gathered = flat.view(world, buf.numel())
    total = gathered[0].clone()
    counts = gathered[:, 3:5].contiguous().view(torch.int64)
    for r in range(1, world):
        total[0:2] += gathered[r, 0:2]
        total[2] = torch.maximum(total[2], gathered[r, 2])
        total[5:] += gathered[r, 5:]
    total[3:5] = counts.sum(dim=0).view(torch.float64)
    result.copy_(total[:5].reshape(result.shape))
    hist.copy_(total[5:].reshape(hist.shape))


def run_config(proc, wl=None, capacity=0, stream=None, alpha=W.VEGAS_ALPHA, grid=None, hists=None, rank=0, world=1,
               weak=False, drain=None):
    """Runs every iteration of `wl` (default: proc.wl) on the GPU.  Returns a RunResult.
    `hists`, if a list, receives a host copy of each iteration's histogram (tests).
    world > 1: this rank processes its shard of each iteration's events (weak=False: wl.n_events split over
    the ranks; weak=True: wl.n_events PER rank) and the per-iteration sums are combined with
    combine_across_ranks before the (replicated, identical) grid refinement; records stay rank-local.
    `drain` (lhe.LheDrain): the records of every unweighting iteration are handed to it right after the call (the
    record buffer is then reused by the next iteration; out.n_records counts all drained events).
    `stream` (torch.cuda.Stream or None): every kernel, helper op and host read of the run is issued on it (the body
    runs with it as torch's current stream, so the small device->host reads of the w_max policy are ordered after the
    passes they depend on)."""
    import torch
    if stream is not None and stream != torch.cuda.current_stream():
        with torch.cuda.stream(stream):
            return run_config(proc, wl, capacity, None, alpha, grid, hists, rank, world, weak, drain)
    wl = proc.wl if wl is None else wl
    if world > 1:
        n_total = wl.n_events * world if weak else wl.n_events
        first_event, n_local = shard_range(n_total, rank, world)
    else:
        n_total, first_event, n_local = wl.n_events, 0, wl.n_events
    grid = proc.new_grid() if grid is None else grid
    hist = proc.new_hist()
    results = [proc.new_result() for _ in range(wl.n_iterations)]
    out = RunResult(grid=grid)
    count = None
    if wl.unweight:
        count = torch.zeros(1, dtype=torch.int64, device="cuda")
        out.records = torch.zeros(max(capacity, 1) * proc.record_size, dtype=torch.uint8, device="cuda")
    w_max_used = [0.0] * wl.n_iterations
    running_max = 0.0
    for k in range(wl.n_iterations):
        frozen = k >= wl.n_adapt
        if frozen and wl.unweight:
            # the running max needs the previous iteration's result: one small device->host read
            if k == wl.n_adapt:
                running_max = api.Process.result_to_host(results[k - 1]).max_abs_w if k > 0 else 0.0
            else:
                running_max = max(running_max, api.Process.result_to_host(results[k - 1]).max_abs_w)
            if not running_max > 0.0:
                raise api.MfError("unweighting needs a positive w_max from the last adapting iteration")
            w_max_used[k] = running_max
            if drain is not None:
                count.zero_()
            proc.unweight(grid, wl.seed, k, first_event, n_local, running_max, out.records, capacity, count, hist,
                          results[k], stream)
            if drain is not None:
                out.n_records += drain.push(out.records, count, running_max, capacity, stream)
        else:
            proc.vegas_iterate(grid, wl.seed, k, first_event, n_local, hist, results[k], stream)
        if world > 1:
            combine_across_ranks(hist, results[k])
        if hists is not None:
            hists.append(hist.cpu().numpy().copy())
        if not frozen:
            proc.refine_grid(grid, hist, alpha, stream)
    torch.cuda.synchronize()
    for k in range(wl.n_iterations):
        r = api.Process.result_to_host(results[k])
        out.iterations.append(IterationRecord(k, n_total, r.sum_w, r.sum_w2, r.max_abs_w, r.n_pass, r.n_accept,
                                              w_max_used[k]))
    if count is not None and drain is None:
        out.n_records = int(count.item())
    return out


def main(argv=None):
    """python -m paper_2106_10279_b200.integrate [--config C0..C4] [--events N]: runs every iteration of a
    BASELINE.json configuration on cuda:0 and prints the per-iteration and combined estimates with timings."""
    import argparse
    import json
    import time
    import torch
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", default="C3")
    ap.add_argument("--events", type=int, default=0, help="events per iteration (default: the configuration's)")
    ap.add_argument("--capacity", type=int, default=1 << 20, help="record buffer capacity (unweighting configs)")
    ap.add_argument("--observables", type=int, default=0, metavar="NBINS",
                    help="also accumulate d sigma / d pT and d sigma / d eta of the first final-state particle "
                         "(PAPER.md Fig. 2) in NBINS bins over the frozen-grid / last iteration and print them")
    ap.add_argument("--lhe", default="", metavar="FILE", help="unweighting configs (C4): drain the accepted events of every "
                    "frozen iteration asynchronously into this LHE 3.0 file (.gz = compressed; PAPER.md L81)")
    ap.add_argument("--dynamic-scale", action="store_true",
                    help="mu^2 = m_t^2 + pT(top)^2 per event with one-loop running alpha_s (mf_set_dynamic_scale)")
    ap.add_argument("--pt-max", type=float, default=600.0)
    ap.add_argument("--eta-max", type=float, default=3.0)
    args = ap.parse_args(argv)
    wl = {"C0": W.C0, "C1": W.C1, "C2": W.C2, "C3": W.C3, "C4": W.C4, **W.EXTRA_CONFIGS}[args.config]
    if args.events > 0:
        wl = wl.scaled(args.events)
    proc = api.Process(wl, W.pdf_for(wl.process))
    if args.dynamic_scale:
        proc.set_dynamic_scale(True)
    run_config(proc, wl.scaled(min(wl.n_events, 1 << 16)), capacity=args.capacity if wl.unweight else 0)   # warm-up
    torch.cuda.synchronize()
    drain = None
    if args.lhe and wl.unweight:
        from . import lhe
        drain = lhe.LheDrain(args.lhe, proc)
    t0 = time.perf_counter()
    run = run_config(proc, wl, capacity=args.capacity if wl.unweight else 0, drain=drain)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    if drain is not None:
        mean, err, _ = run.combined()
        print("LHE: %d events written to %s" % (drain.close(mean, err), args.lhe))
    for r in run.iterations:
        print("iteration %2d  I = %.8g +- %.3g pb  max|w| = %.4g  pass %.4f  accepted %d" %
              (r.iteration, r.integral, r.sigma, r.max_abs_w, r.n_pass / r.n_events, r.n_accept))
    mean, err, chi2 = run.combined()
    n_tot = sum(r.n_events for r in run.iterations)
    if args.observables > 0:
        # one more iteration on the final grid with the observable histograms attached (mf_set_observables)
        nb = args.observables
        obs = torch.zeros((2, nb + 1), dtype=torch.float64, device="cuda")
        proc.set_observables(obs, nb, args.pt_max, args.eta_max)
        res = proc.new_result()
        proc.vegas_iterate(run.grid, wl.seed, wl.n_iterations, 0, wl.n_events, None, res)
        torch.cuda.synchronize()
        proc.set_observables(None)
        h = (obs / wl.n_events).cpu().numpy()
        dpt, deta = args.pt_max / nb, 2 * args.eta_max / nb
        print("pT bin [GeV]      d sigma / d pT [pb / GeV]   |   eta bin          d sigma / d eta [pb]")
        for i in range(nb):
            print("%7.1f - %-7.1f  %-12.5g               |   %+5.2f - %+5.2f    %-12.5g" %
                  (i * dpt, (i + 1) * dpt, h[0, i] / dpt, -args.eta_max + i * deta, -args.eta_max + (i + 1) * deta,
                   h[1, i] / deta))
        print("outside the ranges: %.5g pb (pT), %.5g pb (eta)" % (h[0, nb], h[1, nb]))
    print(json.dumps({"config": args.config, "workload": wl.name, "integral_pb": mean, "error_pb": err,
                      "chi2_per_dof": chi2, "iterations": len(run.iterations), "events_per_iteration": wl.n_events,
                      "wall_s": dt, "events_per_s": n_tot / dt, "unweighted_events": run.n_records}))
    proc.close()


if __name__ == "__main__":
    main()
