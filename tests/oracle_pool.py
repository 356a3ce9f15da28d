"""The oracle as P independent single-threaded processes on disjoint event-index ranges (SURVEY.md §8(c) parity protocol
(iii)): possible because the RNG is counter based; the oracle itself stays as it is, one event at a time on one thread.
Partials are added in index order (math.fsum), accepted records are concatenated in index order, so the result is the
single-process result up to the rounding of P partial sums (1e-16 relative; the parity tolerances are 1e-9).

Test infrastructure only: imports oracle/, never the CUDA binding.  Workers are SPAWNED (not forked), so a parent that
holds a CUDA context is safe."""
import math
import multiprocessing as mp
import os

import numpy as np

_PROC = {}


def _handle(wl):
    from oracle import mfo
    from paper_2106_10279_b200 import workloads as W
    key = (wl.process, wl.sqrt_s, wl.alpha_s, wl.m_top, wl.mu2, wl.ptmin, wl.etamax, wl.drmin, wl.n_bins)
    if key not in _PROC:
        _PROC[key] = mfo.Process(wl, W.pdf_for(wl.process))
    return _PROC[key]


def _work(task):
    kind, wl, grid, seed, it, first, n, w_max, dyn = task
    op = _handle(wl)
    if dyn:
        op.set_dynamic_scale(True)
    try:
        if kind == "rows":
            return op.debug_eval(grid, seed, it, first, n)
        if kind == "iterate":
            hist, r = op.vegas_iterate(grid, seed, it, first, n)
            return hist, (r.sum_w, r.sum_w2, r.max_abs_w, r.n_pass, 0), None
        rec, cnt, hist, r = op.unweight(grid, seed, it, first, n, w_max, n)
        return hist, (r.sum_w, r.sum_w2, r.max_abs_w, r.n_pass, r.n_accept), op.records_array(rec, cnt).copy()
    finally:
        if dyn:
            op.set_dynamic_scale(False)


class IterSums:
    def __init__(self, sum_w, sum_w2, max_abs_w, n_pass, n_accept):
        self.sum_w, self.sum_w2, self.max_abs_w, self.n_pass, self.n_accept = sum_w, sum_w2, max_abs_w, n_pass, n_accept


class OraclePool:
    def __init__(self, n_procs=None):
        self.n = n_procs or max(1, os.cpu_count() or 1)
        self.pool = mp.get_context("spawn").Pool(self.n)

    def close(self):
        self.pool.terminate()
        self.pool.join()

    def _chunks(self, first, n):
        per = max(1, -(-n // (4 * self.n)))          # 4 chunks per worker: the cut pass rate varies along the stream
        out, a = [], first
        while a < first + n:
            m = min(per, first + n - a)
            out.append((a, m))
            a += m
        return out

    def debug_eval(self, wl, grid, seed, it, first, n, dyn=False):
        parts = self.pool.map(_work, [("rows", wl, grid, seed, it, a, m, 0.0, dyn) for a, m in self._chunks(first, n)])
        return np.concatenate(parts, axis=0)

    def windows(self, wl, grid, seed, it, firsts, n):
        """debug rows of several windows [f, f + n) at once; returns a list of arrays"""
        return self.pool.map(_work, [("rows", wl, grid, seed, it, int(f), n, 0.0, False) for f in firsts])

    def iterate(self, wl, grid, seed, it, first, n, w_max=None, dyn=False):
        """mfo_vegas_iterate (w_max None) or mfo_unweight over [first, first + n): (hist, IterSums, records or None)"""
        kind = "iterate" if w_max is None else "unweight"
        parts = self.pool.map(_work, [(kind, wl, grid, seed, it, a, m, w_max or 0.0, dyn) for a, m in self._chunks(first, n)])
        if not parts:
            D = wl.n_dims
            return np.zeros((D, wl.n_bins)), IterSums(0.0, 0.0, 0.0, 0, 0), None
        hist = np.zeros_like(parts[0][0])
        for h, _, _ in parts:
            hist += h
        s = IterSums(math.fsum(p[1][0] for p in parts), math.fsum(p[1][1] for p in parts), max(p[1][2] for p in parts),
                     sum(p[1][3] for p in parts), sum(p[1][4] for p in parts))
        rec = np.concatenate([p[2] for p in parts]) if w_max is not None else None
        return hist, s, rec
