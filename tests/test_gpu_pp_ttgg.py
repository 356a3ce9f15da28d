"""GPU <-> oracle parity for pp -> ttbar gg = g g -> t tbar g g + q qbar -> t tbar g g of four flavours (process 7; SURVEY.md
8(f2); Table 1: 267 diagrams) through the two C ABIs.  The gluon channel is the cooperative program of
process 3, the quark channel the current-based csrc/mf_me_qqttgg.cuh by one warp per event in a kernel ahead of it; the oracle is the 36 diagrams with
explicit colour tensors (oracle/amplitude_qq.hpp, 13 ms per event: it runs through tests/oracle_pool.py).  Tolerances of
tests/test_gpu_parity.py: uniforms, bins, accept and channel draws bit-exact; |M|^2 and weights 1e-10; iteration sums 1e-9."""
import math

import numpy as np
import pytest

from conftest import adapted_grid
from paper_2106_10279_b200 import workloads as W
from test_gpu_parity import _check_sums, _cols, _compare_rows, _iterate_gpu

pytestmark = pytest.mark.gpu
PID = W.MF_PP_TTGG
WL = W.C8


def _torch():
    import torch
    return torch


def test_me2_both_channels(gpu_procs, oracle_procs):
    from oracle import mfo
    from paper_2106_10279_b200 import api
    rng = np.random.default_rng(71)
    pts = []
    for _ in range(70):                        # more than one 64-thread debug block
        w = 500.0 + 5000.0 * rng.random() ** 2
        k, _ = mfo.rambo([173.0, 173.0, 0.0, 0.0], w, rng.random(16))
        pts.append(np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k]))
    pts = np.array(pts)
    # the gluon channel is process 3's matrix element
    g = gpu_procs[PID].debug_me2(pts)
    assert np.array_equal(g, gpu_procs[W.MF_GG_TTGG].debug_me2(pts))
    for i in range(0, 70, 7):
        assert abs(g[i] / oracle_procs[PID].me2(pts[i]) - 1) < 1e-10, i
    # the quark channel, quark from beam 1 and from beam 2
    for swap in (False, True):
        p = pts[:, [1, 0, 2, 3, 4, 5]] if swap else pts
        q = api.debug_me2_quark_gluon(3, WL.m_top, WL.alpha_s, p)
        for i in range(len(p)):
            assert abs(q[i] / mfo.me2_qq_ttbar_gg(p[i], WL.m_top, WL.alpha_s) - 1) < 1e-10, (swap, i)


@pytest.mark.parametrize("grid_kind", ["uniform", "adapted"])
def test_per_event_rows(grid_kind, gpu_procs, oracle_procs, oracle_pool):
    gp, op = gpu_procs[PID], oracle_procs[PID]
    grid = W.uniform_grid(WL.n_dims) if grid_kind == "uniform" else adapted_grid(op, WL)
    dgrid = _torch().from_numpy(grid).cuda()
    n = 1000                                   # sixteen debug blocks, ragged
    for seed, it, first in [(0, 0, 0), (3, 5, (1 << 33) + 11)]:
        g = gp.debug_eval(dgrid, seed, it, first, n)
        o = oracle_pool.debug_eval(WL, grid, seed, it, first, n)
        assert _compare_rows(WL, g, o) <= 1
        c = _cols(WL)
        ok = o[:, c["pas"]] > 0
        assert 0.3 < ok.mean() < 1.0
        share = (o[ok, c["lum_qq"]] * o[ok, c["me2_qq"]]).sum() / (o[ok, c["lum"]] * o[ok, c["me2"]]).sum()
        assert 1e-3 < share < 0.2                # the quark channel is there and is the smaller one


def test_iteration_sums_edges_and_unweighting(gpu_procs, oracle_procs, oracle_pool):
    torch = _torch()
    gp, op = gpu_procs[PID], oracle_procs[PID]
    grid = adapted_grid(op, WL)
    n = 148 * 384 // 16 + 77                   # a ragged piece of one round of the fused pass over several blocks
    hg, rg = _iterate_gpu(gp, grid, 0, 2, 17, n)
    ho, ro, _ = oracle_pool.iterate(WL, grid, 0, 2, 17, n)
    _check_sums(n, hg, rg, ho, ro)
    h0, r0 = _iterate_gpu(gp, grid, 0, 0, 0, 0)
    assert r0.sum_w == 0 and r0.n_pass == 0 and not h0.any()
    for m, first in [(1, 3), (31, (1 << 40) + 3)]:
        hg, rg = _iterate_gpu(gp, grid, 9, 1, first, m)
        ho, ro, _ = oracle_pool.iterate(WL, grid, 9, 1, first, m)
        _check_sums(m, hg, rg, ho, ro)
    # unweighting with a small w_max: many accepted events, so that quark channels are drawn
    n = 3000
    rows = oracle_pool.debug_eval(WL, grid, 0, 5, 3, 300)
    absw = np.abs(rows[:, _cols(WL)["w"]])
    w_max = float(np.quantile(absw[absw > 0], 0.2))
    ho, ro, rec_o = oracle_pool.iterate(WL, grid, 0, 5, 3, n, w_max=w_max)
    assert ro.n_accept > 1000
    dgrid = torch.from_numpy(grid).cuda()
    for capacity, start in [(n, 0), (ro.n_accept // 2, 0), (n, 4)]:
        records = torch.zeros(max(capacity, 1) * gp.record_size, dtype=torch.uint8, device="cuda")
        count = torch.full((1,), start, dtype=torch.int64, device="cuda")
        hist, res = gp.new_hist(), gp.new_result()
        gp.unweight(dgrid, 0, 5, 3, n, w_max, records, capacity, count, hist, res)
        torch.cuda.synchronize()
        r = gp.result_to_host(res)
        assert int(count.item()) == start + ro.n_accept and r.n_accept == ro.n_accept
        _check_sums(n, hist.cpu().numpy(), r, ho, ro)
        n_written = min(capacity, start + ro.n_accept) - start
        rec_g = gp.records_array(records[start * gp.record_size:], max(n_written, 0))
        if capacity >= start + ro.n_accept:
            order = np.argsort(rec_g["id"])
            assert np.array_equal(rec_g["id"][order], rec_o["id"])
            np.testing.assert_allclose(rec_g["w"][order], rec_o["w"], rtol=1e-10)
            scale = np.abs(rec_o["mom"]).max(axis=(1, 2), keepdims=True)
            assert np.max(np.abs(rec_g["mom"][order] - rec_o["mom"]) / scale) < 1e-11
            # R22: the partonic channel, an integer decided in fp64 on both sides
            assert np.array_equal(rec_g["channel"][order], rec_o["channel"])
            ch = rec_o["channel"].astype(np.int64)
            assert ch.max() <= 2 * W.N_FLAVOURS and (ch == 0).any() and (ch > 0).sum() >= 3
        else:
            assert int(count.item()) > capacity and set(rec_g["id"].tolist()) <= set(rec_o["id"].tolist())


def test_pipeline_reduced_n(gpu_procs, oracle_procs, oracle_pool):
    """three adapting iterations of 4096 events, each side refining its own grid"""
    from paper_2106_10279_b200 import integrate
    n, n_it = 1 << 12, 3
    wl = WL.scaled(n, n_it, n_it)
    gp, op = gpu_procs[PID], oracle_procs[PID]
    hists = []
    run = integrate.run_config(gp, wl, hists=hists)
    grid = W.uniform_grid(wl.n_dims)
    for k in range(n_it):
        ho, ro, _ = oracle_pool.iterate(wl, grid, wl.seed, k, 0, n)
        rec = run.iterations[k]
        assert rec.n_pass == ro.n_pass
        Io = ro.sum_w / n
        so = np.sqrt((ro.sum_w2 / n - Io * Io) / (n - 1))
        assert abs(rec.integral - Io) <= 1e-9 * abs(Io) and abs(rec.sigma - so) <= 1e-9 * so
        np.testing.assert_allclose(hists[k], ho, rtol=1e-8, atol=1e-14 * ho.max())
        grid = op.refine_grid(grid, ho, W.VEGAS_ALPHA)
    np.testing.assert_allclose(run.grid.cpu().numpy(), grid, rtol=0, atol=1e-10)


def test_full_size_sampled(gpu_procs, oracle_procs, oracle_pool):
    """the 2^22-event launch bench.py --config C8 times: additivity, determinism, 32 oracle windows of 64 events"""
    gp, op = gpu_procs[PID], oracle_procs[PID]
    n = WL.n_events
    grid = adapted_grid(op, WL)
    hg, rg = _iterate_gpu(gp, grid, 0, 3, 0, n)
    hg2, rg2 = _iterate_gpu(gp, grid, 0, 3, 0, n)
    assert (rg.sum_w, rg.sum_w2, rg.n_pass) == (rg2.sum_w, rg2.sum_w2, rg2.n_pass)
    cut = n // 3 + 7
    ha, ra = _iterate_gpu(gp, grid, 0, 3, 0, cut)
    hb, rb = _iterate_gpu(gp, grid, 0, 3, cut, n - cut)
    assert ra.n_pass + rb.n_pass == rg.n_pass
    assert abs(ra.sum_w + rb.sum_w - rg.sum_w) <= 1e-11 * abs(rg.sum_w)
    assert abs(ra.sum_w2 + rb.sum_w2 - rg.sum_w2) <= 1e-11 * rg.sum_w2
    np.testing.assert_allclose(ha + hb, hg, rtol=1e-9, atol=1e-12 * hg.max())
    # the quark channel raises the cross section over process 3's on the same grid and stream
    _, r3 = _iterate_gpu(gpu_procs[W.MF_GG_TTGG], grid, 0, 3, 0, n)
    assert r3.n_pass == rg.n_pass and 1.001 < rg.sum_w / r3.sum_w < 1.2
    rng = np.random.default_rng(6)
    wn = 64
    firsts = [int(f) for f in rng.integers(0, n - wn, 32)]
    dgrid = _torch().from_numpy(grid).cuda()
    c = _cols(WL)
    for first, o in zip(firsts, oracle_pool.windows(WL, grid, 0, 3, firsts, wn)):
        g = gp.debug_eval(dgrid, 0, 3, first, wn)
        _compare_rows(WL, g, o)
        _, rw = _iterate_gpu(gp, grid, 0, 3, first, wn)
        wo = o[:, c["w"]]
        assert rw.n_pass == int(o[:, c["pas"]].sum())
        assert abs(rw.sum_w - math.fsum(wo)) <= 1e-9 * abs(math.fsum(wo))


def test_call_larger_than_the_quark_term_buffer(gpu_procs, oracle_procs):
    """more than 2^22 events in one call: the library runs it as consecutive pieces (its per-event quark terms live in a buffer
    made at create: the hot calls never allocate) and adds their sums in piece order; records and channels span the pieces"""
    torch = _torch()
    gp, op = gpu_procs[PID], oracle_procs[PID]
    grid = adapted_grid(op, WL)
    n1 = 1 << 22
    n = n1 + 100_003
    hg, rg = _iterate_gpu(gp, grid, 0, 4, 0, n)
    ha, ra = _iterate_gpu(gp, grid, 0, 4, 0, n1)
    hb, rb = _iterate_gpu(gp, grid, 0, 4, n1, n - n1)
    assert rg.n_pass == ra.n_pass + rb.n_pass
    assert rg.sum_w == ra.sum_w + rb.sum_w and rg.sum_w2 == ra.sum_w2 + rb.sum_w2      # the same two numbers, added once
    assert rg.max_abs_w == max(ra.max_abs_w, rb.max_abs_w)
    np.testing.assert_allclose(hg, ha + hb, rtol=1e-12, atol=1e-14 * hg.max())
    # unweighting through both pieces: one cursor, channels drawn for the records of both
    dgrid = torch.from_numpy(grid).cuda()
    w_max = 300.0 * rg.sum_w / n          # 300 x the mean weight: about one event in 300 survives
    cap = 200_000
    out = []
    for first, m in [(0, n), (0, n1), (n1, n - n1)]:
        records = torch.zeros(cap * gp.record_size, dtype=torch.uint8, device="cuda")
        count = torch.zeros(1, dtype=torch.int64, device="cuda")
        res = gp.new_result()
        gp.unweight(dgrid, 0, 4, first, m, w_max, records, cap, count, None, res)
        torch.cuda.synchronize()
        k = int(count.item())
        assert 0 < k < cap and gp.result_to_host(res).n_accept == k
        rec = gp.records_array(records, k)
        out.append(rec[np.argsort(rec["id"])])
    whole, parts = out[0], np.concatenate(out[1:])
    assert len(whole) == len(parts) > 100 and (whole["id"] >= n1).any()
    assert np.array_equal(whole["id"], parts["id"]) and np.array_equal(whole["channel"], parts["channel"])
    assert np.array_equal(whole["w"], parts["w"]) and np.array_equal(whole["mom"], parts["mom"])
    assert (whole["channel"] > 0).any()
