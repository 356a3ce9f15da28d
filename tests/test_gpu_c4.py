"""BASELINE.json configs[4] (C4): gg -> ttbar gg, 5 grid-adapting iterations, then 5 frozen-grid iterations with
hit-or-miss unweighting against the running maximum weight, stream-compacted into a device buffer (
SURVEY.md O15).  (i) the whole 5 + 5 schedule through integrate.run_config at reduced N against an oracle-side replay
of the same w_max policy written out here; (ii) one launch at the config's full 2^26 events checked by additivity,
determinism and oracle parity on sampled windows of the same Philox stream."""
import numpy as np
import pytest

from conftest import adapted_grid
from paper_2106_10279_b200 import workloads as W

pytestmark = pytest.mark.gpu

REL_EVENT, REL_ITER = 1e-10, 1e-9


def _tie_ids(op, wl, grid, seed, it, ids, w_max):
    """of the event ids given, those whose accept decision lies within rounding: |r w_max - |w|| < 1e-10 |w| (O15)"""
    c = wl.n_dims + 4 * (wl.n_final + 2)
    out = set()
    for e in ids:
        row = op.debug_eval(grid, seed, it, int(e), 1)[0]
        w, r = abs(row[c + 6]), row[c + 8]
        if abs(r * w_max - w) < 1e-10 * w:
            out.add(int(e))
    return out


def test_c4_schedule(gpu_procs, oracle_procs, oracle_pool):
    from paper_2106_10279_b200 import integrate
    n = 1 << 13
    wl = W.C4.scaled(n)                      # 10 iterations, 5 adapting, unweighting on the frozen ones
    assert wl.n_iterations == 10 and wl.n_adapt == 5 and wl.unweight
    gp, op = gpu_procs[3], oracle_procs[3]
    hists = []
    run = integrate.run_config(gp, wl, capacity=4 * n, hists=hists)
    rec_g = gp.records_array(run.records, min(run.n_records, 4 * n))
    assert run.n_records <= 4 * n
    # ---- the oracle's replay of the same schedule (policy: SURVEY.md O15 / DESIGN.md R15) -------------------------------
    # Adapting iterations: each side refines its OWN grid (sums 1e-9; a single event's weight, max|w|, follows the two
    # grids' rounding differences amplified by the narrowest bin: 1e-8).  Frozen iterations: the grid is caller-owned, so
    # the oracle takes the GPU's final grid (checked equal to its own within 1e-11) and the GPU's w_max (the policy
    # itself is checked exactly on the GPU's own numbers): same inputs, so weights 1e-10 and decisions bit-exact.
    grid = W.uniform_grid(wl.n_dims)
    cursor = 0
    for k in range(10):
        frozen = k >= 5
        it = run.iterations[k]
        if frozen:
            w_max = max(r.max_abs_w for r in run.iterations[4:k])       # the largest max|w| returned by iterations 4 .. k-1
            assert it.w_max_used == w_max
            ho, ro, rec_o = oracle_pool.iterate(wl, grid, wl.seed, k, 0, n, w_max=w_max)
        else:
            assert it.w_max_used == 0.0 and it.n_accept == 0
            ho, ro, rec_o = oracle_pool.iterate(wl, grid, wl.seed, k, 0, n)
        assert it.n_pass == ro.n_pass
        Io = ro.sum_w / n
        so = np.sqrt((ro.sum_w2 / n - Io * Io) / (n - 1))
        assert abs(it.integral - Io) <= REL_ITER * abs(Io), (k, it.integral, Io)
        assert abs(it.sigma - so) <= REL_ITER * so, (k, it.sigma, so)
        assert abs(it.max_abs_w - ro.max_abs_w) <= (REL_EVENT if frozen else 1e-8) * ro.max_abs_w
        np.testing.assert_allclose(hists[k], ho, rtol=1e-8, atol=1e-14 * ho.max())
        if frozen:
            mine = rec_g[cursor:cursor + it.n_accept]          # iteration k's records follow those of k-1 in the buffer
            cursor += it.n_accept
            ids_g, ids_o = set(mine["id"].tolist()), set(rec_o["id"].tolist())
            assert len(ids_g) == it.n_accept
            if ids_g != ids_o:
                diff = ids_g ^ ids_o
                assert diff == _tie_ids(op, wl, grid, wl.seed, k, diff, w_max), "accept decisions differ away from a tie"
            else:
                assert it.n_accept == ro.n_accept
            order = np.argsort(mine["id"])
            common = np.isin(mine["id"][order], rec_o["id"])
            sel_o = np.isin(rec_o["id"], mine["id"])
            np.testing.assert_allclose(mine["w"][order][common], rec_o["w"][sel_o], rtol=REL_EVENT)
            scale = np.abs(rec_o["mom"][sel_o]).max(axis=(1, 2), keepdims=True)
            assert np.max(np.abs(mine["mom"][order][common] - rec_o["mom"][sel_o]) / scale) < 1e-11
        else:
            grid = op.refine_grid(grid, ho, W.VEGAS_ALPHA)
            if k == 4:
                g_grid = run.grid.cpu().numpy()
                # two independent pipelines, five refinements each: the edges drift apart by the histograms' 1e-9
                # differences (with the SAME histogram in, the refined edges agree to 2e-14: test_refine_grid)
                np.testing.assert_allclose(g_grid, grid, rtol=0, atol=5e-10)
                grid = g_grid
    assert cursor == run.n_records > 0
    assert sum(r.n_accept for r in run.iterations[5:]) == run.n_records


def test_c4_full_size_launch(gpu_procs, oracle_procs, oracle_pool):
    """One mf_unweight launch over the 2^26 events of a C4 iteration, in the launch configuration bench.py times."""
    import torch
    wl = W.C4
    n = wl.n_events
    assert n == 1 << 26
    gp, op = gpu_procs[3], oracle_procs[3]
    grid = adapted_grid(op, W.C3)
    dgrid = torch.from_numpy(grid).cuda()
    seed, it = 0, 7
    cap = 1 << 20

    def launch(first, m, w_max, with_hist=True):
        records = torch.zeros(cap * gp.record_size, dtype=torch.uint8, device="cuda")
        count = torch.zeros(1, dtype=torch.int64, device="cuda")
        hist, res = (gp.new_hist() if with_hist else None), gp.new_result()
        gp.unweight(dgrid, seed, it, first, m, w_max, records, cap, count, hist, res)
        torch.cuda.synchronize()
        c = int(count.item())
        assert c <= cap
        return gp.result_to_host(res), (hist.cpu().numpy() if with_hist else None), gp.records_array(records, c)

    # w_max = 500 x the mean weight of a 2^22-event pass over the head of the stream: ~0.1 % of the events are accepted,
    # the heavy tail of the weight distribution above w_max always (overweight events); then the full launch
    r0, _, _ = launch(0, 1 << 22, 1e300)
    w_max = 500.0 * r0.sum_w / (1 << 22)
    assert 0 < w_max < r0.max_abs_w
    rf, hf, recf = launch(0, n, w_max)
    assert rf.n_accept == len(recf) > 10000 and rf.n_pass < n and rf.n_pass > 0.5 * n
    assert (np.abs(recf["w"]) >= w_max).sum() > 10
    # determinism: sums bit-identical, same accepted set
    rf2, hf2, recf2 = launch(0, n, w_max)
    assert (rf.sum_w, rf.sum_w2, rf.max_abs_w, rf.n_pass, rf.n_accept) == (rf2.sum_w, rf2.sum_w2, rf2.max_abs_w, rf2.n_pass, rf2.n_accept)
    assert np.array_equal(np.sort(recf["id"]), np.sort(recf2["id"]))
    np.testing.assert_allclose(hf, hf2, rtol=1e-12)
    # additivity over index ranges
    cut = n // 3 + 5
    ra, ha, reca = launch(0, cut, w_max)
    rb, hb, recb = launch(cut, n - cut, w_max)
    assert ra.n_pass + rb.n_pass == rf.n_pass and ra.n_accept + rb.n_accept == rf.n_accept
    assert abs(ra.sum_w + rb.sum_w - rf.sum_w) <= 1e-11 * abs(rf.sum_w)
    assert abs(ra.sum_w2 + rb.sum_w2 - rf.sum_w2) <= 1e-11 * rf.sum_w2
    assert max(ra.max_abs_w, rb.max_abs_w) == rf.max_abs_w
    np.testing.assert_allclose(ha + hb, hf, rtol=1e-9, atol=1e-12 * hf.max())
    assert np.array_equal(np.sort(np.concatenate([reca["id"], recb["id"]])), np.sort(recf["id"]))
    # records are self-consistent: ids unique and in range, momentum conserved, |w| > 0
    assert len(np.unique(recf["id"])) == len(recf) and recf["id"].max() < n
    mom = recf["mom"]
    assert np.max(np.abs(mom[:, 0] + mom[:, 1] - mom[:, 2:].sum(axis=1))) < 1e-8 * 6500
    assert np.all(np.abs(recf["w"]) > 0)
    # sampled windows of the same stream against the oracle: per-event rows, and the accepted ids inside each window
    rng = np.random.default_rng(4)
    wn, n_win = 256, 64
    firsts = [int(f) for f in rng.integers(0, n - wn, n_win)]
    # plus windows around accepted events, so that the accepted set is tested where it is not empty
    firsts += [max(0, int(e) - 100) for e in np.sort(recf["id"])[:: max(1, len(recf) // 16)][:16]]
    rows_o = oracle_pool.windows(W.C3, grid, seed, it, firsts, wn)
    from test_gpu_parity import _compare_rows, _cols
    c = _cols(W.C3)
    ids_f = np.sort(recf["id"])
    n_acc_windows = 0
    for first, o in zip(firsts, rows_o):
        g = gp.debug_eval(dgrid, seed, it, first, wn)
        assert _compare_rows(W.C3, g, o) <= 1
        w, r = np.abs(o[:, c["w"]]), o[:, c["r"]]
        acc_o = first + np.where(r * w_max < w)[0]
        tie = np.abs(r * w_max - w) < 1e-10 * w
        assert not tie[w > 0].any()
        acc_g = ids_f[(ids_f >= first) & (ids_f < first + wn)]
        assert np.array_equal(acc_g, acc_o)
        n_acc_windows += len(acc_o) > 0
        sel = np.isin(recf["id"], acc_o)
        if sel.any():
            wg = recf["w"][sel][np.argsort(recf["id"][sel])]
            np.testing.assert_allclose(wg, o[acc_o - first, c["w"]], rtol=REL_EVENT)
    assert n_acc_windows >= 16


def test_run_config_on_a_side_stream(gpu_procs):
    """run_config(stream=...) must give the default-stream result (every host read ordered on that stream)."""
    import torch
    from paper_2106_10279_b200 import integrate
    gp = gpu_procs[1]
    wl = W.C5.scaled(1 << 15, 6, 3)
    wl = type(wl)(**{**wl.__dict__, "process": 1, "name": "C1 with unweighting"})
    a = integrate.run_config(gp, wl, capacity=1 << 15)
    side = torch.cuda.Stream()
    filler = torch.empty(64 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(20):
        filler.fill_(1)                       # keep the default stream busy: an unordered read would be stale
    b = integrate.run_config(gp, wl, capacity=1 << 15, stream=side)
    assert a.n_records == b.n_records > 0
    # (the refined grids agree to rounding only: the w^2 histograms are accumulated with shared-memory atomics)
    for x, y in zip(a.iterations, b.iterations):
        assert (x.n_pass, x.n_accept) == (y.n_pass, y.n_accept)
        for u, v in ((x.sum_w, y.sum_w), (x.sum_w2, y.sum_w2), (x.max_abs_w, y.max_abs_w), (x.w_max_used, y.w_max_used)):
            assert abs(u - v) <= 1e-11 * abs(u)
    assert a.iterations[0].sum_w == b.iterations[0].sum_w          # same grid in: bit-identical sums
    assert torch.allclose(a.grid, b.grid, rtol=0, atol=1e-12)


_NCCL_WORKER = r"""
import os, sys
sys.path.insert(0, os.environ["MF_ROOT"])
import torch, torch.distributed as dist
from paper_2106_10279_b200 import api, integrate, workloads as W
rank = int(os.environ["RANK"])
torch.cuda.set_device(rank)
dist.init_process_group("nccl", device_id=torch.device("cuda", rank))
wl = W.C1.scaled(40001, 4, 3)
gp = api.Process(wl, W.pdf_table())
run = integrate.run_config(gp, wl, rank=rank, world=dist.get_world_size())
if rank == 0:
    ref = integrate.run_config(gp, wl)          # the same events on one rank
    for a, b in zip(run.iterations, ref.iterations):
        assert a.n_pass == b.n_pass and a.n_events == b.n_events
        assert abs(a.sum_w - b.sum_w) <= 1e-11 * abs(b.sum_w) and abs(a.sum_w2 - b.sum_w2) <= 1e-11 * b.sum_w2
        assert a.max_abs_w == b.max_abs_w or abs(a.max_abs_w - b.max_abs_w) <= 1e-9 * b.max_abs_w
    assert torch.allclose(run.grid, ref.grid, rtol=0, atol=1e-10)
# every rank refined identically
g = [torch.empty_like(run.grid) for _ in range(dist.get_world_size())]
dist.all_gather(g, run.grid)
assert all(torch.equal(g[0], x) for x in g)
dist.destroy_process_group()
"""


def test_run_config_sharded_over_two_gpus_nccl(tmp_path):
    """events sharded by index range over two ranks, ONE exchange per iteration over NCCL; the combined sums
    are the single-rank sums and every rank refines the same grid.  Needs two GPUs (this pool has one per box: skipped)."""
    import os
    import subprocess
    import sys
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    script = tmp_path / "worker.py"
    script.write_text(_NCCL_WORKER)
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MF_ROOT=root)
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
                        "127.0.0.1", "--master-port", "29631", str(script)], env=env, stdout=subprocess.PIPE,
                       stderr=subprocess.STDOUT, text=True, timeout=600)
    assert r.returncode == 0, r.stdout[-3000:]
