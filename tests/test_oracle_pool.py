"""The multi-process oracle harness (tests/oracle_pool.py, SURVEY.md §8(c) protocol iii) against the plain
single-process oracle: same rows, same accepted events, sums equal up to the rounding of the partial sums."""
import numpy as np

from paper_2106_10279_b200 import workloads as W


def test_pool_equals_single_process(oracle_procs, oracle_pool):
    for wl, n in ((W.C1, 6001), (W.C3, 301)):
        op = oracle_procs[wl.process]
        grid = W.uniform_grid(wl.n_dims)
        h1, r1 = op.vegas_iterate(grid, 3, 1, 11, n)
        grid = op.refine_grid(grid, h1, W.VEGAS_ALPHA)
        h1, r1 = op.vegas_iterate(grid, 3, 2, 11, n)
        hp, rp, rec = oracle_pool.iterate(wl, grid, 3, 2, 11, n)
        assert rec is None and rp.n_pass == r1.n_pass and rp.max_abs_w == r1.max_abs_w
        assert abs(rp.sum_w - r1.sum_w) <= 1e-14 * abs(r1.sum_w) and abs(rp.sum_w2 - r1.sum_w2) <= 1e-14 * r1.sum_w2
        np.testing.assert_allclose(hp, h1, rtol=1e-13, atol=0)
        assert np.array_equal(oracle_pool.debug_eval(wl, grid, 3, 2, 11, n), op.debug_eval(grid, 3, 2, 11, n))
        w_max = 0.3 * r1.max_abs_w
        rec1, cnt1, hu, ru = op.unweight(grid, 3, 2, 11, n, w_max, n)
        hq, rq, recp = oracle_pool.iterate(wl, grid, 3, 2, 11, n, w_max=w_max)
        a1 = op.records_array(rec1, cnt1)
        assert rq.n_accept == ru.n_accept == cnt1 == len(recp) > 0
        assert np.array_equal(recp["id"], a1["id"]) and np.array_equal(recp["w"], a1["w"])
        assert np.array_equal(recp["mom"], a1["mom"])
    # empty range
    h, r, rec = oracle_pool.iterate(W.C1, W.uniform_grid(4), 0, 0, 5, 0)
    assert r.n_pass == 0 and r.sum_w == 0.0 and not h.any()
