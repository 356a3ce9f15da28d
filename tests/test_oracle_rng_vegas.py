"""Pins for the oracle's O1-O3, O13-O15: Philox4x32-10, uniform conversion, VEGAS map,
grid refinement, iteration sums, unweighting.  CPU only.  Every expected value here comes from the published
known-answer vectors, from exact arithmetic, or from an invariant - never from the CUDA path."""
import math
import os

import numpy as np
import pytest

from oracle import mfo
from paper_2106_10279_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _kat_rows():
    rows = []
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answer_vectors():
    """O1: the three published Philox4x32-10 test vectors (Salmon et al., SC'11)."""
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert mfo.philox4x32_10(ctr, key) == out


def test_philox_python_bigint_reimplementation():
    """O1 again, against an independent arbitrary-precision integer restatement of the round function,
    on random counters/keys (catches a wrong word order that the three KATs might not)."""
    M0, M1, W0, W1, MASK = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85, 0xFFFFFFFF

    def ref(c, k):
        c = list(c); k = list(k)
        for r in range(10):
            p0, p1 = M0 * c[0], M1 * c[2]
            c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & MASK, (p0 >> 32) ^ c[3] ^ k[1], p0 & MASK]
            k = [(k[0] + W0) & MASK, (k[1] + W1) & MASK]
        return c
    rng = np.random.default_rng(7)
    for _ in range(200):
        c = [int(v) for v in rng.integers(0, 2 ** 32, 4)]
        k = [int(v) for v in rng.integers(0, 2 ** 32, 2)]
        assert mfo.philox4x32_10(c, k) == ref(c, k)


def test_stream_layout():
    """Reading R1: key = seed words, counter = (event lo, event hi, iteration, block)."""
    seed, it, ev, blk = 0x0123456789ABCDEF, 7, 0xFEDCBA9876543210, 3
    got = mfo.philox_block(seed, it, ev, blk)
    want = mfo.philox4x32_10([ev & 0xFFFFFFFF, ev >> 32, it, blk], [seed & 0xFFFFFFFF, seed >> 32])
    assert got == want


def test_uniform_conversion():
    """O2: u = (2m+1) 2^-53 with m the top 52 bits; exact values and range."""
    assert mfo.uniform_from_words(0, 0) == 2.0 ** -53
    assert mfo.uniform_from_words(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    assert mfo.uniform_from_words(0x80000000, 0) == 0.5 + 2.0 ** -53
    assert mfo.uniform_from_words(0, 0xFFF) == 2.0 ** -53          # low 12 bits are dropped
    assert mfo.uniform_from_words(0, 0x1000) == 3 * 2.0 ** -53
    assert math.floor((1.0 - 2.0 ** -53) * 50) == 49
    # seed 0, iteration 0, event 0 (follows from the first KAT vector): SURVEY.md §8(c) O2
    w = mfo.philox_block(0, 0, 0, 0)
    assert w == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert mfo.uniform_from_words(w[0], w[1]) == pytest.approx(0.3990464708489646, abs=1e-16)
    assert mfo.uniform_from_words(w[2], w[3]) == pytest.approx(0.7357127844834425, abs=1e-16)
    # exact rational check
    m = (0x6627e8d5 << 20) | (0xe169c58d >> 12)
    assert mfo.uniform_from_words(w[0], w[1]) == (2 * m + 1) / 2 ** 53


def _random_grid(rng, D, nb=50):
    e = np.sort(rng.random((D, nb - 1)), axis=1)
    return np.concatenate([np.zeros((D, 1)), e, np.ones((D, 1))], axis=1)


def test_vegas_map_uniform_grid_is_identity():
    rng = np.random.default_rng(1)
    g = W.uniform_grid(6)
    for _ in range(100):
        u = rng.random(6)
        x, j, b = mfo.vegas_map(g, u)
        assert np.allclose(x, u, rtol=0, atol=2e-16)
        assert j == pytest.approx(1.0, abs=1e-13)  # 6 widths i/50, each rounded
        assert list(b) == [int(math.floor(v * 50)) for v in u]


def test_vegas_map_jacobian_integrates_to_one_and_is_monotone():
    """O3: for any grid, int_0^1 J du = 1 per dimension, and x(u) is monotone and hits the edges."""
    rng = np.random.default_rng(2)
    g = _random_grid(rng, 1)
    nb = 50
    # midpoint rule with an integer number of points per bin is exact for the piecewise-constant J
    pts = (np.arange(nb * 8) + 0.5) / (nb * 8)
    tot = 0.0
    xs = []
    for u in pts:
        x, j, b = mfo.vegas_map(g, [u])
        tot += j / len(pts)
        xs.append(x[0])
        assert g[0, b[0]] <= x[0] <= g[0, b[0] + 1]
    assert tot == pytest.approx(1.0, abs=1e-13)
    assert np.all(np.diff(xs) > 0)
    # bin index depends on u only
    g2 = _random_grid(rng, 1)
    for u in rng.random(50):
        assert mfo.vegas_map(g, [u])[2][0] == mfo.vegas_map(g2, [u])[2][0] == int(u * nb)


def test_vegas_map_edge_values():
    g = _random_grid(np.random.default_rng(3), 2)
    u = [2.0 ** -53, 1 - 2.0 ** -53]
    x, j, b = mfo.vegas_map(g, u)
    assert list(b) == [0, 49]
    assert 0 < x[0] < g[0, 1] and g[1, 49] < x[1] < 1


# ---- O14 grid refinement -----------------------------------------------------------------------------
def _refine(proc, grid, hist, alpha=1.5, prec=0):
    return proc.refine_grid(grid, hist, alpha, prec)


def test_refine_flat_histogram_leaves_grid_unchanged(oracle_procs):
    P = oracle_procs[0]
    g = W.uniform_grid(2)
    h = np.full((2, 50), 3.7)
    g2 = _refine(P, g, h)
    assert np.allclose(g2, g, rtol=0, atol=1e-14)
    # also on a non-uniform grid: a density flat in the *bins* keeps every edge
    rng = np.random.default_rng(5)
    g = _random_grid(rng, 2)
    assert np.allclose(_refine(P, g, h), g, rtol=0, atol=1e-14)


def test_refine_zero_histogram_dimension_untouched(oracle_procs):
    P = oracle_procs[0]
    g = _random_grid(np.random.default_rng(6), 2)
    h = np.zeros((2, 50))
    h[1] = np.random.default_rng(6).random(50)
    g2 = _refine(P, g, h)
    assert np.array_equal(g2[0], g[0])
    assert not np.array_equal(g2[1], g[1])


def test_refine_equalises_damped_density(oracle_procs):
    """O14: new bins hold equal integrals of the piecewise-constant damped density r (Lepage)."""
    P = oracle_procs[0]
    rng = np.random.default_rng(8)
    g = _random_grid(rng, 2)
    h = rng.random((2, 50)) ** 4 * 10
    h[0, 10:14] = 0.0
    for alpha in (1.5, 0.5):
        g2 = _refine(P, g, h, alpha)
        assert np.all(np.diff(g2, axis=1) > 0) and np.all(g2[:, 0] == 0) and np.all(g2[:, -1] == 1)
        for d in range(2):
            # independent restatement in exact-ish arithmetic: the cumulative of r over old bins, linear
            # inside a bin, evaluated at the new edges must be i * delta
            s = np.empty(50)
            s[0] = (h[d, 0] + h[d, 1]) / 2
            s[-1] = (h[d, -2] + h[d, -1]) / 2
            s[1:-1] = (h[d, :-2] + h[d, 1:-1] + h[d, 2:]) / 3
            s /= s.sum()
            r = np.where(s > 0, ((s - 1) / np.log(np.where(s > 0, s, 0.5))) ** alpha, 0.0)
            cum = np.concatenate([[0.0], np.cumsum(r)])
            F = np.interp(g2[d], g[d], cum)
            assert np.allclose(F, np.arange(51) * cum[-1] / 50, rtol=0, atol=1e-12 * cum[-1])


def test_refine_referee_precision(oracle_procs):
    P = oracle_procs[0]
    rng = np.random.default_rng(9)
    g = _random_grid(rng, 2)
    h = rng.random((2, 50))
    a, b = _refine(P, g, h, prec=0), _refine(P, g, h, prec=2)
    assert np.allclose(a, b, rtol=0, atol=1e-14)


# ---- O13 iteration sums / O15 unweighting -------------------------------------------------------------
@pytest.mark.parametrize("pid,n", [(0, 3000), (1, 1500), (2, 300)])
def test_iteration_sums_match_per_event_rows(oracle_procs, pid, n):
    """O13: sum_w, sum_w2, max, n_pass and the w^2 histograms are what the per-event rows add up to."""
    P = oracle_procs[pid]
    D = P.n_dims
    g = _random_grid(np.random.default_rng(10), D)
    hist, res = P.vegas_iterate(g, 5, 2, 1000, n)
    rows = P.debug_eval(g, 5, 2, 1000, n)
    nm = 4 * (P.n_final + 2)
    w = rows[:, D + nm + 6]
    passed = rows[:, D + nm + 7]
    bins = rows[:, 2 * D + nm + 9:].astype(int)
    assert res.sum_w == pytest.approx(math.fsum(w), rel=1e-14)
    assert res.sum_w2 == pytest.approx(math.fsum(w * w), rel=1e-14)
    assert res.max_abs_w == np.abs(w).max()
    assert res.n_pass == int(passed.sum())
    h = np.zeros((D, 50))
    for d in range(D):
        np.add.at(h[d], bins[:, d], w * w)
    assert np.allclose(hist, h, rtol=1e-13, atol=0)
    # counter-based RNG: sub-ranges add up
    h1, r1 = P.vegas_iterate(g, 5, 2, 1000, n // 3)
    h2, r2 = P.vegas_iterate(g, 5, 2, 1000 + n // 3, n - n // 3)
    assert r1.sum_w + r2.sum_w == pytest.approx(res.sum_w, rel=1e-14)
    assert r1.n_pass + r2.n_pass == res.n_pass
    assert np.allclose(h1 + h2, hist, rtol=1e-13)


def test_constant_integrand_through_vegas_weights():
    """O3/O13 special case: sum over events of J is an unbiased estimate of 1 for any grid (f = 1)."""
    rng = np.random.default_rng(11)
    g = _random_grid(rng, 3)
    n = 20000
    tot = 0.0
    tot2 = 0.0
    for e in range(n):
        u = []
        for b in range(2):
            w = mfo.philox_block(1, 0, e, b)
            u += [mfo.uniform_from_words(w[0], w[1]), mfo.uniform_from_words(w[2], w[3])]
        _, j, _ = mfo.vegas_map(g, u[:3])
        tot += j
        tot2 += j * j
    mean = tot / n
    err = math.sqrt((tot2 / n - mean * mean) / (n - 1))
    assert abs(mean - 1.0) < 4 * err


def test_unweighting_replay(oracle_procs):
    """O15: accept iff r * w_max < |w|, r from Philox block 0xFFFFFFFF; records in event order, signed w and id;
    *count keeps advancing past capacity."""
    P = oracle_procs[2]
    D = P.n_dims
    g = W.uniform_grid(D)
    n, seed, it, first = 600, 3, 6, 12345
    rows = P.debug_eval(g, seed, it, first, n)
    nm = 4 * (P.n_final + 2)
    w = rows[:, D + nm + 6]
    r = rows[:, D + nm + 8]
    # r is the documented draw
    for k in (0, 17, n - 1):
        ww = mfo.philox_block(seed, it, first + k, 0xFFFFFFFF)
        assert r[k] == mfo.uniform_from_words(ww[0], ww[1])
    w_max = np.abs(w).max() * 0.05
    want = np.nonzero(r * w_max < np.abs(w))[0]
    assert 5 < len(want) < n
    rec, count, hist, res = P.unweight(g, seed, it, first, n, w_max, capacity=n, count=0)
    assert count == len(want) == res.n_accept
    mom, ww, ids = P.records_view(rec, count)
    assert list(ids) == [first + k for k in want]
    assert np.array_equal(ww, w[want])
    assert np.array_equal(mom.reshape(count, -1), rows[want, D:D + nm])
    # overweight events are always accepted, zero-weight never
    assert set(np.nonzero(np.abs(w) >= w_max)[0]).issubset(set(want))
    assert not set(np.nonzero(w == 0)[0]) & set(want)
    # same sums as the plain iteration
    h0, r0 = P.vegas_iterate(g, seed, it, first, n)
    assert (r0.sum_w, r0.sum_w2, r0.max_abs_w, r0.n_pass) == (res.sum_w, res.sum_w2, res.max_abs_w, res.n_pass)
    assert np.array_equal(h0, hist)
    # overflow protocol: capacity 3, cursor starts at 2 -> one record written, count still advances
    rec2, count2, _, _ = P.unweight(g, seed, it, first, n, w_max, capacity=3, count=2)
    assert count2 == 2 + len(want)
    _, w2, id2 = P.records_view(rec2, 3)
    assert id2[2] == first + want[0] and id2[0] == 0 and id2[1] == 0


def test_unweighting_expected_acceptance(oracle_procs):
    """O15 pin: E[n_accept] = sum min(1, |w|/w_max)."""
    P = oracle_procs[1]
    g = W.uniform_grid(4)
    n = 20000
    rows = P.debug_eval(g, 0, 0, 0, n)
    w = rows[:, 4 + 16 + 6]
    w_max = np.abs(w).max()
    p = np.minimum(1.0, np.abs(w) / w_max)
    _, count, _, res = P.unweight(g, 0, 0, 0, n, w_max, capacity=0)
    sd = math.sqrt((p * (1 - p)).sum())
    assert abs(count - p.sum()) < 4 * sd
    assert res.n_accept == count
