"""Pins for the oracle's observable histograms ("histogram accumulation"; L109-119, Fig. 2).  CPU only.
The oracle function is the definition written out on the oracle's own per-event rows; it is pinned here by a hand
computed example, by closure (every weighted event lands in exactly one bin of each histogram) and by the closed
form of d sigma / d eta for e+e- -> mu+mu- (d sigma / d cos theta ~ 1 + cos^2 theta, eta = atanh cos theta)."""
import math

import numpy as np
import pytest

from oracle import mfo
from paper_2106_10279_b200 import workloads as W


def _row(n_dims, n_final, p_first, w):
    row = np.zeros(3 * n_dims + 4 * (n_final + 2) + 9)
    row[n_dims + 8:n_dims + 12] = p_first
    row[n_dims + 4 * (n_final + 2) + 6] = w
    return row


def test_hand_computed_bins():
    # pT = 5 (3-4-5), pz = 5 sinh(1.0): eta = 1.0 exactly by construction
    p = [0.0, 3.0, 4.0, 5.0 * math.sinh(1.0)]
    rows = np.array([_row(4, 2, p, 2.5), _row(4, 2, [0, 30.0, 40.0, -50.0 * math.sinh(2.2)], -1.0),
                     _row(4, 2, [0, 300.0, 400.0, 0.0], 7.0), _row(4, 2, p, 0.0)])
    obs = mfo.observable_histograms(rows, 4, 2, n_bins=10, pt_max=100.0, eta_max=2.5)
    want = np.zeros((2, 11))
    want[0, 0] += 2.5      # pT 5 of [0, 100) in 10 bins -> bin 0
    want[1, 7] += 2.5      # eta 1.0: (1.0 + 2.5) / 5 * 10 = 7.0 -> bin 7
    want[0, 5] += -1.0     # pT 50 -> bin 5
    want[1, 0] += -1.0     # eta -2.2: (0.3 / 5) * 10 = 0.6 -> bin 0
    want[0, 10] += 7.0     # pT 500 >= pt_max -> overflow
    want[1, 5] += 7.0      # eta 0 -> bin 5
    assert np.array_equal(obs, want)          # the w = 0 event is not entered


@pytest.mark.parametrize("wl,n", [(W.C0, 4000), (W.C1, 2000), (W.C2, 600)], ids=["C0", "C1", "C2"])
def test_closure(wl, n, oracle_procs):
    op = oracle_procs[wl.process]
    grid = W.uniform_grid(wl.n_dims)
    rows = op.debug_eval(grid, 3, 0, 0, n)
    obs = mfo.observable_histograms(rows, wl.n_dims, wl.n_final, 25, 400.0, 3.0)
    _, res = op.vegas_iterate(grid, 3, 0, 0, n)
    for h in obs:
        assert h.sum() == pytest.approx(res.sum_w, rel=1e-12)


def test_ee_mumu_eta_distribution(oracle_procs):
    """(1/sigma) d sigma / d eta integrated over a bin = [F(tanh eta_hi) - F(tanh eta_lo)], F(c) = (3 c + c^3) / 8."""
    wl = W.C0
    n, nb, eta_max = 40000, 12, 3.0
    rows = oracle_procs[0].debug_eval(W.uniform_grid(wl.n_dims), 11, 0, 0, n)
    obs = mfo.observable_histograms(rows, wl.n_dims, wl.n_final, nb, 60.0, eta_max)
    tot = obs[1].sum()
    F = lambda c: (3 * c + c ** 3) / 8.0
    edges = -eta_max + 2 * eta_max * np.arange(nb + 1) / nb
    frac = F(np.tanh(edges[1:])) - F(np.tanh(edges[:-1]))
    got = obs[1][:nb] / tot
    # uniform grid: weights ~ (1 + c^2), binomial-like errors; 5 sigma
    sig = np.sqrt(frac * (1 - frac) / n) * 1.3
    assert np.all(np.abs(got - frac) < 5 * sig + 1e-12)
    assert obs[1][nb] / tot == pytest.approx(1 - (F(math.tanh(eta_max)) - F(-math.tanh(eta_max))), abs=5e-4)
    # pT = 50 sin(theta) < 50 always: nothing beyond 50 GeV
    assert obs[0][int(50.0 / 60.0 * nb) + 1:].sum() == 0.0
