"""Pins for the oracle's flavour-summed pp -> ttbar (process 4; "pp -> ttbar (7
diagrams)" = 3 gg + one q qbar diagram for each of four flavours).  CPU only.

What fixes the oracle here, none of it the oracle's own arithmetic retyped:
  * |M|^2(q qbar -> t tbar) against the textbook closed form (Combridge 1979; Ellis-Stirling-Webber table 10.2 with
    a heavy quark):  (4 g^4 / 9) [ (m^2 - t)^2 + (m^2 - u)^2 + 2 m^2 s ] / s^2, which also pins the colour factor the
    oracle sums from the explicit generators (2, i.e. 2/36 after averaging);
  * basis independence and the q <-> qbar orientation symmetry of the helicity sum;
  * the multi-flavour tables: the interpolant reproduces every table at its knots (a wrong table offset fails);
  * the flavour sum of the luminosity spelt out from single-table lookups, pairing q with qbar of the other beam;
  * w(process 4) - w(process 1) = the quark-channel term reassembled from the row's factors;
  * the quark-channel part of the integral against a 2-D quadrature of luminosity x the closed-form partonic
    cross section  sigma(q qbar -> t tbar) = (4 pi alpha_s^2 / (27 s)) beta (2 + rho),  rho = 4 m^2 / s.
"""
import math

import numpy as np
import pytest
from scipy import integrate

from oracle import mfo
from paper_2106_10279_b200 import workloads as W

MT, AS = 173.0, 0.118
S = 13000.0 ** 2


@pytest.fixture(scope="module")
def table():
    return W.pdf_table_flavours()


@pytest.fixture(scope="module")
def P4(table):
    return mfo.Process(W.C5, table)


def mdot(a, b):
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]


def closed_form_qq(mom, m=MT, alpha_s=AS):
    g4 = (4 * math.pi * alpha_s) ** 2
    s = mdot(mom[0] + mom[1], mom[0] + mom[1])
    t = mdot(mom[0] - mom[2], mom[0] - mom[2])
    u = mdot(mom[0] - mom[3], mom[0] - mom[3])
    return 4 * g4 / 9 * ((m * m - t) ** 2 + (m * m - u) ** 2 + 2 * m * m * s) / s ** 2


def cm_point(shat, cos_t, phi, m=MT):
    E = 0.5 * math.sqrt(shat)
    p = math.sqrt(E * E - m * m)
    st = math.sqrt(1 - cos_t * cos_t)
    k = np.array([E, p * st * math.cos(phi), p * st * math.sin(phi), p * cos_t])
    return np.array([[E, 0, 0, E], [E, 0, 0, -E], k, [E, -k[1], -k[2], -k[3]]])


def test_me2_closed_form_basis_and_orientation(P4):
    rng = np.random.default_rng(5)
    for _ in range(40):
        shat = (2 * MT) ** 2 * (1.0 + 10 ** rng.uniform(-3, 2.5))
        mom = cm_point(shat, rng.uniform(-1, 1), rng.uniform(0, 2 * math.pi))
        ref = closed_form_qq(mom)
        v0, v1 = P4.me2_qq(mom, basis=0), P4.me2_qq(mom, basis=1)
        assert v0 == pytest.approx(ref, rel=1e-12)
        assert v1 == pytest.approx(ref, rel=1e-12)
        assert P4.me2_qq(mom, prec=1) == pytest.approx(ref, rel=1e-13)
        swapped = mom[[1, 0, 2, 3]]
        assert P4.me2_qq(swapped) == pytest.approx(closed_form_qq(swapped), rel=1e-12)
        assert P4.me2_qq(swapped) == pytest.approx(v0, rel=1e-12)        # t <-> u symmetry of the helicity sum
    # threshold value: t = u = -m^2 ... at beta -> 0 the closed form tends to (4 g^4 / 9) (1/2 + 1/2) = 4 g^4 / 9
    mom = cm_point((2 * MT) ** 2 * (1 + 1e-10), 0.3, 1.0)
    assert P4.me2_qq(mom) == pytest.approx(4 * (4 * math.pi * AS) ** 2 / 9, rel=1e-8)


def test_massless_limit_is_the_light_quark_result():
    """m -> 0: (4 g^4 / 9) (t^2 + u^2) / s^2, the q qbar -> q' qbar' entry of every QCD textbook"""
    from dataclasses import replace
    P = mfo.Process(replace(W.C5, m_top=1.0, mu2=100.0), W.pdf_table_flavours())
    mom = cm_point(5000.0 ** 2, 0.37, 0.4, m=1.0)
    s = 5000.0 ** 2
    t = mdot(mom[0] - mom[2], mom[0] - mom[2])
    u = mdot(mom[0] - mom[3], mom[0] - mom[3])
    assert P.me2_qq(mom) == pytest.approx(4 * (4 * math.pi * AS) ** 2 / 9 * (t * t + u * u) / s ** 2, rel=1e-6)


def test_tables_are_reproduced_at_the_knots(P4, table):
    lnx, lnq2, xf = table
    assert xf.shape == (1 + 2 * W.N_FLAVOURS, len(lnx), len(lnq2))
    rng = np.random.default_rng(1)
    for t in range(xf.shape[0]):
        for _ in range(12):
            i, j = rng.integers(0, len(lnx) - 1), rng.integers(0, len(lnq2) - 1)
            v = P4.pdf_xf_table(t, math.exp(lnx[i]), math.exp(lnq2[j]))
            assert v == pytest.approx(xf[t, i, j], rel=1e-9, abs=1e-300)
    # the tables differ from one another (a constant offset bug would make two of them agree)
    x, q2 = 0.02, 3e4
    vals = [P4.pdf_xf_table(t, x, q2) for t in range(xf.shape[0])]
    assert len({round(v, 12) for v in vals[:3]}) == 3
    assert vals[1] > vals[2] and vals[3] > vals[4]              # valence: d > dbar, u > ubar
    assert vals[5] == vals[6] and vals[7] == vals[8]            # s = sbar, c = cbar in this table


def test_gluon_channel_is_process_1(P4, oracle_procs):
    """columns lum, me2 of process 4 are the gg channel: identical to process 1 on the same stream"""
    grid = W.uniform_grid(4)
    a = P4.debug_eval(grid, 3, 1, 10, 64)
    b = oracle_procs[1].debug_eval(grid, 3, 1, 10, 64)
    assert a.shape[1] == b.shape[1] + 2
    keep = [c for c in range(b.shape[1]) if c != 4 + 16 + 6]        # everything but w
    assert np.array_equal(a[:, keep], b[:, keep])


def test_event_rows_from_parts(P4, oracle_procs):
    rng = np.random.default_rng(0)
    e = np.sort(rng.random((4, 49)), axis=1)
    grid = np.concatenate([np.zeros((4, 1)), e, np.ones((4, 1))], axis=1)
    rows = P4.debug_eval(grid, 9, 3, 77, 60)
    rows1 = oracle_procs[1].debug_eval(grid, 9, 3, 77, 60)
    mu2 = MT ** 2
    tau_min = 4 * MT ** 2 / S
    for r, r1 in zip(rows, rows1):
        x = r[0:4]
        mom = r[4:20].reshape(4, 4)
        x1, x2, lum, me2, phi, jv, w, passed = r[20:28]
        lum_qq, me2_qq = r[-2], r[-1]
        # flavour sum written out: quark i from beam 1 with antiquark i from beam 2, and the other way round
        L = 0.0
        for i in range(W.N_FLAVOURS):
            q1, qb1 = P4.pdf_xf_table(1 + 2 * i, x1, mu2), P4.pdf_xf_table(2 + 2 * i, x1, mu2)
            q2, qb2 = P4.pdf_xf_table(1 + 2 * i, x2, mu2), P4.pdf_xf_table(2 + 2 * i, x2, mu2)
            L += (q1 * qb2 + qb1 * q2) / (x1 * x2)
        assert lum_qq == pytest.approx(L, rel=1e-12)
        assert me2_qq == pytest.approx(closed_form_qq(mom), rel=1e-10)      # Lorentz invariant: lab momenta do
        Lt = math.log(tau_min)
        tau = math.exp((1 - x[0]) * Lt)
        jac = (-tau * Lt) * (-math.log(tau))
        common = jv / (2 * x1 * x2 * S) * phi * jac * 0.3894e9
        assert w == pytest.approx(common * (lum * me2 + lum_qq * me2_qq), rel=1e-12)
        assert w - r1[26] == pytest.approx(common * lum_qq * me2_qq, rel=1e-9, abs=1e-12 * abs(w))


def sigma_hat_qq(shat, m=MT, alpha_s=AS):
    rho = 4 * m * m / shat
    beta = math.sqrt(1 - rho)
    return 4 * math.pi * alpha_s ** 2 / (27 * shat) * beta * (2 + rho)


def test_sigma_hat_is_the_angular_integral_of_the_closed_form():
    """the two textbook formulas agree: sigma = (1 / 2s) int |M|^2 dPhi_2, dPhi_2 = beta / (16 pi) dcos"""
    shat = 700.0 ** 2
    beta = math.sqrt(1 - 4 * MT * MT / shat)
    val, _ = integrate.quad(lambda c: closed_form_qq(cm_point(shat, c, 0.0)), -1, 1, epsrel=1e-12)
    assert val * beta / (16 * math.pi) / (2 * shat) == pytest.approx(sigma_hat_qq(shat), rel=1e-10)


@pytest.fixture(scope="module")
def qq_quadrature(P4):
    tau_min = 4 * MT ** 2 / S
    mu2 = MT ** 2

    def inner(lt):
        tau = math.exp(lt)
        ymax = -0.5 * lt

        def lum(y):
            x1, x2 = math.sqrt(tau) * math.exp(y), math.sqrt(tau) * math.exp(-y)
            L = 0.0
            for i in range(W.N_FLAVOURS):
                L += P4.pdf_xf_table(1 + 2 * i, x1, mu2) * P4.pdf_xf_table(2 + 2 * i, x2, mu2)
                L += P4.pdf_xf_table(2 + 2 * i, x1, mu2) * P4.pdf_xf_table(1 + 2 * i, x2, mu2)
            return L / (x1 * x2)
        val, _ = integrate.quad(lum, -ymax, ymax, epsabs=0, epsrel=1e-6, limit=400)
        return val * tau * sigma_hat_qq(tau * S)
    val, _ = integrate.quad(inner, math.log(tau_min), 0, epsabs=0, epsrel=1e-5, limit=400)
    return val * 0.3894e9


def test_vegas_quark_part_agrees_with_quadrature(P4, oracle_procs, oracle_pool, qq_quadrature):
    """whole chain: (process 4 - process 1) event by event on the same stream is the quark channel's integrand
    (the rows come from the multi-process oracle harness: the same single-threaded code on disjoint index ranges)"""
    n = 2 ** 15
    grid = W.uniform_grid(4)
    I, var = [], []
    for it in range(5):
        hist, res = P4.vegas_iterate(grid, 0, it, 0, n)
        if it >= 2:
            r4 = oracle_pool.debug_eval(W.C5, grid, 0, it, 0, n)
            r1 = oracle_pool.debug_eval(W.C1, grid, 0, it, 0, n)
            d = r4[:, 26] - r1[:, 26]
            I.append(d.mean())
            var.append(d.var(ddof=1) / n)
            assert res.sum_w == pytest.approx(r4[:, 26].sum(), rel=1e-12)
        grid = P4.refine_grid(grid, hist, W.VEGAS_ALPHA)
    I, var = np.array(I), np.array(var)
    wsum = (1 / var).sum()
    Ic, sc = (I / var).sum() / wsum, wsum ** -0.5
    assert sc / Ic < 1e-2
    assert abs(Ic - qq_quadrature) < 4 * sc
    assert 100.0 < qq_quadrature < 1000.0          # about a tenth of the gg channel with this synthetic table


def test_channel_of_accepted_events(P4):
    """R18: the channel code of an accepted event, recomputed here from single-table lookups, the closed-form matrix
    elements and the raw Philox words; and its frequencies against their expectation."""
    from test_oracle_amplitudes import esw_gg_ttbar
    n = 6000
    grid = W.uniform_grid(4)
    rows = P4.debug_eval(grid, 2, 4, 100, n)
    w = rows[:, 26]
    w_max = float(np.quantile(np.abs(w), 0.7))
    rec, cnt, _, res = P4.unweight(grid, 2, 4, 100, n, w_max, n)
    mom, wr, ids = P4.records_view(rec, cnt)
    chan = P4.records_array(rec, cnt)["channel"]
    assert cnt == res.n_accept and cnt > 1500 and len(chan) == cnt
    mu2 = MT ** 2
    expect = np.zeros(1 + 2 * W.N_FLAVOURS)
    for k in range(n):                         # expected channel counts: P(accept) x channel share, event by event
        r = rows[k]
        x1, x2, lum = r[20], r[21], r[22]
        a = [abs(lum * r[23])]
        for i in range(W.N_FLAVOURS):
            q1, qb1 = P4.pdf_xf_table(1 + 2 * i, x1, mu2), P4.pdf_xf_table(2 + 2 * i, x1, mu2)
            q2, qb2 = P4.pdf_xf_table(1 + 2 * i, x2, mu2), P4.pdf_xf_table(2 + 2 * i, x2, mu2)
            a += [abs(q1 * qb2 / (x1 * x2) * r[-1]), abs(qb1 * q2 / (x1 * x2) * r[-1])]
        a = np.array(a)
        expect += min(1.0, abs(w[k]) / w_max) * a / a.sum()
        hit = np.nonzero(ids == 100 + k)[0]
        if len(hit):                           # this event was accepted: its channel from the raw words
            words = mfo.philox_block(2, 4, 100 + k, 0xFFFFFFFF)
            v = mfo.uniform_from_words(words[2], words[3]) * a.sum()
            cum = np.cumsum(a)
            if np.min(np.abs(cum - v)) > 1e-9 * a.sum():
                assert chan[hit[0]] == int(np.argmax(cum > v)), k
    assert abs(expect.sum() - cnt) < 5 * math.sqrt(cnt)
    got = np.bincount(chan.astype(int), minlength=len(expect))
    for c in range(len(expect)):
        assert abs(got[c] - expect[c]) < 5 * math.sqrt(expect[c] + 1), (c, got[c], expect[c])
    assert got[0] > 0.8 * cnt and got[1:].sum() > 30          # mostly gg; the quark channels do occur
    assert got[3] + got[4] > 2 * (got[7] + got[8])             # u ubar (valence + a large sea) against c cbar (a small sea)
