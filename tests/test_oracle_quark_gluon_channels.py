"""Pins for the oracle's q qbar -> t tbar g and q g -> t tbar q matrix elements (the quark channels of pp -> ttbar g,
PAPER.md L101; R19) and of the process that sums them with g g -> t tbar g.  CPU only.

The oracle sums the five Feynman diagrams with explicit SU(3) generators and structure constants.  What fixes it:
  * the Ward identity: with the gluon's polarisation vector replaced by its momentum the colour-summed |M|^2 vanishes
    (any wrong relative sign, factor of i, propagator momentum or colour order among the five diagrams breaks it);
  * independence of the spinor and polarisation bases, charge conjugation;
  * the collinear limits, which fix the overall normalisation against matrix elements pinned elsewhere:
      k_g || p_q    in q qbar -> ttbar g :  8 pi alpha_s / (2 p.k)  P_qq(z) / z  |M(q qbar -> ttbar)|^2,  P_qq = C_F (1+z^2)/(1-z)
      p_q' || p_g   in q g -> ttbar q    :  8 pi alpha_s / (2 p.k)  P_qg(z) / z  |M(q qbar -> ttbar)|^2,  P_qg = T_R (z^2+(1-z)^2)
      p_q' || p_q   in q g -> ttbar q    :  8 pi alpha_s / (2 p.k)  P_gq(z) / z  |M(g g -> ttbar)|^2 after averaging over the
                                            azimuth of the splitting,                                   P_gq = C_F (1+(1-z)^2)/z
    (Altarelli-Parisi kernels; z = momentum fraction entering the hard process); the Born matrix elements are the
    textbook closed forms, typed out in the tests.
"""
import math

import numpy as np
import pytest

from oracle import mfo
from paper_2106_10279_b200 import workloads as W
from test_oracle_amplitudes import esw_gg_ttbar
from test_oracle_quark_channel import closed_form_qq, mdot

MT, AS = 173.0, 0.118
E, Z, CT, PH = 1000.0, 0.6, 0.3, 1.1
P1, P2 = np.array([E, 0, 0, E]), np.array([E, 0, 0, -E])


def boost(p, q):
    """p from the rest frame of q to the frame in which q is given"""
    M = math.sqrt(mdot(q, q))
    b, g = q[1:] / M, q[0] / M
    bp = float(np.dot(b, p[1:]))
    return np.concatenate([[g * p[0] + bp], p[1:] + b * (bp / (g + 1) + p[0])])


def decay(q, ct=CT, ph=PH):
    M = math.sqrt(mdot(q, q))
    En = M / 2
    pp = math.sqrt(En * En - MT * MT)
    st = math.sqrt(1 - ct * ct)
    k = np.array([En, pp * st * math.cos(ph), pp * st * math.sin(ph), pp * ct])
    return boost(k, q), boost(np.array([En, -k[1], -k[2], -k[3]]), q)


def generic_point(seed=0):
    rng = np.random.default_rng(seed)
    k, _ = mfo.rambo([MT, MT, 0.0], 900.0 + 400 * rng.random(), rng.random(12))
    w = k[:, 0].sum() / 2
    return np.vstack([[w, 0, 0, w], [w, 0, 0, -w], k])


@pytest.mark.parametrize("kind", [0, 1])
def test_ward_identity_bases_and_precision(kind):
    for seed in range(6):
        mom = generic_point(seed)
        v = mfo.me2_light_line_ttbar_g(kind, mom, MT, AS)
        assert v > 0
        # eps -> k makes every diagram ~ (k / 1)^2 ~ 1e5 times larger; the sum cancels to rounding
        assert abs(mfo.me2_light_line_ttbar_g(kind, mom, MT, AS, subst=1)) < 1e-8 * v
        for basis in (1, 2, 3):
            assert mfo.me2_light_line_ttbar_g(kind, mom, MT, AS, basis=basis) == pytest.approx(v, rel=1e-12)
        assert mfo.me2_light_line_ttbar_g(kind, mom, MT, AS, prec=1) == pytest.approx(v, rel=1e-12)


def test_charge_conjugation_and_alpha_s_power():
    mom = generic_point(3)
    v = mfo.me2_light_line_ttbar_g(0, mom, MT, AS)
    assert mfo.me2_light_line_ttbar_g(0, mom[[1, 0, 3, 2, 4]], MT, AS) == pytest.approx(v, rel=1e-12)
    assert mfo.me2_light_line_ttbar_g(0, mom, MT, 2 * AS) == pytest.approx(8 * v, rel=1e-12)


def _collinear(direction, th, az):
    """the massless momentum (1 - Z) E (1, sin th cos az, sin th sin az, +-cos th)"""
    return (1 - Z) * E * np.array([1, math.sin(th) * math.cos(az), math.sin(th) * math.sin(az), direction * math.cos(th)])


def test_collinear_limit_gluon_along_the_quark():
    born = closed_form_qq(np.array([Z * P1, P2, *decay(Z * P1 + P2)]), MT, AS)
    P = 4 / 3 * (1 + Z * Z) / (1 - Z)
    prev = None
    for th in (1e-3, 1e-4):
        k5 = _collinear(+1, th, 0.7)
        v = mfo.me2_light_line_ttbar_g(0, np.array([P1, P2, *decay(P1 + P2 - k5), k5]), MT, AS)
        ratio = v / (8 * math.pi * AS / (2 * mdot(P1, k5)) * P / Z * born)
        assert abs(ratio - 1) < 1.5 * th          # approaches 1 linearly in the angle
        if prev is not None:
            assert abs(ratio - 1) < 0.2 * abs(prev - 1)
        prev = ratio


def test_collinear_limit_gluon_splits_into_quark_pair():
    born = closed_form_qq(np.array([P1, Z * P2, *decay(P1 + Z * P2)]), MT, AS)
    P = 0.5 * (Z * Z + (1 - Z) ** 2)
    for th in (1e-3, 1e-4):
        p5 = _collinear(-1, th, 0.7)
        v = mfo.me2_light_line_ttbar_g(1, np.array([P1, P2, *decay(P1 + P2 - p5), p5]), MT, AS)
        ratio = v / (8 * math.pi * AS / (2 * mdot(P2, p5)) * P / Z * born)
        assert abs(ratio - 1) < 1.5 * th


def test_collinear_limit_quark_radiates_into_gluon_gluon_channel():
    born = esw_gg_ttbar(np.array([Z * P1, P2, *decay(Z * P1 + P2)]), MT, AS)
    P = 4 / 3 * (1 + (1 - Z) ** 2) / Z
    th = 1e-4
    vals = []
    for ia in range(8):                      # the gluon entering g g -> ttbar is linearly polarised: average the azimuth
        p5 = _collinear(+1, th, 0.3 + ia * 2 * math.pi / 8)
        vals.append(mfo.me2_light_line_ttbar_g(1, np.array([P1, P2, *decay(P1 + P2 - p5), p5]), MT, AS))
    pref = 8 * math.pi * AS / (2 * mdot(P1, _collinear(+1, th, 0.0))) * P / Z * born
    assert np.mean(vals) / pref == pytest.approx(1.0, abs=5e-4)
    assert max(vals) / min(vals) > 1.02        # and the azimuthal correlation is really there


def test_antiquark_gluon_channel_is_the_charge_conjugate():
    """kind 2 (qbar g -> ttbar qbar, from its own diagrams: the light line runs backwards) = kind 1 with t <-> tbar"""
    for seed in range(4):
        mom = generic_point(20 + seed)
        v2 = mfo.me2_light_line_ttbar_g(2, mom, MT, AS)
        assert v2 == pytest.approx(mfo.me2_light_line_ttbar_g(1, mom[[0, 1, 3, 2, 4]], MT, AS), rel=1e-12)
        assert abs(mfo.me2_light_line_ttbar_g(2, mom, MT, AS, subst=1)) < 1e-8 * v2
        assert v2 != pytest.approx(mfo.me2_light_line_ttbar_g(1, mom, MT, AS), rel=1e-3)     # and differs from q g


def test_process_rows_from_parts(oracle_procs):
    """process 5 (pp -> ttbar j): the gg columns are process 2's; the six quark-channel terms and the weight are
    reassembled from single-table PDF lookups and matrix-element calls at the row's (lab-frame) momenta"""
    P5 = mfo.Process(W.C6, W.pdf_table_flavours())
    grid = W.uniform_grid(14)
    rows = P5.debug_eval(grid, 5, 2, 40, 120)
    rows2 = oracle_procs[2].debug_eval(grid, 5, 2, 40, 120)
    n2 = rows2.shape[1]
    assert rows.shape[1] == n2 + 6
    o = 14 + 20
    keep = [c for c in range(n2) if c != o + 6]
    assert np.array_equal(rows[:, keep], rows2[:, keep])
    mu2 = MT ** 2
    nf = W.N_FLAVOURS
    n_pass = 0
    for r, r2 in zip(rows, rows2):
        x1, x2, lum, me2, phi, jv, w, passed = r[o:o + 8]
        if not passed:
            assert w == 0 and not r[-6:].any()
            continue
        n_pass += 1
        mom = r[14:o].reshape(5, 4)
        f = lambda t, x: P5.pdf_xf_table(t, x, mu2)
        Q1, Qb1 = sum(f(1 + 2 * i, x1) for i in range(nf)), sum(f(2 + 2 * i, x1) for i in range(nf))
        Q2, Qb2 = sum(f(1 + 2 * i, x2) for i in range(nf)), sum(f(2 + 2 * i, x2) for i in range(nf))
        D12 = sum(f(1 + 2 * i, x1) * f(2 + 2 * i, x2) for i in range(nf))
        D21 = sum(f(2 + 2 * i, x1) * f(1 + 2 * i, x2) for i in range(nf))
        g1, g2 = f(0, x1), f(0, x2)
        swapped = mom[[1, 0, 2, 3, 4]]
        want = [D12 * mfo.me2_light_line_ttbar_g(0, mom, MT, AS), D21 * mfo.me2_light_line_ttbar_g(0, swapped, MT, AS),
                Q1 * g2 * mfo.me2_light_line_ttbar_g(1, mom, MT, AS), g1 * Q2 * mfo.me2_light_line_ttbar_g(1, swapped, MT, AS),
                Qb1 * g2 * mfo.me2_light_line_ttbar_g(2, mom, MT, AS), g1 * Qb2 * mfo.me2_light_line_ttbar_g(2, swapped, MT, AS)]
        np.testing.assert_allclose(r[-6:], np.array(want) / (x1 * x2), rtol=1e-9)
        # w(5) / w(2) = (gg + quark terms) / gg
        assert w / r2[o + 6] == pytest.approx((lum * me2 + r[-6:].sum()) / (lum * me2), rel=1e-11)
    assert n_pass > 60


def test_channel_of_accepted_events():
    """R20: every accepted event of pp -> ttbar j carries its partonic channel: code 0 = gg, code 1 + 6 i + c =
    flavour i in class c (q qbar, qbar q, q g, g q, qbar g, g qbar), drawn in proportion to |luminosity x |M|^2| in code
    order with the second uniform of the accept block.  Recomputed here from single-table lookups, the component
    matrix-element calls and the raw Philox words; the frequencies against their expectation."""
    P5 = mfo.Process(W.C6, W.pdf_table_flavours())
    n = 1500
    grid = W.uniform_grid(14)
    rows = P5.debug_eval(grid, 2, 4, 100, n)
    o = 14 + 20
    w = rows[:, o + 6]
    w_max = float(np.quantile(np.abs(w[w != 0]), 0.6))
    rec, cnt, _, res = P5.unweight(grid, 2, 4, 100, n, w_max, n)
    arr = P5.records_array(rec, cnt)
    chan, ids = arr["channel"], arr["id"]
    assert cnt == res.n_accept and cnt > 300 and P5.record_size == 5 * 32 + 16 + 8
    mu2, nf = MT ** 2, W.N_FLAVOURS
    expect = np.zeros(1 + 6 * nf)
    for k in range(n):
        r = rows[k]
        x1, x2, lum, me2 = r[o:o + 4]
        if not r[o + 7]:
            continue
        mom = r[14:o].reshape(5, 4)
        sw = mom[[1, 0, 2, 3, 4]]
        M = [mfo.me2_light_line_ttbar_g(0, mom, MT, AS), mfo.me2_light_line_ttbar_g(0, sw, MT, AS),
             mfo.me2_light_line_ttbar_g(1, mom, MT, AS), mfo.me2_light_line_ttbar_g(1, sw, MT, AS),
             mfo.me2_light_line_ttbar_g(2, mom, MT, AS), mfo.me2_light_line_ttbar_g(2, sw, MT, AS)]
        f = lambda t, x: P5.pdf_xf_table(t, x, mu2)
        g1, g2 = f(0, x1), f(0, x2)
        terms = [lum * me2]
        for i in range(nf):
            q1, qb1, q2, qb2 = f(1 + 2 * i, x1), f(2 + 2 * i, x1), f(1 + 2 * i, x2), f(2 + 2 * i, x2)
            lumf = [q1 * qb2, qb1 * q2, q1 * g2, g1 * q2, qb1 * g2, g1 * qb2]
            terms += [lumf[c] / (x1 * x2) * M[c] for c in range(6)]
        terms = np.array(terms)
        a = np.abs(terms)
        # the class sums of the row are the flavour sums of these (signed) terms
        np.testing.assert_allclose([terms[1 + c::6].sum() for c in range(6)], r[-6:], rtol=1e-9, atol=1e-12 * a.max())
        expect += min(1.0, abs(w[k]) / w_max) * a / a.sum()
        hit = np.nonzero(ids == 100 + k)[0]
        if len(hit):
            words = mfo.philox_block(2, 4, 100 + k, 0xFFFFFFFF)
            v = mfo.uniform_from_words(words[2], words[3]) * a.sum()
            cum = np.cumsum(a)
            if np.min(np.abs(cum - v)) > 1e-9 * a.sum():
                assert chan[hit[0]] == int(np.argmax(cum > v)), k
    assert abs(expect.sum() - cnt) < 5 * math.sqrt(cnt)
    got = np.bincount(chan.astype(int), minlength=len(expect))
    by_class = lambda v: np.array([v[0]] + [v[1 + c::6].sum() for c in range(6)])
    for g, e in zip(by_class(got), by_class(expect)):
        assert abs(g - e) < 5 * math.sqrt(e + 1), (g, e)
    assert got[0] > 0.5 * cnt and got[1:].sum() > 30 and chan.max() <= 6 * nf
    # q g (valence quarks against the large gluon density) dominates the quark channels
    assert by_class(got)[3] + by_class(got)[4] > by_class(got)[1] + by_class(got)[2]
