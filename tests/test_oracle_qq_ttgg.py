"""Pins of the oracle's q qbar -> t tbar g g matrix element and of process 7 = pp -> ttbar gg (PAPER.md L101 and
Table 1: 267 diagrams = 123 gg + 4 x 36).  oracle/amplitude_qq.hpp writes the 36 diagrams out with explicit colour tensors;
nothing here re-types its formulae: the pins are a second, diagram-free method (colour-dressed subset recursion), gauge invariance,
basis independence, the symmetries of the process and its two collinear limits onto the separately pinned q qbar -> t tbar g."""
import math

import numpy as np
import pytest

from oracle import mfo
from paper_2106_10279_b200 import workloads as W

MT, AS = 173.0, 0.118
GS = math.sqrt(4 * math.pi * AS)


def _point(seed, w=1500.0):
    rng = np.random.default_rng(seed)
    k, _ = mfo.rambo([MT, MT, 0.0, 0.0], w, rng.random(16))
    return np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k])


def _boost(p, Q):
    """p given in the rest frame of Q (mass M) -> the frame where the system moves with Q"""
    M = math.sqrt(Q[0] ** 2 - Q[1:] @ Q[1:])
    b, gam = Q[1:] / Q[0], Q[0] / M
    bp = b @ p[1:]
    return np.array([gam * (p[0] + bp), *(p[1:] + b * (gam * gam / (gam + 1) * bp + gam * p[0]))])


def test_diagram_sum_equals_the_dressed_recursion():
    """for explicit helicities and colours, sum_d (colour tensor)_d x kin_d of the 36 diagrams = the amplitude of a recursion over
    subsets of {g, g, light pair} that enumerates no diagram; colour conservation makes many assignments vanish on both sides"""
    rng = np.random.default_rng(11)
    n_nonzero, scale = 0, 0.0
    pairs = []
    for seed in (1, 2, 3):
        mom = _point(seed, 900.0 + 700.0 * seed)
        for _ in range(150):
            lam = rng.choice([-1, 1], 6)
            col = [*rng.integers(0, 3, 4), *rng.integers(0, 8, 2)]
            a, b = mfo.qq_ttbar_gg_amplitude(mom, MT, GS, lam, col, basis=int(rng.integers(0, 4)))
            pairs.append((a, b))
            scale = max(scale, abs(b))
    for a, b in pairs:
        assert abs(a - b) <= 1e-11 * scale
        n_nonzero += abs(b) > 1e-6 * scale
    assert n_nonzero >= 30


@pytest.mark.parametrize("gluon", [0, 1])
def test_ward_identity(gluon):
    """polarisation -> momentum: the colour-summed square vanishes (all 36 diagrams and their colour factors enter); what is left
    is rounding, which shrinks with the precision"""
    mom = _point(5)
    m = mfo.me2_qq_ttbar_gg(mom, MT, AS)
    assert m > 0
    assert abs(mfo.me2_qq_ttbar_gg(mom, MT, AS, subst=gluon)) < 1e-7 * m
    assert abs(mfo.me2_qq_ttbar_gg(mom, MT, AS, subst=gluon, prec=1)) < 1e-10 * m


def test_basis_independence_and_symmetries():
    mom = _point(7)
    m = mfo.me2_qq_ttbar_gg(mom, MT, AS)
    for basis in (1, 2, 3):
        assert mfo.me2_qq_ttbar_gg(mom, MT, AS, basis=basis) == pytest.approx(m, rel=1e-11)
    assert mfo.me2_qq_ttbar_gg(mom, MT, AS, prec=1) == pytest.approx(m, rel=1e-12)
    # Bose symmetry of the two gluons
    assert mfo.me2_qq_ttbar_gg(mom[[0, 1, 2, 3, 5, 4]], MT, AS) == pytest.approx(m, rel=1e-11)
    # charge conjugation: q <-> qbar together with t <-> tbar
    assert mfo.me2_qq_ttbar_gg(mom[[1, 0, 3, 2, 4, 5]], MT, AS) == pytest.approx(m, rel=1e-11)
    # ... but not either exchange alone (the charge asymmetry of q qbar -> t tbar + gluons)
    assert abs(mfo.me2_qq_ttbar_gg(mom[[1, 0, 2, 3, 4, 5]], MT, AS) / m - 1) > 1e-3
    # parity: all three-momenta reflected
    refl = mom * np.array([1.0, -1.0, -1.0, -1.0])
    assert mfo.me2_qq_ttbar_gg(refl, MT, AS) == pytest.approx(m, rel=1e-11)
    # coupling power
    assert mfo.me2_qq_ttbar_gg(mom, MT, 2 * AS) == pytest.approx(16 * m, rel=1e-12)


def test_final_state_collinear_limit_onto_qq_ttg():
    """g g collinear (m56 -> 0), averaged over the azimuth: |M|^2 -> (2 g^2 / m56^2) P_gg(z) |M(q qbar -> t tbar g)|^2 with
    P_gg = 2 C_A [z/(1-z) + (1-z)/z + z(1-z)]; the averaged matrix elements carry 1/2! against 1/1!"""
    rng = np.random.default_rng(65)
    w, m56 = 1000.0, 0.25
    rho = rng.random(16)
    k3, _ = mfo.rambo([MT, MT, 0.0], w, rho[:12])
    kc, _ = mfo.rambo([MT, MT, m56], w, rho[:12])
    beams = [[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2]]
    me3 = mfo.me2_light_line_ttbar_g(0, np.vstack([beams, k3]), MT, AS)
    G = kc[2]
    nb = G[1:] / np.linalg.norm(G[1:])
    e1 = np.cross(nb, [0.0, 0.0, 1.0])
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(nb, e1)
    g2 = 4 * math.pi * AS
    for cth in (0.3, -0.55):
        sth = math.sqrt(1 - cth * cth)
        vals, zs = [], []
        for iphi in range(8):
            phi = 2 * math.pi * (iphi + 0.3) / 8
            d = sth * (math.cos(phi) * e1 + math.sin(phi) * e2) + cth * nb
            out = [_boost(np.array([m56 / 2, *(sgn * m56 / 2 * d)]), G) for sgn in (1, -1)]
            mom = np.vstack([beams, kc[:2], out])
            assert np.allclose(mom[0] + mom[1], mom[2:].sum(axis=0), atol=1e-9 * w)
            vals.append(mfo.me2_qq_ttbar_gg(mom, MT, AS))
            zs.append(out[0][0] / G[0])
        z = float(np.mean(zs))
        pgg = 2 * 3.0 * (z / (1 - z) + (1 - z) / z + z * (1 - z))
        want = 2 * g2 / m56 ** 2 * pgg * me3 / 2.0
        assert np.mean(vals) == pytest.approx(want, rel=0.02)
        assert np.std(vals) / np.mean(vals) > 1e-3


def test_initial_state_collinear_limit_onto_qq_ttg():
    """a gluon collinear with the incoming quark, k = (1 - z) p1 + O(theta):
        |M|^2 -> g^2 / (z p1.k) P_qq(z) |M(q(z p1) qbar -> t tbar g)|^2,   P_qq = C_F (1 + z^2)/(1 - z)
    (no azimuthal correlation: the quark's helicity is conserved); 1/2! against 1/1! for the identical gluons"""
    rng = np.random.default_rng(8)
    E, z = 600.0, 0.6
    p1, p2 = np.array([E, 0, 0, E]), np.array([E, 0, 0, -E])
    rho = rng.random(12)
    g2 = 4 * math.pi * AS
    ratios = []
    for theta in (3e-3, 3e-4):
        om = (1 - z) * E
        k = om * np.array([1.0, math.sin(theta) * math.cos(0.7), math.sin(theta) * math.sin(0.7), math.cos(theta)])
        Q = p1 + p2 - k
        M = math.sqrt(Q[0] ** 2 - Q[1:] @ Q[1:])
        kr, _ = mfo.rambo([MT, MT, 0.0], M, rho)
        rest = np.array([_boost(q, Q) for q in kr])
        mom = np.vstack([p1, p2, rest[0], rest[1], k, rest[2]])
        assert np.allclose(mom[0] + mom[1], mom[2:].sum(axis=0), atol=1e-9 * E)
        full = mfo.me2_qq_ttbar_gg(mom, MT, AS)
        Q0 = z * p1 + p2
        M0 = math.sqrt(Q0[0] ** 2 - Q0[1:] @ Q0[1:])
        k0, _ = mfo.rambo([MT, MT, 0.0], M0, rho)
        red = mfo.me2_light_line_ttbar_g(0, np.vstack([z * p1, p2, [_boost(q, Q0) for q in k0]]), MT, AS)
        p1k = p1[0] * k[0] - p1[1:] @ k[1:]
        want = g2 / (z * p1k) * (4.0 / 3.0) * (1 + z * z) / (1 - z) * red / 2.0
        ratios.append(full / want)
    assert abs(ratios[0] - 1) < 0.03 and abs(ratios[1] - 1) < 0.003


def test_process_rows_and_channels(oracle_procs):
    """process 7 = process 3 + the flavour-summed q qbar terms at the same points: every column of the g g -> t tbar g g row is
    reproduced, the weight is the sum of the two luminosity x |M|^2 terms, and accepted events carry a channel drawn from them"""
    P7, P3 = oracle_procs[W.MF_PP_TTGG], oracle_procs[W.MF_GG_TTGG]
    grid = W.uniform_grid(18)
    r7, r3 = P7.debug_eval(grid, 2, 1, 5, 48), P3.debug_eval(grid, 2, 1, 5, 48)
    n3 = r3.shape[1]
    assert r7.shape[1] == n3 + 2
    o = 18 + 4 * 6                                   # x[D], momenta, then x1, x2, lum, me2, phi, jac, w, pass, r, u[D], bin[D]
    c = {"x1": o, "x2": o + 1, "lum": o + 2, "me2": o + 3, "w": o + 6, "pas": o + 7}
    same = [j for j in range(n3) if j != c["w"]]
    assert np.array_equal(r7[:, same], r3[:, same])
    ok = r3[:, c["pas"]] > 0
    assert ok.sum() > 20
    lum_qq, me_qq = r7[ok, n3], r7[ok, n3 + 1]
    assert (me_qq > 0).all() and (lum_qq > 0).sum() > 15       # the interpolated table dips below zero near x = 1 (R8)
    gg = r3[ok, c["lum"]] * r3[ok, c["me2"]]
    np.testing.assert_allclose(r7[ok, c["w"]] / r3[ok, c["w"]], (gg + lum_qq * me_qq) / gg, rtol=1e-12)
    # the q qbar matrix element of the row is the luminosity-weighted mean of the two beam assignments at the row's momenta
    i = int(np.flatnonzero(ok)[0])
    lab = r7[i, 18:o].reshape(6, 4)
    y = 0.5 * math.log(r7[i, c["x1"]] / r7[i, c["x2"]])
    cm = np.array([mfo.boost_z(-y, p) for p in lab])
    ma = mfo.me2_qq_ttbar_gg(cm, MT, AS)
    mb = mfo.me2_qq_ttbar_gg(cm[[1, 0, 2, 3, 4, 5]], MT, AS)
    assert min(ma, mb) * (1 - 1e-9) <= r7[i, n3 + 1] <= max(ma, mb) * (1 + 1e-9)
    # unweighting with a vanishing w_max accepts every event that passes the cuts: channel codes 0 (gg) or 1 + 2 i (+1: the
    # quark comes from beam 2); the quark share of this synthetic proton at these points is ~1 %
    rec, count, hist, res = P7.unweight(grid, 0, 0, 0, 400, 1e-30, 400)
    assert res.n_accept == res.n_pass == count > 250
    ch = P7.records_array(rec, count)["channel"].astype(np.int64)
    assert ch.min() == 0 and ch.max() <= 2 * W.N_FLAVOURS and 0 < (ch > 0).sum() < 0.1 * count
