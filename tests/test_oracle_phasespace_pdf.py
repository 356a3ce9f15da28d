"""Pins for the oracle's O4-O8: parton fractions, 2-body phase space, RAMBO, boost and cuts,
log-bicubic PDF.  CPU only; expected values are closed forms, invariants, quadratures and the golden points
of tests/golden/me2_points.txt (which no code in this repository produced)."""
import math
import os

import numpy as np
import pytest
from scipy import integrate

from oracle import mfo
from paper_2106_10279_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def mink(a, b):
    return a[..., 0] * b[..., 0] - a[..., 1] * b[..., 1] - a[..., 2] * b[..., 2] - a[..., 3] * b[..., 3]


def golden_points():
    out = {3: {"K": {}}, 4: {"K": {}}}
    for line in open(os.path.join(GOLD, "me2_points.txt")):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        if t[0] == "K":
            out[int(t[1])]["K"][int(t[2])] = [float(v) for v in t[3:7]]
        else:
            out[int(t[1])][t[0]] = float(t[2])
    return out


# ---- O4 ---------------------------------------------------------------------------------------------
def test_parton_fractions_identities():
    s = 13000.0 ** 2
    tau_min = 4 * 173.0 ** 2 / s
    assert tau_min == pytest.approx(7.08378698e-4, rel=1e-8)
    rng = np.random.default_rng(0)
    for x0, x1 in rng.random((50, 2)):
        k = mfo.parton_fractions(x0, x1, tau_min, s)
        assert k["x1"] * k["x2"] == pytest.approx(k["tau"], rel=1e-14)
        assert 0.5 * math.log(k["x1"] / k["x2"]) == pytest.approx(k["y"], abs=1e-13)
        assert tau_min * (1 - 1e-14) <= k["tau"] <= 1 and 0 < k["x1"] <= 1 + 1e-15 and 0 < k["x2"] <= 1 + 1e-15
        assert k["shat"] == pytest.approx(k["tau"] * s, rel=1e-15)
        assert abs(k["y"]) <= -0.5 * math.log(k["tau"]) * (1 + 1e-15)
    assert mfo.parton_fractions(0.0, 0.5, tau_min, s)["tau"] == pytest.approx(tau_min, rel=1e-14)
    assert mfo.parton_fractions(1.0, 0.5, tau_min, s)["tau"] == 1.0


def test_parton_fraction_jacobian_integral():
    """O4 pin: int dx1 dx2 Theta(x1 x2 > tau_min) = 1 - tau_min + tau_min ln tau_min."""
    for tau_min in (7.08378698e-4, (346 + 60.0) ** 2 / 13000.0 ** 2, 0.2):
        f = lambda x0: mfo.parton_fractions(x0, 0.3, tau_min, 1.0)["jac"]
        val, _ = integrate.quad(f, 0, 1, epsabs=0, epsrel=1e-13)
        assert val == pytest.approx(1 - tau_min + tau_min * math.log(tau_min), rel=1e-11)


# ---- O5 ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("m", [0.0, 173.0])
def test_two_body(m):
    rng = np.random.default_rng(1)
    for xc, xphi in rng.random((20, 2)):
        shat = (2 * m + 50 + 3000 * rng.random()) ** 2
        mom, wt = mfo.two_body(shat, m, xc, xphi)
        E = math.sqrt(shat) / 2
        assert np.allclose(mom[0] + mom[1], mom[2] + mom[3], atol=1e-12 * E)
        assert np.allclose(mom[0] + mom[1], [2 * E, 0, 0, 0], atol=1e-12 * E)
        assert np.allclose(mink(mom[2:], mom[2:]), m * m, atol=1e-10 * shat)
        assert np.allclose(mink(mom[:2], mom[:2]), 0, atol=1e-12 * shat)
        assert mom[0][3] > 0 > mom[1][3]
        assert mom[2][3] / np.linalg.norm(mom[2][1:]) == pytest.approx(2 * xc - 1, abs=1e-12)
        assert math.atan2(mom[2][2], mom[2][1]) % (2 * math.pi) == pytest.approx(2 * math.pi * xphi, abs=1e-12)
        beta = math.sqrt(1 - 4 * m * m / shat)
        assert wt == pytest.approx(beta / (8 * math.pi), rel=1e-13)  # int dPhi_2 = beta/(8 pi)


# ---- O6 ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("masses", [[0, 0], [0, 0, 0], [0, 0, 0, 0], [173, 173], [173, 173, 0], [173, 173, 0, 0],
                                    [173, 173, 0, 0, 0], [10, 20, 30, 40]])
def test_rambo_momentum_conservation_and_mass_shell(masses):
    rng = np.random.default_rng(2)
    n = len(masses)
    for w in (sum(masses) + 1.0, sum(masses) + 80.0, 1000.0, 9000.0):
        for _ in range(10):
            k, V = mfo.rambo(masses, w, rng.random(4 * n))
            assert np.allclose(k.sum(axis=0), [w, 0, 0, 0], rtol=0, atol=2e-12 * w)
            assert np.allclose(mink(k, k), np.square(masses), rtol=0, atol=1e-11 * w * w)
            assert V > 0 and np.all(k[:, 0] > 0)


def test_rambo_massless_weight_is_the_flat_volume():
    """O6 pin: massless weight = (pi/2)^(n-1) w^(2n-4) / ((n-1)!(n-2)!) for every point."""
    rng = np.random.default_rng(3)
    for n in (2, 3, 4, 5):
        w = 777.0
        want = (math.pi / 2) ** (n - 1) * w ** (2 * n - 4) / (math.factorial(n - 1) * math.factorial(n - 2))
        for _ in range(5):
            _, V = mfo.rambo([0.0] * n, w, rng.random(4 * n))
            assert V == pytest.approx(want, rel=1e-13)
    # n = 2 massless: the textbook two-body volume pi/2
    assert mfo.rambo([0, 0], 10.0, rng.random(8))[1] == pytest.approx(math.pi / 2, rel=1e-14)


def test_rambo_two_body_massive_volume_exact():
    """O6 pin: n=2 massive: V = pi |k| / w for every event (two-body phase space is a number)."""
    rng = np.random.default_rng(4)
    for w, m1, m2 in ((1000.0, 173.0, 173.0), (400.0, 173.0, 173.0), (100.0, 10.0, 60.0)):
        lam = (w * w - (m1 + m2) ** 2) * (w * w - (m1 - m2) ** 2)
        kabs = math.sqrt(lam) / (2 * w)
        for _ in range(5):
            k, V = mfo.rambo([m1, m2], w, rng.random(8))
            assert V == pytest.approx(math.pi * kabs / w, rel=1e-12)
            assert np.linalg.norm(k[0, 1:]) == pytest.approx(kabs, rel=1e-12)
    assert mfo.rambo([173.0, 173.0], 1000.0, rng.random(8))[1] == pytest.approx(1.47377532553376, rel=1e-12)


def test_rambo_three_body_massive_volume_vs_quadrature():
    """O6 pin: the mean of the massive RAMBO weight is the phase-space volume
    int ds12 R2(s; s12, 0) R2(s12; m^2, m^2), R2(s; a, b) = pi lambda^(1/2)(s, a, b) / (2 s)."""
    w, m = 1000.0, 173.0
    s = w * w

    def lam(a, b, c):
        return a * a + b * b + c * c - 2 * a * b - 2 * a * c - 2 * b * c

    def R2(S, a, b):
        return math.pi * math.sqrt(max(lam(S, a, b), 0.0)) / (2 * S)
    vol, _ = integrate.quad(lambda s12: R2(s, s12, 0.0) * R2(s12, m * m, m * m), 4 * m * m, s, epsrel=1e-11)
    assert vol == pytest.approx(733039.12, rel=1e-7)
    rng = np.random.default_rng(5)
    n = 40000
    V = np.array([mfo.rambo([m, m, 0.0], w, rng.random(12))[1] for _ in range(n)])
    err = V.std(ddof=1) / math.sqrt(n)
    assert abs(V.mean() - vol) < 4 * err
    assert err / vol < 2e-3


@pytest.mark.parametrize("n", [2, 3, 4, 5])
def test_two_pi_power_gives_the_textbook_massless_phase_space(n):
    """O6 step 6: dPhi_n = (2 pi)^(4-3n) V.  The oracle's OWN two_pi_power(n) times the volume its own
    RAMBO returns for massless particles must be the textbook integrated n-body phase space
    Phi_n(s) = s^(n-2) / (2 (4 pi)^(2n-3) (n-1)! (n-2)!): 1/(8 pi), s/(256 pi^3), s^2/(24576 pi^5), s^3/(4718592 pi^7).
    An exponent that is off by one is a factor 2 pi."""
    w = 730.0
    s = w * w
    literal = {2: 1 / (8 * math.pi), 3: s / (256 * math.pi ** 3), 4: s * s / (24576 * math.pi ** 5),
               5: s ** 3 / (4718592 * math.pi ** 7)}[n]
    general = s ** (n - 2) / (2 * (4 * math.pi) ** (2 * n - 3) * math.factorial(n - 1) * math.factorial(n - 2))
    assert literal == pytest.approx(general, rel=1e-14)
    rng = np.random.default_rng(40 + n)
    for _ in range(5):
        _, V0 = mfo.rambo([0.0] * n, w, rng.random(4 * n))
        assert mfo.two_pi_power(n) * V0 == pytest.approx(literal, rel=1e-13)
    # and the massive two-body case against the two-body routine's own weight: beta / (8 pi)
    m = 173.0
    _, V = mfo.rambo([m, m], w, rng.random(8))
    beta = math.sqrt(1 - 4 * m * m / s)
    assert mfo.two_pi_power(2) * V == pytest.approx(beta / (8 * math.pi), rel=1e-13)
    _, phi2 = mfo.two_body(s, m, 0.3, 0.6)
    assert mfo.two_pi_power(2) * V == pytest.approx(phi2, rel=1e-13)


def test_rambo_isotropy_and_energy_spectrum():
    """Massless n=2: directions must be isotropic (c = 2 rho1 - 1 is the cosine, phi = 2 pi rho2)."""
    k, _ = mfo.rambo([0, 0], 2.0, [0.75, 0.25, 0.3, 0.6, 0.1, 0.9, 0.5, 0.5])
    # for n=2 the boost only flips/aligns: the two momenta are back to back with |k| = 1
    assert np.allclose(k[0, 1:], -k[1, 1:], atol=1e-14) and np.linalg.norm(k[0, 1:]) == pytest.approx(1.0)


def test_rambo_golden_points():
    g = golden_points()
    for n in (3, 4):
        masses = [173.0, 173.0] + [0.0] * (n - 2)
        k, V = mfo.rambo(masses, 1000.0, W.rambo_test_point(n))
        assert V == pytest.approx(g[n]["V"], rel=1e-12)
        assert (2 * math.pi) ** (4 - 3 * n) * V == pytest.approx(g[n]["PHI"], rel=1e-12)
        for i in range(n):
            assert np.allclose(k[i], g[n]["K"][i], rtol=1e-12, atol=1e-10)
        kq, Vq = mfo.rambo(masses, 1000.0, W.rambo_test_point(n), prec=2)
        assert V == pytest.approx(Vq, rel=1e-13) and np.allclose(k, kq, rtol=1e-13, atol=1e-11)


# ---- O7 ---------------------------------------------------------------------------------------------
def test_boost_z():
    rng = np.random.default_rng(6)
    for _ in range(20):
        p3 = rng.normal(size=3) * 100
        m = rng.random() * 200
        p = np.array([math.sqrt(m * m + p3 @ p3), *p3])
        y = rng.normal() * 2
        q = mfo.boost_z(y, p)
        assert mink(q, q) == pytest.approx(m * m, abs=1e-9 * p[0] ** 2 * math.cosh(y) ** 2)
        assert q[1] == p[1] and q[2] == p[2]
        rap = lambda v: 0.5 * math.log((v[0] + v[3]) / (v[0] - v[3]))
        assert rap(q) == pytest.approx(rap(p) + y, abs=1e-10)
    # partonic CM beams map onto lab beams: E = x_i sqrt(s)/2
    s = 13000.0 ** 2
    k = mfo.parton_fractions(0.4, 0.8, 1e-3, s)
    E = math.sqrt(k["shat"]) / 2
    a = mfo.boost_z(k["y"], [E, 0, 0, E])
    b = mfo.boost_z(k["y"], [E, 0, 0, -E])
    assert a[0] == pytest.approx(k["x1"] * 6500.0, rel=1e-13) and b[0] == pytest.approx(k["x2"] * 6500.0, rel=1e-13)
    assert a[3] == pytest.approx(a[0], rel=1e-13) and b[3] == pytest.approx(-b[0], rel=1e-13)


def test_cut_observables_and_decisions():
    rng = np.random.default_rng(7)
    npass = 0
    for _ in range(300):
        g = []
        for i in range(2):
            pt = 10 + 100 * rng.random()
            eta = rng.normal() * 1.8
            phi = rng.uniform(-math.pi, math.pi)
            g.append([pt * math.cosh(eta), pt * math.cos(phi), pt * math.sin(phi), pt * math.sinh(eta), pt, eta, phi])
        g = np.array(g)
        ok, obs = mfo.cuts(g[:, :4], 30.0, 2.5, 0.4)
        assert np.allclose(obs[:, 0], g[:, 4], rtol=1e-13)
        assert np.allclose(obs[:, 1], g[:, 5], atol=1e-12)
        # pseudorapidity through the polar angle: eta = -ln tan(theta/2)
        theta = np.arctan2(g[:, 4], g[:, 3])
        assert np.allclose(obs[:, 1], -np.log(np.tan(theta / 2)), atol=1e-10)
        dphi = abs(g[0, 6] - g[1, 6])
        dphi = min(dphi, 2 * math.pi - dphi)
        dr = math.hypot(g[0, 5] - g[1, 5], dphi)
        want = bool(np.all(g[:, 4] > 30) and np.all(np.abs(g[:, 5]) < 2.5) and dr > 0.4)
        assert ok == want
        npass += ok
        # single-gluon variant (C2) ignores dR; disabled cuts pass everything
        ok1, _ = mfo.cuts(g[:1, :4], 30.0, 2.5, 0.0)
        assert ok1 == bool(g[0, 4] > 30 and abs(g[0, 5]) < 2.5)
        assert mfo.cuts(g[:, :4], 0.0, 0.0, 0.0)[0]
    assert 20 < npass < 280
    # strict inequalities
    pt = 30.0
    p = [[pt, pt, 0, 0]]
    assert not mfo.cuts(p, 30.0, 2.5, 0.0)[0] and mfo.cuts(p, math.nextafter(30.0, 0), 2.5, 0.0)[0]
    # delta-phi wraps: two gluons at phi = +-3.1 are close
    a = [50 * math.cosh(0.1), 50 * math.cos(3.1), 50 * math.sin(3.1), 50 * math.sinh(0.1)]
    b = [50 * math.cosh(0.1), 50 * math.cos(-3.1), 50 * math.sin(-3.1), 50 * math.sinh(0.1)]
    assert not mfo.cuts([a, b], 30.0, 2.5, 0.4)[0] and mfo.cuts([a, b], 30.0, 2.5, 0.05)[0]


def test_golden_points_pass_the_cuts_at_y0():
    g = golden_points()
    k = np.array([g[4]["K"][i] for i in range(4)])
    ok, obs = mfo.cuts(k[2:], 30.0, 2.5, 0.4)
    assert ok
    assert obs[0, 0] == pytest.approx(150.3, abs=0.5) and obs[1, 0] == pytest.approx(235.1, abs=0.5)
    dphi = abs(obs[0, 2] - obs[1, 2])
    dphi = min(dphi, 2 * math.pi - dphi)
    assert math.hypot(obs[0, 1] - obs[1, 1], dphi) == pytest.approx(1.347, abs=2e-3)  # SURVEY.md golden points


# ---- O8 ---------------------------------------------------------------------------------------------
class _WL:
    pass


def _proc_with_table(lnx, lnq2, xf):
    wl = W.C1
    return mfo.Process(wl, (lnx, lnq2, xf))


def test_pdf_table_recipe(pdf):
    lnx, lnq2, xf = pdf
    assert len(lnx) == 100 and len(lnq2) == 50 and xf.shape == (100, 50)
    assert math.exp(lnx[0]) == pytest.approx(1e-9, rel=1e-13) and lnx[-1] == 0.0
    assert math.exp(lnq2[0]) == pytest.approx(2.72, rel=1e-13) and math.exp(lnq2[-1]) == pytest.approx(1e10, rel=1e-12)
    assert np.allclose(np.diff(lnx), np.diff(lnx)[0]) and np.allclose(np.diff(lnq2), np.diff(lnq2)[0])
    assert np.all(xf[-1] == 0.0)
    x, q2 = math.exp(lnx[40]), math.exp(lnq2[20])
    assert xf[40, 20] == pytest.approx(3 * x ** -0.1 * (1 - x) ** 5 * (1 + 0.1 * math.log(q2 / 100)), rel=1e-13)


def test_pdf_exact_at_knots(pdf, oracle_procs):
    lnx, lnq2, xf = pdf
    P = oracle_procs[1]
    for i in (0, 1, 37, 98):
        for j in (0, 1, 20, 48, 49):
            assert P.pdf_xf(math.exp(lnx[i]), math.exp(lnq2[j])) == pytest.approx(xf[i, j], rel=1e-11, abs=1e-13)


def test_pdf_reproduces_bilinear_and_quadratic_tables(pdf):
    lnx, lnq2, _ = pdf
    rng = np.random.default_rng(8)
    # bilinear in (ln x, ln Q^2): reproduced everywhere, edges included
    a, b, c, d = 2.0, 0.3, -0.07, 0.011
    xf = a + b * lnx[:, None] + c * lnq2[None, :] + d * lnx[:, None] * lnq2[None, :]
    P = _proc_with_table(lnx, lnq2, xf)
    for _ in range(200):
        lx = rng.uniform(lnx[0], 0.0)
        lq = rng.uniform(lnq2[0], lnq2[-1])
        want = a + b * lx + c * lq + d * lx * lq
        assert P.pdf_xf(math.exp(lx), math.exp(lq)) == pytest.approx(want, rel=1e-12)
    # quadratic in ln x (uniform spacing): central-difference derivatives are exact in interior cells
    xf = (1.0 + 0.2 * lnx[:, None] + 0.03 * lnx[:, None] ** 2) * (1 + 0.05 * lnq2[None, :])
    P = _proc_with_table(lnx, lnq2, xf)
    for _ in range(200):
        lx = rng.uniform(lnx[1], lnx[-2])
        lq = rng.uniform(lnq2[0], lnq2[-1])
        want = (1.0 + 0.2 * lx + 0.03 * lx * lx) * (1 + 0.05 * lq)
        assert P.pdf_xf(math.exp(lx), math.exp(lq)) == pytest.approx(want, rel=1e-11)
    # quadratic in ln Q^2 in interior cells
    xf = (1 + 0.1 * lnx[:, None]) * (2.0 - 0.3 * lnq2[None, :] + 0.02 * lnq2[None, :] ** 2)
    P = _proc_with_table(lnx, lnq2, xf)
    for _ in range(200):
        lx = rng.uniform(lnx[0], 0.0)
        lq = rng.uniform(lnq2[1], lnq2[-2])
        want = (1 + 0.1 * lx) * (2.0 - 0.3 * lq + 0.02 * lq * lq)
        assert P.pdf_xf(math.exp(lx), math.exp(lq)) == pytest.approx(want, rel=1e-11)


def test_pdf_continuity_across_cells(pdf, oracle_procs):
    """A cubic Hermite interpolant is C1: value and slope are continuous across knots in both directions."""
    lnx, lnq2, _ = pdf
    P = oracle_procs[1]
    q2 = 173.0 ** 2
    for i in (5, 50, 90):
        x = math.exp(lnx[i])
        eps = 1e-7
        lo, hi, mid = P.pdf_xf(x * (1 - eps), q2), P.pdf_xf(x * (1 + eps), q2), P.pdf_xf(x, q2)
        assert lo == pytest.approx(mid, rel=1e-5) and hi == pytest.approx(mid, rel=1e-5)
        assert (hi - mid) == pytest.approx(mid - lo, rel=2e-3)
    x = 0.01
    for j in (3, 25, 40):
        q = math.exp(lnq2[j])
        eps = 1e-6
        lo, hi, mid = P.pdf_xf(x, q * (1 - eps)), P.pdf_xf(x, q * (1 + eps)), P.pdf_xf(x, q)
        assert (hi - mid) == pytest.approx(mid - lo, rel=2e-3)


def test_pdf_vs_generating_formula(pdf, oracle_procs):
    """Sanity only (the PDF is the interpolant, not the formula): SURVEY.md O8 quotes 6e-7 at x = 0.0123,
    4e-3 at x = 0.5 and a NEGATIVE interpolant at x = 0.9, mu^2 = m_t^2."""
    P = oracle_procs[1]
    q2 = 173.0 ** 2
    f = lambda x: 3 * x ** -0.1 * (1 - x) ** 5 * (1 + 0.1 * math.log(q2 / 100))
    assert abs(P.pdf_xf(0.0123, q2) / f(0.0123) - 1) < 2e-6
    assert abs(P.pdf_xf(0.5, q2) / f(0.5) - 1) < 1e-2
    assert P.pdf_xf(0.9, q2) == pytest.approx(-7.2e-4, rel=0.05) and f(0.9) == pytest.approx(4.8e-5, rel=0.05)
    for prec in (1, 2):
        assert P.pdf_xf(0.0123, q2, prec) == pytest.approx(P.pdf_xf(0.0123, q2), rel=1e-13)


def test_create_rejects_out_of_range_scale(pdf):
    import dataclasses
    with pytest.raises(ValueError):
        mfo.Process(dataclasses.replace(W.C1, mu2=1.0), pdf)
    with pytest.raises(ValueError):
        mfo.Process(dataclasses.replace(W.C1, mu2=1e11), pdf)
