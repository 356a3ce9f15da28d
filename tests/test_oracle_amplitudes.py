"""Pins for the oracle's O9-O11: external wavefunctions, tree amplitudes, colour sum.
CPU only.  Expected values: Dirac algebra written out with numpy, textbook closed forms (e+e- -> mu+mu-,
Ellis-Stirling-Webber gg -> ttbar), gauge / Lorentz / Bose invariance, an explicit colour sum, closed-form
colour-matrix entries and the golden points of tests/golden/me2_points.txt."""
import itertools
import math

import numpy as np
import pytest

from oracle import mfo
from paper_2106_10279_b200 import workloads as W
from test_oracle_phasespace_pdf import golden_points, mink

# Dirac representation, written out independently of the oracle
_s = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], complex)]
_Z = np.zeros((2, 2))
GAMMA = [np.block([[np.eye(2), _Z], [_Z, -np.eye(2)]]).astype(complex)] + \
        [np.block([[_Z, s], [-s, _Z]]) for s in _s]


def slash(p):
    return p[0] * GAMMA[0] - p[1] * GAMMA[1] - p[2] * GAMMA[2] - p[3] * GAMMA[3]


def rand_mom(rng, m, scale=300.0):
    p3 = rng.normal(size=3) * scale
    return np.array([math.sqrt(m * m + p3 @ p3), *p3])


# ---- O9 ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("basis", [0, 1])
@pytest.mark.parametrize("m", [0.0, 173.0])
def test_spinors_solve_dirac_equation_and_are_complete(m, basis):
    rng = np.random.default_rng(0)
    moms = [rand_mom(rng, m) for _ in range(5)] + [np.array([math.sqrt(m * m + 2500), 0, 0, 50.0]),
                                                    np.array([math.sqrt(m * m + 2500), 0, 0, -50.0])]
    for p in moms:
        E = p[0]
        uu = np.zeros((4, 4), complex)
        vv = np.zeros((4, 4), complex)
        for lam in (-1, 1):
            u = mfo.spinor(p, m, lam, basis, 0)
            v = mfo.spinor(p, m, lam, basis, 1)
            assert np.allclose((slash(p) - m * np.eye(4)) @ u, 0, atol=1e-11 * E ** 1.5)
            assert np.allclose((slash(p) + m * np.eye(4)) @ v, 0, atol=1e-11 * E ** 1.5)
            assert (u.conj() @ u).real == pytest.approx(2 * E, rel=1e-13)
            assert (v.conj() @ v).real == pytest.approx(2 * E, rel=1e-13)
            uu += np.outer(u, u.conj() @ GAMMA[0])
            vv += np.outer(v, v.conj() @ GAMMA[0])
        assert np.allclose(uu, slash(p) + m * np.eye(4), atol=1e-11 * E)
        assert np.allclose(vv, slash(p) - m * np.eye(4), atol=1e-11 * E)


def test_helicity_spinors_are_helicity_eigenstates():
    rng = np.random.default_rng(1)
    for m in (0.0, 173.0):
        p = rand_mom(rng, m)
        n = p[1:] / np.linalg.norm(p[1:])
        sig = sum(n[i] * np.block([[_s[i], _Z], [_Z, _s[i]]]) for i in range(3))  # Sigma.p-hat
        for lam in (-1, 1):
            u = mfo.spinor(p, m, lam, 0, 0)
            v = mfo.spinor(p, m, lam, 0, 1)
            assert np.allclose(sig @ u, lam * u, atol=1e-10)
            assert np.allclose(sig @ v, -lam * v, atol=1e-10)   # v(p, lambda) has spin -lambda along p


@pytest.mark.parametrize("basis", [0, 1])
def test_polarisation_vectors(basis):
    rng = np.random.default_rng(2)
    moms = [rand_mom(rng, 0.0) for _ in range(6)] + [np.array([50.0, 0, 0, 50.0]), np.array([50.0, 0, 0, -50.0])]
    g = np.diag([1.0, -1, -1, -1])
    for p in moms:
        e = {lam: mfo.polarisation(p, lam, basis) for lam in (-1, 1)}
        for lam in (-1, 1):
            assert abs(e[lam][0]) == 0
            assert abs(e[lam] @ g @ p) < 1e-12 * p[0]
            assert e[lam] @ g @ e[lam].conj() == pytest.approx(-1.0, abs=1e-13)
        assert abs(e[1] @ g @ e[-1].conj()) < 1e-13
        # completeness on the transverse plane: sum eps^i eps^j* = delta^ij - n^i n^j
        n = p[1:] / p[0]
        tot = sum(np.outer(e[l][1:], e[l][1:].conj()) for l in (-1, 1))
        assert np.allclose(tot, np.eye(3) - np.outer(n, n), atol=1e-13)
        if basis == 0:  # circular: rotation generator eigenstate, (n.S) eps = lambda eps, (S_k)_ij = -i eps_ijk
            for lam in (-1, 1):
                rot = 1j * np.cross(n, e[lam][1:])
                assert np.allclose(rot, lam * e[lam][1:], atol=1e-13)


# ---- O10 C0 -----------------------------------------------------------------------------------------
@pytest.mark.parametrize("basis", [0, 1])
def test_ee_mumu_closed_form(oracle_procs, basis):
    """(1/4) sum |M|^2 = e^4 (1 + cos^2 theta) for massless e+e- -> gamma* -> mu+mu-."""
    P = oracle_procs[0]
    e4 = (4 * math.pi / 132.507) ** 2
    for xc, xphi in np.random.default_rng(3).random((10, 2)):
        mom, _ = mfo.two_body(100.0 ** 2, 0.0, xc, xphi)
        c = 2 * xc - 1
        v, per = P.me2(mom, basis=basis, want_per_hel=True)
        assert v == pytest.approx(e4 * (1 + c * c), rel=1e-13)
        if basis == 0:  # massless chirality: only 4 of the 16 helicity combinations survive
            assert np.sum(per > 1e-20 * v) == 4
            assert sorted(per)[-4:] == pytest.approx(sorted([e4 * (1 + c) ** 2] * 2 + [e4 * (1 - c) ** 2] * 2), rel=1e-12)


# ---- O10/O11 C1 -------------------------------------------------------------------------------------
def esw_gg_ttbar(mom, m, alpha_s):
    """Ellis-Stirling-Webber: (1/256) sum |M|^2 = gs^4 [1/(6 t1 t2) - 3/8][t1^2 + t2^2 + rho - rho^2/(4 t1 t2)]."""
    shat = mink(mom[0] + mom[1], mom[0] + mom[1])
    t1 = 2 * mink(mom[0], mom[2]) / shat
    t2 = 2 * mink(mom[1], mom[2]) / shat
    rho = 4 * m * m / shat
    gs4 = (4 * math.pi * alpha_s) ** 2
    return gs4 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1 * t1 + t2 * t2 + rho - rho * rho / (4 * t1 * t2))


@pytest.mark.parametrize("basis", [0, 1, 2, 3])
def test_gg_ttbar_analytic(oracle_procs, basis):
    P = oracle_procs[1]
    rng = np.random.default_rng(4)
    for _ in range(8):
        shat = (346.0 + 0.5 + 3000 * rng.random() ** 2) ** 2
        mom, _ = mfo.two_body(shat, 173.0, rng.random(), rng.random())
        assert P.me2(mom, basis=basis) == pytest.approx(esw_gg_ttbar(mom, 173.0, 0.118), rel=2e-12)


def test_gg_ttbar_partonic_cross_section(oracle_procs):
    """sigma-hat_gg = (pi alpha_s^2 / 3 s)[(1 + rho + rho^2/16) ln((1+beta)/(1-beta)) - beta (7/4 + 31 rho/16)]
    from the oracle's helicity amplitudes integrated over the oracle's two-body phase space."""
    from scipy import integrate
    P = oracle_procs[1]
    for rs in (400.0, 1000.0, 4000.0):
        shat = rs * rs
        rho = 4 * 173.0 ** 2 / shat
        beta = math.sqrt(1 - rho)
        want = math.pi * 0.118 ** 2 / (3 * shat) * ((1 + rho + rho * rho / 16) * math.log((1 + beta) / (1 - beta))
                                                    - beta * (7.0 / 4 + 31 * rho / 16))

        def f(xc):
            mom, wt = mfo.two_body(shat, 173.0, xc, 0.3)
            return P.me2(mom) * wt / (2 * shat)
        got, _ = integrate.quad(f, 0, 1, epsabs=0, epsrel=1e-11, limit=200)
        assert got == pytest.approx(want, rel=1e-9)


# ---- O10/O11 C2, C3 ---------------------------------------------------------------------------------
def _rambo_event(n, w, rng):
    masses = [173.0, 173.0] + [0.0] * (n - 2)
    k, _ = mfo.rambo(masses, w, rng.random(4 * n))
    return np.vstack([[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2], k])


def test_golden_me2_points(oracle_procs):
    g = golden_points()
    for n, pid in ((3, 2), (4, 3)):
        k = np.array([g[n]["K"][i] for i in range(n)])
        mom = np.vstack([[500, 0, 0, 500.0], [500, 0, 0, -500.0], k])
        assert oracle_procs[pid].me2(mom) == pytest.approx(g[n]["ME2"], rel=2e-11)
        # and through the oracle's own RAMBO
        kk, _ = mfo.rambo([173.0, 173.0] + [0.0] * (n - 2), 1000.0, W.rambo_test_point(n))
        mom = np.vstack([[500, 0, 0, 500.0], [500, 0, 0, -500.0], kk])
        assert oracle_procs[pid].me2(mom) == pytest.approx(g[n]["ME2"], rel=1e-11)


@pytest.mark.parametrize("pid,n", [(1, 2), (2, 3), (3, 4)])
def test_gauge_invariance(oracle_procs, pid, n):
    """Replacing one gluon's polarisation by its momentum makes every ordered amplitude vanish."""
    P = oracle_procs[pid]
    rng = np.random.default_rng(5)
    mom = _rambo_event(n, 900.0, rng)
    v, amps = P.me2(mom, want_amps=True)
    scale = np.abs(amps).max()
    for gl in range(n):  # n = ng here: 2 beams + (n-2) final gluons = n gluons
        v0, a0 = P.me2(mom, subst_gluon=gl, want_amps=True)
        # eps -> k is O(E) larger than a unit polarisation: compare to scale * E
        assert np.abs(a0).max() < 1e-11 * scale * 900.0
        assert v0 < 1e-20 * v * 900.0 ** 2


@pytest.mark.parametrize("pid,n", [(1, 2), (2, 3), (3, 4)])
def test_basis_independence(oracle_procs, pid, n):
    P = oracle_procs[pid]
    mom = _rambo_event(n, 1200.0, np.random.default_rng(6))
    v = P.me2(mom, prec=1)
    for basis in (0, 1, 2, 3):
        assert P.me2(mom, basis=basis) == pytest.approx(v, rel=1e-12)


def _lorentz(rng):
    # random rotation (QR) times a boost along a random axis
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] *= -1
    R = np.eye(4)
    R[1:, 1:] = q
    b = rng.normal(size=3)
    b *= 0.6 / np.linalg.norm(b)
    g = 1 / math.sqrt(1 - b @ b)
    B = np.eye(4)
    B[0, 0] = g
    B[0, 1:] = B[1:, 0] = g * b
    B[1:, 1:] += (g - 1) * np.outer(b, b) / (b @ b)
    return B @ R


@pytest.mark.parametrize("pid,n", [(1, 2), (2, 3), (3, 4)])
def test_lorentz_invariance(oracle_procs, pid, n):
    P = oracle_procs[pid]
    rng = np.random.default_rng(7)
    mom = _rambo_event(n, 800.0, rng)
    v = P.me2(mom)
    for _ in range(2):
        L = _lorentz(rng)
        mom2 = mom @ L.T
        assert mink(mom2[2], mom2[2]) == pytest.approx(173.0 ** 2, rel=1e-10)
        assert P.me2(mom2) == pytest.approx(v, rel=1e-10)
    # pure rotation about z: exact symmetry of the beam setup
    c, s = math.cos(0.7), math.sin(0.7)
    Rz = np.array([[1, 0, 0, 0], [0, c, -s, 0], [0, s, c, 0], [0, 0, 0, 1.0]])
    assert P.me2(mom @ Rz.T) == pytest.approx(v, rel=1e-12)


def test_bose_and_beam_exchange_symmetry(oracle_procs):
    rng = np.random.default_rng(8)
    P = oracle_procs[3]
    mom = _rambo_event(4, 1000.0, rng)
    v = P.me2(mom)
    assert P.me2(mom[[0, 1, 2, 3, 5, 4]]) == pytest.approx(v, rel=1e-12)   # final gluons exchanged
    assert P.me2(mom[[1, 0, 2, 3, 4, 5]]) == pytest.approx(v, rel=1e-12)   # beams exchanged
    # charge conjugation: t <-> tbar
    assert P.me2(mom[[0, 1, 3, 2, 4, 5]]) == pytest.approx(v, rel=1e-12)
    P = oracle_procs[2]
    mom = _rambo_event(3, 1000.0, rng)
    assert P.me2(mom[[1, 0, 3, 2, 4]]) == pytest.approx(P.me2(mom), rel=1e-12)


@pytest.mark.parametrize("pid,n", [(1, 2), (2, 3), (3, 4)])
def test_dressed_recursion_equals_ordered_sum(oracle_procs, pid, n):
    """Colour-dressed Feynman-rule recursion (f^{abc}, T^a explicit) = sum_sigma (T..T)_ij A(sigma)."""
    P = oracle_procs[pid]
    rng = np.random.default_rng(9)
    mom = _rambo_event(n, 1000.0, rng)
    _, amps = P.me2(mom, want_amps=True)
    scale = np.abs(amps).max()      # size of an ordered amplitude at this point; |(T..T)_ij| <= 1
    nz = 0
    for _ in range(40 if n < 4 else 25):
        hel = rng.choice([-1, 1], size=2 + n)
        col = rng.integers(0, 8, size=n)
        i, j = rng.integers(0, 3, size=2)
        a = P.dressed_amplitude(mom, hel, col, i, j)
        b = P.ordered_amplitude_coloured(mom, hel, col, i, j)
        assert abs(a - b) <= 1e-12 * scale
        nz += abs(a) > 1e-6 * scale
    assert nz >= 5


def test_explicit_colour_sum_equals_colour_matrix_contraction(oracle_procs):
    """sum over all 8^3 x 3 x 3 colours of |M|^2 (dressed) = A^dagger C A (gg -> ttbar g, two helicities)."""
    P = oracle_procs[2]
    mom = _rambo_event(3, 1000.0, np.random.default_rng(10))
    _, amps = P.me2(mom, want_amps=True)
    C = mfo.colour_matrix(3)
    for hel in ([1, -1, 1, -1, 1], [-1, -1, 1, 1, -1]):
        hidx = int("".join("1" if h > 0 else "0" for h in hel), 2)
        A = amps[hidx]
        want = (A.conj() @ C @ A).real
        tot = 0.0
        for col in itertools.product(range(8), repeat=3):
            for i in range(3):
                for j in range(3):
                    tot += abs(P.dressed_amplitude(mom, hel, col, i, j)) ** 2
        assert tot == pytest.approx(want, rel=1e-12)


def test_helicity_index_convention_and_average(oracle_procs):
    """|M|^2_avg = 1/(4 * 64 * (ng-2)!) sum_h A_h^dagger C A_h, recomputed here from the exported amplitudes."""
    for pid, n in ((1, 2), (2, 3), (3, 4)):
        P = oracle_procs[pid]
        mom = _rambo_event(n, 1000.0, np.random.default_rng(11))
        v, amps = P.me2(mom, want_amps=True)
        C = mfo.colour_matrix(n)
        tot = sum((A.conj() @ C @ A).real for A in amps)
        assert v == pytest.approx(tot / (4 * 64 * math.factorial(n - 2)), rel=1e-13)
        assert amps.shape == (4 << n, math.factorial(n))


@pytest.mark.parametrize("pid,n", [(1, 2), (2, 3), (3, 4)])
def test_quark_spin_flip_symmetry(oracle_procs, pid, n):
    """Flipping BOTH quark spins leaves A^dagger C A unchanged once the gluon polarisations are summed (Kramers
    conjugation: B u* is the spin-flipped spinor, B gamma^mu* B^-1 = gamma^mu).  With real (linear) polarisations
    it holds polarisation by polarisation, which is what the cooperative CUDA kernel relies on when it evaluates
    one top spin state and doubles the sum; with circular polarisations all helicities flip together."""
    P = oracle_procs[pid]
    C = mfo.colour_matrix(n)
    rng = np.random.default_rng(23)
    for _ in range(3):
        mom = _rambo_event(n, 500.0 + 2500.0 * rng.random(), rng)
        for basis in (3, 1, 0, 2):            # bit 0: z-spin / helicity spinors, bit 1: linear / circular pols
            _, amps = P.me2(mom, basis=basis, want_amps=True)
            q = np.array([(A.conj() @ C @ A).real for A in amps])
            nh = len(q)
            flip_quarks = 3 << n                # helicity index: bits (t, tbar, g0, g1, ...), t highest
            scale = q.max()
            for h in range(nh):
                partner = h ^ flip_quarks if basis & 2 else (nh - 1) ^ h
                assert abs(q[h] - q[partner]) <= 1e-11 * scale
            # hence: sum over one top spin state, doubled, is the full sum
            assert 2 * q[: nh // 2].sum() == pytest.approx(q.sum(), rel=1e-12)


def test_colour_matrix_closed_forms():
    """O11 pins: diagonal N_c C_F^n; the distinct entries quoted in SURVEY.md; symmetry; rank (the n! orderings
    are linearly dependent only from n >= ... none for n <= 4 in this basis, but C must be positive semidefinite)."""
    want = {2: (3, [16, -2]), 3: (9, [64, -8, 1, 10]), 4: (54, [512, -64, -28, -10, -1, 8, 62, 71, 80])}
    for n, (den, nums) in want.items():
        C = mfo.colour_matrix(n)
        assert np.allclose(C, C.T, atol=1e-13)
        assert np.allclose(np.diag(C), 3 * (4.0 / 3) ** n, rtol=1e-13)
        got = sorted(set(np.round(C.ravel() * den, 9)))
        assert got == sorted(float(v) for v in nums)
        assert np.linalg.eigvalsh(C).min() > -1e-12
    # n = 1: Tr(T^a T^a) summed = N_c C_F = 4
    assert mfo.colour_matrix(1)[0, 0] == pytest.approx(4.0)
    # textbook: Tr(T^a T^b T^a T^b) = -2/3 (n = 2 off-diagonal), sum over sigma' of a row (n=2): 16/3 - 2/3
    assert mfo.colour_matrix(2)[0, 1] == pytest.approx(-2.0 / 3, rel=1e-13)


def test_operation_counts_reported(oracle_procs):
    """§8(d): the algorithmic flop count comes from the oracle run on an operation-counting scalar."""
    g = golden_points()
    k = np.array([g[4]["K"][i] for i in range(4)])
    mom = np.vstack([[500, 0, 0, 500.0], [500, 0, 0, -500.0], k])
    c = oracle_procs[3].count_ops_me2(mom)
    assert c["add"] > 1e6 and c["mul"] > 1e6 and c["trans"] == 0
