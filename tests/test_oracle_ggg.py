"""Pins for the oracle's g g -> t tbar g g g (process 6; the paper's heaviest
process, 1240 gg diagrams).  CPU only.  The amplitude code is the n-gluon recursion already pinned for n = 2, 3, 4; what
is new at n = 5 is pinned here: gauge invariance for each of the five gluons, Bose symmetry among the three final
gluons, the colour-dressed Feynman-rule recursion on random colours, Lorentz and basis invariance, the spin-flip
symmetry the kernel relies on, the collinear limit onto the (pinned) g g -> t tbar g g matrix element, and the
120 x 120 colour matrix against its definition."""
import itertools
import math

import numpy as np
import pytest

from oracle import mfo
from paper_2106_10279_b200 import workloads as W
from test_oracle_amplitudes import _lorentz, _rambo_event
from test_oracle_phasespace_pdf import mink

N = 5
PID = W.MF_GG_TTGGG


def test_diagram_count_of_the_recursion():
    """counting every term of the colour-dressed recursion once gives 3 / 16 / 123 / 1240 Feynman diagrams
    for g g -> t tbar + 0, 1, 2, 3 gluons (PAPER.md L101 quotes pp totals 3 + 4, 16 + 20, 123 + 144, ...)."""
    from math import comb
    g = {1: 1}
    for n in range(2, 6):        # gluon current of n external gluons: unordered 2- and 3-partitions
        tot = 0
        for a in range(1, n // 2 + 1):
            ways = comb(n, a) // (2 if 2 * a == n else 1)
            tot += ways * g[a] * g[n - a]
        for a in range(1, n):
            for b in range(a, n):
                c = n - a - b
                if c < b:
                    continue
                ways = comb(n, a) * comb(n - a, b)
                if a == b == c:
                    ways //= 6
                elif a == b or b == c:
                    ways //= 2
                tot += ways * g[a] * g[b] * g[c]
        g[n] = tot
    assert [g[n] for n in range(1, 6)] == [1, 1, 4, 25, 220]
    q = {0: 1}
    for n in range(1, 6):        # quark line with n gluons attached through gluon currents
        q[n] = sum(comb(n, k) * g[k] * q[n - k] for k in range(1, n + 1))
    assert [q[n] for n in range(2, 6)] == [3, 16, 123, 1240]


def test_colour_matrix_five_gluons():
    C = mfo.colour_matrix(N)
    assert C.shape == (120, 120)
    assert np.allclose(C, C.T, atol=1e-12)
    assert np.allclose(np.diag(C), 3 * (4.0 / 3) ** 5, rtol=1e-13)             # N_c C_F^5 = 1024 / 81
    assert np.linalg.eigvalsh(C).min() > -1e-10
    # every row is a permutation of the first one (relabelling invariance), and the entries are multiples of 1/324
    r0 = np.sort(C[0])
    for i in (1, 7, 55, 119):
        assert np.allclose(np.sort(C[i]), r0, atol=1e-12)
    assert np.allclose(C * 324, np.round(C * 324), atol=1e-8)
    # sampled entries straight from the definition (sum over all 8^5 colour assignments)
    perms = list(itertools.permutations(range(N)))
    rng = np.random.default_rng(55)
    for _ in range(24):
        i, j = rng.integers(0, 120, 2)
        assert C[i, j] == pytest.approx(mfo.colour_matrix_entry(N, perms[i], perms[j]), abs=1e-11)


@pytest.mark.parametrize("n", [2, 3, 4])
def test_colour_entry_by_table_equals_the_plain_loop(n):
    """the table lookup M_sigma(a) = M(a o sigma) used for n = 5, against the plain n <= 4 loop, every entry"""
    C = mfo.colour_matrix(n)
    perms = list(itertools.permutations(range(n)))
    for i, s in enumerate(perms):
        for j, t in enumerate(perms):
            assert C[i, j] == pytest.approx(mfo.colour_matrix_entry(n, s, t), abs=1e-13)


def test_gauge_invariance_for_each_of_the_five_gluons(oracle_procs):
    P = oracle_procs[PID]
    mom = _rambo_event(N, 1100.0, np.random.default_rng(61))
    v, amps = P.me2(mom, want_amps=True)
    assert amps.shape == (128, 120)
    scale = np.abs(amps).max()
    for gl in range(N):
        v0, a0 = P.me2(mom, subst_gluon=gl, want_amps=True)
        assert np.abs(a0).max() < 1e-10 * scale * 1100.0
        assert v0 < 1e-19 * v * 1100.0 ** 2


def test_basis_lorentz_and_exchange_symmetries(oracle_procs):
    P = oracle_procs[PID]
    rng = np.random.default_rng(62)
    mom = _rambo_event(N, 1300.0, rng)
    v = P.me2(mom)
    for basis in (1, 2, 3):
        assert P.me2(mom, basis=basis) == pytest.approx(v, rel=1e-11)
    L = _lorentz(rng)
    mom2 = mom @ L.T
    assert mink(mom2[3], mom2[3]) == pytest.approx(173.0 ** 2, rel=1e-10)
    assert P.me2(mom2) == pytest.approx(v, rel=1e-9)
    for perm in itertools.permutations((4, 5, 6)):          # Bose symmetry among the three final gluons
        assert P.me2(mom[[0, 1, 2, 3] + list(perm)]) == pytest.approx(v, rel=1e-11)
    assert P.me2(mom[[1, 0, 2, 3, 4, 5, 6]]) == pytest.approx(v, rel=1e-11)     # beams exchanged
    assert P.me2(mom[[0, 1, 3, 2, 4, 5, 6]]) == pytest.approx(v, rel=1e-11)     # t <-> tbar


def test_dressed_recursion_equals_ordered_sum(oracle_procs):
    P = oracle_procs[PID]
    rng = np.random.default_rng(63)
    mom = _rambo_event(N, 1000.0, rng)
    _, amps = P.me2(mom, want_amps=True)
    scale = np.abs(amps).max()
    nz = 0
    for _ in range(120):         # most random colour assignments of five gluons vanish by colour conservation
        hel = rng.choice([-1, 1], size=2 + N)
        col = rng.integers(0, 8, size=N)
        i, j = rng.integers(0, 3, size=2)
        a = P.dressed_amplitude(mom, hel, col, i, j)
        b = P.ordered_amplitude_coloured(mom, hel, col, i, j)
        assert abs(a - b) <= 1e-11 * scale
        nz += abs(a) > 1e-6 * scale
    assert nz >= 3


def test_average_and_spin_flip_symmetry(oracle_procs):
    P = oracle_procs[PID]
    C = mfo.colour_matrix(N)
    mom = _rambo_event(N, 900.0, np.random.default_rng(64))
    v, amps = P.me2(mom, basis=3, want_amps=True)          # z-axis spins, linear polarisations: the kernel's choice
    q = np.array([(A.conj() @ C @ A).real for A in amps])
    assert v == pytest.approx(q.sum() / (4 * 64 * 6), rel=1e-12)          # 4 helicities x 64 colours x 3! identical gluons
    flip = 3 << N
    for h in range(len(q)):
        assert abs(q[h] - q[h ^ flip]) <= 1e-10 * q.max()
    assert 2 * q[:64].sum() == pytest.approx(q.sum(), rel=1e-11)
    assert P.me2(mom) == pytest.approx(v, rel=1e-11)


def test_collinear_limit_onto_gg_ttgg(oracle_procs):
    """Two final gluons collinear (invariant mass m45 -> 0): averaged over the azimuth of the splitting,
        |M_5|^2 -> (2 g_s^2 / m45^2) P_gg(z) |M_4|^2,   P_gg(z) = 2 C_A [ z/(1-z) + (1-z)/z + z(1-z) ],
    colour and spin summed for labelled gluons; with the 1/(n_g - 2)! of the averaged matrix elements the ratio carries
    2!/3!.  |M_4|^2 is the separately pinned g g -> t tbar g g matrix element (golden points, gauge invariance)."""
    P5, P4 = oracle_procs[PID], oracle_procs[W.MF_GG_TTGG]
    rng = np.random.default_rng(65)
    w, mt, m45 = 1000.0, 173.0, 0.25
    rho = rng.random(16)
    k4, _ = mfo.rambo([mt, mt, 0.0, 0.0], w, rho)                 # the massless parent: t, tbar, g, G
    kc, _ = mfo.rambo([mt, mt, 0.0, m45], w, rho)                 # the same point with G -> a cluster of mass m45
    beams = [[w / 2, 0, 0, w / 2], [w / 2, 0, 0, -w / 2]]
    me4 = P4.me2(np.vstack([beams, k4]))
    G = kc[3]
    b = G[1:] / G[0]                                              # boost from the cluster rest frame
    gam = G[0] / m45
    g2 = 4 * math.pi * 0.118
    for cth in (0.3, -0.55):
        sth = math.sqrt(1 - cth * cth)
        vals, zs = [], []
        for iphi in range(8):
            phi = 2 * math.pi * (iphi + 0.3) / 8
            nb = b / np.linalg.norm(b)                         # polar angle measured from the cluster's direction
            e1 = np.cross(nb, [0.0, 0.0, 1.0])
            e1 /= np.linalg.norm(e1)
            e2 = np.cross(nb, e1)
            d = sth * (math.cos(phi) * e1 + math.sin(phi) * e2) + cth * nb
            out = []
            for sgn in (1, -1):
                q = np.array([m45 / 2, *(sgn * m45 / 2 * d)])
                bq = b @ q[1:]
                E = gam * (q[0] + bq)
                p3 = q[1:] + b * (gam * gam / (gam + 1) * bq + gam * q[0])
                out.append(np.array([E, *p3]))
            mom = np.vstack([beams, kc[:3], out])
            assert np.allclose(mom[0] + mom[1], mom[2:].sum(axis=0), atol=1e-9 * w)
            vals.append(P5.me2(mom))
            zs.append(out[0][0] / G[0])
        z = float(np.mean(zs))
        assert max(zs) - min(zs) < 1e-3                             # the energy fraction does not depend on the azimuth (boost along G)
        pgg = 2 * 3.0 * (z / (1 - z) + (1 - z) / z + z * (1 - z))
        want = 2 * g2 / m45 ** 2 * pgg * me4 / 3.0
        assert np.mean(vals) == pytest.approx(want, rel=0.02)
        assert np.std(vals) / np.mean(vals) > 1e-3                  # the azimuthal (spin) correlation is there and averages out
