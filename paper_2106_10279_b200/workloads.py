"""Seeded, synthetic workload definitions shared by the CUDA path, the oracle, the tests and bench.py.

This module holds INPUTS only — process descriptors, the synthetic gluon PDF table and the initial VEGAS
grid — and none of the method's arithmetic.  It imports neither the CUDA binding nor the oracle.

The five configurations are BASELINE.json `configs[0..4]` (C0..C4).  They stand in for the
paper's workloads, pp -> t tbar (+jets) at sqrt(s) = 13 TeV with an LHAPDF set through PDFFlow and
pT > 30 GeV cuts, which cannot be run here (no LHAPDF grids, no MG5_aMC).
"""
from dataclasses import dataclass, replace
import math

import numpy as np

MF_EE_MUMU, MF_GG_TT, MF_GG_TTG, MF_GG_TTGG = 0, 1, 2, 3
MF_PP_TTG = 5              # gg -> ttbar g + the q qbar, q g and qbar g channels (36 diagrams with four flavours)
MF_GG_TTGGG = 6            # gg -> ttbar ggg: the paper's heaviest process
MF_PP_TTGG = 7             # gg -> ttbar gg + q qbar -> ttbar gg of four flavours: 123 + 4 x 36 = the 267 diagrams of PAPER.md L101, L140
MF_PP_TT = 4               # gg -> ttbar + the q qbar -> ttbar channels of four flavours
GEV2_TO_PB = 0.3894e9  # BASELINE.json configs[0]: use this literal everywhere
N_BINS = 50
N_DIMS = {MF_EE_MUMU: 2, MF_GG_TT: 4, MF_GG_TTG: 14, MF_GG_TTGG: 18, MF_PP_TT: 4, MF_PP_TTG: 14, MF_GG_TTGGG: 22, MF_PP_TTGG: 18}
N_FINAL = {MF_EE_MUMU: 2, MF_GG_TT: 2, MF_GG_TTG: 3, MF_GG_TTGG: 4, MF_PP_TT: 2, MF_PP_TTG: 3, MF_GG_TTGGG: 5, MF_PP_TTGG: 4}
N_FLAVOURS = 4             # quark flavours of the multi-flavour table: d, u, s, c (3 gg + 4 q qbar = the 7 diagrams of PAPER.md L101)
VEGAS_ALPHA = 1.5


@dataclass(frozen=True)
class Workload:
    name: str
    process: int
    sqrt_s: float
    alpha_em: float = 1.0 / 132.507
    alpha_s: float = 0.118
    m_top: float = 173.0
    mu2: float = 173.0 ** 2
    ptmin: float = 0.0
    etamax: float = 0.0
    drmin: float = 0.0
    gev2_to_pb: float = GEV2_TO_PB
    n_bins: int = N_BINS
    n_events: int = 0          # events per iteration
    n_iterations: int = 0      # total iterations
    n_adapt: int = 0           # iterations after which the grid is refined (the rest run on a frozen grid)
    unweight: bool = False     # frozen iterations run mf_unweight
    seed: int = 0

    @property
    def n_dims(self):
        return N_DIMS[self.process]

    @property
    def n_final(self):
        return N_FINAL[self.process]

    def scaled(self, n_events, n_iterations=None, n_adapt=None):
        """Same physics at a reduced size (parity tests run the oracle at sizes it finishes in seconds)."""
        it = self.n_iterations if n_iterations is None else n_iterations
        ad = min(self.n_adapt, it) if n_adapt is None else n_adapt
        return replace(self, n_events=n_events, n_iterations=it, n_adapt=ad)


C0 = Workload("C0 e+e- -> mu+mu-", MF_EE_MUMU, sqrt_s=100.0, n_events=1_000_000, n_iterations=5, n_adapt=5)
C1 = Workload("C1 gg -> ttbar", MF_GG_TT, sqrt_s=13000.0, n_events=2 ** 20, n_iterations=10, n_adapt=10)
C2 = Workload("C2 gg -> ttbar g", MF_GG_TTG, sqrt_s=13000.0, ptmin=30.0, etamax=2.5, n_events=2 ** 22,
              n_iterations=10, n_adapt=10)
C3 = Workload("C3 gg -> ttbar gg", MF_GG_TTGG, sqrt_s=13000.0, ptmin=30.0, etamax=2.5, drmin=0.4,
              n_events=2 ** 22, n_iterations=10, n_adapt=10)
C4 = Workload("C4 gg -> ttbar gg + unweighting", MF_GG_TTGG, sqrt_s=13000.0, ptmin=30.0, etamax=2.5, drmin=0.4,
              n_events=2 ** 26, n_iterations=10, n_adapt=5, unweight=True)
CONFIGS = [C0, C1, C2, C3, C4]
# beyond BASELINE.json: the flavour-summed pp -> ttbar of PAPER.md L101 ("pp -> ttbar (7 diagrams)":
# 3 gg + one q qbar diagram for each of 4 flavours), gluon and quark channels in ONE pass over the same points
C5 = Workload("C5 pp -> ttbar (gg + q qbar)", MF_PP_TT, sqrt_s=13000.0, n_events=2 ** 20, n_iterations=10, n_adapt=5,
              unweight=True)
C6 = Workload("C6 pp -> ttbar j (gg + q qbar, q g, qbar g)", MF_PP_TTG, sqrt_s=13000.0, ptmin=30.0, etamax=2.5,
              n_events=2 ** 22, n_iterations=10, n_adapt=10)
# gg -> ttbar ggg (1240 diagrams, 128 helicity states, 120 x 120 colour matrix; RAMBO n = 5, 22-dim VEGAS),
# cuts as for gg -> ttbar gg on all three gluons; the paper ran its heaviest process at <= 1M events
C7 = Workload("C7 gg -> ttbar ggg", MF_GG_TTGGG, sqrt_s=13000.0, ptmin=30.0, etamax=2.5, drmin=0.4, n_events=2 ** 18,
              n_iterations=10, n_adapt=10)
# pp -> ttbar gg (Table 1: the 267-diagram row): C3's sizes and cuts
C8 = Workload("C8 pp -> ttbar gg (gg + q qbar)", MF_PP_TTGG, sqrt_s=13000.0, ptmin=30.0, etamax=2.5, drmin=0.4,
              n_events=2 ** 22, n_iterations=10, n_adapt=10)
EXTRA_CONFIGS = {"C5": C5, "C6": C6, "C7": C7, "C8": C8}


def pdf_table(nx=100, nq=50):
    """Synthetic gluon table of BASELINE.json configs[1]:
    x g(x,Q) = 3 x^-0.1 (1-x)^5 (1 + 0.1 ln(Q^2/100 GeV^2)) on nx log-spaced x knots in [1e-9, 1] and
    nq log-spaced Q^2 knots in [2.72, 1e10] GeV^2.  Returns (lnx[nx], lnq2[nq], xf[nx, nq]) in fp64.
    The PDF the method uses is the INTERPOLANT of this table, not the formula."""
    i = np.arange(nx, dtype=np.float64)
    lnx = math.log(1e-9) * (1.0 - i / (nx - 1))
    lnx[-1] = 0.0
    j = np.arange(nq, dtype=np.float64)
    lnq2 = math.log(2.72) + j * (math.log(1e10) - math.log(2.72)) / (nq - 1)
    x = np.exp(lnx)
    x[-1] = 1.0
    q2 = np.exp(lnq2)
    xf = 3.0 * x[:, None] ** -0.1 * (1.0 - x[:, None]) ** 5 * (1.0 + 0.1 * np.log(q2[None, :] / 100.0))
    return np.ascontiguousarray(lnx), np.ascontiguousarray(lnq2), np.ascontiguousarray(xf)


def pdf_table_flavours(nx=100, nq=50):
    """Synthetic multi-flavour table for MF_PP_TT on the knots of pdf_table: xf[1 + 2 N_FLAVOURS][nx][nq] with
    table 0 the gluon of pdf_table, table 1 + 2 i the quark of flavour i (d, u, s, c) and table 2 + 2 i its
    antiquark.  With L = ln(Q^2 / 100 GeV^2):
        sea_i   = c_i x^-0.1 (1-x)^7 (1 + 0.15 L),     c = (0.20, 0.18, 0.10, 0.03)
        valence = 1.1 x^0.6 (1-x)^4 (1 + 0.05 L) for d,  2.2 x^0.6 (1-x)^3 (1 + 0.05 L) for u,  0 otherwise
        x qbar_i = sea_i,   x q_i = valence_i + sea_i
    (shapes of the kind a proton set has: valence peaks, a steep sea; the numbers are this repository's own)."""
    lnx, lnq2, xg = pdf_table(nx, nq)
    x = np.exp(lnx)[:, None]
    x[-1] = 1.0
    L = np.log(np.exp(lnq2)[None, :] / 100.0)
    c = (0.20, 0.18, 0.10, 0.03)
    val = (1.1 * x ** 0.6 * (1.0 - x) ** 4 * (1.0 + 0.05 * L), 2.2 * x ** 0.6 * (1.0 - x) ** 3 * (1.0 + 0.05 * L))
    xf = np.zeros((1 + 2 * N_FLAVOURS, nx, nq))
    xf[0] = xg
    for i in range(N_FLAVOURS):
        sea = c[i] * x ** -0.1 * (1.0 - x) ** 7 * (1.0 + 0.15 * L)
        xf[2 + 2 * i] = sea
        xf[1 + 2 * i] = sea + (val[i] if i < 2 else 0.0)
    return lnx, lnq2, np.ascontiguousarray(xf)


def pdf_for(process, nx=100, nq=50):
    """the table a process needs: None, the gluon table, or the multi-flavour table"""
    if process == MF_EE_MUMU:
        return None
    return pdf_table_flavours(nx, nq) if process in (MF_PP_TT, MF_PP_TTG, MF_PP_TTGG) else pdf_table(nx, nq)


def uniform_grid(n_dims, n_bins=N_BINS):
    """Initial VEGAS grid: edges e_{d,i} = i / n_bins, shape [n_dims, n_bins + 1]."""
    e = np.arange(n_bins + 1, dtype=np.float64) / n_bins
    e[-1] = 1.0
    return np.ascontiguousarray(np.tile(e, (n_dims, 1)))


def rambo_test_point(n):
    """The fixed uniforms of SURVEY.md §8(c) 'golden points': for final particle i,
    (rho1..rho4) = (0.15+0.2i, 0.35+0.15i, 0.55-0.1i, 0.25+0.1i)."""
    rho = []
    for i in range(n):
        rho += [0.15 + 0.2 * i, 0.35 + 0.15 * i, 0.55 - 0.1 * i, 0.25 + 0.1 * i]
    return np.array(rho, dtype=np.float64)
