#!/usr/bin/env python3
"""Build-time generator of the index tables of the g g -> t tbar g g g matrix element (one event per thread block,
mf_me_cta5.cuh; the paper's heaviest process).

The colour-ordered recursion (R10) for five gluons, organised for a whole CTA per event:

  * real polarisations, hatted currents, top spin 0 only (spin-flip symmetry), helicity recycling: a current is
    computed once per polarisation assignment of the gluons it contains;
  * gluon currents J(seq) for the CANONICAL sequences (seq[0] < seq[-1]; J(reversed) = (-1)^(k+1) J) of length 2..5:
    10 x 4 + 30 x 8 + 60 x 16 + 60 x 32 = 3160 real 4-vectors, one work item each, level by level;
  * quark currents only up to two gluons on either side of the line (Y1, Y2 from ubar; X1, X2 from v): the amplitude of an
    ordering sigma is summed over the gluon-current block M that contains the MIDDLE gluon of the ordering,
        Ahat(sigma) = sum_{i <= 3 <= j} Y(sigma_1 .. sigma_{i-1}) Jslash(sigma_i .. sigma_j) X(sigma_{j+1} .. sigma_5),
    nine terms, so no quark current of more than two gluons is ever needed;
  * the 120 x 120 colour contraction of the 64 x 2 (helicity, real / imaginary part) amplitude vectors is a dense
    real matrix product and runs on the FP64 tensor path (DMMA) in two halves of 64 columns.

This file emits the tables only (operand indices of every work item, the bit-compress tables, the colour matrix); the
arithmetic is hand written in mf_me_cta5.cuh.  Imports nothing from oracle/.
"""
import itertools
import math
import os

import numpy as np

from gen_me import gell_mann_half, FLOPS

HERE = os.path.dirname(os.path.abspath(__file__))
N = 5
LABELS = list(range(N))

# ---- scratch layout (item indices; a VEC item is 4 doubles, a SPIN item 8 doubles) ------------------------------------
SEQS = {k: [s for s in itertools.permutations(LABELS, k) if s[0] < s[-1]] for k in range(2, N + 1)}
SEQ_INDEX = {k: {s: i for i, s in enumerate(SEQS[k])} for k in SEQS}
ORDERED_PAIRS = list(itertools.permutations(LABELS, 2))
PAIR_INDEX = {p: i for i, p in enumerate(ORDERED_PAIRS)}
V_P, V_QX, V_QY, V_EPS = 0, 32, 64, 96
V_J = {2: V_EPS + 2 * N}
for k in range(3, N + 1):
    V_J[k] = V_J[k - 1] + len(SEQS[k - 1]) * (1 << (k - 1))
N_VEC = V_J[N] + len(SEQS[N]) * (1 << N)
S_UB, S_V, S_Y1 = 0, 1, 3
S_X1 = S_Y1 + 2 * N
S_Y2 = S_X1 + 4 * N
S_X2 = S_Y2 + 4 * len(ORDERED_PAIRS)
N_SPIN = S_X2 + 8 * len(ORDERED_PAIRS)
XM_STRIDE = 68            # row stride of the amplitude matrix [ordering][64 columns]: conflict-free DMMA fragment loads


def mask_of(seq):
    m = 0
    for g in seq:
        m |= 1 << g
    return m


def canon(seq):
    seq = tuple(seq)
    if len(seq) > 1 and seq[0] > seq[-1]:
        return seq[::-1], (-1) ** (len(seq) + 1)
    return seq, 1


def ref(seq):
    """(base VEC index, mask, sign) of Jhat(seq): the item is base + pext(pols, mask)"""
    seq = tuple(seq)
    if len(seq) == 1:
        return V_EPS + 2 * seq[0], 1 << seq[0], 1
    c, s = canon(seq)
    return V_J[len(c)] + SEQ_INDEX[len(c)][c] * (1 << len(c)), mask_of(c), s


def pext(pw, mask):
    v, i = 0, 0
    for g in range(N):
        if mask >> g & 1:
            v |= (pw >> g & 1) << i
            i += 1
    return v


def pdep(v, mask):
    pw, i = 0, 0
    for g in range(N):
        if mask >> g & 1:
            pw |= (v >> i & 1) << g
            i += 1
    return pw


# ---- tables ---------------------------------------------------------------------------------------------------------
def gluon_tables():
    """per level k = 2..5 and canonical sequence: [mask, out base, offset into the split table, n3 | n4 << 8]; the split
    table holds, per sequence, its V3 splits [bL, mL, bR, mR, sign] and then its V4 splits [bA, mA, bB, mB, bC, mC, sign]
    (sign includes the reflection signs of the operands and the vertex sign: Jhat = (-sum V3 + sum V4) / P^2)"""
    desc, split, flops = {}, [], 0
    for k in range(2, N + 1):
        rows = []
        for s in SEQS[k]:
            off = len(split)
            n3 = n4 = 0
            for j in range(1, k):
                (bl, ml, sl), (br, mr, sr) = ref(s[:j]), ref(s[j:])
                split += [bl, ml, br, mr, -sl * sr]
                n3 += 1
            for j in range(1, k):
                for l in range(j + 1, k):
                    (ba, ma, sa), (bb, mb, sb), (bc, mc, sc) = ref(s[:j]), ref(s[j:l]), ref(s[l:])
                    split += [ba, ma, bb, mb, bc, mc, sa * sb * sc]
                    n4 += 1
            rows.append([mask_of(s), ref(s)[0], off, n3 | (n4 << 8)])
            flops += (1 << k) * (n3 * FLOPS["v3_acc"] + n4 * FLOPS["v4_acc"] + 4)
        desc[k] = rows
    return desc, split, flops


def amp_table():
    """per ordering sigma (lexicographic): the nine blocks sigma[i..j], i <= 3 <= j (entry (j - 3) * 3 + (i - 1):
    base, mask, sign), then sigma itself"""
    rows = []
    for sg in itertools.permutations(LABELS):
        r = []
        for j in (3, 4, 5):
            for i in (1, 2, 3):
                r += list(ref(sg[i - 1:j]))
        r += list(sg)
        rows.append(r)
    return rows


def colour_matrix5():
    """C[s][t] = sum over colours of Tr(T^{a_s0} .. T^{a_s4} (T^{a_t0} .. T^{a_t4})^dagger) as integer numerators over 324:
    the products M(a) = T^{a_0} .. T^{a_4} for all 8^5 colour assignments once; M_s(a) = M(a o s) is a gather."""
    T = gell_mann_half()
    M = T
    for _ in range(N - 1):
        M = np.einsum('...ij,ajk->...aik', M, T)          # index order: a_0 slowest ... a_4 fastest
    M = M.reshape([8] * N + [9])
    perms = list(itertools.permutations(LABELS))
    # M_s(a)[a_0..a_4] = M[a_{s0}, .., a_{s4}]: axis i of the result is a_i, so take M's axis order inverse(s)... written out:
    def permuted(s):
        # result[a_0, .., a_4] = M[a_{s[0]}, .., a_{s[4]}]  <=>  result = M.transpose(axes) with axes[s[i]] = i
        axes = [0] * N
        for i in range(N):
            axes[s[i]] = i
        return M.transpose(axes + [N]).reshape(-1)
    V = np.stack([permuted(s) for s in perms])             # 120 x (8^5 * 9)
    C = (V @ V.conj().T).real
    den = 324
    num = np.rint(C * den).astype(np.int64)
    assert np.abs(C * den - num).max() < 1e-7, "colour matrix is not a multiple of 1/%d" % den
    assert (num == num.T).all() and num[0][0] == 4096
    return perms, num, den


def fmt_rows(vals, per_line=32):
    return ["  " + ", ".join("%d" % v for v in vals[i:i + per_line]) + "," for i in range(0, len(vals), per_line)]


def main():
    desc, split, gl_flops = gluon_tables()
    amp = amp_table()
    perms, cnum, cden = colour_matrix5()
    assert perms == list(itertools.permutations(LABELS))
    assert max(split) < 32768 and N_VEC < 32768
    o = []
    w = o.append
    w("// GENERATED by gen_cta5.py — do not edit.  Index tables of the g g -> t tbar g g g matrix element (one event per")
    w("// thread block; arithmetic in mf_me_cta5.cuh).  A FRAGMENT: included inside namespace mf::g5.")
    w("")
    w("// scratch items: VEC (4 doubles): P[mask] | q of the right / left quark currents [mask] | eps[g][p] | J2 | J3 | J4 | J5")
    w("constexpr int kVP = %d, kVQX = %d, kVQY = %d, kVEps = %d, kVJ2 = %d, kVJ3 = %d, kVJ4 = %d, kVJ5 = %d, kNVec = %d;" %
      (V_P, V_QX, V_QY, V_EPS, V_J[2], V_J[3], V_J[4], V_J[5], N_VEC))
    w("// SPIN (8 doubles): ubar | v[hb] | Y1[a][pa] | X1[d][hb][pd] | Y2[pair][pa | pb << 1] | X2[pair][hb][pc | pd << 1]")
    w("constexpr int kSUb = %d, kSV = %d, kSY1 = %d, kSX1 = %d, kSY2 = %d, kSX2 = %d, kNSpin = %d;" %
      (S_UB, S_V, S_Y1, S_X1, S_Y2, S_X2, N_SPIN))
    w("constexpr int kNSeq2 = %d, kNSeq3 = %d, kNSeq4 = %d, kNSeq5 = %d, kNPerm = %d, kXmStride = %d;" %
      (len(SEQS[2]), len(SEQS[3]), len(SEQS[4]), len(SEQS[5]), len(perms), XM_STRIDE))
    w("constexpr double kCden = %d.0;         // kColour holds 2 x numerator above the diagonal, 1 x on it: x^T C x = x^T kColour x / kCden" % cden)
    # static operation count (adds + multiplies, FMA = 2) of one matrix element
    q_flops = (2 * N * (FLOPS["slash_row"] + FLOPS["prop_row"]) + 4 * N * (FLOPS["slash_col"] + FLOPS["prop_col"]) +
               80 * (FLOPS["slash_row"] + 50 + FLOPS["prop_row"] + 4) + 160 * (FLOPS["slash_col"] + 50 + FLOPS["prop_col"] + 4))
    amp_flops = len(perms) * 32 * (9 * (48 + 4) + 6 * 32)
    col_flops = 2 * (2 * 8 * 8 * 4 * 8 * 240 + 2 * 120 * 64)        # 240 (row tile, k-step) pairs x 8 column tiles per half
    s0_flops = 31 * 40 + 200
    total = s0_flops + gl_flops + q_flops + amp_flops + col_flops
    w("// static fp64 operation count per matrix element: S0 %d + gluon currents %d + quark currents %d + amplitudes %d +" %
      (s0_flops, gl_flops, q_flops, amp_flops))
    w("// colour contraction (DMMA on the upper triangle: 2 halves x 240 x 8 instructions of 512 flop) %d" % col_flops)
    w("constexpr double kFlopsMe2Cta_3g = %d.0;" % total)
    w("")
    w("// canonical gluon sequences of length k = 2..5 (row k - 2): mask, output base, offset into kSplit, n3 | n4 << 8")
    w("MF_CTABLE short kSeqDesc[4][%d][4] = {" % len(SEQS[5]))
    for k in range(2, N + 1):
        rows = desc[k] + [[0, 0, 0, 0]] * (len(SEQS[5]) - len(desc[k]))
        w("  {" + ", ".join("{%d, %d, %d, %d}" % tuple(r) for r in rows) + "},")
    w("};")
    w("// V3 splits [bL, mL, bR, mR, sign] then V4 splits [bA, mA, bB, mB, bC, mC, sign] of every sequence")
    w("MF_CTABLE short kSplit[%d] = {" % len(split))
    o.extend(fmt_rows(split))
    w("};")
    w("// per ordering: nine blocks (base, mask, sign), entry (j - 3) * 3 + (i - 1) = sigma[i..j]; then sigma")
    w("MF_CTABLE short kAmp[%d][32] = {" % len(amp))
    for r in amp:
        w("  {" + ", ".join("%d" % v for v in r) + "},")
    w("};")
    w("// kPext[mask][pw]: the bits of pw at the positions of mask, compressed; kPdep: the inverse")
    w("MF_TABLE unsigned char kPext[32][32] = {")
    for m in range(32):
        w("  {" + ", ".join("%d" % pext(pw, m) for pw in range(32)) + "},")
    w("};")
    w("MF_TABLE unsigned char kPdep[32][32] = {")
    for m in range(32):
        w("  {" + ", ".join("%d" % pdep(v, m) for v in range(32)) + "},")
    w("};")
    w("// index of the canonical pair (min, max) among the J2 sequences")
    w("MF_TABLE unsigned char kJ2Idx[5][5] = {")
    for a in LABELS:
        w("  {" + ", ".join("%d" % (SEQ_INDEX[2][(min(a, b), max(a, b))] if a != b else 0) for b in LABELS) + "},")
    w("};")
    w("// colour matrix (orderings in lexicographic order), UPPER triangle, numerators over kCden:")
    w("// (off-diagonal entries doubled, so x^T C x = x^T kColour x), and row tile m of the DMMA contraction only needs the columns >= 8 m")
    cup = np.triu(2 * cnum, 1) + np.diag(np.diag(cnum))          # doubled: the halved diagonal stays an integer
    assert (cup + cup.T == 2 * cnum).all()
    w("MF_TABLE double kColour[%d] = {" % (len(perms) ** 2))
    flat = [int(v) for v in cup.reshape(-1)]
    for i in range(0, len(flat), 30):
        w("  " + ", ".join("%d." % v for v in flat[i:i + 30]) + ",")
    w("};")
    text = "\n".join(o) + "\n"
    path = os.path.join(HERE, "mf_me_ttggg_tables_generated.cuh")
    old = open(path).read() if os.path.exists(path) else None
    if old != text:
        with open(path, "w") as f:
            f.write(text)
    return path


if __name__ == "__main__":
    print(main())
