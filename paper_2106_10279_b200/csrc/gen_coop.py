#!/usr/bin/env python3
"""Build-time generator of the COOPERATIVE matrix element of g g -> t tbar g g (64 threads per event).

The straight-line code of gen_me.py keeps one event per thread; for 4 gluons its working set (30 gluon
currents, 32 quark currents, 21 bilinears per polarisation combination) spills ~80 kB per thread.  This
generator re-organises the same colour-ordered recursion (R10) as a STAGED program over a
shared-memory scratch, executed by 64 threads per event:

  * helicity recycling: a current is computed once per polarisation assignment of the gluons IT contains
    (J2: 4 variants, J3: 8, J4: 16; X(cd): 2 spins x 4; ...), not once per full helicity combination;
  * stages S1..S3 are table driven: one task = one current; the tables (operand indices into the scratch)
    are emitted here, so the kernel's interpreter has no index arithmetic;
  * stage S4 is generated straight-line code: thread (pols, h, hb) forms its 24 colour-ordered amplitudes from
    the staged currents and contracts them with the colour matrix.

Emits mf_me_ttgg_coop_generated.cuh.  Imports nothing from oracle/.
"""
import itertools
import os

import numpy as np

from gen_me import colour_matrix

HERE = os.path.dirname(os.path.abspath(__file__))
N = 4           # gluons: 0, 1 beams; 2, 3 final
P_CUT = N // 2  # the quark line is cut after P_CUT gluons
LABELS = list(range(N))


def mask_of(seq):
    m = 0
    for g in seq:
        m |= 1 << g
    return m


def canon(seq):
    """canonical orientation of a gluon sequence and the reflection sign J(rev) = (-1)^(k+1) J"""
    seq = tuple(seq)
    if len(seq) > 1 and seq[0] > seq[-1]:
        return seq[::-1], (-1) ** (len(seq) + 1)
    return seq, 1


def polidx(gluons, pols):
    """compressed polarisation index: bit i = pol of the i-th smallest label in `gluons`"""
    v = 0
    for i, g in enumerate(sorted(gluons)):
        v |= ((pols >> g) & 1) << i
    return v


def pol_variants(gluons):
    """all full 4-bit pol words restricted to `gluons` (other bits zero), in polidx order"""
    gl = sorted(gluons)
    out = []
    for v in range(1 << len(gl)):
        p = 0
        for i, g in enumerate(gl):
            p |= ((v >> i) & 1) << g
        out.append(p)
    return out


class Layout:
    """component-major arrays: VEC[4][NV], SPIN[8][NS], CVEC[8][NC], SCAL[NSC]"""

    def __init__(self):
        self.idx = {"V": {}, "S": {}, "C": {}, "X": {}}
        self.bases = {}

    def add(self, arr, key):
        d = self.idx[arr]
        assert key not in d, key
        d[key] = len(d)
        return d[key]

    def get(self, arr, key):
        return self.idx[arr][key]

    def n(self, arr):
        return len(self.idx[arr])


def build_layout():
    L = Layout()
    for m in range(1, 1 << N):
        L.add("V", ("P", m))
    for m in range(1, 1 << N):
        if bin(m).count("1") <= N - P_CUT:
            L.add("V", ("qX", m))
    for m in range(1, 1 << N):
        if bin(m).count("1") <= P_CUT - 1:
            L.add("V", ("qY", m))
    for g in LABELS:
        for p in range(2):
            L.add("V", ("eps", g, p))
    # gluon currents, canonical sequences, family-contiguous so S4 can index them arithmetically
    seqs = {k: [s for s in itertools.permutations(LABELS, k) if canon(s)[0] == s] for k in range(2, N + 1)}
    for k in range(2, N + 1):
        L.bases["J%d" % k] = L.n("V")
        for s in seqs[k]:
            for pv in pol_variants(s):
                L.add("V", ("J", s, pv))
    for m in range(1, 1 << N):
        if bin(m).count("1") >= 2:
            L.add("X", ("iP2", m))
        if bin(m).count("1") <= N - P_CUT:
            L.add("X", ("idX", m))
        if bin(m).count("1") <= P_CUT - 1:
            L.add("X", ("idY", m))
    for h in range(2):
        L.add("S", ("ub", h))
    for hb in range(2):
        L.add("S", ("v", hb))
    L.bases["X1"] = L.n("S")
    for hb in range(2):
        for d in LABELS:
            for pv in pol_variants((d,)):
                L.add("S", ("X", (d,), hb, pv))
    L.bases["Y1"] = L.n("S")
    for h in range(2):
        for a in LABELS:
            for pv in pol_variants((a,)):
                L.add("S", ("Y", (a,), h, pv))
    ordered_pairs = list(itertools.permutations(LABELS, 2))
    L.bases["X2"] = L.n("S")
    for hb in range(2):
        for cd in ordered_pairs:
            for pv in pol_variants(cd):
                L.add("S", ("X", cd, hb, pv))
    L.bases["Yt"] = L.n("S")
    for h in range(2):
        for ab in ordered_pairs:
            for pv in pol_variants(ab):
                L.add("S", ("Yt", ab, h, pv))
    L.bases["c0"] = L.n("C")
    for h in range(2):
        for hb in range(2):
            L.add("C", ("c", (), (), h, hb, 0))
    L.bases["cR"] = L.n("C")
    for h in range(2):
        for hb in range(2):
            for d in LABELS:
                for pv in pol_variants((d,)):
                    L.add("C", ("c", (), (d,), h, hb, pv))
    L.bases["cL"] = L.n("C")
    for h in range(2):
        for hb in range(2):
            for a in LABELS:
                for pv in pol_variants((a,)):
                    L.add("C", ("c", (a,), (), h, hb, pv))
    L.bases["cLR"] = L.n("C")
    for h in range(2):
        for hb in range(2):
            for ad in ordered_pairs:
                for pv in pol_variants(ad):
                    L.add("C", ("c", (ad[0],), (ad[1],), h, hb, pv))
    L.seqs = seqs
    L.ordered_pairs = ordered_pairs
    return L


# ---- operand lookup ----------------------------------------------------------------------------------------
def J_ref(L, seq, pols):
    """(VEC index, sign) of Jhat(seq) for the polarisation word `pols`"""
    seq = tuple(seq)
    if len(seq) == 1:
        return L.get("V", ("eps", seq[0], (pols >> seq[0]) & 1)), 1
    c, s = canon(seq)
    pv = pols & mask_of(seq)
    return L.get("V", ("J", c, pv)), s


def P_ref(L, seq):
    return L.get("V", ("P", mask_of(seq)))


# ---- tasks ---------------------------------------------------------------------------------------------------
# op codes of the interpreter (mf_me_coop.cuh)
OP_J, OP_XCOL, OP_YROW, OP_BIL = 0, 1, 2, 3


def task_J(L, seq, pols):
    k = len(seq)
    v3, v4 = [], []
    for j in range(1, k):
        a, sa = J_ref(L, seq[:j], pols)
        b, sb = J_ref(L, seq[j:], pols)
        v3.append((a, P_ref(L, seq[:j]), b, P_ref(L, seq[j:]), -sa * sb))
    for j in range(1, k):
        for l in range(j + 1, k):
            a, sa = J_ref(L, seq[:j], pols)
            b, sb = J_ref(L, seq[j:l], pols)
            c, sc = J_ref(L, seq[l:], pols)
            v4.append((a, b, c, sa * sb * sc))
    out = L.get("V", ("J", tuple(seq), pols & mask_of(seq)))
    fields = [out, L.get("X", ("iP2", mask_of(seq)))]
    signs = 0
    for i, t in enumerate(v3):
        fields += list(t[:4])
        signs |= (1 if t[4] < 0 else 0) << i
    for i, t in enumerate(v4):
        fields += list(t[:3])
        signs |= (1 if t[3] < 0 else 0) << (len(v3) + i)
    fields.append(signs)
    flops = 53 * len(v3) + 49 * len(v4) + 4
    return dict(op=OP_J, a=len(v3), b=len(v4), fields=fields, flops=flops)


def task_X(L, seq, hb, pols):
    """Xhat(seq) = -(qslash+m)/(q^2-m^2) sum_j Jslash(seq[:j]) Xhat(seq[j:]),  Xhat() = v"""
    k = len(seq)
    terms = []
    for j in range(1, k + 1):
        jv, js = J_ref(L, seq[:j], pols)
        rest = tuple(seq[j:])
        sp = L.get("S", ("v", hb)) if not rest else L.get("S", ("X", rest, hb, pols & mask_of(rest)))
        terms.append((jv, sp, js))
    m = mask_of(seq)
    fields = [L.get("S", ("X", tuple(seq), hb, pols & m)), L.get("V", ("qX", m)), L.get("X", ("idX", m))]
    signs = 0
    for i, t in enumerate(terms):
        fields += [t[0], t[1]]
        signs |= (1 if t[2] < 0 else 0) << i
    fields.append(signs)
    return dict(op=OP_XCOL, a=len(terms), b=1, fields=fields, flops=42 * len(terms) + 8 * (len(terms) - 1) + 66)


def task_Y(L, seq, h, pols, propagate):
    """Ytilde(seq) = sum_j Yhat(seq[:j]) Jslash(seq[j:]);  Yhat = Ytilde (-(qslash+m)/(q^2-m^2)),  Yhat() = ubar"""
    k = len(seq)
    terms = []
    for j in range(0, k):
        left = tuple(seq[:j])
        sp = L.get("S", ("ub", h)) if not left else L.get("S", ("Y", left, h, pols & mask_of(left)))
        jv, js = J_ref(L, seq[j:], pols)
        terms.append((sp, jv, js))
    m = mask_of(seq)
    if propagate:
        fields = [L.get("S", ("Y", tuple(seq), h, pols & m)), L.get("V", ("qY", m)), L.get("X", ("idY", m))]
    else:
        fields = [L.get("S", ("Yt", tuple(seq), h, pols & m)), 0, 0]
    signs = 0
    for i, t in enumerate(terms):
        fields += [t[0], t[1]]
        signs |= (1 if t[2] < 0 else 0) << i
    fields.append(signs)
    return dict(op=OP_YROW, a=len(terms), b=1 if propagate else 0, fields=fields,
                flops=42 * len(terms) + 8 * (len(terms) - 1) + (66 if propagate else 0))


def task_bil(L, left, right, h, hb, pols):
    row = L.get("S", ("ub", h)) if not left else L.get("S", ("Y", tuple(left), h, pols & mask_of(left)))
    col = L.get("S", ("v", hb)) if not right else L.get("S", ("X", tuple(right), hb, pols & mask_of(right)))
    out = L.get("C", ("c", tuple(left), tuple(right), h, hb, pols & (mask_of(left) | mask_of(right))))
    return dict(op=OP_BIL, a=0, b=0, fields=[out, row, col], flops=72)


def build_stages(L):
    s1, s2, s3 = [], [], []
    for s in L.seqs[2]:
        for pv in pol_variants(s):
            s1.append(task_J(L, s, pv))
    for hb in range(2):
        for d in LABELS:
            for pv in pol_variants((d,)):
                s1.append(task_X(L, (d,), hb, pv))
    for h in range(2):
        for a in LABELS:
            for pv in pol_variants((a,)):
                s1.append(task_Y(L, (a,), h, pv, True))
    for h in range(2):
        for hb in range(2):
            s1.append(task_bil(L, (), (), h, hb, 0))
    for s in L.seqs[3]:
        for pv in pol_variants(s):
            s2.append(task_J(L, s, pv))
    for hb in range(2):
        for cd in L.ordered_pairs:
            for pv in pol_variants(cd):
                s2.append(task_X(L, cd, hb, pv))
    for h in range(2):
        for ab in L.ordered_pairs:
            for pv in pol_variants(ab):
                s2.append(task_Y(L, ab, h, pv, False))
    for h in range(2):
        for hb in range(2):
            for d in LABELS:
                for pv in pol_variants((d,)):
                    s2.append(task_bil(L, (), (d,), h, hb, pv))
                    s2.append(task_bil(L, (d,), (), h, hb, pv))
            for ad in L.ordered_pairs:
                for pv in pol_variants(ad):
                    s2.append(task_bil(L, (ad[0],), (ad[1],), h, hb, pv))
    for s in L.seqs[4]:
        for pv in pol_variants(s):
            s3.append(task_J(L, s, pv))
    return [s1, s2, s3]


# tasks a lane may interleave in one round, by task shape (op, a, b): independent instruction streams hide the
# FP64 and shared-memory latencies that two warps per scheduler cannot
MAX_MULT = {(OP_J, 1, 0): 1, (OP_J, 2, 1): 2, (OP_J, 3, 3): 2, (OP_XCOL, 1, 1): 1, (OP_XCOL, 2, 1): 2,
            (OP_YROW, 1, 1): 1, (OP_YROW, 2, 0): 2, (OP_BIL, 0, 0): 4}


def schedule(stage_tasks, n_warps=2):
    """Splits the tasks of a stage into warp rounds.  A round = up to 32 * m tasks of equal shape; lane l runs tasks
    l, 32 + l, ... of the round interleaved (m <= MAX_MULT).  Large groups are halved between the two warps, small
    ones go whole to the less loaded warp."""
    groups = {}
    for t in stage_tasks:
        groups.setdefault((t["op"], t["a"], t["b"]), []).append(t)
    warps = [[] for _ in range(n_warps)]
    load = [0] * n_warps

    def add_rounds(w, key, ts):
        cap = 32 * MAX_MULT[key]
        for i in range(0, len(ts), cap):
            chunk = ts[i:i + cap]
            m = (len(chunk) + 31) // 32
            warps[w].append((key, m, chunk))
            load[w] += chunk[0]["flops"] * m

    for key in sorted(groups, key=lambda k: -groups[k][0]["flops"] * len(groups[k])):
        ts = groups[key]
        if len(ts) >= 64:
            half = (len(ts) // 2 + 31) // 32 * 32 if len(ts) % 64 else len(ts) // 2
            lo = load.index(min(load))          # the less loaded warp takes the larger part
            add_rounds(lo, key, ts[:half])
            add_rounds(1 - lo, key, ts[half:])
        else:
            add_rounds(load.index(min(load)), key, ts)
    return warps, load


# ---- stage S4: generated straight-line code --------------------------------------------------------------------
def pair_name(a, b):
    return "pp%d%d" % (min(a, b), max(a, b))


def emit_s4(L):
    perms = list(itertools.permutations(LABELS))
    perms_c, Cnum, Cden = colour_matrix(N)
    assert perms_c == perms
    o = []
    w = o.append
    w("// S4: thread (pols, h, hb) forms its %d colour-ordered amplitudes and contracts them with the colour matrix." % len(perms))
    w("// Returns sum_{s,s'} conj(Ahat_s) Cnum_{ss'} Ahat_s'  (colour matrix numerators; the caller divides by kCoopCden).")
    w("MF_HD double coop_s4(const double* V, const double* S, const double* C, int pols, int h, int hb) {")
    w("  const int hs = h * 2 + hb;")
    for g in LABELS:
        w("  const int ps%d = (pols >> %d) & 1;" % (g, g))
    for a, b in itertools.combinations(LABELS, 2):
        w("  const int %s = ps%d | (ps%d << 1);" % (pair_name(a, b), a, b))
    for m in LABELS:
        rest = [g for g in LABELS if g != m]
        w("  const int pt%d = ps%d | (ps%d << 1) | (ps%d << 2);" % (m, rest[0], rest[1], rest[2]))
    opi = {p: i for i, p in enumerate(L.ordered_pairs)}
    amp = {}
    # term 1: Ytilde(ab) . Xhat(cd)
    for a, b in itertools.combinations(LABELS, 2):
        c, d = [g for g in LABELS if g not in (a, b)]
        w("  {")
        for (x, y) in ((a, b), (b, a)):
            w("    const spin yt%d%d = coop_ld_spin(S, %d + (h * 12 + %d) * 4 + %s);" % (x, y, L.bases["Yt"], opi[(x, y)], pair_name(x, y)))
        for (x, y) in ((c, d), (d, c)):
            w("    const spin x%d%d = coop_ld_spin(S, %d + (hb * 12 + %d) * 4 + %s);" % (x, y, L.bases["X2"], opi[(x, y)], pair_name(x, y)))
        for (x, y) in ((a, b), (b, a)):
            for (u, v) in ((c, d), (d, c)):
                nm = "%d%d%d%d" % (x, y, u, v)
                w("    const cplx t%s = sdot(yt%d%d, x%d%d);" % (nm, x, y, u, v))
                w("    A%sr = t%s.re; A%si = t%s.im;" % (nm, nm, nm, nm))
                amp[(x, y, u, v)] = True
        w("  }")
    decl = "  double " + ", ".join("A%d%d%d%dr, A%d%d%d%di" % (p + p) for p in perms) + ";"
    # the declarations must precede the blocks: insert after the index preamble
    first_block = next(i for i, l in enumerate(o) if l == "  {")
    o.insert(first_block, decl)

    def add(perm, z, sign):
        nm = "%d%d%d%d" % perm
        w("    A%sr %s= %s.re; A%si %s= %s.im;" % (nm, "+" if sign > 0 else "-", z, nm, "+" if sign > 0 else "-", z))

    # term 2: c0 . J4(sigma)
    w("  {")
    w("    const cvec c0 = coop_ld_cvec(C, %d + hs);" % L.bases["c0"])
    for i, s in enumerate(L.seqs[4]):
        w("    { const cplx z = cdot_r(c0, coop_ld_vec(V, %d + %d * 16 + pols));" % (L.bases["J4"], i))
        add(s, "z", 1)
        add(s[::-1], "z", (-1) ** (4 + 1))
        w("    }")
    w("  }")
    # terms 3 and 4: c(., d) . J3(abc)  and  c(a, .) . J3(bcd)
    seq3_index = {s: i for i, s in enumerate(L.seqs[3])}
    for g in LABELS:
        w("  {")
        w("    const cvec cr = coop_ld_cvec(C, %d + (hs * 4 + %d) * 2 + ps%d);" % (L.bases["cR"], g, g))
        w("    const cvec cl = coop_ld_cvec(C, %d + (hs * 4 + %d) * 2 + ps%d);" % (L.bases["cL"], g, g))
        for s in L.seqs[3]:
            if g in s:
                continue
            w("    { const rvec j = coop_ld_vec(V, %d + %d * 8 + pt%d);" % (L.bases["J3"], seq3_index[s], g))
            w("      const cplx zr = cdot_r(cr, j), zl = cdot_r(cl, j);")
            add(s + (g,), "zr", 1)
            add(s[::-1] + (g,), "zr", 1)
            add((g,) + s, "zl", 1)
            add((g,) + s[::-1], "zl", 1)
            w("    }")
        w("  }")
    # term 5: c(a, d) . J2(bc)
    seq2_index = {s: i for i, s in enumerate(L.seqs[2])}
    for (a, d) in L.ordered_pairs:
        b, c = [g for g in LABELS if g not in (a, d)]
        w("  { const cvec clr = coop_ld_cvec(C, %d + (hs * 12 + %d) * 4 + %s);" % (L.bases["cLR"], opi[(a, d)], pair_name(a, d)))
        w("    const cplx z = cdot_r(clr, coop_ld_vec(V, %d + %d * 4 + %s));" % (L.bases["J2"], seq2_index[(b, c)], pair_name(b, c)))
        add((a, b, c, d), "z", 1)
        add((a, c, b, d), "z", -1)
        w("  }")
    # colour contraction grouped by distinct matrix entry
    groups = {}
    for i in range(len(perms)):
        for j in range(i, len(perms)):
            v = int(Cnum[i, j]) * (1 if i == j else 2)
            if v:
                groups.setdefault(v, []).append((i, j))
    w("  double acc = 0.0, g;")
    for v in sorted(groups):
        first = True
        for (i, j) in groups[v]:
            a, b = "A%d%d%d%d" % perms[i], "A%d%d%d%d" % perms[j]
            if first:
                w("  g = fma(%si, %si, %sr * %sr);" % (a, b, a, b))
            else:
                w("  g = fma(%si, %si, fma(%sr, %sr, g));" % (a, b, a, b))
            first = False
        w("  acc = fma(%.1f, g, acc);" % v)
    w("  return acc;")
    w("}")
    npairs = sum(len(v) for v in groups.values())
    flops = 24 * 30 + 48 * 14 + 4 * 2 * 24 + 4 * npairs + len(groups)
    return "\n".join(o), Cden, flops


def emit_tables(L, stages):
    """Per warp ONE flat list of rounds over all stages (the last round of a stage carries the barrier flag).  The
    operand indices of a round are stored as 16-byte vectors of 8 shorts, vector (t, v) of all 32 lanes contiguous
    (t = task slot of the lane, v = vector of the task), so a warp fetches them with conflict-free 128-bit loads."""
    o = []
    w = o.append
    words = []          # the table as shorts, later grouped into uint4 (8 shorts)
    w("struct CoopRound { short variant, m, nvec, stage, sync, pad; int offset; };  // offset in 16-byte vectors")
    sched = [schedule(st) for st in stages]
    n_warps = 2
    variants = []       # (op, a, b, m) in order of first use
    rows, counts = [], []
    for wi in range(n_warps):
        row = []
        for si, (warps, load) in enumerate(sched):
            rounds = warps[wi]
            assert rounds, "every warp needs a round in every stage (it carries the barrier)"
            for ri, (key, m, tasks) in enumerate(rounds):
                nf = len(tasks[0]["fields"])
                nvec = 1
                while nvec * 8 < nf:
                    nvec *= 2
                assert nvec <= 4
                var = key + (m,)
                if var not in variants:
                    variants.append(var)
                off = len(words) // 8
                for t in range(m):
                    for v in range(nvec):
                        for lane in range(32):
                            i = t * 32 + lane
                            f = list(tasks[i]["fields"]) if i < len(tasks) else [-1]
                            f += [0] * (nvec * 8 - len(f))
                            words.extend(f[8 * v:8 * v + 8])
                row.append("{%d, %d, %d, %d, %d, 0, %d}" % (variants.index(var), m, nvec, si, 1 if ri == len(rounds) - 1 else 0, off))
        counts.append(len(row))
        rows.append(row)
    max_rounds = max(counts)
    w("constexpr int kCoopStages = %d, kCoopWarps = %d, kCoopMaxRounds = %d;" % (len(stages), n_warps, max_rounds))
    w("MF_CONST CoopRound kCoopRounds[kCoopWarps][kCoopMaxRounds] = {")
    for wi, row in enumerate(rows):
        row = row + ["{-1, 0, 0, 0, 0, 0, 0}"] * (max_rounds - len(row))
        w("  {" + ", ".join(row) + "},  // warp %d: ~%s flop/lane per stage" % (wi, "/".join(str(ld[wi]) for _, ld in sched)))
    w("};")
    w("MF_CONST int kCoopNumRounds[kCoopWarps] = {%s};" % ", ".join(map(str, counts)))
    names = {OP_J: "CoopTaskJ<%d, %d>", OP_XCOL: "CoopTaskX<%d>", OP_YROW: "CoopTaskY<%d, %s>", OP_BIL: "CoopTaskBil"}
    w("// the (task shape, tasks per lane) combinations the rounds use: X(variant id, tasks per lane, task type)")
    w("#define MF_COOP_VARIANTS(X) \\")
    for i, (op, a, b, m) in enumerate(variants):
        if op == OP_J:
            nm = names[op] % (a, b)
        elif op == OP_XCOL:
            nm = names[op] % a
        elif op == OP_YROW:
            nm = names[op] % (a, "true" if b else "false")
        else:
            nm = names[op]
        w("  X(%d, %d, %s)%s" % (i, m, nm.replace(", ", " MF_COMMA "), " \\" if i + 1 < len(variants) else ""))
    assert max(words) < 32768 and len(words) % 8 == 0
    w("// operand indices: vector (offset + (t * nvec + v) * 32 + lane) holds fields 8 v .. 8 v + 7 of task slot t of the lane")
    w("// (-1 in field 0 = idle slot)")
    w("constexpr int kCoopTableVecs = %d;" % (len(words) // 8))
    w("__align__(16) MF_TABLE short kCoopTable[%d] = {" % len(words))
    for i in range(0, len(words), 32):
        w("  " + ", ".join("%d" % v for v in words[i:i + 32]) + ",")
    w("};")
    return "\n".join(o), sched


def main():
    L = build_layout()
    stages = build_stages(L)
    s4, Cden, s4_flops = emit_s4(L)
    tables, sched = emit_tables(L, stages)
    staged = sum(t["flops"] for st in stages for t in st)
    s0_flops = 15 * 30 + 200
    total = s0_flops + staged + 64 * s4_flops
    hdr = ["// GENERATED by gen_coop.py — do not edit.  Cooperative (64 threads per event) matrix element of",
           "// g g -> t tbar g g: scratch layout, task tables of stages S1-S3, straight-line stage S4.",
           "#pragma once", '#include "mf_me_prims.cuh"', "",
           "#if defined(__CUDA_ARCH__)", "#define MF_TABLE static __device__ const", "#define MF_CONST static __constant__ const",
           "#else", "#define MF_TABLE static const", "#define MF_CONST static const", "#endif",
           "#if !defined(__CUDACC__)", "#define __align__(n) alignas(n)", "#endif", "",
           "namespace mf {", "",
           "// scratch layout (doubles): VEC 4*kCoopNV | SPIN 8*kCoopNS | CVEC 8*kCoopNC | SCAL kCoopNX (each region 16-byte aligned)",
           "constexpr int kCoopNV = %d, kCoopNS = %d, kCoopNC = %d, kCoopNX = %d;" % (L.n("V"), L.n("S"), L.n("C"), L.n("X")),
           "constexpr int kCoopScratchDoubles = 4 * kCoopNV + 8 * kCoopNS + 8 * kCoopNC + kCoopNX;",
           "constexpr double kCoopCden = %.1f;" % Cden,
           "// item indices the hand-written stage S0 needs"]
    for m in range(1, 1 << N):
        hdr.append("//   P[mask %2d] = VEC %d" % (m, L.get("V", ("P", m))))
    hdr.append("constexpr int kCoopP0 = %d, kCoopQX0 = %d, kCoopQY0 = %d, kCoopEps0 = %d;" %
               (L.get("V", ("P", 1)), L.get("V", ("qX", 1)), L.get("V", ("qY", 1)), L.get("V", ("eps", 0, 0))))
    hdr.append("constexpr int kCoopUb0 = %d, kCoopV0 = %d;" % (L.get("S", ("ub", 0)), L.get("S", ("v", 0))))

    def tab(name, arr, key_of):
        vals = []
        for m in range(1, 1 << N):
            k = key_of(m)
            vals.append(str(L.idx[arr].get(k, -1)))
        return "MF_TABLE short %s[15] = {%s};" % (name, ", ".join(vals))

    hdr.append(tab("kCoopQXofMask", "V", lambda m: ("qX", m)))
    hdr.append(tab("kCoopQYofMask", "V", lambda m: ("qY", m)))
    hdr.append(tab("kCoopIP2ofMask", "X", lambda m: ("iP2", m)))
    hdr.append(tab("kCoopIdXofMask", "X", lambda m: ("idX", m)))
    hdr.append(tab("kCoopIdYofMask", "X", lambda m: ("idY", m)))
    hdr.append("// static fp64 operation count per event (adds + multiplies, FMA = 2): S0 %d + S1-S3 %d + 64 x S4 %d" %
               (s0_flops, staged, s4_flops))
    hdr.append("constexpr double kFlopsMe2Coop_2g = %d.0;" % total)
    hdr.append("")
    loaders = '''// Scratch items are stored as planes of double2 so that consecutive lanes reading consecutive items issue
// conflict-free 128-bit shared-memory loads: VEC plane p = components (2p, 2p+1); SPIN / CVEC plane c = (re[c], im[c]).
MF_HD rvec coop_ld_vec(const double* V, int i) {
  const double2* q = reinterpret_cast<const double2*>(V);
  const double2 a = q[i], b = q[kCoopNV + i];
  rvec r;
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = b.x; r.v[3] = b.y;
  return r;
}
MF_HD void coop_st_vec(double* V, int i, const rvec& r) {
  double2* q = reinterpret_cast<double2*>(V);
  q[i] = make_double2(r.v[0], r.v[1]);
  q[kCoopNV + i] = make_double2(r.v[2], r.v[3]);
}
MF_HD spin coop_ld_spin(const double* S, int i) {
  const double2* q = reinterpret_cast<const double2*>(S);
  spin r;
#pragma unroll
  for (int c = 0; c < 4; ++c) { const double2 t = q[c * kCoopNS + i]; r.re[c] = t.x; r.im[c] = t.y; }
  return r;
}
MF_HD void coop_st_spin(double* S, int i, const spin& r) {
  double2* q = reinterpret_cast<double2*>(S);
#pragma unroll
  for (int c = 0; c < 4; ++c) q[c * kCoopNS + i] = make_double2(r.re[c], r.im[c]);
}
MF_HD cvec coop_ld_cvec(const double* C, int i) {
  const double2* q = reinterpret_cast<const double2*>(C);
  cvec r;
#pragma unroll
  for (int c = 0; c < 4; ++c) { const double2 t = q[c * kCoopNC + i]; r.re[c] = t.x; r.im[c] = t.y; }
  return r;
}
MF_HD void coop_st_cvec(double* C, int i, const cvec& r) {
  double2* q = reinterpret_cast<double2*>(C);
#pragma unroll
  for (int c = 0; c < 4; ++c) q[c * kCoopNC + i] = make_double2(r.re[c], r.im[c]);
}
'''
    text = "\n".join(hdr) + "\n" + loaders + "\n" + tables + "\n\n" + s4 + "\n\n}  // namespace mf\n"
    path = os.path.join(HERE, "mf_me_ttgg_coop_generated.cuh")
    old = open(path).read() if os.path.exists(path) else None
    if old != text:
        with open(path, "w") as f:
            f.write(text)
    return path


if __name__ == "__main__":
    print(main())
