#!/usr/bin/env python3
"""Build-time generator of the COOPERATIVE matrix element of g g -> t tbar g g (64 threads per event).

The straight-line code of gen_me.py keeps one event per thread; for 4 gluons its working set spills ~80 kB per
thread.  This generator re-organises the same colour-ordered recursion (R10) as a STAGED program over a
shared-memory scratch, executed by a team of 64 threads (2 warps) per event:

  * spin-flip symmetry: with real gluon polarisation vectors the amplitudes of the quark spin assignment
    (-s, -sbar) are, up to a common phase, the complex conjugates of those of (s, sbar) (B u* with
    B = gamma^0 gamma^1 gamma^3 is the spin-flipped solution and B gamma^mu* B^-1 = gamma^mu), so
    A^dagger C A is the same for both: only the top spin state 0 is evaluated and the sum is doubled;
  * helicity recycling: a current is computed once per polarisation assignment of the gluons IT contains
    (J2: 4 variants, J3: 8; X(cd): 2 spins x 4; ...), not once per full helicity combination;
  * polarisation siblings: one lane computes M = 2 or 4 variants of a current that differ in the polarisation of
    its first / last gluon, loading the shared operands (and forming the shared dot products) once: the program
    is co-limited by shared-memory bandwidth, so operand reuse in registers matters as much as flops;
  * S4 needs a four-gluon current only contracted with the fermion bilinear ubar gamma^mu v, and the bilinears
    Y(a) gamma^mu X(d) only contracted with J(bc): the tasks store those complex SCALARS (z2, z5), not the vectors;
  * stages S1, A, B are table driven: one lane-task = M sibling currents; the tables (operand indices into the
    scratch) are emitted here, so the kernel's interpreter has no index arithmetic;
  * stage S4 is generated straight-line code: thread (pols, hb, k) forms the real (k = 0) or imaginary (k = 1)
    parts of its 24 colour-ordered amplitudes and contracts them with the colour matrix
    (A^dagger C A = Re A^T C Re A + Im A^T C Im A for real symmetric C), so the two warps of a team share S4
    without exchanging anything.

Emits mf_me_ttgg_coop_generated.cuh.  Imports nothing from oracle/.
"""
import itertools
import os

from gen_me import colour_matrix

HERE = os.path.dirname(os.path.abspath(__file__))
N = 4           # gluons: 0, 1 beams; 2, 3 final
LABELS = list(range(N))

# ---- schedule knobs (tuned on B200; any setting gives the same result up to rounding) -------------------------
# number of sibling groups computed by the wide lane-task of a family; the rest use the next narrower one
WIDE_GROUPS = {"J3": 32, "X2": 32, "Yt": 24, "z5": 32, "J4": 32}
ROUND_OVERHEAD = 60      # cost-model flops per round and lane (field fetch, dispatch)


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


def pol_words(gluons):
    """all full 4-bit pol words with zero bits outside `gluons`, in polidx order"""
    gl = sorted(gluons)
    out = []
    for v in range(1 << len(gl)):
        p = 0
        for i, g in enumerate(gl):
            p |= ((v >> i) & 1) << g
        out.append(p)
    return out


class Layout:
    """VEC items (real 4-vectors), SPIN items (Dirac spinors), X scalars; Z = two planes of complex scalars"""

    def __init__(self):
        self.idx = {"V": {}, "S": {}, "X": {}}
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


ORDERED_PAIRS = list(itertools.permutations(LABELS, 2))
PAIR_INDEX = {p: i for i, p in enumerate(ORDERED_PAIRS)}
SEQS = {k: [s for s in itertools.permutations(LABELS, k) if canon(s)[0] == s] for k in range(2, N + 1)}
SEQ_INDEX = {k: {s: i for i, s in enumerate(SEQS[k])} for k in SEQS}
# z arrays: rows of 16 polarisation words, padded, and with the word's bits PERMUTED per row so that the lanes of a
# producing round (which differ in the sequence / pair and in the polarisations of the inner gluons) store to
# different banks: z2 row (seq = (a, b, c, d), hb): bit order (b, c, a, d), stride 18; z5 row (pair (a, d), hb),
# b < c the other two gluons: bit order (a, b, c, d), stride 17.  The reading S4 threads of a half warp cover one
# whole row, in any order.
Z_ROW = 18                  # z2 row stride (also the hb stride the J4 tasks use)
Z5_ROW = 17
Z5_OFF = 12 * 2 * Z_ROW
Z_PLANE = Z5_OFF + 12 * 2 * Z5_ROW   # doubles per re / im plane
SPIN_ROW = 13               # X2 / Ytilde: rows of 12 ordered pairs, padded (bank spread for the S4 readers)
J2_STRIDE = len([0 for _ in itertools.combinations(LABELS, 2)])   # J2 stored polarisation-major: [4][6 sequences]


def permuted_word(order, pols):
    """bit i of the result = polarisation of gluon order[i]"""
    v = 0
    for i, g in enumerate(order):
        v |= ((pols >> g) & 1) << i
    return v


def z2_order(seq):
    a, b, c, d = seq
    return (b, c, a, d)


def z5_order(pair):
    a, d = pair
    b, c = [g for g in LABELS if g not in pair]
    return (a, b, c, d)


def build_layout():
    L = Layout()
    for m in range(1, 1 << N):
        L.add("V", ("P", m))
    for m in range(1, 1 << N):
        if bin(m).count("1") <= 2:
            L.add("V", ("qX", m))
    for m in range(1, 1 << N):
        if bin(m).count("1") == 1:
            L.add("V", ("qY", m))
    for g in LABELS:
        for p in range(2):
            L.add("V", ("eps", g, p))
    # gluon currents, canonical sequences, family-contiguous so S4 and the z5 tasks can index them arithmetically:
    # J2 [polidx][seq] (the z5 tasks read all four variants of one sequence), J3 [seq][polidx]
    L.bases["J2"] = L.n("V")
    for v in range(4):
        for s in SEQS[2]:
            L.add("V", ("J", s, pol_words(s)[v]))
    L.bases["J3"] = L.n("V")
    for s in SEQS[3]:
        for pw in pol_words(s):
            L.add("V", ("J", s, pw))
    # fermion bilinears as pairs of real vectors (k = 0 real part, 1 imaginary part)
    L.bases["c0"] = L.n("V")
    for hb in range(2):
        for k in range(2):
            L.add("V", ("c0", hb, k))
    for nm in ("cR", "cL"):
        L.bases[nm] = L.n("V")
        for g in LABELS:
            for hb in range(2):
                for p in range(2):
                    for k in range(2):
                        L.add("V", (nm, g, hb, p, k))
    for m in range(1, 1 << N):
        if bin(m).count("1") >= 2:
            L.add("X", ("iP2", m))
        if bin(m).count("1") <= 2:
            L.add("X", ("idX", m))
        if bin(m).count("1") == 1:
            L.add("X", ("idY", m))
    L.add("S", ("ub",))
    for hb in range(2):
        L.add("S", ("v", hb))
    L.bases["X1"] = L.n("S")
    for hb in range(2):
        for d in LABELS:
            for p in range(2):
                L.add("S", ("X1", d, hb, p))
    L.bases["Y1"] = L.n("S")
    for a in LABELS:
        for p in range(2):
            L.add("S", ("Y1", a, p))
    L.bases["X2"] = L.n("S")       # [hb][polidx][pair, padded to SPIN_ROW]
    for hb in range(2):
        for v in range(4):
            for cd in ORDERED_PAIRS:
                L.add("S", ("X2", cd, hb, pol_words(cd)[v]))
            for i in range(SPIN_ROW - len(ORDERED_PAIRS)):
                L.add("S", ("pad", "X2", hb, v, i))
    L.bases["Yt"] = L.n("S")       # [polidx][pair, padded]
    for v in range(4):
        for ab in ORDERED_PAIRS:
            L.add("S", ("Yt", ab, pol_words(ab)[v]))
        for i in range(SPIN_ROW - len(ORDERED_PAIRS)):
            L.add("S", ("pad", "Yt", v, i))
    return L


# ---- operand lookup ----------------------------------------------------------------------------------------
def J_ref(L, seq, pols):
    """(VEC index, sign) of Jhat(seq) for the polarisation word `pols`"""
    seq = tuple(seq)
    if len(seq) == 1:
        return L.get("V", ("eps", seq[0], (pols >> seq[0]) & 1)), 1
    c, s = canon(seq)
    return L.get("V", ("J", c, pols & mask_of(seq))), s


def P_ref(L, seq):
    return L.get("V", ("P", mask_of(seq)))


def z2_index(seq, pols):
    return (SEQ_INDEX[4][seq] * 2) * Z_ROW + permuted_word(z2_order(seq), pols)   # hb = 0, k = 0; hb stride Z_ROW


def z5_index(pair, hb, pols):
    return Z5_OFF + (PAIR_INDEX[pair] * 2 + hb) * Z5_ROW + permuted_word(z5_order(pair), pols)


# ---- flop model of the task templates of mf_me_coop.cuh (adds + multiplies, FMA = 2; shared dot products of
# sibling currents counted once, as the templates compute them once) ------------------------------------------
def flops_v3(ma, md):
    mm = ma * md
    return 7 * (mm + ma + md) + (ma + md) + 4 + 24 * mm


def flops_v4(ma, md):
    mm = ma * md
    return 7 * (mm + ma + md) + mm + 24 * mm


F_SLASH, F_SLASH_ACC, F_PROP, F_BIL, F_CDOT = 42, 50, 66, 72, 14


# ---- lane-tasks ---------------------------------------------------------------------------------------------
def task_J2(L, s, pw):
    a, b = s
    return dict(fam="J2", M=1, flops=flops_v3(1, 1) + 4,
                fields=[L.get("V", ("J", s, pw)), L.get("X", ("iP2", mask_of(s))), J_ref(L, (a,), pw)[0], P_ref(L, (a,)),
                        J_ref(L, (b,), pw)[0], P_ref(L, (b,))])


def task_X1c(L, d, hb, p):
    pw = p << d
    return dict(fam="X1c", M=1, flops=F_SLASH + F_PROP + F_BIL,
                fields=[L.get("S", ("X1", d, hb, p)), L.get("V", ("qX", 1 << d)), L.get("X", ("idX", 1 << d)),
                        J_ref(L, (d,), pw)[0], L.get("S", ("v", hb)), L.get("S", ("ub",)),
                        L.get("V", ("cR", d, hb, p, 0)), L.get("V", ("cR", d, hb, p, 1))])


def task_Y1c(L, a, p):
    pw = p << a
    return dict(fam="Y1c", M=1, flops=F_SLASH + F_PROP + 2 * F_BIL,
                fields=[L.get("S", ("Y1", a, p)), L.get("V", ("qY", 1 << a)), L.get("X", ("idY", 1 << a)),
                        L.get("S", ("ub",)), J_ref(L, (a,), pw)[0], L.get("S", ("v", 0)), L.get("S", ("v", 1)),
                        L.get("V", ("cL", a, 0, p, 0)), L.get("V", ("cL", a, 0, p, 1)),
                        L.get("V", ("cL", a, 1, p, 0)), L.get("V", ("cL", a, 1, p, 1))])


def task_J3(L, s, pw_ab, m):
    """J3(abc) for the polarisations pw_ab of (a, b) and pc = 0..m-1 (m = 2) or pc given in pw_ab (m = 1)"""
    a, b, c = s
    pcs = [0, 1] if m == 2 else [(pw_ab >> c) & 1]
    base = pw_ab & ~(1 << c)
    pws = [base | (pc << c) for pc in pcs]
    j2bc = [J_ref(L, (b, c), pw) for pw in pws]
    j2ab = J_ref(L, (a, b), base)
    signs = (1 if j2bc[0][1] < 0 else 0) | (2 if j2ab[1] < 0 else 0)
    f = [L.get("V", ("J", s, pw)) for pw in pws]
    f += [L.get("X", ("iP2", mask_of(s))), J_ref(L, (a,), base)[0], P_ref(L, (a,))]
    f += [x[0] for x in j2bc] + [P_ref(L, (b, c)), j2ab[0], P_ref(L, (a, b))]
    f += [J_ref(L, (c,), pw)[0] for pw in pws] + [P_ref(L, (c,)), J_ref(L, (b,), base)[0], signs]
    fl = 2 * (7 * (2 * m + 1) + (1 + m) + 4 + 24 * m) + 7 * (2 * m + 1) + 25 * m + 4 * m
    return dict(fam="J3", M=m, fields=f, flops=fl)


def task_J4(L, s, pw_bc, ma, md, pa=0, pd=0):
    """z2 = c0 . J4(abcd) for the polarisations pw_bc of (b, c) and (pa, pd) in ma x md variants"""
    a, b, c, d = s
    base = pw_bc & ((1 << b) | (1 << c))
    pas = [0, 1] if ma == 2 else [pa]
    pds = [0, 1] if md == 2 else [pd]
    wa = [base | (x << a) for x in pas]        # words seen by operands containing a (not d)
    wd = [base | (x << d) for x in pds]
    j2ab = [J_ref(L, (a, b), w) for w in wa]
    j2cd = [J_ref(L, (c, d), w) for w in wd]
    j2bc = J_ref(L, (b, c), base)
    signs = (1 if j2ab[0][1] < 0 else 0) | (2 if j2cd[0][1] < 0 else 0) | (4 if j2bc[1] < 0 else 0)
    f = [z2_index(s, base | (x << a) | (y << d)) for y in pds for x in pas]      # out[ia + ma * id]
    f += [L.get("X", ("iP2", mask_of(s)))]
    f += [J_ref(L, (a,), w)[0] for w in wa] + [x[0] for x in j2ab] + [J_ref(L, (a, b, c), w)[0] for w in wa]
    f += [J_ref(L, (d,), w)[0] for w in wd] + [x[0] for x in j2cd] + [J_ref(L, (b, c, d), w)[0] for w in wd]
    f += [J_ref(L, (b,), base)[0], J_ref(L, (c,), base)[0], j2bc[0]]
    f += [P_ref(L, (a,)), P_ref(L, (b, c, d)), P_ref(L, (a, b)), P_ref(L, (c, d)), P_ref(L, (a, b, c)), P_ref(L, (d,))]
    f += [L.get("V", ("c0", 0, 0)), signs]
    mm = ma * md
    fl = 3 * flops_v3(ma, md) + 3 * flops_v4(ma, md) + 16 + 4 * 7 * mm
    return dict(fam="J4", M=mm, MA=ma, MD=md, fields=f, flops=fl)


def task_X2(L, cd, hb, pd, m, pc=0):
    """X2(cd) = prop [eps_c-slash X1(d) + J2(cd)-slash v] for pc = 0..m-1"""
    c, d = cd
    pcs = [0, 1] if m == 2 else [pc]
    pws = [(x << c) | (pd << d) for x in pcs]
    j2 = [J_ref(L, cd, w) for w in pws]
    f = [L.get("S", ("X2", cd, hb, w)) for w in pws]
    f += [L.get("V", ("qX", mask_of(cd))), L.get("X", ("idX", mask_of(cd))), L.get("S", ("X1", d, hb, pd)),
          L.get("S", ("v", hb))]
    f += [J_ref(L, (c,), w)[0] for w in pws] + [x[0] for x in j2] + [1 if j2[0][1] < 0 else 0]
    return dict(fam="X2", M=m, fields=f, flops=m * (F_SLASH + F_SLASH_ACC + F_PROP))


def task_Yt(L, ab, pa, m, pb=0):
    """Ytilde(ab) = ubar J2(ab)-slash + Y1(a) eps_b-slash for pb = 0..m-1"""
    a, b = ab
    pbs = [0, 1] if m == 2 else [pb]
    pws = [(pa << a) | (x << b) for x in pbs]
    j2 = [J_ref(L, ab, w) for w in pws]
    f = [L.get("S", ("Yt", ab, w)) for w in pws]
    f += [L.get("S", ("ub",)), L.get("S", ("Y1", a, pa))]
    f += [x[0] for x in j2] + [J_ref(L, (b,), w)[0] for w in pws] + [1 if j2[0][1] < 0 else 0]
    return dict(fam="Yt", M=m, fields=f, flops=m * (F_SLASH + F_SLASH_ACC))


def task_z5(L, ad, hb, pa, m, pd=0):
    """z5 = [Y1(a) gamma X1(d)] . J2(bc) for the 4 polarisations of (b, c), b < c, and pd = 0..m-1"""
    a, d = ad
    b, c = [g for g in LABELS if g not in ad]
    pds = [0, 1] if m == 2 else [pd]
    f = [z5_index(ad, hb, (pa << a) | (x << d)) for x in pds]
    f += [2, 4, L.get("S", ("Y1", a, pa))]              # bits of pb, pc in the permuted z5 word
    f += [L.get("S", ("X1", d, hb, x)) for x in pds]
    f += [L.get("V", ("J", (b, c), 0))]
    return dict(fam="z5", M=m, fields=f, flops=m * (F_BIL + 4 * F_CDOT))


def build_rounds(L):
    """lane-tasks grouped into rounds of <= 32 equal-shaped lane-tasks; each round knows the phases it may run in"""
    rounds = []

    def add(phases, tasks):
        for i in range(0, len(tasks), 32):
            chunk = tasks[i:i + 32]
            t0 = chunk[0]
            key = (t0["fam"], t0.get("MA", 0), t0.get("MD", 0), t0["M"])
            rounds.append(dict(key=key, tasks=chunk, phases=phases, cost=t0["flops"] + ROUND_OVERHEAD))

    # S1
    add(["S1"], [task_J2(L, s, pw) for s in SEQS[2] for pw in pol_words(s)])
    add(["S1"], [task_X1c(L, d, hb, p) for hb in range(2) for d in LABELS for p in range(2)])
    add(["S1"], [task_Y1c(L, a, p) for a in LABELS for p in range(2)])
    # J3: sibling groups (seq, pa, pb)
    groups = [(s, pw) for s in SEQS[3] for pw in pol_words(s[:2])]
    w = WIDE_GROUPS["J3"]
    add(["A"], [task_J3(L, s, pw, 2) for s, pw in groups[:w]])
    add(["A"], [task_J3(L, s, pw | (pc << s[2]), 1) for s, pw in groups[w:] for pc in range(2)])
    # J4: sibling groups (seq, pb, pc) of 4 (pa, pd)
    groups = [(s, pw) for s in SEQS[4] for pw in pol_words(s[1:3])]
    w = WIDE_GROUPS["J4"]
    add(["B"], [task_J4(L, s, pw, 2, 2) for s, pw in groups[:w]])
    add(["B"], [task_J4(L, s, pw, 1, 2, pa=pa) for s, pw in groups[w:] for pa in range(2)])
    # X2: sibling groups (pair, hb, pd)
    groups = [(cd, hb, pd) for hb in range(2) for pd in range(2) for cd in ORDERED_PAIRS]   # pair fastest: the lanes'
    # spinor stores then go to consecutive items
    w = WIDE_GROUPS["X2"]
    add(["A", "B"], [task_X2(L, cd, hb, pd, 2) for cd, hb, pd in groups[:w]])
    add(["A", "B"], [task_X2(L, cd, hb, pd, 1, pc) for cd, hb, pd in groups[w:] for pc in range(2)])
    # Yt: sibling groups (pair, pa)
    groups = [(ab, pa) for pa in range(2) for ab in ORDERED_PAIRS]
    w = WIDE_GROUPS["Yt"]
    add(["A", "B"], [task_Yt(L, ab, pa, 2) for ab, pa in groups[:w]])
    add(["A", "B"], [task_Yt(L, ab, pa, 1, pb) for ab, pa in groups[w:] for pb in range(2)])
    # z5: sibling groups (pair, hb, pa)
    groups = [(ad, hb, pa) for hb in range(2) for ad in ORDERED_PAIRS for pa in range(2)]
    w = WIDE_GROUPS["z5"]
    add(["A", "B"], [task_z5(L, ad, hb, pa, 2) for ad, hb, pa in groups[:w]])
    add(["A", "B"], [task_z5(L, ad, hb, pa, 1, pd) for ad, hb, pa in groups[w:] for pd in range(2)])
    return [r for r in rounds if r["tasks"]]


PHASES = ["S1", "A", "B"]


def schedule(rounds, n_warps=2):
    """assigns every round to (phase, warp) minimising sum over phases of the slower warp (exhaustive over the
    rounds that may move, greedy for the rest)"""
    fixed = [r for r in rounds if len(r["phases"]) == 1]
    flex = [r for r in rounds if len(r["phases"]) > 1]
    slots = [(p, w) for p in PHASES for w in range(n_warps)]

    def total(load):
        return sum(max(load[(p, w)] for w in range(n_warps)) for p in PHASES)

    best = None
    fixed_sorted = sorted(fixed, key=lambda r: -r["cost"])
    for combo in itertools.product(*[[(p, w) for p in r["phases"] for w in range(n_warps)] for r in flex]):
        load = {s: 0 for s in slots}
        for r, s in zip(flex, combo):
            load[s] += r["cost"]
        assign = list(combo)
        fa = []
        for r in fixed_sorted:
            p = r["phases"][0]
            w = min(range(n_warps), key=lambda x: load[(p, x)])
            load[(p, w)] += r["cost"]
            fa.append((p, w))
        t = total(load)
        if best is None or t < best[0]:
            best = (t, assign, fa, dict(load))
    _, assign, fa, load = best
    plan = {s: [] for s in slots}
    for r, s in zip(fixed_sorted, fa):
        plan[s].append(r)
    for r, s in zip(flex, assign):
        plan[s].append(r)
    for s in slots:   # producers of a phase first is irrelevant inside a phase; keep heavy rounds first
        plan[s].sort(key=lambda r: -r["cost"])
    return plan, load


# ---- stage S4: generated straight-line code --------------------------------------------------------------------
def pair_name(a, b):
    return "pp%d%d" % (min(a, b), max(a, b))


def emit_s4(L):
    perms = list(itertools.permutations(LABELS))
    perms_c, Cnum, Cden = colour_matrix(N)
    assert perms_c == perms
    o = []
    w = o.append
    flops = 0
    w("// S4: thread (pols, hb, k) forms the real (k = 0) or imaginary (k = 1) parts of its %d colour-ordered amplitudes" % len(perms))
    w("// and contracts them with the colour matrix: returns sum_{s,s'} x_s Cnum_{ss'} x_s' (the caller divides by kCoopCden).")
    w("// Team thread tid: warp = hb, lane = ps2 | ps3 << 1 | k << 2 | ps0 << 3 | ps1 << 4 (the output-fragment layout of")
    w("// the DMMA blocks of the first pair of gluon pairs; the other two pairs' results are moved to it by lane shuffles).")
    w("// EVERY lane of the warp must call it (mma.sync / shfl.sync).")
    w("MF_HD double coop_s4_tid(const double* V, const double* S, const double* Z, int tid) {")
    w("  const int hb = tid >> 5, lane = tid & 31;")
    w("  const int ps2 = lane & 1, ps3 = (lane >> 1) & 1, k = (lane >> 2) & 1, ps0 = (lane >> 3) & 1, ps1 = (lane >> 4) & 1;")
    for a, b in itertools.combinations(LABELS, 2):
        w("  const int %s = ps%d | (ps%d << 1);" % (pair_name(a, b), a, b))
    for m in LABELS:
        rest = [g for g in LABELS if g != m]
        w("  const int pt%d = ps%d | (ps%d << 1) | (ps%d << 2);" % (m, rest[0], rest[1], rest[2]))
    w("  const double* Zk = Z + k * %d;" % Z_PLANE)

    def word_expr(order):
        return " | ".join("ps%d" % g if i == 0 else "(ps%d << %d)" % (g, i) for i, g in enumerate(order))
    w("  double " + ", ".join("A%d%d%d%d" % p for p in perms) + ";")
    # term 1: Ytilde(ab) . Xhat(cd), the real (k = 0) or imaginary (k = 1) part of the product.
    # Device: per pair of gluon pairs {ab | cd} two complex 8 x 8 x 4 products as DMMA.884 blocks (real 16 x 8 x 8):
    #   block N: rows Ytilde(ab / ba; pa, pb; part k), columns Xhat(cd / dc; pc, pd)        -> A[(ab)(cd)]
    #   block T: rows Xhat(ab / ba; pa, pb; part k),  columns Ytilde(cd / dc; pc, pd)       -> A[(cd)(ab)] (transposed, so
    #            that both blocks leave the helicity (pa, pb, pc, pd) and the part k in the same lane)
    # fragment lane = t | g << 2 with g = (k, pa, pb), t = (pc, pd); see coop_s4_block.
    pairs3 = [((0, 1), (2, 3)), ((0, 2), (1, 3)), ((0, 3), (1, 2))]
    w("#if defined(__CUDA_ARCH__)")
    w("  {")
    w("    double c[2][2];")
    for pi_, ((a, b), (c, d)) in enumerate(pairs3):
        # lane layout of this pair: bit 0 = ps_c, bit 1 = ps_d, bit 2 = k, bit 3 = ps_a, bit 4 = ps_b
        names_n = [["A%d%d%d%d" % (x + u) for u in ((c, d), (d, c))] for x in ((a, b), (b, a))]
        names_t = [["A%d%d%d%d" % (u + x) for u in ((c, d), (d, c))] for x in ((a, b), (b, a))]
        if pi_ == 0:
            tgt_n, tgt_t = names_n, names_t
        else:
            w("    // lane of this pair's layout that holds this thread's helicity")
            w("    const int src%d = ps%d | (ps%d << 1) | (k << 2) | (ps%d << 3) | (ps%d << 4);" % (pi_, c, d, a, b))
        w("    coop_s4_block<%d, %d, %d, %d, %d, %d>(S, lane, 0, hb * %d, c);    // Ytilde(%d%d) x Xhat(%d%d)" %
          (L.bases["Yt"], L.bases["X2"], PAIR_INDEX[(a, b)], PAIR_INDEX[(b, a)], PAIR_INDEX[(c, d)], PAIR_INDEX[(d, c)], 4 * SPIN_ROW, a, b, c, d))
        for mt in range(2):
            for j in range(2):
                if pi_ == 0:
                    w("    %s = c[%d][%d];" % (names_n[mt][j], mt, j))
                else:
                    w("    %s = __shfl_sync(0xFFFFFFFFu, c[%d][%d], src%d);" % (names_n[mt][j], mt, j, pi_))
        w("    coop_s4_block<%d, %d, %d, %d, %d, %d>(S, lane, hb * %d, 0, c);    // Xhat(%d%d) x Ytilde(%d%d), transposed" %
          (L.bases["X2"], L.bases["Yt"], PAIR_INDEX[(a, b)], PAIR_INDEX[(b, a)], PAIR_INDEX[(c, d)], PAIR_INDEX[(d, c)], 4 * SPIN_ROW, a, b, c, d))
        for mt in range(2):
            for j in range(2):
                if pi_ == 0:
                    w("    %s = c[%d][%d];" % (names_t[mt][j], mt, j))
                else:
                    w("    %s = __shfl_sync(0xFFFFFFFFu, c[%d][%d], src%d);" % (names_t[mt][j], mt, j, pi_))
        flops += 8 * 16
    w("  }")
    w("#else   // host emulation (tests/host_shim): the same products thread by thread")
    flops_dev = flops
    for a, b in itertools.combinations(LABELS, 2):
        c, d = [g for g in LABELS if g not in (a, b)]
        w("  {")
        for (x, y) in ((a, b), (b, a)):
            w("    const spin yt%d%d = coop_row_part(coop_ld_spin(S, %d + %s * %d + %d), k);" % (x, y, L.bases["Yt"], pair_name(x, y), SPIN_ROW, PAIR_INDEX[(x, y)]))
        for (x, y) in ((c, d), (d, c)):
            w("    const spin x%d%d = coop_col_part(coop_ld_spin(S, %d + (hb * 4 + %s) * %d + %d), k);" % (x, y, L.bases["X2"], pair_name(x, y), SPIN_ROW, PAIR_INDEX[(x, y)]))
        for (x, y) in ((a, b), (b, a)):
            for (u, v) in ((c, d), (d, c)):
                w("    A%d%d%d%d = sdot_part(yt%d%d, x%d%d);" % (x, y, u, v, x, y, u, v))
        w("  }")
    w("#endif")

    def add(perm, z, sign):
        nonlocal flops
        w("    A%d%d%d%d %s= %s;" % (perm + ("+" if sign > 0 else "-", z)))
        flops += 1

    # term 2: z2 = c0 . J4(sigma), stored by the J4 tasks
    w("  {")
    for i, s in enumerate(SEQS[4]):
        w("    { const double z = Zk[%d + hb * %d + (%s)];" % (i * 2 * Z_ROW, Z_ROW, word_expr(z2_order(s))))
        add(s, "z", 1)
        add(s[::-1], "z", (-1) ** (4 + 1))
        w("    }")
    w("  }")
    # terms 3 and 4: c(., g) . J3(abc)  and  c(g, .) . J3(bcd)
    for g in LABELS:
        w("  {")
        w("    const rvec cr = coop_ld_vec(V, %d + ((%d * 2 + hb) * 2 + ps%d) * 2 + k);" % (L.bases["cR"], g, g))
        w("    const rvec cl = coop_ld_vec(V, %d + ((%d * 2 + hb) * 2 + ps%d) * 2 + k);" % (L.bases["cL"], g, g))
        for s in SEQS[3]:
            if g in s:
                continue
            w("    { const rvec j = coop_ld_vec(V, %d + %d * 8 + pt%d);" % (L.bases["J3"], SEQ_INDEX[3][s], g))
            w("      const double zr = rdot(cr, j), zl = rdot(cl, j);")
            flops += 14
            add(s + (g,), "zr", 1)
            add(s[::-1] + (g,), "zr", 1)
            add((g,) + s, "zl", 1)
            add((g,) + s[::-1], "zl", 1)
            w("    }")
        w("  }")
    # term 5: z5 = c(a, d) . J2(bc), stored by the z5 tasks
    for (a, d) in ORDERED_PAIRS:
        b, c = [g for g in LABELS if g not in (a, d)]
        w("  { const double z = Zk[%d + hb * %d + (%s)];" % (Z5_OFF + PAIR_INDEX[(a, d)] * 2 * Z5_ROW, Z5_ROW, word_expr(z5_order((a, d)))))
        add((a, b, c, d), "z", 1)
        add((a, c, b, d), "z", -1)
        w("  }")
    # Colour contraction in a symmetry-adapted basis.  The colour matrix is invariant under relabelling the gluons,
    # C[rho s][rho s'] = C[s][s'], in particular under the Klein four-group V4 = {e, (01)(23), (02)(13), (03)(12)}:
    # in the basis y(chi, orbit) = sum_{rho in V4} chi(rho) x[rho s] (4 characters x 6 orbits, add/subtract
    # butterflies only) it is block diagonal, x^T C x = sum_chi y_chi^T M_chi y_chi / 16, and sequence reversal
    # (which also leaves C invariant and maps every V4 orbit to itself) empties most of the three non-trivial
    # blocks: 57 products instead of 300.  Exact integer arithmetic here; the /16 is folded into the literals.
    V4 = [(0, 1, 2, 3), (1, 0, 3, 2), (2, 3, 0, 1), (3, 2, 1, 0)]
    pidx = {p: i for i, p in enumerate(perms)}
    seen, orbits = set(), []
    for sgm in perms:
        if sgm in seen:
            continue
        orb = [tuple(r[x] for x in sgm) for r in V4]
        orbits.append(orb)
        seen.update(orb)
    for r in V4:   # the invariance the transformation relies on
        for s1 in perms:
            for s2 in perms:
                assert Cnum[pidx[tuple(r[x] for x in s1)]][pidx[tuple(r[x] for x in s2)]] == Cnum[pidx[s1]][pidx[s2]]
    chars = [(1, 1, 1, 1), (1, 1, -1, -1), (1, -1, 1, -1), (1, -1, -1, 1)]
    T = [[0] * len(perms) for _ in range(len(perms))]
    for ci, ch in enumerate(chars):
        for oi, orb in enumerate(orbits):
            for gi, sgm in enumerate(orb):
                T[ci * len(orbits) + oi][pidx[sgm]] = ch[gi]
    nP = len(perms)
    CT = [[sum(int(Cnum[i][k]) * T[j][k] for k in range(nP)) for j in range(nP)] for i in range(nP)]
    M = [[sum(T[i][k] * CT[k][j] for k in range(nP)) for j in range(nP)] for i in range(nP)]
    nO = len(orbits)
    for i in range(nP):
        for j in range(nP):
            assert M[i][j] == M[j][i] and (i // nO == j // nO or M[i][j] == 0)
    for oi, orb in enumerate(orbits):
        x = ["A%d%d%d%d" % p for p in orb]
        w("  const double s%da = %s + %s, d%da = %s - %s, s%db = %s + %s, d%db = %s - %s;" %
          (oi, x[0], x[1], oi, x[0], x[1], oi, x[2], x[3], oi, x[2], x[3]))
        w("  const double y0_%d = s%da + s%db, y1_%d = s%da - s%db, y2_%d = d%da + d%db, y3_%d = d%da - d%db;" %
          (oi, oi, oi, oi, oi, oi, oi, oi, oi, oi, oi, oi))
        flops += 8
    w("  double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;")
    n_acc = 0
    for ci in range(len(chars)):
        for i in range(nO):
            row = ci * nO + i
            terms = [(j, M[row][ci * nO + j] * (1 if j == i else 2)) for j in range(i, nO) if M[row][ci * nO + j]]
            assert terms and terms[0][0] == i
            expr = "%r * y%d_%d" % (terms[0][1] / 16.0, ci, i)
            flops += 1
            for j, v in terms[1:]:
                expr = "fma(%r, y%d_%d, %s)" % (v / 16.0, ci, j, expr)
                flops += 2
            w("  acc%d = fma(y%d_%d, %s, acc%d);" % (n_acc % 4, ci, i, expr, n_acc % 4))
            flops += 2
            n_acc += 1
    w("  const double acc = (acc0 + acc1) + (acc2 + acc3);")
    flops += 3
    w("  return acc;")
    w("}")
    return "\n".join(o), Cden, flops


VARIANT_NAMES = {"J2": "CoopTaskJ2", "X1c": "CoopTaskX1c", "Y1c": "CoopTaskY1c", "J3": "CoopTaskJ3<%(M)d>",
                 "J4": "CoopTaskJ4<%(MA)d MF_COMMA %(MD)d>", "X2": "CoopTaskX2<%(M)d>", "Yt": "CoopTaskYt<%(M)d>",
                 "z5": "CoopTaskZ5<%(M)d>"}


def emit_tables(L, rounds):
    """Per warp a straight-line program of rounds over all phases (macro MF_COOP_WARPn: R(offset, task type) per round,
    S() at the end of a phase = team barrier).  The operand indices of a round are stored as 16-byte vectors of 8
    shorts, vector v of all 32 lanes contiguous, so a warp fetches them with conflict-free 128-bit loads."""
    o = []
    w = o.append
    words = []
    n_warps = 2
    plan, load = schedule(rounds, n_warps)
    progs = []
    for wi in range(n_warps):
        prog = []
        for ph in PHASES:
            for r in plan[(ph, wi)]:
                nf = max(len(t["fields"]) for t in r["tasks"])
                nvec = (nf + 7) // 8
                off = len(words) // 8
                for v in range(nvec):
                    for lane in range(32):
                        f = list(r["tasks"][lane]["fields"]) if lane < len(r["tasks"]) else [-1]
                        f += [0] * (nvec * 8 - len(f))
                        words.extend(f[8 * v:8 * v + 8])
                key = r["key"]
                prog.append("R(%d, %s)" % (off, (VARIANT_NAMES[key[0]] % dict(MA=key[1], MD=key[2], M=key[3])).replace(" MF_COMMA", ",")))
            prog.append("S()")
        progs.append(prog)
    w("constexpr int kCoopPhases = %d, kCoopWarps = %d;" % (len(PHASES), n_warps))
    w("// the program of each warp of a team: R(table offset in 16-byte vectors, task type) = one round of 32 lane-tasks,")
    w("// S() = end of a phase (barrier of the team's two warps)")
    for wi, prog in enumerate(progs):
        cost = "/".join(str(load[(p, wi)]) for p in PHASES)
        w("// warp %d: ~%s flop/lane per phase" % (wi, cost))
        w("#define MF_COOP4_WARP%d(R, S) \\" % wi)
        w("  " + " \\\n  ".join(prog))
    assert max(words) < 32768 and min(words) >= -1 and len(words) % 8 == 0
    w("// operand indices: vector (offset + v * 32 + lane) holds fields 8 v .. 8 v + 7 of the lane's task")
    w("// (-1 in field 0 = idle lane)")
    w("constexpr int kCoopTableVecs = %d;" % (len(words) // 8))
    w("__align__(16) MF_TABLE short kCoopTable[%d] = {" % len(words))
    for i in range(0, len(words), 32):
        w("  " + ", ".join("%d" % v for v in words[i:i + 32]) + ",")
    w("};")
    return "\n".join(o), plan, load


def main():
    L = build_layout()
    rounds = build_rounds(L)
    s4, Cden, s4_flops = emit_s4(L)
    tables, plan, load = emit_tables(L, rounds)
    staged = sum(t["flops"] for r in rounds for t in r["tasks"])
    s0_flops = 15 * 30 + 250
    total = s0_flops + staged + 64 * s4_flops
    hdr = ["// GENERATED by gen_coop.py — do not edit.  Cooperative (64 threads per event) matrix element of",
           "// g g -> t tbar g g: scratch layout, task tables of phases S1 / A / B, straight-line stage S4.",
           "// A FRAGMENT: included by mf_me_coop.cuh inside namespace mf::g4 (no include guard, no namespace of its own).",
           "",
           "// scratch layout (doubles): VEC 4*kCoopNV | SPIN 8*kCoopNS | Z 2*kCoopZPlane | SCAL kCoopNX (each region 16-byte aligned)",
           "constexpr int kCoopNV = %d, kCoopNS = %d, kCoopZPlane = %d, kCoopZRow = %d, kCoopNX = %d, kCoopJ2Stride = %d, kCoopSpinRow = %d;" % (L.n("V"), L.n("S"), Z_PLANE, Z_ROW, L.n("X"), J2_STRIDE, SPIN_ROW),
           "constexpr int kCoopScratchDoubles = 4 * kCoopNV + 8 * kCoopNS + 2 * kCoopZPlane + kCoopNX;",
           "constexpr double kCoopCden = %.1f;" % Cden,
           "// item indices the hand-written stage S0 needs"]
    hdr.append("constexpr int kCoopP0 = %d, kCoopEps0 = %d, kCoopC0 = %d;" %
               (L.get("V", ("P", 1)), L.get("V", ("eps", 0, 0)), L.get("V", ("c0", 0, 0))))
    hdr.append("constexpr int kCoopUb = %d, kCoopV0 = %d;" % (L.get("S", ("ub",)), L.get("S", ("v", 0))))

    # S0 lane table: lane l < kCoopS0Lanes computes v = P(mask) (kind 0), P(mask) - p4 (kind 1) or p3 - P(mask) (kind 2),
    # stores it as VEC item `vec` and, if x >= 0, 1 / (v.v - [kind > 0] m_t^2) as scalar item `x`
    s0 = []
    for m in range(1, 1 << N):
        s0.append((0, m, L.get("V", ("P", m)), L.idx["X"].get(("iP2", m), -1)))
    for m in range(1, 1 << N):
        if ("qX", m) in L.idx["V"]:
            s0.append((1, m, L.get("V", ("qX", m)), L.get("X", ("idX", m))))
    for m in range(1, 1 << N):
        if ("qY", m) in L.idx["V"]:
            s0.append((2, m, L.get("V", ("qY", m)), L.get("X", ("idY", m))))
    assert len(s0) <= 32
    hdr.append("constexpr int kCoopS0Lanes = %d, kCoopS0Spin0 = 30, kCoopS0Pol0 = 32, kCoopS0Beam0 = 36;   // S0 lane assignment" % len(s0))
    hdr.append("constexpr int kCoopNGF = 2, kCoopPolBits = 4;     // final-state gluons; polarisation bits of an S4 thread")
    hdr.append("MF_TABLE short kCoopS0Tab[%d][4] = {%s};   // kind, mask, vec, x" %
               (len(s0), ", ".join("{%d, %d, %d, %d}" % t for t in s0)))
    hdr.append("// static fp64 operation count per event (adds + multiplies, FMA = 2): S0 %d + S1/A/B %d + 64 x S4 %d" %
               (s0_flops, staged, s4_flops))
    hdr.append("constexpr double kFlopsMe2Coop_2g = %d.0;" % total)
    hdr.append("")
    text = "\n".join(hdr) + "\n" + LOADERS + "\n" + tables + "\n\n" + s4 + "\n"
    path = os.path.join(HERE, "mf_me_ttgg_coop_generated.cuh")
    old = open(path).read() if os.path.exists(path) else None
    if old != text:
        with open(path, "w") as f:
            f.write(text)
    return path


LOADERS = '''// Scratch items are stored as planes of double2 so that consecutive lanes reading consecutive items issue
// conflict-free 128-bit shared-memory loads: VEC plane p = components (2p, 2p+1); SPIN plane c = (re[c], im[c]).
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
// x or -x without touching the FP64 pipe (sign-bit flip)
MF_HD double mf_flip(double x, int neg) {
#if defined(__CUDA_ARCH__)
  return __hiloint2double(__double2hiint(x) ^ (neg << 31), __double2loint(x));
#else
  return neg ? -x : x;
#endif
}
// Part k (0 = real, 1 = imaginary) of row . column = sum_m r.re x_a + r.im' x_b with the row prepared by
// coop_row_part (imaginary parts negated for k = 0) and the column by coop_col_part ((re, im) swapped for k = 1).
MF_HD spin coop_row_part(spin r, int k) {
#pragma unroll
  for (int m = 0; m < 4; ++m) r.im[m] = mf_flip(r.im[m], k ^ 1);
  return r;
}
MF_HD spin coop_col_part(const spin& c, int k) {
  spin o;
#pragma unroll
  for (int m = 0; m < 4; ++m) { o.re[m] = k ? c.im[m] : c.re[m]; o.im[m] = k ? c.re[m] : c.im[m]; }
  return o;
}
MF_HD double sdot_part(const spin& r, const spin& c) {
  double acc = r.re[0] * c.re[0];
  acc = fma(r.im[0], c.im[0], acc);
#pragma unroll
  for (int m = 1; m < 4; ++m) { acc = fma(r.re[m], c.re[m], acc); acc = fma(r.im[m], c.im[m], acc); }
  return acc;
}
#if defined(__CUDA_ARCH__)
// D = A B + C on the FP64 tensor path (DMMA.884): A 8 x 4 (lane holds A[lane >> 2][lane & 3]), B 4 x 8 (B[lane & 3][lane >> 2]),
// C / D 8 x 8 (lane holds rows lane >> 2, columns 2 (lane & 3) and 2 (lane & 3) + 1).  Full FP64 rate on B200 (37.0 TFLOP/s
// measured, profiles/r2_dmma_probe.md) with one instruction per 256 FMAs and the operands read once per fragment.
__device__ __forceinline__ void coop_dmma(double& c0, double& c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// One block of the S4 spinor contraction: rows = the two spinor items (ROWBASE + rowoff + pp kSpinRow + PR0 / PR1) for the
// polarisations pp = (pa, pb) and the part k of the lane's g = lane >> 2 = (k, pa, pb); columns = the items (COLBASE + coloff
// + pp' kSpinRow + PC0 / PC1), column n = j + 2 pp'.  The inner index runs over (component c, re / im): K = 8 = two DMMA
// steps s, c = 2 s + (t & 1), part r = t >> 1, with t = lane & 3:
//   row element  = r ^ k ? im : re of the row spinor, negated for (k = 0, r = 1)     [Re: yr xr - yi xi;  Im: yi xr + yr xi]
//   column element = r ? im : re of the column spinor.
// Result c[m][j]: row item m, column item j, for the helicity (pa, pb) of g and (pc, pd) = t.
template <int ROWBASE, int COLBASE, int PR0, int PR1, int PC0, int PC1>
__device__ __forceinline__ void coop_s4_block(const double* S, int lane, int rowoff, int coloff, double (&c)[2][2]) {
  const int t = lane & 3, kb = (lane >> 2) & 1, pp = lane >> 3, r = t >> 1;
  const int plane = (t & 1) * kCoopNS;
  const int row0 = 2 * (plane + ROWBASE + rowoff + pp * kCoopSpinRow) + (r ^ kb);
  const int col = 2 * (plane + COLBASE + coloff + pp * kCoopSpinRow + (kb ? PC1 : PC0)) + r;
  const int neg = r & (kb ^ 1);
  c[0][0] = c[0][1] = c[1][0] = c[1][1] = 0.0;
#pragma unroll
  for (int s = 0; s < 2; ++s) {
    const double b = S[col + 4 * s * kCoopNS];
    coop_dmma(c[0][0], c[0][1], mf_flip(S[row0 + 2 * PR0 + 4 * s * kCoopNS], neg), b);
    coop_dmma(c[1][0], c[1][1], mf_flip(S[row0 + 2 * PR1 + 4 * s * kCoopNS], neg), b);
  }
}
#endif
'''


if __name__ == "__main__":
    print(main())
