#!/usr/bin/env python3
"""Build-time generator of the COOPERATIVE matrix element of g g -> t tbar g (one WARP per event).

Same construction as gen_coop.py (real polarisations, hatted currents, helicity recycling, spin-flip symmetry,
polarisation siblings, real / imaginary S4 threads), for three gluons and with the quark line cut after ONE gluon:

    Ahat(abc) = Ytilde(a) . Xhat(bc)  +  cR(c) . Jhat(ab)  +  c0 . Jhat(abc)
    Ytilde(a) = ubar eps_a-slash,   Xhat(bc) = prop [eps_b-slash Xhat(c) + Jhat(bc)-slash v],   Xhat(c) = prop eps_c-slash v
    cR(c) = ubar gamma^mu Xhat(c),  c0 = ubar gamma^mu v

8 gluon polarisation words x 2 antitop spins x (re, im) = 32 S4 threads = one warp, so a team is a warp and its
stages are separated by __syncwarp only.  Emits mf_me_ttg_coop_generated.cuh (a fragment included by
mf_me_coop.cuh inside namespace mf::g3).  Imports nothing from oracle/.
"""
import itertools
import os

import gen_coop as G
from gen_me import colour_matrix

HERE = os.path.dirname(os.path.abspath(__file__))
N = 3
LABELS = list(range(N))
PAIRS = list(itertools.permutations(LABELS, 2))          # ordered pairs (b, c)
PAIR_INDEX = {p: i for i, p in enumerate(PAIRS)}
SEQ2 = [s for s in itertools.permutations(LABELS, 2) if G.canon(s)[0] == s]
SEQ3 = [s for s in itertools.permutations(LABELS, 3) if G.canon(s)[0] == s]
SPIN_ROW = 7                # X2 rows of 6 ordered pairs, padded
Z_HB = 3 * 8                # z3[k][hb][seq][8 polarisation words]: hb stride
Z_PLANE = 2 * Z_HB
ROUND_OVERHEAD = 60


def build_layout():
    L = G.Layout()
    for m in range(1, 1 << N):
        L.add("V", ("P", m))
    for m in range(1, 1 << N):
        if bin(m).count("1") <= 2:
            L.add("V", ("qX", m))
    for g in LABELS:
        for p in range(2):
            L.add("V", ("eps", g, p))
    L.bases["J2"] = L.n("V")           # [polidx][seq]
    for v in range(4):
        for s in SEQ2:
            L.add("V", ("J", s, G.pol_words(s)[v]))
    L.bases["c0"] = L.n("V")
    for hb in range(2):
        for k in range(2):
            L.add("V", ("c0", hb, k))
    L.bases["cR"] = L.n("V")
    for g in LABELS:
        for hb in range(2):
            for p in range(2):
                for k in range(2):
                    L.add("V", ("cR", g, hb, p, k))
    for m in range(1, 1 << N):
        if bin(m).count("1") >= 2:
            L.add("X", ("iP2", m))
        if bin(m).count("1") <= 2:
            L.add("X", ("idX", m))
    L.add("S", ("ub",))
    for hb in range(2):
        L.add("S", ("v", hb))
    L.bases["X1"] = L.n("S")
    for hb in range(2):
        for d in LABELS:
            for p in range(2):
                L.add("S", ("X1", d, hb, p))
    L.bases["Yt"] = L.n("S")           # Ytilde(a): [a][pa]
    for a in LABELS:
        for p in range(2):
            L.add("S", ("Yt", (a,), p << a))
    L.bases["X2"] = L.n("S")           # [hb][polidx][pair, padded]
    for hb in range(2):
        for v in range(4):
            for cd in PAIRS:
                L.add("S", ("X2", cd, hb, G.pol_words(cd)[v]))
            for i in range(SPIN_ROW - len(PAIRS)):
                L.add("S", ("pad", "X2", hb, v, i))
    return L


def z3_index(seq, pols):
    return SEQ3.index(seq) * 8 + pols      # hb = 0, k = 0


def task_Yt1(L, a, p):
    return dict(fam="Yt1", M=1, flops=G.F_SLASH,
                fields=[L.get("S", ("Yt", (a,), p << a)), L.get("S", ("ub",)), G.J_ref(L, (a,), p << a)[0]])


def task_J3z(L, s, pw):
    """z3 = c0 . J3(abc) for one polarisation word"""
    a, b, c = s
    j2bc = G.J_ref(L, (b, c), pw)
    j2ab = G.J_ref(L, (a, b), pw)
    signs = (1 if j2bc[1] < 0 else 0) | (2 if j2ab[1] < 0 else 0)
    f = [z3_index(s, pw), L.get("X", ("iP2", G.mask_of(s))), G.J_ref(L, (a,), pw)[0], G.P_ref(L, (a,)),
         j2bc[0], G.P_ref(L, (b, c)), j2ab[0], G.P_ref(L, (a, b)), G.J_ref(L, (c,), pw)[0], G.P_ref(L, (c,)),
         G.J_ref(L, (b,), pw)[0], signs, L.get("V", ("c0", 0, 0))]
    fl = 2 * (7 * 3 + 2 + 4 + 24) + 7 * 3 + 25 + 16 + 28
    return dict(fam="J3z", M=1, fields=f, flops=fl)


def build_program(L):
    """the single warp's program: phases S1 (J2, X1 + cR, Ytilde) and A (X2, z3)"""
    def rounds_of(tasks):
        return [tasks[i:i + 32] for i in range(0, len(tasks), 32)]

    s1 = []
    s1 += rounds_of([G.task_J2(L, s, pw) for s in SEQ2 for pw in G.pol_words(s)])
    s1 += rounds_of([G.task_X1c(L, d, hb, p) for hb in range(2) for d in LABELS for p in range(2)])
    s1 += rounds_of([task_Yt1(L, a, p) for a in LABELS for p in range(2)])
    a = []
    a += rounds_of([G.task_X2(L, cd, hb, pd, 2) for hb in range(2) for pd in range(2) for cd in PAIRS])
    a += rounds_of([task_J3z(L, s, pw) for s in SEQ3 for pw in range(8)])
    return [s1, a]


NAMES = {"J2": "CoopTaskJ2", "X1c": "CoopTaskX1c", "Yt1": "CoopTaskYt1", "X2": "CoopTaskX2<%d>", "J3z": "CoopTaskJ3z<%d>"}


def emit_tables(phases):
    o, words, prog = [], [], []
    w = o.append
    for rounds in phases:
        for tasks in rounds:
            nf = max(len(t["fields"]) for t in tasks)
            nvec = (nf + 7) // 8
            off = len(words) // 8
            for v in range(nvec):
                for lane in range(32):
                    f = list(tasks[lane]["fields"]) if lane < len(tasks) else [-1]
                    f += [0] * (nvec * 8 - len(f))
                    words.extend(f[8 * v:8 * v + 8])
            nm = NAMES[tasks[0]["fam"]]
            prog.append("R(%d, %s)" % (off, nm % tasks[0]["M"] if "%" in nm else nm))
        prog.append("S()")
    w("constexpr int kCoopPhases = %d, kCoopWarps = 1;" % len(phases))
    w("// the program of the team's warp: R(table offset in 16-byte vectors, task type) = one round of <= 32 lane-tasks,")
    w("// S() = end of a phase (__syncwarp)")
    w("#define MF_COOP3_WARP0(R, S) \\")
    w("  " + " \\\n  ".join(prog))
    w("#define MF_COOP3_WARP1(R, S)")
    assert max(words) < 32768 and min(words) >= -1 and len(words) % 8 == 0
    w("constexpr int kCoopTableVecs = %d;" % (len(words) // 8))
    w("__align__(16) MF_TABLE short kCoopTable[%d] = {" % len(words))
    for i in range(0, len(words), 32):
        w("  " + ", ".join("%d" % v for v in words[i:i + 32]) + ",")
    w("};")
    return "\n".join(o)


def pair_name(a, b):
    return "pp%d%d" % (min(a, b), max(a, b))


def emit_s4(L):
    perms, Cnum, Cden = colour_matrix(N)
    o = []
    w = o.append
    flops = 0
    w("// S4: thread (pols, hb, k) forms the real (k = 0) or imaginary (k = 1) parts of its %d colour-ordered amplitudes" % len(perms))
    w("// and contracts them with the colour matrix: returns sum_{s,s'} x_s Cnum_{ss'} x_s' (the caller divides by kCoopCden).")
    w("MF_HD double coop_s4(const double* V, const double* S, const double* Z, int pols, int hb, int k) {")
    for g in LABELS:
        w("  const int ps%d = (pols >> %d) & 1;" % (g, g))
    for a, b in itertools.combinations(LABELS, 2):
        w("  const int %s = ps%d | (ps%d << 1);" % (pair_name(a, b), a, b))
    w("  const double* Zk = Z + k * %d + hb * %d + pols;" % (Z_PLANE, Z_HB))
    w("  double " + ", ".join("A%d%d%d" % p for p in perms) + ";")
    # term 1: Ytilde(a) . Xhat(bc)
    w("  {")
    for a in LABELS:
        w("    const spin yt%d = coop_row_part(coop_ld_spin(S, %d + %d + ps%d), k);" % (a, L.bases["Yt"], 2 * a, a))
    for (b, c) in PAIRS:
        a = [g for g in LABELS if g not in (b, c)][0]
        w("    A%d%d%d = sdot_part(yt%d, coop_col_part(coop_ld_spin(S, %d + (hb * 4 + %s) * %d + %d), k));" %
          (a, b, c, a, L.bases["X2"], pair_name(b, c), SPIN_ROW, PAIR_INDEX[(b, c)]))
        flops += 15
    w("  }")
    # term 2: cR(c) . J2(ab), antisymmetric in (a, b)
    for c in LABELS:
        a, b = [g for g in LABELS if g != c]
        w("  { const double z = rdot(coop_ld_vec(V, %d + ((%d * 2 + hb) * 2 + ps%d) * 2 + k), coop_ld_vec(V, %d + %s * %d + %d));" %
          (L.bases["cR"], c, c, L.bases["J2"], pair_name(a, b), len(SEQ2), SEQ2.index((a, b))))
        w("    A%d%d%d += z; A%d%d%d -= z; }" % (a, b, c, b, a, c))
        flops += 7 + 2
    # term 3: z3 = c0 . J3(abc); J3(cba) = + J3(abc)
    for i, s in enumerate(SEQ3):
        r = s[::-1]
        w("  { const double z = Zk[%d]; A%d%d%d += z; A%d%d%d += z; }" % ((i * 8,) + s + r))
        flops += 2
    # colour contraction, row by row with literal coefficients, four independent accumulators
    w("  double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;")
    for i in range(len(perms)):
        terms = [(j, int(Cnum[i][j]) * (1 if i == j else 2)) for j in range(i, len(perms)) if Cnum[i][j]]
        expr = "%.1f * A%d%d%d" % ((float(terms[0][1]),) + perms[terms[0][0]])
        flops += 1
        for j, v in terms[1:]:
            expr = "fma(%.1f, A%d%d%d, %s)" % ((float(v),) + perms[j] + (expr,))
            flops += 2
        w("  acc%d = fma(A%d%d%d, %s, acc%d);" % ((i % 4,) + perms[i] + (expr, i % 4)))
        flops += 2
    w("  return (acc0 + acc1) + (acc2 + acc3);")
    flops += 3
    w("}")
    w("// team thread tid = pols | hb << kCoopPolBits | k << (kCoopPolBits + 1)")
    w("MF_HD double coop_s4_tid(const double* V, const double* S, const double* Z, int tid) {")
    w("  return coop_s4(V, S, Z, tid & %d, (tid >> %d) & 1, (tid >> %d) & 1);" % ((1 << N) - 1, N, N + 1))
    w("}")
    return "\n".join(o), Cden, flops


def main():
    L = build_layout()
    phases = build_program(L)
    s4, Cden, s4_flops = emit_s4(L)
    tables = emit_tables(phases)
    staged = sum(t["flops"] for rounds in phases for tasks in rounds for t in tasks)
    s0_flops = 13 * 30 + 250
    total = s0_flops + staged + 32 * s4_flops
    s0 = []
    for m in range(1, 1 << N):
        s0.append((0, m, L.get("V", ("P", m)), L.idx["X"].get(("iP2", m), -1)))
    for m in range(1, 1 << N):
        if ("qX", m) in L.idx["V"]:
            s0.append((1, m, L.get("V", ("qX", m)), L.get("X", ("idX", m))))
    hdr = ["// GENERATED by gen_coop3.py — do not edit.  Cooperative (one warp per event) matrix element of",
           "// g g -> t tbar g: scratch layout, task tables of phases S1 / A, straight-line stage S4.",
           "// A FRAGMENT: included by mf_me_coop.cuh inside namespace mf::g3 (no include guard, no namespace of its own).",
           "",
           "// scratch layout (doubles): VEC 4*kCoopNV | SPIN 8*kCoopNS | Z 2*kCoopZPlane | SCAL kCoopNX",
           "// kCoopZRow = the hb stride of the z3 array; kCoopJ2Stride is unused here (the z5 tasks do not exist)",
           "constexpr int kCoopNV = %d, kCoopNS = %d, kCoopZPlane = %d, kCoopZRow = %d, kCoopNX = %d, kCoopJ2Stride = %d;" %
           (L.n("V"), L.n("S"), Z_PLANE, Z_HB, L.n("X") + (L.n("X") & 1), len(SEQ2)),
           "constexpr int kCoopScratchDoubles = 4 * kCoopNV + 8 * kCoopNS + 2 * kCoopZPlane + kCoopNX;",
           "constexpr double kCoopCden = %.1f;" % Cden,
           "constexpr int kCoopP0 = %d, kCoopEps0 = %d, kCoopC0 = %d;" %
           (L.get("V", ("P", 1)), L.get("V", ("eps", 0, 0)), L.get("V", ("c0", 0, 0))),
           "constexpr int kCoopUb = %d, kCoopV0 = %d;" % (L.get("S", ("ub",)), L.get("S", ("v", 0))),
           "constexpr int kCoopS0Lanes = %d, kCoopS0Spin0 = 14, kCoopS0Pol0 = 16, kCoopS0Beam0 = 20;   // S0 lane assignment" % len(s0),
           "constexpr int kCoopNGF = 1, kCoopPolBits = 3;     // final-state gluons; polarisation bits of an S4 thread",
           "MF_TABLE short kCoopS0Tab[%d][4] = {%s};   // kind, mask, vec, x" %
           (len(s0), ", ".join("{%d, %d, %d, %d}" % t for t in s0)),
           "// static fp64 operation count per event (adds + multiplies, FMA = 2): S0 %d + S1/A %d + 32 x S4 %d" %
           (s0_flops, staged, s4_flops),
           "constexpr double kFlopsMe2Coop_1g = %d.0;" % total, ""]
    assert len(s0) <= 14
    text = "\n".join(hdr) + "\n" + G.LOADERS + "\n" + tables + "\n\n" + s4 + "\n"
    path = os.path.join(HERE, "mf_me_ttg_coop_generated.cuh")
    old = open(path).read() if os.path.exists(path) else None
    if old != text:
        with open(path, "w") as f:
            f.write(text)
    return path


if __name__ == "__main__":
    print(main())
