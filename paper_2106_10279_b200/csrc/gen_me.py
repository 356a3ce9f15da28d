#!/usr/bin/env python3
"""Build-time generator of the straight-line matrix-element code for g g -> t tbar + (n-2) g, n = 2, 3, 4.

It plays the role of the paper's exporter plugin (MG5_aMC writes one Matrix class and
its ALOHA routines per process): it unrolls the colour-ordered recursion (R10) for a fixed
process into calls to the primitives of mf_me_prims.cuh, sharing every sub-current between the n! colour
orderings, and folds the exact colour matrix (R11) into the code.

    python gen_me.py            # writes mf_me_ggtt_generated.cuh next to this file

Decomposition used (n gluons, labels 0,1 = beams, 2.. = final; all gluon momenta incoming):

    Ahat(sigma) = Ytilde(sigma[:p]) . Xhat(sigma[p:])
                + sum_{a<p, b>p} c(sigma[:a], sigma[b:]) . Jhat(sigma[a:b])        p = n // 2
    Jhat(seq)   = [ -sum_j V3(Jhat(seq[:j]), Jhat(seq[j:])) + sum_{j<l} V4(...) ] / P_seq^2     (real vectors)
    Xhat(seq)   = -(qslash+m)/(q^2-m^2) sum_j Jhat-slash(seq[:j]) Xhat(seq[j:]),  q = P_seq - p4, Xhat() = v
    Yhat(seq)   = -[sum_j Yhat(seq[:j]) Jhat-slash(seq[j:])] (qslash+m)/(q^2-m^2), q = p3 - P_seq, Yhat() = ubar
    Ytilde      = the same sum without the trailing propagator
    c(L, R)^mu  = Yhat(L) gamma^mu Xhat(R)

i.e. the quark line is cut between positions p and p+1: orderings where a propagator sits there factorise
into a left row current times a right column current; in all others one gluon current bridges the cut and
is contracted with a fermion bilinear.  Reflection J(reversed) = (-1)^(k+1) J halves the gluon currents.
This module imports nothing from oracle/ and the oracle does not use its output.
"""
import itertools
import math
import os
from fractions import Fraction

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))


# ----------------------------------------------------------------------------------------------------
# colour matrix C_{sigma sigma'} = sum_a Tr(T^{a_s1}..T^{a_sn} (T^{a_s'1}..T^{a_s'n})^dagger), exact rationals
def gell_mann_half():
    l = np.zeros((8, 3, 3), dtype=complex)
    l[0][0, 1] = l[0][1, 0] = 1
    l[1][0, 1] = -1j; l[1][1, 0] = 1j
    l[2][0, 0] = 1; l[2][1, 1] = -1
    l[3][0, 2] = l[3][2, 0] = 1
    l[4][0, 2] = -1j; l[4][2, 0] = 1j
    l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2] = -1j; l[6][2, 1] = 1j
    l[7][0, 0] = l[7][1, 1] = 1 / math.sqrt(3); l[7][2, 2] = -2 / math.sqrt(3)
    return l / 2


def colour_matrix(n):
    """n! x n! integer numerators and the common denominator (3^(n-1) * 2 for n = 4, ...)."""
    T = gell_mann_half()
    perms = list(itertools.permutations(range(n)))
    # chains[s][a_0..a_{n-1}] = T^{a_{s0}} ... T^{a_{s,n-1}}, flattened over the colour assignment
    vecs = []
    for s in perms:
        M = None
        for pos in range(n):
            g = s[pos]
            shape = [1] * n
            shape[g] = 8
            Tg = T.reshape(shape + [3, 3])
            M = Tg if M is None else np.einsum('...ij,...jk->...ik', M, Tg)
        M = np.broadcast_to(M, [8] * n + [3, 3])
        vecs.append(M.reshape(-1))
    V = np.stack(vecs)
    C = (V @ V.conj().T).real
    den = 2 * 3 ** (n - 1)
    num = np.rint(C * den).astype(int)
    assert np.abs(C * den - num).max() < 1e-9, "colour matrix is not a multiple of 1/%d" % den
    g = 0
    for v in num.flatten():
        g = math.gcd(g, int(v))
    g = math.gcd(g, den)
    return perms, num // g, den // g


# ----------------------------------------------------------------------------------------------------
# fp64 operations (adds + multiplies as written; an FMA counts 2) of each primitive of mf_me_prims.cuh
FLOPS = {"rdot": 7, "radd": 4, "rsub": 4, "rscale": 4, "v3_acc": 53, "v4_acc": 49, "slash_col": 42, "slash_row": 42,
         "spin_acc": 8, "prop_col": 66, "prop_row": 66, "sdot": 30, "bilinear": 72, "cdot_r": 14}


def count_flops(line):
    """static operation count of one emitted source line"""
    import re
    n = sum(FLOPS[f] * len(re.findall(r"\b%s\(" % f, line)) for f in FLOPS)
    if line.lstrip().startswith(("const double Ar", "const double Ai")):
        n += line.count(" + ") + line.count(" - ")          # amplitude = signed sum of terms
    if line.lstrip().startswith(("g =", "g +=")):
        n += 3 + (1 if "+=" in line else 0)                  # Ar*Ar + Ai*Ai (+ accumulate)
    if "acc +=" in line or "total +=" in line:
        n += 2 if "*" in line else 1
    return n


class Emitter:
    def __init__(self, n):
        self.n = n
        self.p = n // 2
        self.lines = []
        self.done = set()

    def emit(self, s):
        self.lines.append(s)

    @staticmethod
    def mask(seq):
        m = 0
        for g in seq:
            m |= 1 << g
        return m

    def P(self, seq):
        return "Pg[%d]" % seq[0] if len(seq) == 1 else "P_%d" % self.mask(seq)

    # ---- gluon currents (real) --------------------------------------------------------------------
    def J(self, seq):
        """(name, sign) of Jhat(seq), emitting its computation on first use."""
        seq = tuple(seq)
        k = len(seq)
        if k == 1:
            return "e%d" % seq[0], 1
        sign = 1
        if seq[0] > seq[-1]:
            seq = seq[::-1]
            sign = (-1) ** (k + 1)
        name = "J_" + "".join(map(str, seq))
        if name not in self.done:
            self.done.add(name)
            parts = []
            for j in range(1, k):
                a, sa = self.J(seq[:j])
                b, sb = self.J(seq[j:])
                parts.append("v3_acc(%s, %s, %s, %s, %s, %s);" % (name, "%+.1f" % (-sa * sb), a, self.P(seq[:j]), b,
                                                                  self.P(seq[j:])))
            for j in range(1, k):
                for l in range(j + 1, k):
                    a, sa = self.J(seq[:j])
                    b, sb = self.J(seq[j:l])
                    c, sc = self.J(seq[l:])
                    parts.append("v4_acc(%s, %s, %s, %s, %s);" % (name, "%+.1f" % (sa * sb * sc), a, b, c))
            self.emit("rvec %s = {{0.0, 0.0, 0.0, 0.0}};" % name)
            for s in parts:
                self.emit(s)
            self.emit("%s = rscale(%s, iP2_%d);" % (name, name, self.mask(seq)))
        return name, sign

    # ---- quark currents ---------------------------------------------------------------------------
    def X(self, seq, hb):
        """propagated column current Xhat(seq) for tbar spin hb"""
        seq = tuple(seq)
        if not seq:
            return "vv[%d]" % hb
        name = "X_%s_%d" % ("".join(map(str, seq)), hb)
        if name not in self.done:
            self.done.add(name)
            k = len(seq)
            terms = []
            for j in range(1, k + 1):
                jn, js = self.J(seq[:j])
                xn = self.X(seq[j:], hb)
                terms.append((jn, js, xn))
            self.emit("spin %s;" % name)
            self.emit("{")
            for i, (jn, js, xn) in enumerate(terms):
                arg = jn if js > 0 else "rscale(%s, -1.0)" % jn
                if i == 0:
                    self.emit("  spin t = slash_col(%s, %s);" % (arg, xn))
                else:
                    self.emit("  spin_acc(t, slash_col(%s, %s));" % (arg, xn))
            m = self.mask(seq)
            self.emit("  %s = prop_col(qX_%d, mt, idX_%d, t);" % (name, m, m))
            self.emit("}")
        return name

    def Yt(self, seq, h):
        """unpropagated row current Ytilde(seq) for t spin h"""
        seq = tuple(seq)
        name = "Yt_%s_%d" % ("".join(map(str, seq)), h)
        if name not in self.done:
            self.done.add(name)
            k = len(seq)
            terms = []
            for j in range(0, k):
                yn = self.Y(seq[:j], h)
                jn, js = self.J(seq[j:])
                terms.append((yn, jn, js))
            self.emit("spin %s;" % name)
            self.emit("{")
            for i, (yn, jn, js) in enumerate(terms):
                arg = jn if js > 0 else "rscale(%s, -1.0)" % jn
                if i == 0:
                    self.emit("  %s = slash_row(%s, %s);" % (name, yn, arg))
                else:
                    self.emit("  spin_acc(%s, slash_row(%s, %s));" % (name, yn, arg))
            self.emit("}")
        return name

    def Y(self, seq, h):
        """propagated row current Yhat(seq) for t spin h"""
        seq = tuple(seq)
        if not seq:
            return "ub[%d]" % h
        name = "Y_%s_%d" % ("".join(map(str, seq)), h)
        if name not in self.done:
            self.done.add(name)
            yt = self.Yt(seq, h)
            m = self.mask(seq)
            self.emit("spin %s = prop_row(%s, qY_%d, mt, idY_%d);" % (name, yt, m, m))
        return name

    def cbil(self, L, R, h, hb):
        name = "c_%s_%s_%d%d" % ("".join(map(str, L)) or "n", "".join(map(str, R)) or "n", h, hb)
        if name not in self.done:
            self.done.add(name)
            self.emit("cvec %s = bilinear(%s, %s);" % (name, self.Y(L, h), self.X(R, hb)))
        return name

    def cJ(self, L, R, mid, h, hb):
        """(name, sign) of the scalar c(L,R).Jhat(mid), shared between orderings"""
        jn, js = self.J(mid)
        cn = self.cbil(L, R, h, hb)
        name = "d_%s_%s" % (cn[2:], jn)
        if name not in self.done:
            self.done.add(name)
            self.emit("cplx %s = cdot_r(%s, %s);" % (name, cn, jn))
        return name, js

    def amplitude(self, sigma, h, hb):
        n, p = self.n, self.p
        terms = []
        yt = self.Yt(sigma[:p], h)
        x = self.X(sigma[p:], hb)
        nm = "s_%s_%d%d" % ("".join(map(str, sigma)), h, hb)
        self.emit("cplx %s = sdot(%s, %s);" % (nm, yt, x))
        terms.append((nm, 1))
        for a in range(0, p):
            for b in range(p + 1, n + 1):
                terms.append(self.cJ(sigma[:a], sigma[b:], sigma[a:b], h, hb))
        re = " ".join("%s %s.re" % ("+" if s > 0 else "-", t) for t, s in terms)
        im = " ".join("%s %s.im" % ("+" if s > 0 else "-", t) for t, s in terms)
        return re, im


def generate(n):
    perms, Cnum, Cden = colour_matrix(n)
    np_ = len(perms)
    E = Emitter(n)
    out = []
    w = out.append
    w("// g g -> t tbar + %d g: %d colour orderings, colour matrix = integers / %d" % (n - 2, np_, Cden))
    w("// Returns sum over gluon polarisations and quark spins of Ahat^dagger C Ahat (no couplings, no averaging).")
    w("MF_HD double me2_ggtt_%dg(const rvec* Pg, const rvec (*eps)[2], const spin* ub, const spin* vv, "
      "const rvec& p3, const rvec& p4, double mt) {" % (n - 2))
    w("  const double mt2 = mt * mt;")
    # momentum sums and propagator denominators (helicity independent)
    full = (1 << n) - 1
    for m in range(1, full + 1):
        gl = [g for g in range(n) if m >> g & 1]
        if len(gl) >= 2:
            w("  const rvec P_%d = radd(%s, Pg[%d]);" % (m, E.P(gl[:-1]), gl[-1]))
            w("  const double iP2_%d = 1.0 / rdot(P_%d, P_%d);" % (m, m, m))
    p = E.p
    for m in range(1, full):
        gl = [g for g in range(n) if m >> g & 1]
        if len(gl) <= n - p:
            w("  const rvec qX_%d = rsub(%s, p4);" % (m, E.P(gl)))
            w("  const double idX_%d = 1.0 / (rdot(qX_%d, qX_%d) - mt2);" % (m, m, m))
        if len(gl) <= p - 1:
            w("  const rvec qY_%d = rsub(p3, %s);" % (m, E.P(gl)))
            w("  const double idY_%d = 1.0 / (rdot(qY_%d, qY_%d) - mt2);" % (m, m, m))
    w("  double total = 0.0;")
    w("#pragma unroll 1")
    w("  for (int gh = 0; gh < %d; ++gh) {" % (1 << n))
    for g in range(n):
        w("    const rvec e%d = eps[%d][(gh >> %d) & 1];" % (g, g, g))
    # body
    # quark spins: only the top spin state 0 (both antitop states); flipping BOTH spins conjugates every colour-ordered
    # amplitude up to a common phase when the gluon polarisation vectors are real (gen_coop.py), so the other
    # half of the spin sum equals this one: the result is doubled below
    for hb in range(2):
        for h in range(1):
            amps = []
            for s in perms:
                re, im = E.amplitude(s, h, hb)
                amps.append((re, im))
            for i, (re, im) in enumerate(amps):
                E.emit("const double Ar%d_%d%d = %s;" % (i, h, hb, re))
                E.emit("const double Ai%d_%d%d = %s;" % (i, h, hb, im))
            # colour contraction grouped by distinct matrix entry
            groups = {}
            for i in range(np_):
                for j in range(i, np_):
                    v = int(Cnum[i, j]) * (1 if i == j else 2)
                    if v:
                        groups.setdefault(v, []).append((i, j))
            E.emit("{")
            E.emit("  double acc = 0.0, g;")
            for v in sorted(groups):
                first = True
                for (i, j) in groups[v]:
                    t = "Ar%d_%d%d * Ar%d_%d%d + Ai%d_%d%d * Ai%d_%d%d" % (i, h, hb, j, h, hb, i, h, hb, j, h, hb)
                    E.emit("  g %s %s;" % ("=" if first else "+=", t))
                    first = False
                E.emit("  acc += %.1f * g;" % v)
            E.emit("  total += acc;")
            E.emit("}")
    pre = sum(count_flops(l) for l in out) + 1 * sum(l.count("1.0 /") for l in out)
    body = sum(count_flops(l) for l in E.lines)
    flops = pre + (1 << n) * body
    for l in E.lines:
        w("    " + l)
    w("  }")
    w("  return total * (2.0 / %.1f);   // x 2: spin-flip symmetry, only top spin 0 was summed" % Cden)
    w("}")
    w("// static fp64 operation count of the code above (adds + multiplies as written, FMA = 2; divisions = 1):")
    w("//   per event %d = preamble %d + %d polarisation combinations x %d" % (flops, pre, 1 << n, body))
    w("constexpr double kFlopsMe2_%dg = %d.0;" % (n - 2, flops))
    return "\n".join(out)


def main():
    hdr = ['// GENERATED by gen_me.py — do not edit.  Straight-line colour-ordered matrix elements (steps a8, a9).',
           '#pragma once', '#include "mf_me_prims.cuh"', '', 'namespace mf {', '']
    body = [generate(n) + "\n" for n in (2, 3, 4)]
    text = "\n".join(hdr + body + ['}  // namespace mf', ''])
    path = os.path.join(HERE, "mf_me_ggtt_generated.cuh")
    old = open(path).read() if os.path.exists(path) else None
    if old != text:
        with open(path, "w") as f:
            f.write(text)
    return path


if __name__ == "__main__":
    print(main())
