// mf_me_qqttgg.cuh — |M|^2 of q qbar -> t tbar g g, the quark channel of pp -> ttbar gg (PAPER.md L101 and
// Table 1: 267 diagrams = 123 of g g -> t tbar g g + 36 for each of four massless flavours).  Used by the fused pass of
// MF_PP_TTGG (mf_kernels_coop.cuh, R22) and by mf_debug_me2_qq_ttgg.
//
// Conventions of mf_me_prims.cuh (chiral two-component spinors, z-axis spin states for the top, helicity = chirality states for
// the massless line, REAL linear gluon polarisations, all factors of i and g pulled out: M = i g^4 sum_s a_s S_s).
// Formulation: currents, not diagrams.  Each quark line (light: column u(p1), row vbar(p2); top: column v(p4), row ubar(p3))
// gives 13 vector currents  row-chain gamma^mu column-chain  with zero, one or both gluons (or their three-gluon merger G)
// attached on either side of the vertex x where the virtual gluon leaves; strings are read from the row to the column:
//    0: x     1: x a   2: a x   3: x b   4: b x     5: x a b   6: x b a   7: a x b   8: b x a   9: a b x   10: b a x
//   11: x G  12: G x
// The amplitude is the contraction of a light-line with a top-line current over the virtual gluon (24 terms), the same with one
// gluon on the virtual gluon (three-gluon vertex, 8 terms) and with both on it (two chains, the merger, the four-gluon vertex).
// Colour: f^{abc} T^c = -i [T^a, T^b] turns every term into the 20 string tensors listed in gen_qq_colour.py (0..5: light x,
// top S; 6..11: light S, top x; 12..19: one gluon on each line); the colour-summed square is the generated reduced quadratic
// form of rank 11.  Derivation of the relative factors: DESIGN.md "q qbar -> t tbar g g".
#pragma once
#include "mf_me_qttg.cuh"


namespace mf {

// propagator momenta and inverse denominators of one quark line (flow momentum pc into the column end, pr out of the row end)
struct QQLineKin {
  rvec qa, qb, qab, ra, rb, rab;
  double ia, ib, iab, ja, jb, jab, m;
};
MF_HD QQLineKin qq_line_kin(const rvec& pc, const rvec& pr, const rvec& ka, const rvec& kb, double m) {
  QQLineKin k;
  k.m = m;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    k.qa.v[i] = pc.v[i] - ka.v[i];
    k.qb.v[i] = pc.v[i] - kb.v[i];
    k.qab.v[i] = pc.v[i] - ka.v[i] - kb.v[i];
    k.ra.v[i] = pr.v[i] + ka.v[i];
    k.rb.v[i] = pr.v[i] + kb.v[i];
    k.rab.v[i] = pr.v[i] + ka.v[i] + kb.v[i];
  }
  const double m2 = m * m;
  k.ia = 1.0 / (rdot(k.qa, k.qa) - m2);
  k.ib = 1.0 / (rdot(k.qb, k.qb) - m2);
  k.iab = 1.0 / (rdot(k.qab, k.qab) - m2);
  k.ja = 1.0 / (rdot(k.ra, k.ra) - m2);
  k.jb = 1.0 / (rdot(k.rb, k.rb) - m2);
  k.jab = 1.0 / (rdot(k.rab, k.rab) - m2);
  return k;
}
// the 13 hatted currents of a line for polarisations ea, eb and the hatted merger G
MF_HD void qq_line_currents(const spin& row, const spin& col, const QQLineKin& k, const rvec& ea, const rvec& eb, const rvec& G,
                            cvec J[13]) {
  const spin ca = prop_col(k.qa, k.m, k.ia, slash_col(ea, col));
  const spin cb = prop_col(k.qb, k.m, k.ib, slash_col(eb, col));
  const spin ra = prop_row(slash_row(row, ea), k.ra, k.m, k.ja);
  const spin rb = prop_row(slash_row(row, eb), k.rb, k.m, k.jb);
  J[0] = bilinear(row, col);
  J[1] = bilinear(row, ca);
  J[2] = bilinear(ra, col);
  J[3] = bilinear(row, cb);
  J[4] = bilinear(rb, col);
  J[5] = bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(ea, cb)));    // x a b: b is met first coming from the column
  J[6] = bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(eb, ca)));    // x b a
  J[7] = bilinear(ra, cb);                                                 // a x b
  J[8] = bilinear(rb, ca);                                                 // b x a
  J[9] = bilinear(prop_row(slash_row(ra, eb), k.rab, k.m, k.jab), col);    // a b x: a next to the row spinor
  J[10] = bilinear(prop_row(slash_row(rb, ea), k.rab, k.m, k.jab), col);   // b a x
  J[11] = bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(G, col)));   // x G
  J[12] = bilinear(prop_row(slash_row(row, G), k.rab, k.m, k.jab), col);   // G x
}

MF_HD cplx cmul(const cplx& a, const cplx& b) { return cplx{a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re}; }
MF_HD void cacc(cplx& o, double s, const cplx& a) { o.re = fma(s, a.re, o.re); o.im = fma(s, a.im, o.im); }
// three-gluon vertex with a complex first leg (J1, incoming momentum P1) and a real second leg (E, P2):
//   V3^r = (J1.E)(P1 - P2)^r + E^r ((P1 + 2 P2).J1) - J1^r ((2 P1 + P2).E)
MF_HD cvec v3c_vec(const cvec& J1, const rvec& P1, const rvec& E, const rvec& P2) {
  rvec d, s1, s2;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    d.v[m] = P1.v[m] - P2.v[m];
    s1.v[m] = P1.v[m] + 2.0 * P2.v[m];
    s2.v[m] = 2.0 * P1.v[m] + P2.v[m];
  }
  const cplx je = cdot_r(J1, E), pj = cdot_r(J1, s1);
  const double pe = rdot(s2, E);
  cvec o;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    o.re[m] = je.re * d.v[m] + E.v[m] * pj.re - J1.re[m] * pe;
    o.im[m] = je.im * d.v[m] + E.v[m] * pj.im - J1.im[m] * pe;
  }
  return o;
}

// the 20 string coefficients a_s for one helicity configuration.  L: the 13 light-line currents (memory); the top line's
// currents are formed one after the other from its chains and contracted at once (never stored: the live set is what limits
// this thread-per-event code).
struct QQKin {
  rvec PL0, PLa, PLb, mka, mkb, K;       // virtual-gluon momenta leaving the light line (nothing / a / b attached to it), -ka, -kb, -(ka+kb)
  double iA, iB, iCa, iCb;               // 1/PL0^2, 1/(p3+p4)^2, 1/PLa^2, 1/PLb^2
};
MF_HD cplx cscale(const cplx& a, double s) { return cplx{a.re * s, a.im * s}; }
MF_HD void qq_assemble(const cvec L[13], const spin& row, const spin& col, const QQLineKin& k, const rvec& ea, const rvec& eb,
                       const rvec& G, const QQKin& q, cplx a[20]) {
  const spin ca = prop_col(k.qa, k.m, k.ia, slash_col(ea, col));
  const spin cb = prop_col(k.qb, k.m, k.ib, slash_col(eb, col));
  const spin ra = prop_row(slash_row(row, ea), k.ra, k.m, k.ja);
  const spin rb = prop_row(slash_row(row, eb), k.rb, k.m, k.jb);
  const cvec L0 = L[0];
  // (I) nothing on the virtual gluon: one term per tensor, plus the merged pair on either line ([T^b, T^a] in its place)
  {
    const cvec T0 = bilinear(row, col);
#pragma unroll
    for (int i = 0; i < 6; ++i) a[6 + i] = cscale(cdot_c(L[5 + i], T0), q.iB);
    const cplx m3 = cdot_c(L[11], T0), m4 = cdot_c(L[12], T0);
    cacc(a[7], q.iB, m3);  cacc(a[6], -q.iB, m3);       // G x on the light line -> b a x - a b x ... (x G: x b a - x a b)
    cacc(a[11], q.iB, m4); cacc(a[10], -q.iB, m4);
    // (II) gluon g on the virtual gluon, the other one on the light line: top string x -> g x - x g
    const double eA = q.iCb * q.iB, eB = q.iCa * q.iB;
    const cplx u1 = cdot_c(v3c_vec(L[3], q.PLb, ea, q.mka), T0), u2 = cdot_c(v3c_vec(L[4], q.PLb, ea, q.mka), T0);
    const cplx u3 = cdot_c(v3c_vec(L[1], q.PLa, eb, q.mkb), T0), u4 = cdot_c(v3c_vec(L[2], q.PLa, eb, q.mkb), T0);
    a[12] = cscale(u3, -eB); a[13] = cscale(u3, eB); a[14] = cscale(u4, -eB); a[15] = cscale(u4, eB);
    a[16] = cscale(u1, -eA); a[17] = cscale(u1, eA); a[18] = cscale(u2, -eA); a[19] = cscale(u2, eA);
    // (III) both on the virtual gluon: a then b, b then a, the merged pair, the four-gluon vertex
    const cvec Wa = v3c_vec(L0, q.PL0, ea, q.mka), Wb = v3c_vec(L0, q.PL0, eb, q.mkb);
    const double d3 = q.iA * q.iB;
    const cplx l0t0 = cdot_c(L0, T0), lea = cdot_r(L0, ea), leb = cdot_r(L0, eb), tea = cdot_r(T0, ea), teb = cdot_r(T0, eb);
    const double eab = rdot(ea, eb);
    const cplx sab = cdot_c(v3c_vec(Wa, q.PLa, eb, q.mkb), T0), sba = cdot_c(v3c_vec(Wb, q.PLb, ea, q.mka), T0);
    const cplx sG = cdot_c(v3c_vec(L0, q.PL0, G, q.K), T0);
    const cplx v0 = cmul(leb, tea), v1 = cmul(lea, teb);
    // [T^b,[T^a,T^x]] = b a x - b x a - a x b + x a b   carries  s_ab / PLa^2 + (L.eb)(ea.T) - (ea.eb)(L.T)
    // [T^a,[T^b,T^x]] = a b x - a x b - b x a + x b a   carries  s_ba / PLb^2 + (L.ea)(eb.T) - (ea.eb)(L.T)
    // [[T^b,T^a],T^x] = b a x - a b x - x b a + x a b   carries  s_G - [(L.ea)(eb.T) - (L.eb)(ea.T)]
    const cplx A = {d3 * (sab.re * q.iCa + v0.re - eab * l0t0.re), d3 * (sab.im * q.iCa + v0.im - eab * l0t0.im)};
    const cplx B = {d3 * (sba.re * q.iCb + v1.re - eab * l0t0.re), d3 * (sba.im * q.iCb + v1.im - eab * l0t0.im)};
    const cplx C = {d3 * (sG.re - (v1.re - v0.re)), d3 * (sG.im - (v1.im - v0.im))};
    a[0] = cplx{A.re + C.re, A.im + C.im};
    a[1] = cplx{B.re - C.re, B.im - C.im};
    a[2] = cplx{-A.re - B.re, -A.im - B.im};
    a[3] = a[2];
    a[4] = cplx{B.re - C.re, B.im - C.im};
    a[5] = cplx{A.re + C.re, A.im + C.im};
    // (II) gluon g on the virtual gluon (T^x -> [T^g, T^x] on the top line), the other one on the top line
    const double dA = q.iA * q.iCa, dB = q.iA * q.iCb;
    {
      const cvec T3 = bilinear(row, cb);                                   // x b
      const cplx t1 = cdot_c(Wa, T3);
      cacc(a[2], dA, t1); cacc(a[0], -dA, t1);                             // -> a x b - x a b
      cacc(a[12], q.iCa, cdot_c(L[1], T3)); cacc(a[14], q.iCa, cdot_c(L[2], T3));
    }
    {
      const cvec T4 = bilinear(rb, col);                                   // b x
      const cplx t2 = cdot_c(Wa, T4);
      cacc(a[5], dA, t2); cacc(a[3], -dA, t2);                             // -> b a x - b x a
      cacc(a[13], q.iCa, cdot_c(L[1], T4)); cacc(a[15], q.iCa, cdot_c(L[2], T4));
    }
    {
      const cvec T1 = bilinear(row, ca);                                   // x a
      const cplx t3 = cdot_c(Wb, T1);
      cacc(a[3], dB, t3); cacc(a[1], -dB, t3);                             // -> b x a - x b a
      cacc(a[16], q.iCb, cdot_c(L[3], T1)); cacc(a[18], q.iCb, cdot_c(L[4], T1));
    }
    {
      const cvec T2 = bilinear(ra, col);                                   // a x
      const cplx t4 = cdot_c(Wb, T2);
      cacc(a[4], dB, t4); cacc(a[2], -dB, t4);                             // -> a b x - a x b
      cacc(a[17], q.iCb, cdot_c(L[3], T2)); cacc(a[19], q.iCb, cdot_c(L[4], T2));
    }
  }
  // (I) the top-line currents with both gluons, against the bare light line
  cacc(a[0], q.iA, cdot_c(L0, bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(ea, cb)))));    // x a b
  cacc(a[1], q.iA, cdot_c(L0, bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(eb, ca)))));    // x b a
  cacc(a[2], q.iA, cdot_c(L0, bilinear(ra, cb)));                                                 // a x b
  cacc(a[3], q.iA, cdot_c(L0, bilinear(rb, ca)));                                                 // b x a
  cacc(a[4], q.iA, cdot_c(L0, bilinear(prop_row(slash_row(ra, eb), k.rab, k.m, k.jab), col)));    // a b x
  cacc(a[5], q.iA, cdot_c(L0, bilinear(prop_row(slash_row(rb, ea), k.rab, k.m, k.jab), col)));    // b a x
  const cplx m1 = cdot_c(L0, bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(G, col))));      // x G -> x b a - x a b
  const cplx m2 = cdot_c(L0, bilinear(prop_row(slash_row(row, G), k.rab, k.m, k.jab), col));      // G x -> b a x - a b x
  cacc(a[1], q.iA, m1);  cacc(a[0], -q.iA, m1);
  cacc(a[5], q.iA, m2);  cacc(a[4], -q.iA, m2);
}

}  // namespace mf
// colour-summed |sum_s a_s S_s|^2: qq_colour_square(a)
#include "mf_me_qqttgg_colour_generated.cuh"
namespace mf {

// kinematics of one phase-space point and beam assignment: everything that does not depend on the helicities
struct QQPoint {
  QQKin q;
  QQLineKin kl, kt;
  rvec Ea[2], Eb[2];
  double isab;
};
MF_HD void qq_point(const double p1[4], const double p2[4], const double p3[4], const double p4[4], const double k5[4],
                    const double k6[4], double mt, QQPoint& pt) {
  rvec ka, kb, pcl, prl, pct, prt;
  QQKin& q = pt.q;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    ka.v[m] = k5[m]; kb.v[m] = k6[m];
    pcl.v[m] = p1[m]; prl.v[m] = -p2[m];
    pct.v[m] = -p4[m]; prt.v[m] = p3[m];
    q.PL0.v[m] = p1[m] + p2[m];
    q.PLa.v[m] = q.PL0.v[m] - k5[m];
    q.PLb.v[m] = q.PL0.v[m] - k6[m];
    q.mka.v[m] = -k5[m]; q.mkb.v[m] = -k6[m];
    q.K.v[m] = -(k5[m] + k6[m]);
  }
  const rvec PT0 = radd(prt, rscale(pct, -1.0));
  q.iA = 1.0 / rdot(q.PL0, q.PL0);
  q.iB = 1.0 / rdot(PT0, PT0);
  q.iCa = 1.0 / rdot(q.PLa, q.PLa);
  q.iCb = 1.0 / rdot(q.PLb, q.PLb);
  pt.isab = 1.0 / rdot(q.K, q.K);
  pt.kl = qq_line_kin(pcl, prl, ka, kb, 0.0);
  pt.kt = qq_line_kin(pct, prt, ka, kb, mt);
  pol_vectors(k5, pt.Ea[0], pt.Ea[1]);
  pol_vectors(k6, pt.Eb[0], pt.Eb[1]);
}
MF_HD rvec qq_merged(const QQKin& q, double isab, const rvec& ea, const rvec& eb) {   // hatted three-gluon merger of the two gluons
  rvec G = {{0.0, 0.0, 0.0, 0.0}};
  v3_acc(G, 1.0, ea, q.mka, eb, q.mkb);
  return rscale(G, isab);
}

// Averaged |M|^2 of q(p1) qbar(p2) -> t(p3) tbar(p4) g(k5) g(k6) at CM-frame momenta: 1/(4 x 9) for spins and colours of the
// initial state, 1/2! for the identical gluons, g2 = 4 pi alpha_s.  Flipping every fermion spin conjugates the amplitude (real
// polarisations), so only the left-handed light line is evaluated and the sum doubled.
MF_HD double me2_qq_ttgg(const double p1[4], const double p2[4], const double p3[4], const double p4[4], const double k5[4],
                         const double k6[4], double mt, double g2) {
  QQPoint pt;
  qq_point(p1, p2, p3, p4, k5, k6, mt, pt);
  const spin lcol = chiral_col(p1, 0, false), lrow = bar_of(chiral_col(p2, 0, true));
  double total = 0.0;
#pragma unroll 1
  for (int pol = 0; pol < 4; ++pol) {
    const rvec ea = pt.Ea[pol & 1], eb = pt.Eb[pol >> 1];
    const rvec G = qq_merged(pt.q, pt.isab, ea, eb);
    cvec L[13];
    qq_line_currents(lrow, lcol, pt.kl, ea, eb, G, L);
#pragma unroll 1
    for (int st = 0; st < 4; ++st) {
      cplx a[20];
      qq_assemble(L, ubar_row(p3, mt, st >> 1), v_col(p4, mt, st & 1), pt.kt, ea, eb, G, pt.q, a);
      total += qq_colour_square(a);
    }
  }
  const double g4 = g2 * g2;
  return 2.0 * total * g4 * g4 / 72.0;
}

// The same 20 coefficients with BOTH lines' currents in memory (the warp kernel below: every current set is formed once per
// (polarisation pair, spin state) and shared).
MF_HD void qq_assemble_mem(const cvec* L, const cvec* T, const rvec& ea, const rvec& eb, const rvec& G, const QQKin& q, cplx a[20]) {
  const cvec L0 = L[0], T0 = T[0];
  // (I) nothing on the virtual gluon: one term per tensor, plus the merged pair on either line ([T^b, T^a] in its place)
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    a[i] = cscale(cdot_c(L0, T[5 + i]), q.iA);
    a[6 + i] = cscale(cdot_c(L[5 + i], T0), q.iB);
  }
  a[12] = cscale(cdot_c(L[1], T[3]), q.iCa); a[13] = cscale(cdot_c(L[1], T[4]), q.iCa);
  a[14] = cscale(cdot_c(L[2], T[3]), q.iCa); a[15] = cscale(cdot_c(L[2], T[4]), q.iCa);
  a[16] = cscale(cdot_c(L[3], T[1]), q.iCb); a[17] = cscale(cdot_c(L[3], T[2]), q.iCb);
  a[18] = cscale(cdot_c(L[4], T[1]), q.iCb); a[19] = cscale(cdot_c(L[4], T[2]), q.iCb);
  const cplx m1 = cdot_c(L0, T[11]), m2 = cdot_c(L0, T[12]), m3 = cdot_c(L[11], T0), m4 = cdot_c(L[12], T0);
  cacc(a[1], q.iA, m1);  cacc(a[0], -q.iA, m1);        // x G   ->  x b a - x a b
  cacc(a[5], q.iA, m2);  cacc(a[4], -q.iA, m2);        // G x   ->  b a x - a b x
  cacc(a[7], q.iB, m3);  cacc(a[6], -q.iB, m3);
  cacc(a[11], q.iB, m4); cacc(a[10], -q.iB, m4);
  // (II) gluon g on the virtual gluon (T^x -> [T^g, T^x] on the top line), the other one on the top line ...
  const cvec Wa = v3c_vec(L0, q.PL0, ea, q.mka), Wb = v3c_vec(L0, q.PL0, eb, q.mkb);
  const double dA = q.iA * q.iCa, dB = q.iA * q.iCb;
  const cplx t1 = cdot_c(Wa, T[3]), t2 = cdot_c(Wa, T[4]), t3 = cdot_c(Wb, T[1]), t4 = cdot_c(Wb, T[2]);
  cacc(a[2], dA, t1); cacc(a[0], -dA, t1);             // (x b) -> a x b - x a b
  cacc(a[5], dA, t2); cacc(a[3], -dA, t2);             // (b x) -> b a x - b x a
  cacc(a[3], dB, t3); cacc(a[1], -dB, t3);             // (x a) -> b x a - x b a
  cacc(a[4], dB, t4); cacc(a[2], -dB, t4);             // (a x) -> a b x - a x b
  // ... or on the light line: top string x -> g x - x g
  const double eA = q.iCb * q.iB, eB = q.iCa * q.iB;
  const cplx u1 = cdot_c(v3c_vec(L[3], q.PLb, ea, q.mka), T0), u2 = cdot_c(v3c_vec(L[4], q.PLb, ea, q.mka), T0);
  const cplx u3 = cdot_c(v3c_vec(L[1], q.PLa, eb, q.mkb), T0), u4 = cdot_c(v3c_vec(L[2], q.PLa, eb, q.mkb), T0);
  cacc(a[17], eA, u1); cacc(a[16], -eA, u1);
  cacc(a[19], eA, u2); cacc(a[18], -eA, u2);
  cacc(a[13], eB, u3); cacc(a[12], -eB, u3);
  cacc(a[15], eB, u4); cacc(a[14], -eB, u4);
  // (III) both on the virtual gluon: a then b, b then a, the merged pair, the four-gluon vertex (see qq_assemble)
  const double d3 = q.iA * q.iB;
  const cplx l0t0 = cdot_c(L0, T0), lea = cdot_r(L0, ea), leb = cdot_r(L0, eb), tea = cdot_r(T0, ea), teb = cdot_r(T0, eb);
  const double eab = rdot(ea, eb);
  const cplx sab = cdot_c(v3c_vec(Wa, q.PLa, eb, q.mkb), T0), sba = cdot_c(v3c_vec(Wb, q.PLb, ea, q.mka), T0);
  const cplx sG = cdot_c(v3c_vec(L0, q.PL0, G, q.K), T0);
  const cplx v0 = cmul(leb, tea), v1 = cmul(lea, teb);
  const cplx A = {d3 * (sab.re * q.iCa + v0.re - eab * l0t0.re), d3 * (sab.im * q.iCa + v0.im - eab * l0t0.im)};
  const cplx B = {d3 * (sba.re * q.iCb + v1.re - eab * l0t0.re), d3 * (sba.im * q.iCb + v1.im - eab * l0t0.im)};
  const cplx C = {d3 * (sG.re - (v1.re - v0.re)), d3 * (sG.im - (v1.im - v0.im))};
  cacc(a[5], 1.0, A); cacc(a[3], -1.0, A); cacc(a[2], -1.0, A); cacc(a[0], 1.0, A);
  cacc(a[4], 1.0, B); cacc(a[2], -1.0, B); cacc(a[3], -1.0, B); cacc(a[1], 1.0, B);
  cacc(a[5], 1.0, C); cacc(a[4], -1.0, C); cacc(a[1], -1.0, C); cacc(a[0], 1.0, C);
}

// thread-per-event evaluation through qq_assemble_mem (tests/host_shim: the arithmetic of the warp kernel, checked on the host)
MF_HD double me2_qq_ttgg_mem(const double p1[4], const double p2[4], const double p3[4], const double p4[4], const double k5[4],
                             const double k6[4], double mt, double g2) {
  QQPoint pt;
  qq_point(p1, p2, p3, p4, k5, k6, mt, pt);
  const spin lcol = chiral_col(p1, 0, false), lrow = bar_of(chiral_col(p2, 0, true));
  double total = 0.0;
  for (int pol = 0; pol < 4; ++pol) {
    const rvec ea = pt.Ea[pol & 1], eb = pt.Eb[pol >> 1];
    const rvec G = qq_merged(pt.q, pt.isab, ea, eb);
    cvec L[13], T[13];
    qq_line_currents(lrow, lcol, pt.kl, ea, eb, G, L);
    for (int st = 0; st < 4; ++st) {
      qq_line_currents(ubar_row(p3, mt, st >> 1), v_col(p4, mt, st & 1), pt.kt, ea, eb, G, T);
      cplx a[20];
      qq_assemble_mem(L, T, ea, eb, G, pt.q, a);
      total += qq_colour_square(a);
    }
  }
  const double g4 = g2 * g2;
  return 2.0 * total * g4 * g4 / 72.0;
}

#if defined(__CUDACC__)
// The same matrix element by ONE WARP per event, both beam assignments at once (quark_prepass_kernel).
// Stage 1: one set of 13 line currents per lane, the same code for both lines (qq_line_kin + the chains + 13 bilinears with the
// lane's spinors, momenta and mass): lanes 0-15 the top line for (polarisation pair, spin state) = 16 sets, lanes 16-31 the light
// line for (beam assignment, polarisation pair) = 8 sets (formed twice, stored once).  All sets go to shared memory.
// Stage 2: lane = (beam assignment o, polarisation pair, top spin state): the 20 string coefficients from its two sets
// (qq_assemble_mem), the colour form in registers; the 16 lanes of an assignment are summed by shuffles.
constexpr int kQQLStride = 106;        // 13 currents x 8 doubles, padded: broadcast reads of different sets fall into different banks
constexpr int kQQWarpSets = 8 + 16;    // light-line sets, then top-line sets
// what does not depend on the lane, nor on the beam assignment (the virtual gluon's kinematics, the polarisation vectors):
// formed by lane 0, read by all from shared memory when needed
struct QQWarpShared {
  QQKin q;
  rvec Ea[2], Eb[2];
  double isab;
};
constexpr int kQQWarpSharedDoubles = (sizeof(QQWarpShared) + 7) / 8;
__device__ __forceinline__ void qq_store(double* dst, const cvec& c) {
#pragma unroll
  for (int m = 0; m < 4; ++m) { dst[m] = c.re[m]; dst[4 + m] = c.im[m]; }
}
// ev = the event's four final-state momenta and shat (17 doubles), sh and Js[kQQWarpSets x kQQLStride]: the warp's shared memory
__device__ __forceinline__ void me2_qq_ttgg_warp(const double* ev, QQWarpShared* sh, double* Js, int lane, double mt, double g2,
                                                 double& m0, double& m1) {
  const double E = 0.5 * sqrt(ev[16]);
  if (lane == 0) {
    const double p1[4] = {E, 0.0, 0.0, E}, p2[4] = {E, 0.0, 0.0, -E};
    QQPoint pt;
    qq_point(p1, p2, ev, ev + 4, ev + 8, ev + 12, mt, pt);      // q, Ea, Eb, isab do not depend on the beam assignment
    sh->q = pt.q; sh->isab = pt.isab;
    sh->Ea[0] = pt.Ea[0]; sh->Ea[1] = pt.Ea[1]; sh->Eb[0] = pt.Eb[0]; sh->Eb[1] = pt.Eb[1];
  }
  __syncwarp();
  {
    const bool top = lane < 16;
    const int c = lane & 15;
    const int pol1 = top ? (c >> 2) : ((c >> 1) & 3);
    const rvec ea = sh->Ea[pol1 & 1], eb = sh->Eb[pol1 >> 1];
    const rvec G = qq_merged(sh->q, sh->isab, ea, eb);
    spin row, col;
    rvec pc, pr, ka, kb;
    double m;
    if (top) {
      row = ubar_row(ev, mt, (c >> 1) & 1);
      col = v_col(ev + 4, mt, c & 1);
      m = mt;
#pragma unroll
      for (int i = 0; i < 4; ++i) { pc.v[i] = -ev[4 + i]; pr.v[i] = ev[i]; }
    } else {
      const double pz = (c >> 3) == 0 ? E : -E;
      const double p1[4] = {E, 0.0, 0.0, pz}, p2[4] = {E, 0.0, 0.0, -pz};
      col = chiral_col(p1, 0, false);
      row = bar_of(chiral_col(p2, 0, true));
      m = 0.0;
#pragma unroll
      for (int i = 0; i < 4; ++i) { pc.v[i] = p1[i]; pr.v[i] = -p2[i]; }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) { ka.v[i] = ev[8 + i]; kb.v[i] = ev[12 + i]; }
    const QQLineKin k = qq_line_kin(pc, pr, ka, kb, m);
    double* dst = Js + (top ? 8 + c : (c >> 1)) * kQQLStride;
    const bool store = top || (c & 1) == 0;
    const spin ca = prop_col(k.qa, k.m, k.ia, slash_col(ea, col)), cb = prop_col(k.qb, k.m, k.ib, slash_col(eb, col));
    const spin ra = prop_row(slash_row(row, ea), k.ra, k.m, k.ja), rb = prop_row(slash_row(row, eb), k.rb, k.m, k.jb);
    auto put = [&](int i, const cvec& v) { if (store) qq_store(dst + 8 * i, v); };
    put(0, bilinear(row, col));
    put(1, bilinear(row, ca));
    put(2, bilinear(ra, col));
    put(3, bilinear(row, cb));
    put(4, bilinear(rb, col));
    put(5, bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(ea, cb))));
    put(6, bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(eb, ca))));
    put(7, bilinear(ra, cb));
    put(8, bilinear(rb, ca));
    put(9, bilinear(prop_row(slash_row(ra, eb), k.rab, k.m, k.jab), col));
    put(10, bilinear(prop_row(slash_row(rb, ea), k.rab, k.m, k.jab), col));
    put(11, bilinear(row, prop_col(k.qab, k.m, k.iab, slash_col(G, col))));
    put(12, bilinear(prop_row(slash_row(row, G), k.rab, k.m, k.jab), col));
  }
  __syncwarp();
  const int o = lane >> 4, pol = (lane >> 2) & 3, st = lane & 3;
  const rvec ea = sh->Ea[pol & 1], eb = sh->Eb[pol >> 1];
  const rvec G = qq_merged(sh->q, sh->isab, ea, eb);
  cplx a[20];
  qq_assemble_mem(reinterpret_cast<const cvec*>(Js + (o * 4 + pol) * kQQLStride),
                  reinterpret_cast<const cvec*>(Js + (8 + pol * 4 + st) * kQQLStride), ea, eb, G, sh->q, a);
  double v = qq_colour_square(a);
#pragma unroll
  for (int d = 1; d < 16; d <<= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
  const double g4 = g2 * g2;
  v *= 2.0 * g4 * g4 / 72.0;
  m0 = __shfl_sync(0xFFFFFFFFu, v, 0);
  m1 = __shfl_sync(0xFFFFFFFFu, v, 16);
  __syncwarp();
}
#endif

}  // namespace mf
