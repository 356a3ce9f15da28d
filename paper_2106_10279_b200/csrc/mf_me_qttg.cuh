// mf_me_qttg.cuh — |M|^2 of the quark channels of pp -> ttbar g ("36 diagrams" = 16 gg + 5
// for each of q qbar -> ttbar g, q g -> ttbar q, ...): one massless quark line, the top line and one gluon, five diagrams.
// Used by the fused pass of MF_PP_TTG (mf_kernels.cuh, R19) and by mf_debug_me2_quark_gluon.
//
// Conventions of mf_me_prims.cuh (chiral two-component spinors, z-axis spin states, REAL linear gluon polarisations).
// The light line is described by its column spinor (incoming quark, momentum pc into the line) and its row spinor with
// momentum pr flowing out of the line, the gluon by its outgoing momentum kg:
//   kind 0  q(p1) qbar(prow) -> t tbar g(pg):  row = vbar(prow), pr = -prow, kg = pg
//   kind 1  q(p1) g(pg) -> t tbar q(prow):     row = ubar(prow), pr = prow,  kg = -pg
// Colour-stripped diagrams (all factors of i and g pulled out: -i g^3 for K_0..K_3, g^3 for K_4):
//   K_0 = [row gamma^mu a1-slash E-slash col] [ubar3 gamma_mu v4] / (a1^2 st)        a1 = pc - kg
//   K_1 = [row E-slash a2-slash gamma^mu col] [ubar3 gamma_mu v4] / (a2^2 st)        a2 = pr + kg
//   K_2 = [row gamma^mu col] [ubar3 E-slash (t1-slash + m) gamma_mu v4] / ((t1^2 - m^2) sl)   t1 = p3 + kg
//   K_3 = [row gamma^mu col] [ubar3 gamma_mu (t2-slash + m) E-slash v4] / ((t2^2 - m^2) sl)   t2 = -p4 - kg
//   K_4 = [(jl.jt)((ql+qt).E) + (jt.E)((kg-qt).jl) + (E.jl)((-kg-ql).jt)] / (sl st)
// with ql = pc - pr, qt = p3 + p4, sl = ql^2, st = qt^2.  Colour: with the tensors (T^b T^a)_{ji} T^b_{kl},
// (T^a T^b)_{ji} T^b_{kl}, T^b_{ji} (T^a T^b)_{kl}, T^b_{ji} (T^b T^a)_{kl} and i f^{bca} T^b_{ji} T^c_{kl} the
// colour-summed square is  sum_{de} S_de Re(conj(K_d) K_e)  with the real symmetric matrix below (csrc/gen_qttg_colour.py).
#pragma once
#include "mf_me_prims.cuh"

namespace mf {

MF_HD spin spin_add_scaled(const spin& a, double m, const spin& c) {   // a + m c
  spin o;
#pragma unroll
  for (int i = 0; i < 4; ++i) { o.re[i] = fma(m, c.re[i], a.re[i]); o.im[i] = fma(m, c.im[i], a.im[i]); }
  return o;
}
MF_HD double re_conj_mul(const cplx& a, const cplx& b) { return a.re * b.re + a.im * b.im; }   // Re(conj(a) b)

// Massless quark: the chirality-c part (c = 0: left, components 0-1; c = 1: right, components 2-3) of u(p) resp. v(p),
// normalised to psi^dagger psi = 2 E: a helicity eigenstate.  A vector current (an odd number of gamma matrices between
// row and column) connects equal chiralities only, so the light line has TWO spin states that contribute, not four
// (the spin-summed |M|^2 does not depend on the basis).  The z-axis spin state that is projected is the one with the
// larger component along the wanted helicity (no 0/0 for momenta along the z axis: the beams).
MF_HD spin chiral_col(const double p[4], int c, bool is_v) {
  const bool up = (c == 0) == (p[3] <= 0.0);          // left part: |(E - p.sigma) xi|^2 = E -+ pz for xi = (1,0) / (0,1)
  spin u = is_v ? v_col(p, 0.0, up ? 0 : 1) : u_col(p, 0.0, up ? 0 : 1);
  const double n2 = p[0] + ((c == 0) == up ? -p[3] : p[3]);
  const double n = sqrt(2.0 * p[0] / n2);
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const bool keep = (k >> 1) == c;
    u.re[k] = keep ? n * u.re[k] : 0.0;
    u.im[k] = keep ? n * u.im[k] : 0.0;
  }
  return u;
}

MF_HD double me2_light_line_ttg(int kind, const double p1[4], const double prow[4], const double p3[4],
                                const double p4[4], const double pg[4], double mt, double g2) {
  const double sr = kind == 0 ? -1.0 : 1.0, sk = kind == 0 ? 1.0 : -1.0;
  rvec ql, qt, a1, a2, t1, t2, k12, k23, k31;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    const double pr = sr * prow[m], kg = sk * pg[m];
    ql.v[m] = p1[m] - pr;
    qt.v[m] = p3[m] + p4[m];
    a1.v[m] = p1[m] - kg;
    a2.v[m] = pr + kg;
    t1.v[m] = p3[m] + kg;
    t2.v[m] = -p4[m] - kg;
    k12.v[m] = ql.v[m] + qt.v[m];
    k23.v[m] = kg - qt.v[m];
    k31.v[m] = -kg - ql.v[m];
  }
  const double sl = rdot(ql, ql), st = rdot(qt, qt);
  const double wA = 1.0 / (rdot(a1, a1) * st), wB = 1.0 / (rdot(a2, a2) * st);
  const double wC = 1.0 / ((rdot(t1, t1) - mt * mt) * sl), wD = 1.0 / ((rdot(t2, t2) - mt * mt) * sl);
  const double wE = 1.0 / (sl * st);
  rvec E[2];
  pol_vectors(pg, E[0], E[1]);
  // colour matrix in units of 1/3: S[d][e] = sum over colours of conj(C_d) C_e of the five colour tensors
  // (T^b T^a)_{ji} T^b_{kl}, (T^a T^b)_{ji} T^b_{kl}, T^b_{ji} (T^a T^b)_{kl}, T^b_{ji} (T^b T^a)_{kl}, i f^{bca} T^b_{ji} T^c_{kl}
  // (checked against the oracle's explicit-generator sum by the parity tests of this matrix element):
  //   3 S = {{8, -1, 7, -2, 9}, {-1, 8, -2, 7, -9}, {7, -2, 8, -1, 9}, {-2, 7, -1, 8, -9}, {9, -9, 9, -9, 18}}
  double total = 0.0;
  for (int lam = 0; lam < 2; ++lam) {
    const rvec& e = E[lam];
    // the top line's three currents for its four spin states (kept in memory), then the light line's, one spin state
    // at a time (kept in registers)
    cvec jt[4], jtC[4], jtD[4];
    for (int a = 0; a < 2; ++a)
      for (int b = 0; b < 2; ++b) {
        const spin ub3 = ubar_row(p3, mt, a), v4 = v_col(p4, mt, b);
        jt[2 * a + b] = bilinear(ub3, v4);
        const spin r1 = slash_row(ub3, e), c1 = slash_col(e, v4);
        jtC[2 * a + b] = bilinear(spin_add_scaled(slash_row(r1, t1), mt, r1), v4);
        jtD[2 * a + b] = bilinear(ub3, spin_add_scaled(slash_col(t2, c1), mt, c1));
      }
    const double k12e = rdot(k12, e);
#pragma unroll 1
    for (int i = 0; i < 2; ++i) {          // the two chiralities of the massless light line
      const spin col = chiral_col(p1, i, false);
      const spin row = bar_of(chiral_col(prow, i, kind == 0));
      const cvec jl = bilinear(row, col);
      const cvec jlA = bilinear(row, slash_col(a1, slash_col(e, col)));
      const cvec jlB = bilinear(slash_row(slash_row(row, e), a2), col);
      const cplx el = cdot_r(jl, e), k23l = cdot_r(jl, k23);
#pragma unroll 1
      for (int j = 0; j < 4; ++j) {
        cplx K[5];
        K[0] = cdot_c(jlA, jt[j]);  K[0].re *= wA; K[0].im *= wA;
        K[1] = cdot_c(jlB, jt[j]);  K[1].re *= wB; K[1].im *= wB;
        K[2] = cdot_c(jl, jtC[j]);  K[2].re *= wC; K[2].im *= wC;
        K[3] = cdot_c(jl, jtD[j]);  K[3].re *= wD; K[3].im *= wD;
        const cplx lt = cdot_c(jl, jt[j]), et = cdot_r(jt[j], e), k31t = cdot_r(jt[j], k31);
        K[4].re = wE * (lt.re * k12e + (et.re * k23l.re - et.im * k23l.im) + (el.re * k31t.re - el.im * k31t.im));
        K[4].im = wE * (lt.im * k12e + (et.re * k23l.im + et.im * k23l.re) + (el.re * k31t.im + el.im * k31t.re));
        // K^dagger (3 S) K with u = K0 + K2, v = K1 + K3, d = u - v, r = (K0 - K2) + (K1 - K3):
        //   6 (|u|^2 + |v|^2) + 1.5 |d|^2 + 18 Re(conj(K4) d) + 18 |K4|^2 + 0.5 |r|^2
        const cplx u = {K[0].re + K[2].re, K[0].im + K[2].im}, v = {K[1].re + K[3].re, K[1].im + K[3].im};
        const cplx dd = {u.re - v.re, u.im - v.im};
        const cplx r = {(K[0].re - K[2].re) + (K[1].re - K[3].re), (K[0].im - K[2].im) + (K[1].im - K[3].im)};
        total += 6.0 * (re_conj_mul(u, u) + re_conj_mul(v, v)) + 1.5 * re_conj_mul(dd, dd) +
                 18.0 * (re_conj_mul(K[4], dd) + re_conj_mul(K[4], K[4])) + 0.5 * re_conj_mul(r, r);
      }
    }
  }
  const double avg = kind == 0 ? 36.0 : 96.0;
  return total * (g2 * g2 * g2) / (3.0 * avg);
}

}  // namespace mf
