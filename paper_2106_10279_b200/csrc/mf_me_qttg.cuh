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

// The top line's three currents for its four spin states and one gluon polarisation e:
//   jt = ubar3 gamma v4,  jtC = ubar3 e-slash (t1-slash + m) gamma v4,  jtD = ubar3 gamma (t2-slash + m) e-slash v4
MF_HD void qttg_top_currents(const double p3[4], const double p4[4], const rvec& t1, const rvec& t2, double mt, const rvec& e,
                             cvec jt[4], cvec jtC[4], cvec jtD[4]) {
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) {
      const spin ub3 = ubar_row(p3, mt, a), v4 = v_col(p4, mt, b);
      jt[2 * a + b] = bilinear(ub3, v4);
      const spin r1 = slash_row(ub3, e), c1 = slash_col(e, v4);
      jtC[2 * a + b] = bilinear(spin_add_scaled(slash_row(r1, t1), mt, r1), v4);
      jtD[2 * a + b] = bilinear(ub3, spin_add_scaled(slash_col(t2, c1), mt, c1));
    }
}
// sum over the two chiralities of the massless light line (one evaluated, doubled) and the four top spin states of K^dagger (3 S) K for one gluon
// polarisation e.  The light line runs from the column spinor (pcol, a v spinor if col_v; flow momentum into the line) to
// the row spinor (prow, a vbar if row_v).  w[5] = the propagator weights of the five diagrams.
MF_HD double qttg_light_sum(const double pcol[4], bool col_v, const double prow[4], bool row_v, const rvec& e, const rvec& a1,
                            const rvec& a2, const rvec& k12, const rvec& k23, const rvec& k31, const cvec jt[4],
                            const cvec jtC[4], const cvec jtD[4], const double w[5]) {
  // colour matrix in units of 1/3: S[d][e] = sum over colours of conj(C_d) C_e of the five colour tensors
  // (T^b T^a)_{ji} T^b_{kl}, (T^a T^b)_{ji} T^b_{kl}, T^b_{ji} (T^a T^b)_{kl}, T^b_{ji} (T^b T^a)_{kl}, i f^{bca} T^b_{ji} T^c_{kl}
  // (checked against the oracle's explicit-generator sum by the parity tests of this matrix element):
  //   3 S = {{8, -1, 7, -2, 9}, {-1, 8, -2, 7, -9}, {7, -2, 8, -1, 9}, {-2, 7, -1, 8, -9}, {9, -9, 9, -9, 18}}
  double total = 0.0;
  const double k12e = rdot(k12, e);
  // Flipping the spin of every fermion conjugates the amplitudes (real polarisation e, real momenta), and the four top spin
  // states below are closed under the flip: the right-handed light line gives the same sum as the left-handed one.
  {
    const int i = 0;
    const spin col = chiral_col(pcol, i, col_v);
    const spin row = bar_of(chiral_col(prow, i, row_v));
    const cvec jl = bilinear(row, col);
    const cvec jlA = bilinear(row, slash_col(a1, slash_col(e, col)));
    const cvec jlB = bilinear(slash_row(slash_row(row, e), a2), col);
    const cplx el = cdot_r(jl, e), k23l = cdot_r(jl, k23);
#pragma unroll 1
    for (int j = 0; j < 4; ++j) {
      cplx K[5];
      K[0] = cdot_c(jlA, jt[j]);  K[0].re *= w[0]; K[0].im *= w[0];
      K[1] = cdot_c(jlB, jt[j]);  K[1].re *= w[1]; K[1].im *= w[1];
      K[2] = cdot_c(jl, jtC[j]);  K[2].re *= w[2]; K[2].im *= w[2];
      K[3] = cdot_c(jl, jtD[j]);  K[3].re *= w[3]; K[3].im *= w[3];
      const cplx lt = cdot_c(jl, jt[j]), et = cdot_r(jt[j], e), k31t = cdot_r(jt[j], k31);
      K[4].re = w[4] * (lt.re * k12e + (et.re * k23l.re - et.im * k23l.im) + (el.re * k31t.re - el.im * k31t.im));
      K[4].im = w[4] * (lt.im * k12e + (et.re * k23l.im + et.im * k23l.re) + (el.re * k31t.im + el.im * k31t.re));
      // K^dagger (3 S) K with u = K0 + K2, v = K1 + K3, d = u - v, r = (K0 - K2) + (K1 - K3):
      //   6 (|u|^2 + |v|^2) + 1.5 |d|^2 + 18 Re(conj(K4) d) + 18 |K4|^2 + 0.5 |r|^2
      const cplx u = {K[0].re + K[2].re, K[0].im + K[2].im}, v = {K[1].re + K[3].re, K[1].im + K[3].im};
      const cplx dd = {u.re - v.re, u.im - v.im};
      const cplx r = {(K[0].re - K[2].re) + (K[1].re - K[3].re), (K[0].im - K[2].im) + (K[1].im - K[3].im)};
      total += 6.0 * (re_conj_mul(u, u) + re_conj_mul(v, v)) + 1.5 * re_conj_mul(dd, dd) +
               18.0 * (re_conj_mul(K[4], dd) + re_conj_mul(K[4], K[4])) + 0.5 * re_conj_mul(r, r);
    }
  }
  return 2.0 * total;
}

// One class at caller-supplied momenta (mf_debug_me2_quark_gluon, tests/host_shim): kind 0 / 1 as in the header comment.
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
  const double w[5] = {1.0 / (rdot(a1, a1) * st), 1.0 / (rdot(a2, a2) * st), 1.0 / ((rdot(t1, t1) - mt * mt) * sl),
                       1.0 / ((rdot(t2, t2) - mt * mt) * sl), 1.0 / (sl * st)};
  rvec E[2];
  pol_vectors(pg, E[0], E[1]);
  double total = 0.0;
  for (int lam = 0; lam < 2; ++lam) {
    cvec jt[4], jtC[4], jtD[4];
    qttg_top_currents(p3, p4, t1, t2, mt, E[lam], jt, jtC, jtD);
    total += qttg_light_sum(p1, false, prow, kind == 0, E[lam], a1, a2, k12, k23, k31, jt, jtC, jtD, w);
  }
  const double avg = kind == 0 ? 36.0 : 96.0;
  return total * (g2 * g2 * g2) / (3.0 * avg);
}

// All six flavour-blind quark-channel classes of pp -> ttbar j at one CM-frame point (beams b1 along +z, b2 along -z; final
// t = p3, tbar = p4, light parton k2):  0 q qbar -> g,  1 qbar q -> g,  2 q g -> q,  3 g q -> q,  4 qbar g -> qbar,  5 g qbar -> qbar
// (first parton from beam 1).  The gluon is k2 (outgoing) for classes 0, 1, beam 2 for 2, 4 and beam 1 for 3, 5: the top line's
// currents depend on the gluon only, so they are formed three times, not six; the antiquark classes run the light line from
// the outgoing antiquark (column v(k2), flow momentum -k2) to the incoming one (row vbar(b), flow -b) instead of exchanging
// t and tbar.  out[c] = averaged |M|^2 of class c.
MF_HD void me2_ttj_quark_classes(const double b1[4], const double b2[4], const double p3[4], const double p4[4],
                                 const double k2[4], double mt, double g2, double out[6]) {
  rvec qt;
#pragma unroll
  for (int m = 0; m < 4; ++m) qt.v[m] = p3[m] + p4[m];
  const double st = rdot(qt, qt);
#pragma unroll
  for (int c = 0; c < 6; ++c) out[c] = 0.0;
#pragma unroll 1
  for (int G = 0; G < 3; ++G) {
    const double* pg = G == 0 ? k2 : G == 1 ? b2 : b1;
    const double sk = G == 0 ? 1.0 : -1.0;
    rvec kg, t1, t2, k23;
#pragma unroll
    for (int m = 0; m < 4; ++m) {
      kg.v[m] = sk * pg[m];
      t1.v[m] = p3[m] + kg.v[m];
      t2.v[m] = -p4[m] - kg.v[m];
      k23.v[m] = kg.v[m] - qt.v[m];
    }
    const double wCt = 1.0 / (rdot(t1, t1) - mt * mt), wDt = 1.0 / (rdot(t2, t2) - mt * mt);
    rvec E[2];
    pol_vectors(pg, E[0], E[1]);
#pragma unroll 1
    for (int lam = 0; lam < 2; ++lam) {
      cvec jt[4], jtC[4], jtD[4];
      qttg_top_currents(p3, p4, t1, t2, mt, E[lam], jt, jtC, jtD);
#pragma unroll 1
      for (int u = 0; u < 2; ++u) {
        const int c = G == 0 ? u : G == 1 ? (u ? 4 : 2) : (u ? 5 : 3);
        // the light line of class c: column (pcol, v spinor?, sign of the flow momentum), row likewise
        const bool anti = c >= 4;
        const double* pcol = anti ? k2 : (c == 1 || c == 3) ? b2 : b1;
        const double* prow = c == 0 ? b2 : c == 1 ? b1 : c == 4 ? b1 : c == 5 ? b2 : k2;
        const double sc = anti ? -1.0 : 1.0, sr = (c == 2 || c == 3) ? 1.0 : -1.0;
        rvec ql, a1, a2, k12, k31;
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          const double pc = sc * pcol[m], pr = sr * prow[m];
          ql.v[m] = pc - pr;
          a1.v[m] = pc - kg.v[m];
          a2.v[m] = pr + kg.v[m];
          k12.v[m] = ql.v[m] + qt.v[m];
          k31.v[m] = -kg.v[m] - ql.v[m];
        }
        const double sl = rdot(ql, ql);
        const double w[5] = {1.0 / (rdot(a1, a1) * st), 1.0 / (rdot(a2, a2) * st), wCt / sl, wDt / sl, 1.0 / (sl * st)};
        out[c] += qttg_light_sum(pcol, anti, prow, c != 2 && c != 3, E[lam], a1, a2, k12, k23, k31, jt, jtC, jtD, w);
      }
    }
  }
  const double f = (g2 * g2 * g2) / 3.0;
  out[0] *= f / 36.0; out[1] *= f / 36.0;
#pragma unroll
  for (int c = 2; c < 6; ++c) out[c] *= f / 96.0;
}

}  // namespace mf
