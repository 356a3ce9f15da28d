// mf_me_qqtt.cuh — |M|^2 of q(p1) qbar(p2) -> t(p3) tbar(p4) through the s-channel gluon, massless q (the quark
// channel of the flavour-summed pp -> ttbar: SURVEY.md 8(f2); "pp -> ttbar (7 diagrams)" = 3 gg + one
// q qbar diagram per flavour; L65: helicities are looped over and summed).
//   iM = [vbar(p2) (i g T^a_{ji} gamma^mu) u(p1)] (-i g_{mu nu} / s) [ubar(p3) (i g T^a_{kl} gamma^nu) v(p4)]
//   colour: sum |T^a_{ji} T^a_{kl}|^2 = tr(T^a T^b) tr(T^a T^b) = (1/2)^2 8 = 2;  average 1 / (4 spins x 9 colours)
//   |M|^2_avg = (2 / 36) (g^2 / s)^2 sum over the 16 spin combinations of |j_q . j_t|^2
// The helicity sum is symmetric under p1 <-> p2 (t <-> u), so one evaluation serves both beam assignments of the quark.
#pragma once
#include "mf_me_prims.cuh"

namespace mf {

// mom: p1, p2 (beams), p3, p4 in the CM frame; g2 = 4 pi alpha_s
MF_HD double me2_qq_tt(const double p1[4], const double p2[4], const double p3[4], const double p4[4], double mt,
                       double g2) {
  double P[4] = {p1[0] + p2[0], p1[1] + p2[1], p1[2] + p2[2], p1[3] + p2[3]};
  double s = P[0] * P[0] - P[1] * P[1] - P[2] * P[2] - P[3] * P[3];
  cvec jq[4], jt[4];
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      jq[2 * a + b] = bilinear(bar_of(v_col(p2, 0.0, b)), u_col(p1, 0.0, a));
      jt[2 * a + b] = bilinear(ubar_row(p3, mt, a), v_col(p4, mt, b));
    }
  double total = 0.0;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      cplx d = cdot_c(jq[i], jt[j]);
      total += d.re * d.re + d.im * d.im;
    }
  double f = g2 / s;
  return (1.0 / 18.0) * f * f * total;
}

}  // namespace mf
