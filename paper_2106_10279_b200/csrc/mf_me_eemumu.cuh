// mf_me_eemumu.cuh — |M|^2 of e-(p1) e+(p2) -> mu-(p3) mu+(p4) through the s-channel photon only, massless
// (BASELINE.json configs[0]; "loops over initial and final state particle helicities and
// aggregates their contribution to the final squared amplitude").
//   iM = [vbar(p2) (i e gamma^mu) u(p1)] (-i g_{mu nu}/s) [ubar(p3) (i e gamma^nu) v(p4)]
//   |M|^2_avg = (1/4) sum over the 16 spin combinations = e^4/(4 s^2) sum |j_e . j_mu|^2
// The two fermion currents depend on two spins each, so the 16-term sum needs 4 + 4 bilinears.
#pragma once
#include "mf_me_prims.cuh"

namespace mf {

// mom: p1, p2 (beams), p3, p4 in the CM frame
MF_HD double me2_ee_mumu(const double p1[4], const double p2[4], const double p3[4], const double p4[4],
                         double alpha_em) {
  double e2 = 4.0 * kPi * alpha_em;
  double P[4] = {p1[0] + p2[0], p1[1] + p2[1], p1[2] + p2[2], p1[3] + p2[3]};
  double s = P[0] * P[0] - P[1] * P[1] - P[2] * P[2] - P[3] * P[3];
  cvec je[4], jm[4];
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      je[2 * a + b] = bilinear(bar_of(v_col(p2, 0.0, b)), u_col(p1, 0.0, a));
      jm[2 * a + b] = bilinear(ubar_row(p3, 0.0, a), v_col(p4, 0.0, b));
    }
  double total = 0.0;
#pragma unroll
  for (int i = 0; i < 4; ++i)
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      cplx d = cdot_c(je[i], jm[j]);
      total += d.re * d.re + d.im * d.im;
    }
  double f = e2 / s;
  return 0.25 * f * f * total;
}

}  // namespace mf
