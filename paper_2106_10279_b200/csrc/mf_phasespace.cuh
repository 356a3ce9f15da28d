// mf_phasespace.cuh — steps a2-a5 of the hot path: VEGAS map, parton fractions, phase space, boost, cuts.
// Everything stays in registers; the VEGAS grid is read from shared memory.
#pragma once
#include "mf_common.cuh"

namespace mf {

// a2. VEGAS importance-sampling map for one dimension (Lepage; PAPER.md L27, L61 via VegasFlow).
// t = u nb, i = min(floor t, nb-1), x = e_i + (t - i)(e_{i+1} - e_i); the Jacobian factor nb (e_{i+1} - e_i)
// is multiplied into jac.  The bin index depends on u only, so it is bit-exact against the oracle.
MF_HD double vegas_map1(const double* edges /* this dimension's nb+1 edges */, int nb, double u, double& jac,
                        int& bin) {
  double t = u * (double)nb;
  int i = (int)t;
  if (i > nb - 1) i = nb - 1;
  double e0 = edges[i], e1 = edges[i + 1];
  double width = e1 - e0;
  jac *= (double)nb * width;
  bin = i;
  return e0 + (t - (double)i) * width;
}

// a3. Parton fractions (R4): tau = exp((1-x0) ln tau_min), y = (x1 - 1/2)(-ln tau),
// x1 = sqrt(tau) e^y, x2 = sqrt(tau) e^-y, shat = tau s; Jacobian (-tau ln tau_min)(-ln tau).
struct Parton { double y, x1, x2, shat, jac; };
MF_HD Parton parton_fractions(double x0, double x1v, double ln_tau_min, double s) {
  Parton k;
  double tau = exp((1.0 - x0) * ln_tau_min);
  double mlt = -log(tau);
  k.y = (x1v - 0.5) * mlt;
  double rt = sqrt(tau);
  double ey = exp(k.y);
  k.x1 = rt * ey;
  k.x2 = rt * exp(-k.y);
  k.shat = tau * s;
  k.jac = -(tau * ln_tau_min) * mlt;
  return k;
}

// a4 (C0, C1). Analytic two-body phase space in the partonic CM frame ("2-body analytic", BASELINE.json).
// Final momenta k[0] = (E, kx, ky, kz), k[1] = (E, -k).  Returns beta/(32 pi^2) * 2 * 2pi, the weight per
// unit (x_c, x_phi).
MF_HD double two_body(double shat, double m, double xc, double xphi, double k[2][4]) {
  double E = 0.5 * sqrt(shat);
  double c = 2.0 * xc - 1.0;
  double sphi, cphi;
  sincos(kTwoPi * xphi, &sphi, &cphi);
  double st = sqrt(1.0 - c * c);
  double kk = sqrt(E * E - m * m);
  k[0][0] = E; k[0][1] = kk * st * cphi; k[0][2] = kk * st * sphi; k[0][3] = kk * c;
  k[1][0] = E; k[1][1] = -k[0][1]; k[1][2] = -k[0][2]; k[1][3] = -k[0][3];
  double beta = kk / E;
  return beta / (32.0 * kPi * kPi) * 2.0 * kTwoPi;
}

// a4 (C2-C4). RAMBO (Kleiss, Stirling, Ellis 1986): N massless isotropic momenta from
// 4 uniforms each, conformally transformed to total momentum (w, 0), then rescaled by xi (Newton, fixed 10
// iterations, R6) to put the first two particles on the top mass shell.  Returns the volume V
// (dPhi_n = (2 pi)^{4-3n} V).  q[] holds the massless momenta on entry and the massive ones on exit.
template <int N>
MF_HD double rambo_finish(double q[N][4], double w, double m_top) {
  double Q0 = 0, Q1 = 0, Q2 = 0, Q3 = 0;
#pragma unroll
  for (int i = 0; i < N; ++i) { Q0 += q[i][0]; Q1 += q[i][1]; Q2 += q[i][2]; Q3 += q[i][3]; }
  double M = sqrt(Q0 * Q0 - Q1 * Q1 - Q2 * Q2 - Q3 * Q3);
  double iM = 1.0 / M;
  double b1 = -Q1 * iM, b2 = -Q2 * iM, b3 = -Q3 * iM;
  double x = w * iM, gamma = Q0 * iM, a = 1.0 / (1.0 + gamma);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    double bq = b1 * q[i][1] + b2 * q[i][2] + b3 * q[i][3];
    double e = q[i][0];
    q[i][0] = x * (gamma * e + bq);
    q[i][1] = x * (q[i][1] + b1 * e + a * bq * b1);
    q[i][2] = x * (q[i][2] + b2 * e + a * bq * b2);
    q[i][3] = x * (q[i][3] + b3 * e + a * bq * b3);
  }
  // massless volume (pi/2)^{N-1} w^{2N-4} / ((N-1)! (N-2)!)
  double V0 = 1.0;
#pragma unroll
  for (int j = 0; j < N - 1; ++j) V0 *= 0.5 * kPi;
#pragma unroll
  for (int j = 0; j < 2 * N - 4; ++j) V0 *= w;
  double fact = 1.0;
#pragma unroll
  for (int j = 2; j <= N - 1; ++j) fact *= (double)j;
#pragma unroll
  for (int j = 2; j <= N - 2; ++j) fact *= (double)j;
  V0 /= fact;
  // masses (m_top, m_top, 0, ...): solve sum_i sqrt(m_i^2 + xi^2 p0_i^2) = w
  double m2 = m_top * m_top;
  double r = 2.0 * m_top / w;
  double xi = sqrt(1.0 - r * r);
#pragma unroll 1
  for (int it = 0; it < 10; ++it) {
    double f = -w, df = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
      double mi2 = i < 2 ? m2 : 0.0;
      double p0 = q[i][0];
      double e = sqrt(mi2 + xi * xi * p0 * p0);
      f += e;
      df += xi * p0 * p0 / e;
    }
    xi -= f / df;
  }
  double prod = 1.0, sum = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    double mi2 = i < 2 ? m2 : 0.0;
    double p0 = q[i][0];
    double e = sqrt(mi2 + xi * xi * p0 * p0);
    double kabs = xi * p0;
    q[i][0] = e;
    q[i][1] *= xi; q[i][2] *= xi; q[i][3] *= xi;
    prod *= kabs / e;
    sum += kabs * kabs / e;
  }
  double xipow = 1.0;
#pragma unroll
  for (int j = 0; j < 2 * N - 3; ++j) xipow *= xi;
  return V0 * xipow * prod * w / sum;
}
// one massless RAMBO momentum from its four mapped uniforms
MF_HD void rambo_q(double r1, double r2, double r3, double r4, double q[4]) {
  double c = 2.0 * r1 - 1.0;
  double sphi, cphi;
  sincos(kTwoPi * r2, &sphi, &cphi);
  double q0 = -log(r3 * r4);
  double st = sqrt(1.0 - c * c);
  q[0] = q0; q[1] = q0 * st * cphi; q[2] = q0 * st * sphi; q[3] = q0 * c;
}
template <int N> MF_HD double two_pi_power() {  // (2 pi)^{4-3N}
  double f = 1.0;
#pragma unroll
  for (int j = 0; j < 3 * N - 4; ++j) f /= kTwoPi;
  return f;
}

// a5. Boost along +z with rapidity y (cosh/sinh from one exp pair), and the cut observables.
struct Boost { double ch, sh; };
MF_HD Boost make_boost(double y) {
  double ep = exp(y), em = exp(-y);
  Boost b;
  b.ch = 0.5 * (ep + em);
  b.sh = 0.5 * (ep - em);
  return b;
}
MF_HD void boost_z(const Boost& b, const double in[4], double out[4]) {
  out[0] = in[0] * b.ch + in[3] * b.sh;
  out[1] = in[1];
  out[2] = in[2];
  out[3] = in[3] * b.ch + in[0] * b.sh;
}
// Fiducial cuts on the final gluons in the lab frame (PAPER.md L25(iii), L123; BASELINE.json configs[2,3]):
// pT > ptmin, |eta| < etamax, DeltaR > drmin, strict; a cut <= 0 is disabled.
template <int NGF>
MF_HD bool pass_cuts(const double g[][4], double ptmin, double etamax, double drmin) {
  double eta[NGF > 0 ? NGF : 1], phi[NGF > 0 ? NGF : 1];
#pragma unroll
  for (int i = 0; i < NGF; ++i) {
    double pt = sqrt(g[i][1] * g[i][1] + g[i][2] * g[i][2]);
    if (ptmin > 0.0 && !(pt > ptmin)) return false;
    eta[i] = asinh(g[i][3] / pt);
    if (etamax > 0.0 && !(fabs(eta[i]) < etamax)) return false;
    phi[i] = atan2(g[i][2], g[i][1]);
  }
  if (drmin > 0.0) {
#pragma unroll
    for (int i = 0; i < NGF; ++i)
#pragma unroll
      for (int j = i + 1; j < NGF; ++j) {
        double dphi = fabs(phi[i] - phi[j]);
        if (dphi > kPi) dphi = kTwoPi - dphi;
        double deta = eta[i] - eta[j];
        if (!(sqrt(deta * deta + dphi * dphi) > drmin)) return false;
      }
  }
  return true;
}

}  // namespace mf
