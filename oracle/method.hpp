// ORACLE — TEST INFRASTRUCTURE ONLY (see real.hpp).  Plain, slow, one event at a time.
//
// method.hpp: steps O1–O8 and O13–O15 of SURVEY.md §8(c), i.e. everything on the hot path except the
// matrix element (amplitude.hpp).  The paper names the methods but prints no formula
// ("generation of random numbers, computation of the phase space kinematics, matrix
// element evaluation and histogram accumulation"; L27 VegasFlow/PDFFlow; L71-75 RAMBO; L81 unweighting),
// so each function cites the published method it restates and the DESIGN.md reading it takes.
#pragma once
#include <cstdint>
#include <vector>
#include "real.hpp"

namespace mfo {

// ---------------------------------------------------------------------------------------------
// O1. Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  BASELINE.json north_star names it;
// PAPER.md L61 only says "generation of random numbers".  Ten rounds of
//   c <- ( hi(M1*c2) ^ c1 ^ k0, lo(M1*c2), hi(M0*c0) ^ c3 ^ k1, lo(M0*c0) ),
// the key being bumped by the Weyl constants between rounds.
inline void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// Stream layout (reading R1): key = (seed lo, seed hi); counter = (event lo, event hi,
// iteration, block).  Block b = 0.. yields dims 2b (words 0,1) and 2b+1 (words 2,3); block
// 0xFFFFFFFF yields the accept draw (words 0,1).
inline void philox_block(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t block, uint32_t out[4]) {
  uint32_t ctr[4] = {(uint32_t)event, (uint32_t)(event >> 32), iteration, block};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  philox4x32_10(ctr, key, out);
}

// O2. Two words -> one uniform in (0,1) (reading R2): m = hi*2^20 | lo>>12 (52 bits), u = (2m+1)*2^-53.
// Every value is an exactly representable double.
inline double uniform_from_words(uint32_t hi, uint32_t lo) {
  uint64_t m = ((uint64_t)hi << 20) | (uint64_t)(lo >> 12);
  return (double)(2 * m + 1) * 0x1.0p-53;
}

inline void uniforms_for_event(uint64_t seed, uint32_t iteration, uint64_t event, int D, double* u) {
  for (int b = 0; 2 * b < D; ++b) {
    uint32_t w[4];
    philox_block(seed, iteration, event, (uint32_t)b, w);
    u[2 * b] = uniform_from_words(w[0], w[1]);
    if (2 * b + 1 < D) u[2 * b + 1] = uniform_from_words(w[2], w[3]);
  }
}
inline double accept_draw(uint64_t seed, uint32_t iteration, uint64_t event) {
  uint32_t w[4];
  philox_block(seed, iteration, event, 0xFFFFFFFFu, w);
  return uniform_from_words(w[0], w[1]);
}
// the second uniform of the same block: picks the partonic channel of an accepted event (process 4, reading R18)
inline double channel_draw(uint64_t seed, uint32_t iteration, uint64_t event) {
  uint32_t w[4];
  philox_block(seed, iteration, event, 0xFFFFFFFFu, w);
  return uniform_from_words(w[2], w[3]);
}

// ---------------------------------------------------------------------------------------------
// O3. VEGAS importance-sampling map (Lepage 1978; PAPER.md L27, L61 by citation to VegasFlow).
// grid[d*(nb+1) + i] = edge e_{d,i}, 0 = e_0 < ... < e_nb = 1.
// t = u*nb, i = min(floor t, nb-1), x = e_i + (t-i)(e_{i+1}-e_i), J = prod_d nb (e_{i+1}-e_i).
template <class R>
inline R vegas_map(const double* grid, int D, int nb, const double* u, R* x, int* bin) {
  R jac = R(1);
  for (int d = 0; d < D; ++d) {
    R t = R(u[d]) * R(nb);
    int i = (int)r_to_double(t);  // t >= 0: truncation is floor
    if (i > nb - 1) i = nb - 1;
    R e0 = R(grid[d * (nb + 1) + i]), e1 = R(grid[d * (nb + 1) + i + 1]);
    R width = e1 - e0;
    x[d] = e0 + (t - R(i)) * width;
    jac = jac * (R(nb) * width);
    bin[d] = i;
  }
  return jac;
}

// ---------------------------------------------------------------------------------------------
// O4. Parton fractions (reading R4).  tau = exp((1-x0) ln tau_min), J_tau = -tau ln tau_min;
// y = (x1 - 1/2)(-ln tau), J_y = -ln tau; x1 = sqrt(tau) e^y, x2 = sqrt(tau) e^-y; shat = tau s.
template <class R> struct PartonKin { R tau, y, x1, x2, shat, jac; };
template <class R>
inline PartonKin<R> parton_fractions(R x0, R x1v, R tau_min, R s) {
  PartonKin<R> k;
  R L = r_log(tau_min);
  k.tau = r_exp((R(1) - x0) * L);
  R jtau = -(k.tau * L);
  R mlt = -r_log(k.tau);
  k.y = (x1v - R(0.5)) * mlt;
  R rt = r_sqrt(k.tau);
  k.x1 = rt * r_exp(k.y);
  k.x2 = rt * r_exp(-k.y);
  k.shat = k.tau * s;
  k.jac = jtau * mlt;
  return k;
}

// ---------------------------------------------------------------------------------------------
// O5. Analytic two-body phase space in the partonic CM frame (BASELINE.json: "2-body analytic").
// mom[0..1] = beams along +z/-z, mom[2], mom[3] = final particles of equal mass m.
// dPhi_2 = beta/(32 pi^2) dcos(theta) dphi; with cos = 2xc-1, phi = 2 pi xphi the weight per unit
// (xc, xphi) is beta/(32 pi^2) * 2 * 2 pi.  Returns that weight.
template <class R>
inline R two_body(R shat, R m, R xc, R xphi, R mom[4][4]) {
  R E = r_sqrt(shat) / R(2);
  R c = R(2) * xc - R(1);
  R phi = R(2) * r_pi<R>() * xphi;
  R st = r_sqrt(R(1) - c * c);
  R k = r_sqrt(E * E - m * m);
  mom[0][0] = E; mom[0][1] = R(0); mom[0][2] = R(0); mom[0][3] = E;
  mom[1][0] = E; mom[1][1] = R(0); mom[1][2] = R(0); mom[1][3] = -E;
  mom[2][0] = E; mom[2][1] = k * st * r_cos(phi); mom[2][2] = k * st * r_sin(phi); mom[2][3] = k * c;
  mom[3][0] = E; mom[3][1] = -mom[2][1]; mom[3][2] = -mom[2][2]; mom[3][3] = -mom[2][3];
  R beta = k / E;
  return beta / (R(32) * r_pi<R>() * r_pi<R>()) * R(2) * (R(2) * r_pi<R>());
}

// ---------------------------------------------------------------------------------------------
// O6. RAMBO (Kleiss, Stirling, Ellis, Comput. Phys. Commun. 40 (1986) 359, ref [25]).
// rho[4*i..4*i+3] are the four uniforms of final particle i.  k[i] = massive momenta in the CM frame
// (total (w,0,0,0)).  Returns the phase-space VOLUME weight V (so that dPhi_n = (2 pi)^{4-3n} V).
template <class R>
inline R rambo(int n, const R* mass, R w, const R* rho, R k[][4]) {
  const R pi = r_pi<R>();
  R q[8][4];
  R Q[4] = {R(0), R(0), R(0), R(0)};
  // step 1: isotropic massless q_i with energies distributed as q0 exp(-q0)
  for (int i = 0; i < n; ++i) {
    R c = R(2) * rho[4 * i] - R(1);
    R phi = R(2) * pi * rho[4 * i + 1];
    R q0 = -r_log(rho[4 * i + 2] * rho[4 * i + 3]);
    R s = r_sqrt(R(1) - c * c);
    q[i][0] = q0; q[i][1] = q0 * s * r_cos(phi); q[i][2] = q0 * s * r_sin(phi); q[i][3] = q0 * c;
    for (int m = 0; m < 4; ++m) Q[m] = Q[m] + q[i][m];
  }
  // step 2: conformal transformation to total momentum (w, 0)
  R M = r_sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
  R b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
  R x = w / M, gamma = Q[0] / M, a = R(1) / (R(1) + gamma);
  R p[8][4];
  for (int i = 0; i < n; ++i) {
    R bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
    p[i][0] = x * (gamma * q[i][0] + bq);
    for (int m = 0; m < 3; ++m) p[i][m + 1] = x * (q[i][m + 1] + b[m] * q[i][0] + a * bq * b[m]);
  }
  // step 3: massless volume
  R V0 = R(1);
  for (int j = 0; j < n - 1; ++j) V0 = V0 * (pi / R(2));
  for (int j = 0; j < 2 * n - 4; ++j) V0 = V0 * w;
  R fact = R(1);
  for (int j = 2; j <= n - 1; ++j) fact = fact * R(j);  // (n-1)!
  for (int j = 2; j <= n - 2; ++j) fact = fact * R(j);  // (n-2)!
  V0 = V0 / fact;
  // step 4: masses.  Solve sum_i sqrt(m_i^2 + xi^2 p0_i^2) = w, Newton, fixed 10 iterations (reading R6).
  R summ = R(0);
  bool any_mass = false;
  for (int i = 0; i < n; ++i) { summ = summ + mass[i]; if (mass[i] != R(0)) any_mass = true; }
  if (!any_mass) {
    for (int i = 0; i < n; ++i) for (int m = 0; m < 4; ++m) k[i][m] = p[i][m];
    return V0;
  }
  R xi = r_sqrt(R(1) - (summ / w) * (summ / w));
  for (int it = 0; it < 10; ++it) {
    R f = -w, df = R(0);
    for (int i = 0; i < n; ++i) {
      R e = r_sqrt(mass[i] * mass[i] + xi * xi * p[i][0] * p[i][0]);
      f = f + e;
      df = df + xi * p[i][0] * p[i][0] / e;
    }
    xi = xi - f / df;
  }
  R prod = R(1), sum = R(0);
  for (int i = 0; i < n; ++i) {
    R e = r_sqrt(mass[i] * mass[i] + xi * xi * p[i][0] * p[i][0]);
    k[i][0] = e;
    for (int m = 1; m < 4; ++m) k[i][m] = xi * p[i][m];
    R kabs = xi * p[i][0];
    prod = prod * (kabs / e);
    sum = sum + kabs * kabs / e;
  }
  // step 5: massive volume
  R xipow = R(1);
  for (int j = 0; j < 2 * n - 3; ++j) xipow = xipow * xi;
  return V0 * xipow * prod * w / sum;
}
// (2 pi)^{4-3n}
template <class R> inline R two_pi_power(int n) {
  R f = R(1);
  for (int j = 0; j < 3 * n - 4; ++j) f = f / (R(2) * r_pi<R>());
  return f;
}

// ---------------------------------------------------------------------------------------------
// O7. Boost to the lab frame along +z with rapidity y, and fiducial cuts on the final gluons
// (PAPER.md L25(iii), L123; BASELINE.json configs[2,3] bind which particles and which cuts).
template <class R> inline void boost_z(R y, const R in[4], R out[4]) {
  R ch = (r_exp(y) + r_exp(-y)) / R(2), sh = (r_exp(y) - r_exp(-y)) / R(2);
  out[0] = in[0] * ch + in[3] * sh;
  out[1] = in[1];
  out[2] = in[2];
  out[3] = in[3] * ch + in[0] * sh;
}
template <class R> struct CutObs { R pt, eta, phi; };
template <class R> inline CutObs<R> cut_observables(const R p[4]) {
  CutObs<R> o;
  o.pt = r_sqrt(p[1] * p[1] + p[2] * p[2]);
  o.eta = r_asinh(p[3] / o.pt);
  o.phi = r_atan2(p[2], p[1]);
  return o;
}
template <class R> inline R delta_r(const CutObs<R>& a, const CutObs<R>& b) {
  R dphi = r_fabs(a.phi - b.phi);
  if (dphi > r_pi<R>()) dphi = R(2) * r_pi<R>() - dphi;
  R deta = a.eta - b.eta;
  return r_sqrt(deta * deta + dphi * dphi);
}
// gluons: lab-frame momenta of the ng final gluons.  Strict inequalities; a cut <= 0 is disabled.
template <class R>
inline bool pass_cuts(int ng, const R gluons[][4], R ptmin, R etamax, R drmin) {
  CutObs<R> o[4];
  for (int i = 0; i < ng; ++i) {
    o[i] = cut_observables(gluons[i]);
    if (ptmin > R(0) && !(o[i].pt > ptmin)) return false;
    if (etamax > R(0) && !(r_fabs(o[i].eta) < etamax)) return false;
  }
  if (drmin > R(0))
    for (int i = 0; i < ng; ++i)
      for (int j = i + 1; j < ng; ++j)
        if (!(delta_r(o[i], o[j]) > drmin)) return false;
  return true;
}

// ---------------------------------------------------------------------------------------------
// O8. PDF: log-bicubic (LHAPDF-style) interpolation of x*g on (ln x, ln Q^2) knots (PAPER.md L27
// PDFFlow by citation; BASELINE.json configs[1] gives the table).  Cubic Hermite in ln x on the rows
// j-1..j+2 that exist, then cubic Hermite in ln Q^2, of the VALUE x*g (not of its logarithm).
// Knot derivative: one-sided difference at an end, mean of the two one-sided differences inside.
struct PdfTable {
  int nx = 0, nq = 0;
  std::vector<double> lnx, lnq2, xf;  // xf[ix*nq + iq]
};
template <class R> inline R hermite(R t, R f0, R d0, R f1, R d1, R h) {
  R t2 = t * t, t3 = t2 * t;
  return (R(2) * t3 - R(3) * t2 + R(1)) * f0 + (t3 - R(2) * t2 + t) * h * d0 + (R(-2) * t3 + R(3) * t2) * f1 +
         (t3 - t2) * h * d1;
}
template <class R> inline R pdf_ddx(const PdfTable& T, int i, int j) {  // dF/dlnx at knot (i, j)
  auto F = [&](int a) { return R(T.xf[a * T.nq + j]); };
  auto X = [&](int a) { return R(T.lnx[a]); };
  if (i == 0) return (F(1) - F(0)) / (X(1) - X(0));
  if (i == T.nx - 1) return (F(i) - F(i - 1)) / (X(i) - X(i - 1));
  R left = (F(i) - F(i - 1)) / (X(i) - X(i - 1)), right = (F(i + 1) - F(i)) / (X(i + 1) - X(i));
  return (left + right) / R(2);
}
template <class R> inline R pdf_xf(const PdfTable& T, R x, R q2) {
  R lx = r_log(x), lq = r_log(q2);
  int i = 0;
  while (i < T.nx - 2 && !(lx < R(T.lnx[i + 1]))) ++i;  // lnx_i <= lx < lnx_{i+1}, clamped
  int j = 0;
  while (j < T.nq - 2 && !(lq < R(T.lnq2[j + 1]))) ++j;
  R h = R(T.lnx[i + 1]) - R(T.lnx[i]);
  R t = (lx - R(T.lnx[i])) / h;
  R g[4];  // x-interpolated values on rows j-1 .. j+2
  bool have[4];
  for (int r = 0; r < 4; ++r) {
    int jj = j - 1 + r;
    have[r] = (jj >= 0 && jj < T.nq);
    if (have[r])
      g[r] = hermite<R>(t, R(T.xf[i * T.nq + jj]), pdf_ddx<R>(T, i, jj), R(T.xf[(i + 1) * T.nq + jj]),
                        pdf_ddx<R>(T, i + 1, jj), h);
  }
  R hq = R(T.lnq2[j + 1]) - R(T.lnq2[j]);
  R uq = (lq - R(T.lnq2[j])) / hq;
  R right0 = (g[2] - g[1]) / hq;  // one-sided difference across the cell
  R d0, d1;
  if (have[0]) {
    R left0 = (g[1] - g[0]) / (R(T.lnq2[j]) - R(T.lnq2[j - 1]));
    d0 = (left0 + right0) / R(2);
  } else d0 = right0;
  if (have[3]) {
    R right1 = (g[3] - g[2]) / (R(T.lnq2[j + 2]) - R(T.lnq2[j + 1]));
    d1 = (right0 + right1) / R(2);
  } else d1 = right0;
  return hermite<R>(uq, g[1], d0, g[2], d1, hq);
}

// ---------------------------------------------------------------------------------------------
// O14. VEGAS grid refinement (Lepage; reading R14): smooth, normalise, damp r = ((s-1)/ln s)^alpha,
// rebin to equal sum of r.  In place, per dimension; a dimension with an all-zero histogram is left alone.
template <class R>
inline void refine_grid(double* grid, const double* hist, int D, int nb, R alpha) {
  for (int d = 0; d < D; ++d) {
    const double* h = hist + d * nb;
    double* e = grid + d * (nb + 1);
    std::vector<R> s(nb), r(nb), enew(nb + 1);
    s[0] = (R(h[0]) + R(h[1])) / R(2);
    for (int i = 1; i < nb - 1; ++i) s[i] = (R(h[i - 1]) + R(h[i]) + R(h[i + 1])) / R(3);
    s[nb - 1] = (R(h[nb - 2]) + R(h[nb - 1])) / R(2);
    R S = R(0);
    for (int i = 0; i < nb; ++i) S = S + s[i];
    if (!(S > R(0))) continue;
    R rsum = R(0);
    for (int i = 0; i < nb; ++i) {
      s[i] = s[i] / S;
      if (!(s[i] > R(0))) r[i] = R(0);
      else if (!(s[i] < R(1))) r[i] = R(1);
      else r[i] = r_pow((s[i] - R(1)) / r_log(s[i]), alpha);
      rsum = rsum + r[i];
    }
    R delta = rsum / R(nb);
    R acc = R(0);
    int j = 0;
    enew[0] = R(0);
    enew[nb] = R(1);
    for (int i = 1; i < nb; ++i) {
      while (acc < delta && j < nb) { acc = acc + r[j]; ++j; }
      acc = acc - delta;
      enew[i] = R(e[j]) - (acc / r[j - 1]) * (R(e[j]) - R(e[j - 1]));
    }
    for (int i = 0; i <= nb; ++i) e[i] = r_to_double(enew[i]);
  }
}

}  // namespace mfo
