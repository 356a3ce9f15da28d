// mf_kernels.cuh — the kernels of the fused pass (steps a1-a12, a14 of SURVEY.md 8(a)).
//
// Layout of one launch:
//   * thread = event, grid-stride over the event range; nothing per event touches HBM;
//   * the VEGAS grid, the collapsed PDF row and its ln x knots, and the block's w^2 histogram live in
//     shared memory; per-thread running sums (sum w, sum w^2, max|w|, n_pass, n_accept) live in registers;
//   * at the end: warp shuffle -> shared -> ONE partial record per block in global memory, and the block's
//     histogram to its own slice of a [blocks][D*nb] scratch; a second tiny kernel adds the partials in a
//     fixed order (so the sums do not depend on scheduling; only the shared-memory fp64 atomics of the
//     histogram are order-dependent, at the 1e-16 level).
#pragma once
#include "mf_event.cuh"

namespace mf {

struct BlockPartial {
  double sum_w, sum_w2, max_abs_w;
  unsigned long long n_pass, n_accept;
};
struct IterResult {  // == mf_iter_result
  double sum_w, sum_w2, max_abs_w;
  unsigned long long n_pass, n_accept;
};

// Everything a launch of the fused pass needs besides Params.
struct PassArgs {
  const double* grid;      // [D][nb+1] device
  const double* pdf_lnx;   // [nx] device (nullptr for e+e-)
  const double* pdf_row;   // [nfl][nx] device: every parton table collapsed at mu2
  const double* pdf_lnq2;  // [nq] device, and the full tables [nfl][nx][nq]: the dynamic-scale path only
  const double* pdf_xf;
  uint64_t seed, first_event, n_events;
  uint32_t iteration;
  double w_max;            // unweighting only
  char* records;           // unweighting only
  uint64_t capacity;
  unsigned long long* count;
  BlockPartial* partials;  // [gridDim.x]
  double* hist_part;       // [gridDim.x][D*nb] or nullptr
  double* obs;             // observable histograms [2][obs_nb + 1] (added to) or nullptr (mf_set_observables)
  int obs_nb;
  double obs_ptmax, obs_etamax;
  const double* quark_terms;  // pp -> ttbar gg: the quark-channel term of every event (quark_prepass_kernel) or nullptr
  double* coop_queue;      // cooperative kernels only: [gridDim.x][blockDim.x][18] momenta queue (mf_kernels_coop.cuh)
};

#define MF_ME_CALL __device__ __forceinline__
// The matrix element is the only large piece of code, with ONE call site per thread-per-event kernel: inlined, so that
// the momenta stay in registers (an out-of-line call passes them through local memory: +4 % / +9 % time for gg -> ttbar /
// e+e- -> mu+mu-).
template <int PROC>
MF_ME_CALL double me2_call(const Params& P, double shat, const double (*k)[4]) {
  return matrix_element<PROC>(P, shat, k);
}

// process 4: both channels in ONE out-of-line call, so that the top-quark spinors are formed once
MF_ME_CALL double me2_pp_call(const Params& P, double shat, const double (*k)[4], double& me_qq) {
  me_qq = matrix_element_qq(P, shat, k);
  return matrix_element<4>(P, shat, k);
}

// process 5: |M|^2 of the six quark-channel classes (0 q qbar, 1 qbar q, 2 q g, 3 g q, 4 qbar g, 5 g qbar; first parton from
// beam 1) at the CM-frame point, in one call that shares the top line's currents between the classes with the same gluon
// (mf_me_qttg.cuh).  Out of line: one copy per kernel.
__device__ __noinline__ void quark_gluon_me2_all(const Params& P, double shat, const double (*k)[4], double M[6]) {
  const double E = 0.5 * sqrt(shat);
  const double b1[4] = {E, 0.0, 0.0, E}, b2[4] = {E, 0.0, 0.0, -E};
  me2_ttj_quark_classes(b1, b2, k[0], k[1], k[2], P.m_top, 4.0 * kPi * P.alpha_s, M);
}

// process 7: |M|^2 of q qbar -> t tbar g g with the quark from beam 1 (Ma) and from beam 2 (Mb) (mf_me_qqttgg.cuh).
// Out of line: one copy per kernel.
__device__ __noinline__ void quark_pair_me2_gg(const Params& P, double shat, const double (*k)[4], double M[2]) {
  const double E = 0.5 * sqrt(shat);
  const double g2 = 4.0 * kPi * P.alpha_s;
#pragma unroll 1
  for (int o = 0; o < 2; ++o) {            // one copy of the code for both assignments
    const double pz = o == 0 ? E : -E;
    const double bq[4] = {E, 0.0, 0.0, pz}, bqbar[4] = {E, 0.0, 0.0, -pz};
    M[o] = me2_qq_ttgg(bq, bqbar, k[0], k[1], k[2], k[3], P.m_top, g2);
  }
}

// Luminosity (step a6): F(x1) F(x2) / (x1 x2) with F the interpolant of the collapsed row in shared memory; and
// the factor that rescales |M|^2 (1 at the fixed scale).  Dynamic scale (R16; mf_set_dynamic_scale):
// mu_F^2 = mu_R^2 = m_t^2 + pT(top)^2 per event, F by the general 2-D lookup in the table (global memory / L2),
// alpha_s running at one loop (n_f = 5) from its value at the descriptor's mu2: |M|^2 ~ alpha_s^{n_g}.
// (the two general 2-D lookups of the rarely used dynamic scale are kept out of line: the fused kernels are
// instruction-cache sensitive)
__device__ __noinline__ double pdf_pair_2d(const Params& P, const PassArgs& A, double x1, double x2, double mu2,
                                           double& f2) {
  f2 = pdf_xf_2d(A.pdf_lnx, A.pdf_lnq2, A.pdf_xf, P.pdf_nx, P.pdf_nq, x2, mu2);
  return pdf_xf_2d(A.pdf_lnx, A.pdf_lnq2, A.pdf_xf, P.pdf_nx, P.pdf_nq, x1, mu2);
}
template <int PROC>
MF_D double luminosity(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                       const Event<PROC>& ev, double& as_factor) {
  as_factor = 1.0;
  if (PROC == 0) return 1.0;
  double f1, f2;
  if (P.dyn_scale) {
    const double mu2 = P.m_top * P.m_top + ev.k[0][1] * ev.k[0][1] + ev.k[0][2] * ev.k[0][2];
    f1 = pdf_pair_2d(P, A, ev.x1, ev.x2, mu2, f2);
    const double ratio = 1.0 / (1.0 + P.alpha_s * (23.0 / (12.0 * kPi)) * log(mu2 / P.mu2));
#pragma unroll
    for (int g = 0; g < Traits<PROC>::NG; ++g) as_factor *= ratio;
  } else {
    f1 = pdf_xf_row(s_lnx, s_row, P.pdf_nx, ev.x1);
    f2 = pdf_xf_row(s_lnx, s_row, P.pdf_nx, ev.x2);
  }
  return f1 * f2 / (ev.x1 * ev.x2);
}

// Process 4 (gg + q qbar channels; R17): x f(x) of every parton table at both beams; rows /
// tables are ordered gluon, q_0, qbar_0, q_1, qbar_1, ...
// Dynamic scale (rare, large code): out of line and rolled, through memory.
__device__ __noinline__ void parton_densities_dyn(const Params& P, const PassArgs& A, double x1, double x2, double mu2,
                                                  double* f1, double* f2) {
  const size_t tab = (size_t)P.pdf_nx * P.pdf_nq;
#pragma unroll 1
  for (int t = 0; t < P.pdf_nfl; ++t) {
    f1[t] = pdf_xf_2d(A.pdf_lnx, A.pdf_lnq2, A.pdf_xf + t * tab, P.pdf_nx, P.pdf_nq, x1, mu2);
    f2[t] = pdf_xf_2d(A.pdf_lnx, A.pdf_lnq2, A.pdf_xf + t * tab, P.pdf_nx, P.pdf_nq, x2, mu2);
  }
}
// Fixed scale (the hot path): one logarithm and one cell search per beam serve all rows; everything in registers.
template <int PROC>
MF_D void parton_densities(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                           const Event<PROC>& ev, double* f1, double* f2, double& as_factor) {
  as_factor = 1.0;
  const int nt = P.pdf_nfl;
  if (P.dyn_scale) {
    const double mu2 = P.m_top * P.m_top + ev.k[0][1] * ev.k[0][1] + ev.k[0][2] * ev.k[0][2];
    double g1[kMaxPartonTables], g2[kMaxPartonTables];
    parton_densities_dyn(P, A, ev.x1, ev.x2, mu2, g1, g2);
#pragma unroll
    for (int t = 0; t < kMaxPartonTables; ++t)
      if (t < nt) { f1[t] = g1[t]; f2[t] = g2[t]; }
    const double ratio = 1.0 / (1.0 + P.alpha_s * (23.0 / (12.0 * kPi)) * log(mu2 / P.mu2));
#pragma unroll
    for (int g = 0; g < Traits<PROC>::NG; ++g) as_factor *= ratio;
  } else {
    const HermiteWeights W1 = hermite_weights(s_lnx, P.pdf_nx, ev.x1), W2 = hermite_weights(s_lnx, P.pdf_nx, ev.x2);
#pragma unroll
    for (int t = 0; t < kMaxPartonTables; ++t)
      if (t < nt) {
        f1[t] = hermite_apply(W1, s_row + t * P.pdf_nx, P.pdf_nx);
        f2[t] = hermite_apply(W2, s_row + t * P.pdf_nx, P.pdf_nx);
      }
  }
}

// the gluon-gluon luminosity (returned) and the flavour-summed quark luminosity
//   lum_qq = sum_i [ q_i(x1) qbar_i(x2) + qbar_i(x1) q_i(x2) ] / (x1 x2)
MF_D double luminosity_pp(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                          const Event<4>& ev, double& as_factor, double& lum_qq, double* f1, double* f2) {
  parton_densities<4>(P, A, s_lnx, s_row, ev, f1, f2, as_factor);
  const int nt = P.pdf_nfl;
  const double inv = 1.0 / (ev.x1 * ev.x2);
  double a = 0.0, b = 0.0;
#pragma unroll
  for (int t = 1; t + 1 < kMaxPartonTables; t += 2)
    if (t + 1 < nt) {
      a = fma(f1[t], f2[t + 1], a);
      b = fma(f1[t + 1], f2[t], b);
    }
  lum_qq = (a + b) * inv;
  return f1[0] * f2[0] * inv;
}

// pp -> ttbar j (R19): the gluon-gluon luminosity (returned) and the sum over the six flavour-summed
// quark-channel classes of luminosity x |M|^2 (x the R16 factor):
//   0: q qbar   1: qbar q   2: q g   3: g q   4: qbar g   5: g qbar      (first parton from beam 1)
// terms (optional): the six products, for the debug rows.
MF_D double pp_ttj_terms(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                         const Event<5>& ev, double& asf, double& quark_sum, double* terms) {
  double f1[kMaxPartonTables], f2[kMaxPartonTables];
  parton_densities<5>(P, A, s_lnx, s_row, ev, f1, f2, asf);
  const int nt = P.pdf_nfl;
  double Q1 = 0.0, Qb1 = 0.0, Q2 = 0.0, Qb2 = 0.0, D12 = 0.0, D21 = 0.0;
#pragma unroll
  for (int t = 1; t + 1 < kMaxPartonTables; t += 2)
    if (t + 1 < nt) {
      Q1 += f1[t]; Qb1 += f1[t + 1]; Q2 += f2[t]; Qb2 += f2[t + 1];
      D12 = fma(f1[t], f2[t + 1], D12);
      D21 = fma(f1[t + 1], f2[t], D21);
    }
  const double inv = 1.0 / (ev.x1 * ev.x2);
  const double l0 = D12 * inv, l1 = D21 * inv, l2 = Q1 * f2[0] * inv, l3 = f1[0] * Q2 * inv, l4 = Qb1 * f2[0] * inv,
               l5 = f1[0] * Qb2 * inv;
  double M[6];
  quark_gluon_me2_all(P, ev.shat, ev.k, M);
  double sum = 0.0;
#pragma unroll
  for (int c = 0; c < 6; ++c) {
    const double lc = c == 0 ? l0 : c == 1 ? l1 : c == 2 ? l2 : c == 3 ? l3 : c == 4 ? l4 : l5;
    const double term = lc * (M[c] * asf);
    if (terms) terms[c] = term;
    sum += term;
  }
  quark_sum = sum;
  return f1[0] * f2[0] * inv;
}

// pp -> ttbar gg (R22): the gluon-gluon luminosity (returned) and the flavour-summed quark term
//   quark_sum = sum_i [ q_i(x1) qbar_i(x2) Ma + qbar_i(x1) q_i(x2) Mb ] / (x1 x2)   (x the R16 factor)
// parts (optional, debug rows): the flavour-summed q qbar luminosity and the luminosity-weighted mean of Ma, Mb.
MF_D double quark_pair_luminosities(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                                    const Event<7>& ev, double& asf, double& La, double& Lb) {
  double f1[kMaxPartonTables], f2[kMaxPartonTables];
  parton_densities<7>(P, A, s_lnx, s_row, ev, f1, f2, asf);
  const int nt = P.pdf_nfl;
  La = 0.0;
  Lb = 0.0;
#pragma unroll
  for (int t = 1; t + 1 < kMaxPartonTables; t += 2)
    if (t + 1 < nt) {
      La = fma(f1[t], f2[t + 1], La);
      Lb = fma(f1[t + 1], f2[t], Lb);
    }
  const double inv = 1.0 / (ev.x1 * ev.x2);
  La *= inv;
  Lb *= inv;
  return f1[0] * f2[0] * inv;
}
MF_D double pp_ttgg_terms(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                          const Event<7>& ev, double& asf, double& quark_sum, double* parts) {
  double La, Lb;
  const double lum = quark_pair_luminosities(P, A, s_lnx, s_row, ev, asf, La, Lb);
  double M[2];
  quark_pair_me2_gg(P, ev.shat, ev.k, M);
  const double both = La * (M[0] * asf) + Lb * (M[1] * asf);
  if (parts) {
    parts[0] = La + Lb;
    parts[1] = (La + Lb) != 0.0 ? both / (La + Lb) : M[0] * asf;
  }
  quark_sum = both;
  return lum;
}

// a6-a10 of one event that passed the cuts (thread-per-event kernels): luminosity, |M|^2, weight.
// parts (optional): lum, me2 [, lum_qq, me2_qq for process 4] for the debug rows.
// channel (optional, process 4; R18): the partonic channel this event gets IF it is accepted, drawn in
// proportion to |luminosity x |M|^2| of the channels, in channel order (0 gg; 1 + 2 i quark i from beam 1; 2 + 2 i quark
// i from beam 2): the first c with sum_{c' <= c} |a_c'| > v sum |a|, v = the second uniform of the accept block.  It
// is formed here, where the densities are in registers (a few dozen flop), not again for the accepted events.
template <int PROC>
MF_D double weigh_event(const Params& P, const PassArgs& A, const double* s_lnx, const double* s_row,
                        const Event<PROC>& ev, double* parts, double v = 0.0, unsigned* channel = nullptr) {
  double asf;
  if constexpr (PROC == 4) {
    double lum_qq, f1[kMaxPartonTables], f2[kMaxPartonTables];
    const double lum = luminosity_pp(P, A, s_lnx, s_row, ev, asf, lum_qq, f1, f2);
    double me_qq;
    const double me_gg = me2_pp_call(P, ev.shat, ev.k, me_qq) * asf;
    me_qq *= asf;
    if (parts) { parts[0] = lum; parts[1] = me_gg; parts[2] = lum_qq; parts[3] = me_qq; }
    if (channel) {
      const int nt = P.pdf_nfl;
      const double inv = 1.0 / (ev.x1 * ev.x2);
      double a[kMaxPartonTables], total;
      a[0] = total = fabs(lum * me_gg);
#pragma unroll
      for (int t = 1; t + 1 < kMaxPartonTables; t += 2)
        if (t + 1 < nt) {
          a[t] = fabs(f1[t] * f2[t + 1] * inv * me_qq);
          a[t + 1] = fabs(f1[t + 1] * f2[t] * inv * me_qq);
          total += a[t];
          total += a[t + 1];
        }
      const double vt = v * total;
      double cum = 0.0;
      unsigned pick = (unsigned)(nt - 1);
      bool found = false;
#pragma unroll
      for (int c = 0; c < kMaxPartonTables; ++c)
        if (c < nt) {
          cum += a[c];
          if (!found && cum > vt) { pick = (unsigned)c; found = true; }
        }
      *channel = pick;
    }
    return event_weight<PROC>(P, ev, 1.0, fma(lum, me_gg, lum_qq * me_qq));
  } else if constexpr (PROC == 5) {
    double quark_sum;
    const double lum = pp_ttj_terms(P, A, s_lnx, s_row, ev, asf, quark_sum, parts ? parts + 2 : nullptr);
    const double me_gg = me2_call<PROC>(P, ev.shat, ev.k) * asf;
    if (parts) { parts[0] = lum; parts[1] = me_gg; }
    return event_weight<PROC>(P, ev, 1.0, fma(lum, me_gg, quark_sum));
  } else {
    const double lum = luminosity<PROC>(P, A, s_lnx, s_row, ev, asf);
    const double me2 = me2_call<PROC>(P, ev.shat, ev.k) * asf;
    if (parts) { parts[0] = lum; parts[1] = me2; }
    return event_weight<PROC>(P, ev, lum, me2);
  }
}

// Lab-frame momenta of an event, beams first (record / debug-row layout).
template <int PROC>
MF_D void lab_momenta(const Event<PROC>& ev, double out[][4]) {
  constexpr int NF = Traits<PROC>::NF;
  Boost b = make_boost(ev.y);
  double E = 0.5 * sqrt(ev.shat);
  double p1[4] = {E, 0.0, 0.0, E}, p2[4] = {E, 0.0, 0.0, -E};
  boost_z(b, p1, out[0]);
  boost_z(b, p2, out[1]);
#pragma unroll
  for (int i = 0; i < NF; ++i) boost_z(b, ev.k[i], out[2 + i]);
}

MF_D double accept_draw(uint64_t seed, uint32_t iteration, uint64_t event) {
  U4 r = philox_block(seed, iteration, event, 0xFFFFFFFFu);
  return uniform52(r.x, r.y);
}

// Observable bins of an event ("histogram accumulation"; L109-119: d sigma / d pT,top, d sigma / d eta,top):
// lab-frame pT and pseudorapidity of the FIRST final-state particle (the top quark; mu- for e+e-).  Returns the pT bin
// in the low 16 bits and the eta bin in the high 16 bits; bin obs_nb = outside [0, pt_max) resp. [-eta_max, eta_max).
template <int PROC>
MF_D int observable_bins(const PassArgs& A, const Event<PROC>& ev) {
  const Boost b = make_boost(ev.y);
  double t[4];
  boost_z(b, ev.k[0], t);
  const int nb = A.obs_nb;
  const double pt = sqrt(t[1] * t[1] + t[2] * t[2]);
  const double eta = asinh(t[3] / pt);
  const double bp = pt / A.obs_ptmax * nb, be = (eta + A.obs_etamax) / (2.0 * A.obs_etamax) * nb;
  const int ip = bp < nb ? (int)bp : nb;
  const int ie = (be >= 0.0 && be < nb) ? (int)be : nb;
  return ip | (ie << 16);
}

constexpr int kThreads = 128;

// pp -> ttbar j (R20): the partonic channel of an ACCEPTED event: code 0 = gg, code 1 + 6 i + c = flavour i in class
// c (0 q qbar, 1 qbar q, 2 q g, 3 g q, 4 qbar g, 5 g qbar; first parton from beam 1), drawn in proportion to
// |luminosity x |M|^2| in code order: the first code whose cumulative sum exceeds v x the total, v = the second uniform of
// the event's accept block.  Accepted events are rare (< 1 %): everything is recomputed here from the
// tables in global memory; the gluon channel's term (the team's matrix element is not kept) is what the event's weight w
// leaves after the quark terms: w = common x (gg term + sum of the signed quark terms).
// (inlined: as an out-of-line function inside the fused pass, with nvcc 12.9 for sm_100a, it received its weight argument as 0,
// by value or through a struct; inlined there it cost 12 % of the step, so it now runs in record_kernel after the pass)
__device__ __forceinline__ unsigned pp_ttj_channel(const Params& P, const PassArgs& A, const Event<5>& ev, double w, double v) {
  double f1[kMaxPartonTables], f2[kMaxPartonTables], asf;
  parton_densities<5>(P, A, A.pdf_lnx, A.pdf_row, ev, f1, f2, asf);
  const int nf = (P.pdf_nfl - 1) / 2;
  const double inv = 1.0 / (ev.x1 * ev.x2);
  double M[6];
  quark_gluon_me2_all(P, ev.shat, ev.k, M);
#pragma unroll
  for (int c = 0; c < 6; ++c) M[c] *= asf;
  auto sterm = [&](int i, int c) {
    const double q1 = f1[1 + 2 * i], qb1 = f1[2 + 2 * i], q2 = f2[1 + 2 * i], qb2 = f2[2 + 2 * i];
    const double l = c == 0 ? q1 * qb2 : c == 1 ? qb1 * q2 : c == 2 ? q1 * f2[0] : c == 3 ? f1[0] * q2 : c == 4 ? qb1 * f2[0] : f1[0] * qb2;
    return l * inv * M[c];
  };
  auto term = [&](int i, int c) { return fabs(sterm(i, c)); };
  double quark_sum = 0.0;
  for (int i = 0; i < nf; ++i)
    for (int c = 0; c < 6; ++c) quark_sum += sterm(i, c);
  const double gg_term = w / event_weight<5>(P, ev, 1.0, 1.0) - quark_sum;
  double total = fabs(gg_term);
  for (int i = 0; i < nf; ++i)
    for (int c = 0; c < 6; ++c) total += term(i, c);
  const double vt = v * total;
  double cum = fabs(gg_term);
  if (cum > vt) return 0u;
  for (int i = 0; i < nf; ++i)
    for (int c = 0; c < 6; ++c) {
      cum += term(i, c);
      if (cum > vt) return (unsigned)(1 + 6 * i + c);
    }
  return (unsigned)(6 * nf);
}

// pp -> ttbar gg (R22): the partonic channel of an ACCEPTED event, codes as for pp -> ttbar (0 gg; 1 + 2 i quark i
// from beam 1; 2 + 2 i quark i from beam 2), drawn as in pp_ttj_channel (the gluon channel's term is what w leaves).
__device__ __forceinline__ unsigned pp_ttgg_channel(const Params& P, const PassArgs& A, const Event<7>& ev, double w, double v) {
  double f1[kMaxPartonTables], f2[kMaxPartonTables], asf;
  parton_densities<7>(P, A, A.pdf_lnx, A.pdf_row, ev, f1, f2, asf);
  const int nt = P.pdf_nfl;
  const double inv = 1.0 / (ev.x1 * ev.x2);
  double M[2];
  quark_pair_me2_gg(P, ev.shat, ev.k, M);
  auto sterm = [&](int t) { return (t & 1) ? f1[t] * f2[t + 1] * inv * (M[0] * asf) : f1[t] * f2[t - 1] * inv * (M[1] * asf); };
  double quark_sum = 0.0;
  for (int t = 1; t < nt; ++t) quark_sum += sterm(t);
  const double gg_term = w / event_weight<7>(P, ev, 1.0, 1.0) - quark_sum;
  double total = fabs(gg_term);
  for (int t = 1; t < nt; ++t) total += fabs(sterm(t));
  const double vt = v * total;
  double cum = fabs(gg_term);
  if (cum > vt) return 0u;
  for (int t = 1; t < nt; ++t) {
    cum += fabs(sterm(t));
    if (cum > vt) return (unsigned)t;
  }
  return (unsigned)(nt - 1);
}

// processes whose accepted records are completed by record_kernel after the pass: the one-warp-team kernels (g g -> t tbar g:
// 9.58 -> 9.26 ms per 2^22 events; pp -> ttbar j: 20.3 -> 19.5 ms) and pp -> ttbar gg (its channel draw); g g -> t tbar g g and
// g g -> t tbar g g g write their records in the pass (no gain from deferring, and one launch fewer per step)
__host__ __device__ constexpr bool defers_record(int proc) { return proc == 2 || proc == 5 || proc == 7; }

// Per-thread running sums of the pass (registers).
struct Accum {
  double sum_w = 0.0, sum_w2 = 0.0, max_w = 0.0;
  unsigned long long n_pass = 0, n_acc = 0;
};

// a11/a12/a14 for one event (called by every thread of a warp, valid or not): running sums, the block's
// shared-memory w^2 histogram, and hit-or-miss unweighting with a warp-aggregated cursor.
template <int PROC, bool UNW>
MF_D void accumulate_event(const Params& P, const PassArgs& A, const double* s_grid, double* s_hist, bool valid,
                           uint64_t event, double w, const Bins<PROC>& bins, Accum& acc, int obs_bins,
                           unsigned channel = 0u, const Event<PROC>* ev_live = nullptr) {
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  const int nb = P.n_bins;
  const double w2 = w * w;
  acc.sum_w += w;
  acc.sum_w2 += w2;
  acc.max_w = fmax(acc.max_w, fabs(w));
  if (w != 0.0) {
#pragma unroll
    for (int d = 0; d < D; ++d) atomicAdd(&s_hist[d * nb + bins.get(d)], w2);
    if (A.obs != nullptr) {   // observable histograms accumulate the weights themselves (global memory, L2 atomics)
      atomicAdd(A.obs + (obs_bins & 0xFFFF), w);
      atomicAdd(A.obs + (A.obs_nb + 1) + (obs_bins >> 16), w);
    }
  }
  if (UNW) {
    // a14: hit-or-miss against w_max; one global atomic per warp with survivors
    bool ok = false;
    if (valid && w != 0.0) ok = accept_draw(A.seed, A.iteration, event) * A.w_max < fabs(w);
    unsigned m = __ballot_sync(0xFFFFFFFFu, ok);
    if (m) {
      const int lane = threadIdx.x & 31;
      unsigned long long base = 0;
      if (lane == __ffs(m) - 1) base = atomicAdd(A.count, (unsigned long long)__popc(m));
      base = __shfl_sync(0xFFFFFFFFu, base, __ffs(m) - 1);
      if (ok) {
        ++acc.n_acc;
        unsigned long long slot = base + __popc(m & ((1u << lane) - 1u));
        if (A.records != nullptr && slot < A.capacity) {
          constexpr int kRec = (NF + 2) * 32 + 16 + ((PROC == 4 || PROC == 5 || PROC == 7) ? 8 : 0);
          double* rec = reinterpret_cast<double*>(A.records + slot * (uint64_t)kRec);
          rec[4 * (NF + 2)] = w;
          reinterpret_cast<unsigned long long*>(rec)[4 * (NF + 2) + 1] = event;
          if constexpr (defers_record(PROC)) {
            // the thread does not hold the event any more (registers), and accepted events are
            // rare (< 1 %): record_kernel, next on the stream, regenerates the event from its id and fills in the momenta
            // (and, for pp -> ttbar j / gg, the partonic channel); here only the weight and the id are written
          } else {
            // the thread-per-event kernels pass the event they still hold; the others regenerate it here
            Event<PROC> ev;
            if (ev_live != nullptr) {
              ev = *ev_live;
            } else {
              Bins<PROC> b2;
              DebugRow dbg = {nullptr, D, NF};
              generate_event<PROC>(P, s_grid, A.seed, A.iteration, event, ev, b2, dbg);
            }
            double mom[NF + 2][4];
            lab_momenta<PROC>(ev, mom);
#pragma unroll
            for (int i = 0; i < NF + 2; ++i)
#pragma unroll
              for (int c = 0; c < 4; ++c) rec[4 * i + c] = mom[i][c];
            if (PROC == 4) reinterpret_cast<unsigned long long*>(rec)[4 * (NF + 2) + 2] = channel;
          }
        }
      }
    }
  }
}

// Completes the records an mf_unweight call of a cooperative / block process has just written (weight and event id), slots
// [*start, min(*A.count, A.capacity)): thread = record; the event is regenerated from its id, its lab-frame momenta stored and,
// for pp -> ttbar j / pp -> ttbar gg (R20 / R22), the partonic channel drawn from the record's weight and the event's accept
// block.  Accepted events are rare (< 1 %), so this costs microseconds; inside the fused pass the same code cost registers
// and instruction cache in a loop that almost never runs it (pp -> ttbar j: 20 % of the step with the channel draw).
template <int PROC>
__global__ void __launch_bounds__(kThreads) record_kernel(const Params P, const PassArgs A, const unsigned long long* start) {
  static_assert(defers_record(PROC), "thread-per-event kernels write their records themselves");
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  constexpr int kRec = (NF + 2) * 32 + 16 + ((PROC == 5 || PROC == 7) ? 8 : 0);
  const unsigned long long first = *start, cnt = *A.count;
  const unsigned long long last = cnt < A.capacity ? cnt : A.capacity;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long slot = first + (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; slot < last; slot += stride) {
    double* rec = reinterpret_cast<double*>(A.records + slot * (uint64_t)kRec);
    const double w = rec[4 * (NF + 2)];
    const unsigned long long event = reinterpret_cast<unsigned long long*>(rec)[4 * (NF + 2) + 1];
    Event<PROC> ev;
    Bins<PROC> bins;
    DebugRow dbg = {nullptr, D, NF};
    generate_event<PROC>(P, A.grid, A.seed, A.iteration, event, ev, bins, dbg);
    double mom[NF + 2][4];
    lab_momenta<PROC>(ev, mom);
#pragma unroll
    for (int i = 0; i < NF + 2; ++i)
#pragma unroll
      for (int c = 0; c < 4; ++c) rec[4 * i + c] = mom[i][c];
    if constexpr (PROC == 5 || PROC == 7) {
      const U4 r = philox_block(A.seed, A.iteration, event, 0xFFFFFFFFu);      // words z, w: the channel draw
      unsigned ch;
      if constexpr (PROC == 5) ch = pp_ttj_channel(P, A, ev, w, uniform52(r.z, r.w));
      else ch = pp_ttgg_channel(P, A, ev, w, uniform52(r.z, r.w));
      reinterpret_cast<unsigned long long*>(rec)[4 * (NF + 2) + 2] = ch;
    }
  }
}

// a11 (warp shuffle -> shared -> ONE partial per block, fixed order) and the a12 histogram flush.
// s_red: 5 * 32 doubles.  Contains a __syncthreads: every thread of the block must call it.
MF_D void block_finish(const PassArgs& A, Accum acc, double* s_red, const double* s_hist, int n_hist) {
  double sum_w = acc.sum_w, sum_w2 = acc.sum_w2, max_w = acc.max_w;
  unsigned long long n_pass = acc.n_pass, n_acc = acc.n_acc;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    sum_w += __shfl_down_sync(0xFFFFFFFFu, sum_w, o);
    sum_w2 += __shfl_down_sync(0xFFFFFFFFu, sum_w2, o);
    max_w = fmax(max_w, __shfl_down_sync(0xFFFFFFFFu, max_w, o));
    n_pass += __shfl_down_sync(0xFFFFFFFFu, n_pass, o);
    n_acc += __shfl_down_sync(0xFFFFFFFFu, n_acc, o);
  }
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  if (lane == 0) {
    s_red[warp] = sum_w;
    s_red[32 + warp] = sum_w2;
    s_red[64 + warp] = max_w;
    s_red[96 + warp] = __longlong_as_double((long long)n_pass);
    s_red[128 + warp] = __longlong_as_double((long long)n_acc);
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    BlockPartial bp = {0.0, 0.0, 0.0, 0ull, 0ull};
    for (int i = 0; i < nwarp; ++i) {
      bp.sum_w += s_red[i];
      bp.sum_w2 += s_red[32 + i];
      bp.max_abs_w = fmax(bp.max_abs_w, s_red[64 + i]);
      bp.n_pass += (unsigned long long)__double_as_longlong(s_red[96 + i]);
      bp.n_accept += (unsigned long long)__double_as_longlong(s_red[128 + i]);
    }
    A.partials[blockIdx.x] = bp;
  }
  if (A.hist_part != nullptr) {
    double* dst = A.hist_part + (size_t)blockIdx.x * n_hist;
    for (int i = threadIdx.x; i < n_hist; i += blockDim.x) dst[i] = s_hist[i];
  }
}

// ---- the fused pass, one thread per event (e+e- -> mu+mu-, gg -> ttbar, pp -> ttbar) ----------------------
// Lock-step: a block barrier at the top of every grid-stride round keeps the four warps of a block on the same part of the
// (straight-line, once-per-event) matrix-element code, so one warp's instruction fetches serve all four (ncu on gg -> ttbar:
// no_instruction 1.19 warps per issue without it).  Measured per 2^20 events (profiles/r2_tpe.md): gg -> ttbar 0.292 -> 0.271 ms,
// with 3 instead of 4 blocks per SM (168 registers: fewer spills) 0.267 ms; pp -> ttbar 0.429 -> 0.402 ms (3 blocks per SM:
// 0.437 ms); e+e- -> mu+mu- 0.112 -> 0.118 ms (its code is small: no barrier there).
#ifndef MF_TPE_BLOCKS1
#define MF_TPE_BLOCKS1 3
#endif
#ifndef MF_TPE_BLOCKS4
#define MF_TPE_BLOCKS4 2
#endif
#ifndef MF_TPE_LOCKSTEP
#define MF_TPE_LOCKSTEP 1
#endif
template <int PROC, bool UNW>
__global__ void __launch_bounds__(kThreads, PROC == 1 ? MF_TPE_BLOCKS1 : PROC == 4 ? MF_TPE_BLOCKS4 : 2)
    fused_pass_kernel(const Params P, const PassArgs A) {
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  extern __shared__ double smem[];
  const int nb = P.n_bins, nx = PROC == 0 ? 0 : P.pdf_nx, nrow = (PROC == 4 || PROC == 5) ? nx * P.pdf_nfl : nx;
  double* s_grid = smem;                    // D*(nb+1)
  double* s_hist = s_grid + D * (nb + 1);   // D*nb
  double* s_lnx = s_hist + D * nb;          // nx
  double* s_row = s_lnx + nx;               // nx (process 4: one row per parton table)
  double* s_red = s_row + nrow;             // 5 * 32
  for (int i = threadIdx.x; i < D * (nb + 1); i += blockDim.x) s_grid[i] = A.grid[i];
  for (int i = threadIdx.x; i < D * nb; i += blockDim.x) s_hist[i] = 0.0;
  for (int i = threadIdx.x; i < nx; i += blockDim.x) s_lnx[i] = A.pdf_lnx[i];
  for (int i = threadIdx.x; i < nrow; i += blockDim.x) s_row[i] = A.pdf_row[i];
  __syncthreads();

  Accum acc;
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  const uint64_t rounds = (A.n_events + stride - 1) / stride;
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (uint64_t rd = 0; rd < rounds; ++rd, idx += stride) {
#if MF_TPE_LOCKSTEP
    if (PROC != 0) __syncthreads();
#endif
    const bool valid = idx < A.n_events;
    const uint64_t event = A.first_event + idx;
    double w = 0.0;
    Bins<PROC> bins;
    bins.clear();
    int obs_bins = 0;
    unsigned channel = 0u;
    Event<PROC> ev;
    if (valid) {
      DebugRow dbg = {nullptr, D, NF};
      generate_event<PROC>(P, s_grid, A.seed, A.iteration, event, ev, bins, dbg);
      if (ev.pass && A.obs != nullptr) obs_bins = observable_bins<PROC>(A, ev);
      if (ev.pass) {
        ++acc.n_pass;
        if (PROC == 4 && UNW) {
          const U4 r = philox_block(A.seed, A.iteration, event, 0xFFFFFFFFu);      // words z, w: the channel draw
          w = weigh_event<PROC>(P, A, s_lnx, s_row, ev, nullptr, uniform52(r.z, r.w), &channel);
        } else {
          w = weigh_event<PROC>(P, A, s_lnx, s_row, ev, nullptr);
        }
      }
    }
    accumulate_event<PROC, UNW>(P, A, s_grid, s_hist, valid, event, w, bins, acc, obs_bins, channel, PROC == 0 ? nullptr : &ev);
  }
  block_finish(A, acc, s_red, s_hist, D * nb);
}

// ---- pp -> ttbar gg: the quark channel, BEFORE the cooperative pass ---------------------------------------------------------
// out[i] = sum over the flavours and the two beam assignments of luminosity x |M(q qbar -> t tbar g g)|^2 (x the R16 factor) of
// event first_event + i (0 if it fails the cuts): the term the cooperative pass adds to  L_gg |M_gg|^2.
// Thread = event for a1-a6; the matrix element of every event that passed is then evaluated by a whole WARP
// (me2_qq_ttgg_warp: lane = beam assignment x polarisation pair x top spin state, the light line's currents shared through
// 7.4 kB of shared memory per warp, everything else in registers).  As thread-per-event code (~4 kB of thread-local state per
// event) it ran from local memory: 350 ms per 2^22 events on the owner threads of the cooperative kernel, 103 ms in a
// thread-per-event kernel of its own (profiles/r2_c8.md).
// The block's warps step through the block's passing events together (ranked queue in shared memory, one block barrier per
// step): the matrix element is ~7000 straight-line instructions executed once per event, and without the lock-step the warps
// of an SM were each waiting for their own instruction fetches (ncu: 5.5 warps per issue stalled on no_instruction).
constexpr int kPrepassThreads = 256;
constexpr int kPrepassWarpDoubles = kQQWarpSharedDoubles + kQQWarpSets * kQQLStride;   // a warp's shared kinematics and line currents
__host__ __device__ inline int prepass_smem_doubles(int D, int nb, int nx, int nfl) {
  (void)D; (void)nb;      // the grid stays in global memory here (two edges per dimension and event: L1 hits)
  return nx + nfl * nx + kPrepassThreads * (17 + 2) + 32 + (kPrepassThreads / 32) * kPrepassWarpDoubles;
}
template <int PROC>
__global__ void __launch_bounds__(kPrepassThreads, 1) quark_prepass_kernel(const Params P, const PassArgs A, double* out) {
  static_assert(PROC == 7, "the prepass serves pp -> ttbar gg");
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF, NW = kPrepassThreads / 32;
  extern __shared__ double smem[];
  const int nx = P.pdf_nx, nrow = nx * P.pdf_nfl;
  double* s_lnx = smem;                     // nx
  double* s_row = s_lnx + nx;               // one row per parton table
  double* s_ev = s_row + nrow;              // [rank][17]: momenta and shat of the block's passing events
  double* s_res = s_ev + kPrepassThreads * 17;                       // [rank][2]
  unsigned* s_cnt = reinterpret_cast<unsigned*>(s_res + kPrepassThreads * 2);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* s_warp = reinterpret_cast<double*>(s_cnt) + 32 + warp * kPrepassWarpDoubles;
  QQWarpShared* s_sh = reinterpret_cast<QQWarpShared*>(s_warp);
  double* s_L = s_warp + kQQWarpSharedDoubles;
  for (int i = threadIdx.x; i < nx; i += blockDim.x) s_lnx[i] = A.pdf_lnx[i];
  for (int i = threadIdx.x; i < nrow; i += blockDim.x) s_row[i] = A.pdf_row[i];
  __syncthreads();
  const double g2 = 4.0 * kPi * P.alpha_s;
  const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
  const uint64_t rounds = (A.n_events + stride - 1) / stride;
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  for (uint64_t rd = 0; rd < rounds; ++rd, idx += stride) {
    const bool valid = idx < A.n_events;
    bool pass = false;
    double La = 0.0, Lb = 0.0, asf = 1.0;
    Event<PROC> ev;
    if (valid) {
      Bins<PROC> bins;
      DebugRow dbg = {nullptr, D, NF};
      generate_event<PROC>(P, A.grid, A.seed, A.iteration, A.first_event + idx, ev, bins, dbg);
      pass = ev.pass;
      if (pass) quark_pair_luminosities(P, A, s_lnx, s_row, ev, asf, La, Lb);
    }
    // rank the block's passing events (ballot + prefix over the warps) and queue their records
    const unsigned bal = __ballot_sync(0xFFFFFFFFu, pass);
    if (lane == 0) s_cnt[warp] = __popc(bal);
    __syncthreads();
    int base = 0, total = 0;
    for (int w = 0; w < NW; ++w) {
      const int c = (int)s_cnt[w];
      if (w < warp) base += c;
      total += c;
    }
    const int rank = base + __popc(bal & ((1u << lane) - 1u));
    if (pass) {
#pragma unroll
      for (int f = 0; f < 4; ++f)
#pragma unroll
        for (int c = 0; c < 4; ++c) s_ev[17 * rank + 4 * f + c] = ev.k[f][c];
      s_ev[17 * rank + 16] = ev.shat;
    }
#pragma unroll 1
    for (int r0 = 0; r0 < total; r0 += NW) {
      __syncthreads();                       // (first turn: the queue is complete) keeps the warps on the same code
      const int r = r0 + warp;
      if (r < total) {
        double m0, m1;
        me2_qq_ttgg_warp(s_ev + 17 * r, s_sh, s_L, lane, P.m_top, g2, m0, m1);
        if (lane == 0) { s_res[2 * r] = m0; s_res[2 * r + 1] = m1; }
      }
    }
    __syncthreads();
    if (valid) out[idx] = pass ? La * (s_res[2 * rank] * asf) + Lb * (s_res[2 * rank + 1] * asf) : 0.0;
    __syncthreads();                         // the queue and the counters are rewritten in the next round
  }
}

// Adds the per-block partials in block order.  Blocks 0..gridDim.x-2 own histogram bins (one thread per
// bin, summing over the pass's blocks); the last block reduces the scalar partials.  accumulate != 0: the outputs already hold
// the earlier pieces of the same call (MF_PP_TTGG calls larger than its quark-term buffer) and are added to.
__global__ void __launch_bounds__(256) finalize_kernel(const BlockPartial* partials, const double* hist_part,
                                                        int n_blocks, int n_hist, double* hist, IterResult* result,
                                                        int accumulate) {
  if (blockIdx.x + 1 < gridDim.x) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (hist != nullptr && i < n_hist) {
      double s = accumulate ? hist[i] : 0.0;
      for (int b = 0; b < n_blocks; ++b) s += hist_part[(size_t)b * n_hist + i];
      hist[i] = s;
    }
    return;
  }
  __shared__ double sw[256], sw2[256], mx[256];
  __shared__ unsigned long long np[256], na[256];
  double a = 0.0, b2 = 0.0, m = 0.0;
  unsigned long long p = 0, q = 0;
  for (int b = threadIdx.x; b < n_blocks; b += blockDim.x) {
    BlockPartial bp = partials[b];
    a += bp.sum_w; b2 += bp.sum_w2; m = fmax(m, bp.max_abs_w); p += bp.n_pass; q += bp.n_accept;
  }
  sw[threadIdx.x] = a; sw2[threadIdx.x] = b2; mx[threadIdx.x] = m; np[threadIdx.x] = p; na[threadIdx.x] = q;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) {
      sw[threadIdx.x] += sw[threadIdx.x + o];
      sw2[threadIdx.x] += sw2[threadIdx.x + o];
      mx[threadIdx.x] = fmax(mx[threadIdx.x], mx[threadIdx.x + o]);
      np[threadIdx.x] += np[threadIdx.x + o];
      na[threadIdx.x] += na[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    if (accumulate) {
      result->sum_w += sw[0]; result->sum_w2 += sw2[0]; result->max_abs_w = fmax(result->max_abs_w, mx[0]);
      result->n_pass += np[0]; result->n_accept += na[0];
    } else {
      result->sum_w = sw[0]; result->sum_w2 = sw2[0]; result->max_abs_w = mx[0];
      result->n_pass = np[0]; result->n_accept = na[0];
    }
  }
}

}  // namespace mf
