// mf_event.cuh — the per-event chain a1..a10 (random numbers -> phase-space kinematics ->
// matrix element -> weight), written once and used by every kernel of the fused pass.
#pragma once
#include "mf_common.cuh"
#include "mf_philox.cuh"
#include "mf_phasespace.cuh"
#include "mf_pdf.cuh"
#include "mf_me_prims.cuh"
#include "mf_me_eemumu.cuh"
#include "mf_me_qqtt.cuh"
#include "mf_me_qttg.cuh"
#include "mf_me_qqttgg.cuh"
#include "mf_me_ggtt_generated.cuh"

namespace mf {

// What the kinematic stage hands to the matrix-element stage (registers only).
template <int PROC> struct Event {
  static constexpr int NF = Traits<PROC>::NF;
  double k[NF][4];    // final-state momenta, partonic CM frame
  double shat, y;     // partonic invariant mass squared, rapidity of the CM frame in the lab
  double x1, x2;      // parton fractions (1, 1 for e+e-)
  double phi;         // phase-space weight per unit hypercube volume
  double jac_parton;  // J_tau J_y (1 for e+e-)
  double jac_vegas;   // prod_d nb (e_{i+1} - e_i)
  bool pass;
};

// Packed VEGAS bin indices: one byte per dimension (n_bins <= 128).
template <int PROC> struct Bins {
  uint32_t w[(Traits<PROC>::D + 3) / 4];
  MF_HD void clear() {
#pragma unroll
    for (int i = 0; i < (Traits<PROC>::D + 3) / 4; ++i) w[i] = 0u;
  }
  MF_HD void set(int d, int b) { w[d >> 2] |= (uint32_t)b << (8 * (d & 3)); }
  MF_HD int get(int d) const { return (int)((w[d >> 2] >> (8 * (d & 3))) & 0xFFu); }
};

// Optional per-event dump (mf_debug_eval): row layout of include/mf.h.
struct DebugRow {
  double* row;  // nullptr = off
  int D, NF;
  MF_HD void x(int d, double v) const { if (row) row[d] = v; }
  MF_HD void u(int d, double v) const { if (row) row[D + 4 * (NF + 2) + 9 + d] = v; }
  MF_HD void bin(int d, int b) const { if (row) row[2 * D + 4 * (NF + 2) + 9 + d] = (double)b; }
};

// a1-a5: Philox -> uniforms -> VEGAS map -> parton fractions -> phase space -> boost + cuts.
// `grid` points at the [D][nb+1] edges (shared memory in the kernels).
template <int PROC>
MF_HD void generate_event(const Params& P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t event,
                          Event<PROC>& ev, Bins<PROC>& bins, const DebugRow& dbg) {
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF, NGF = Traits<PROC>::NGF;
  const int nb = P.n_bins, stride = nb + 1;
  double jac = 1.0;
  bins.clear();
  // dimensions 0, 1 from Philox block 0
  double x0, x1;
  {
    U4 r = philox_block(seed, iteration, event, 0u);
    double u0 = uniform52(r.x, r.y), u1 = uniform52(r.z, r.w);
    int b0, b1;
    x0 = vegas_map1(grid, nb, u0, jac, b0);
    x1 = vegas_map1(grid + stride, nb, u1, jac, b1);
    bins.set(0, b0); bins.set(1, b1);
    dbg.u(0, u0); dbg.u(1, u1); dbg.x(0, x0); dbg.x(1, x1); dbg.bin(0, b0); dbg.bin(1, b1);
  }
  if (PROC == 0) {
    ev.shat = P.s; ev.y = 0.0; ev.x1 = 1.0; ev.x2 = 1.0; ev.jac_parton = 1.0;
    ev.phi = two_body(P.s, 0.0, x0, x1, ev.k);
  } else {
    Parton pk = parton_fractions(x0, x1, P.ln_tau_min, P.s);
    ev.shat = pk.shat; ev.y = pk.y; ev.x1 = pk.x1; ev.x2 = pk.x2; ev.jac_parton = pk.jac;
    if (PROC == 1 || PROC == 4) {
      U4 r = philox_block(seed, iteration, event, 1u);
      double u2 = uniform52(r.x, r.y), u3 = uniform52(r.z, r.w);
      int b2, b3;
      double x2 = vegas_map1(grid + 2 * stride, nb, u2, jac, b2);
      double x3 = vegas_map1(grid + 3 * stride, nb, u3, jac, b3);
      bins.set(2, b2); bins.set(3, b3);
      dbg.u(2, u2); dbg.u(3, u3); dbg.x(2, x2); dbg.x(3, x3); dbg.bin(2, b2); dbg.bin(3, b3);
      ev.phi = two_body(pk.shat, P.m_top, x2, x3, ev.k);
    } else {
      // RAMBO: final particle i uses dimensions 2+4i .. 5+4i = Philox blocks 1+2i, 2+2i
#pragma unroll
      for (int i = 0; i < NF; ++i) {
        double rho[4];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          int d = 2 + 4 * i + 2 * h;
          U4 r = philox_block(seed, iteration, event, (uint32_t)(d >> 1));
          double ua = uniform52(r.x, r.y), ub = uniform52(r.z, r.w);
          int ba, bb;
          rho[2 * h] = vegas_map1(grid + d * stride, nb, ua, jac, ba);
          rho[2 * h + 1] = vegas_map1(grid + (d + 1) * stride, nb, ub, jac, bb);
          bins.set(d, ba); bins.set(d + 1, bb);
          dbg.u(d, ua); dbg.u(d + 1, ub); dbg.x(d, rho[2 * h]); dbg.x(d + 1, rho[2 * h + 1]);
          dbg.bin(d, ba); dbg.bin(d + 1, bb);
        }
        rambo_q(rho[0], rho[1], rho[2], rho[3], ev.k[i]);
      }
      double w = sqrt(pk.shat);
      double V = rambo_finish<NF>(ev.k, w, P.m_top);
      ev.phi = two_pi_power<NF>() * V;
    }
  }
  ev.jac_vegas = jac;
  ev.pass = true;
  if (NGF > 0) {
    Boost b = make_boost(ev.y);
    double gl[NGF > 0 ? NGF : 1][4];
#pragma unroll
    for (int g = 0; g < NGF; ++g) boost_z(b, ev.k[2 + g], gl[g]);
    ev.pass = pass_cuts<NGF>(gl, P.ptmin, P.etamax, P.drmin);
  }
}

// a7-a9: averaged |M|^2 at the CM-frame momenta (beams along +-z with energy sqrt(shat)/2).
template <int PROC>
MF_HD double matrix_element(const Params& P, double shat, const double k[][4]) {
  constexpr int NG = Traits<PROC>::NG;
  double E = 0.5 * sqrt(shat);
  if (PROC == 0) {
    double p1[4] = {E, 0.0, 0.0, E}, p2[4] = {E, 0.0, 0.0, -E};
    return me2_ee_mumu(p1, p2, k[0], k[1], P.alpha_em);
  } else {
    constexpr int N = NG > 0 ? NG : 2;
    rvec Pg[N];
    rvec eps[N][2];
    Pg[0] = {{E, 0.0, 0.0, E}};
    Pg[1] = {{E, 0.0, 0.0, -E}};
    eps[0][0] = {{0.0, 1.0, 0.0, 0.0}}; eps[0][1] = {{0.0, 0.0, 1.0, 0.0}};
    eps[1][0] = {{0.0, 1.0, 0.0, 0.0}}; eps[1][1] = {{0.0, 0.0, -1.0, 0.0}};
#pragma unroll
    for (int g = 2; g < N; ++g) {
      Pg[g] = {{-k[g][0], -k[g][1], -k[g][2], -k[g][3]}};  // outgoing gluon enters with -k
      pol_vectors(k[g], eps[g][0], eps[g][1]);
    }
    spin ub[2], vv[2];
#pragma unroll
    for (int s = 0; s < 2; ++s) { ub[s] = ubar_row(k[0], P.m_top, s); vv[s] = v_col(k[1], P.m_top, s); }
    rvec p3 = {{k[0][0], k[0][1], k[0][2], k[0][3]}}, p4 = {{k[1][0], k[1][1], k[1][2], k[1][3]}};
    double sum;
    if (PROC == 1 || PROC == 4) sum = me2_ggtt_0g(Pg, eps, ub, vv, p3, p4, P.m_top);
    else if (PROC == 2 || PROC == 5) sum = me2_ggtt_1g(Pg, eps, ub, vv, p3, p4, P.m_top);
    else sum = me2_ggtt_2g(Pg, eps, ub, vv, p3, p4, P.m_top);
    return sum * P.me_norm;
  }
}

// a7-a9 for the quark channel of process 4: averaged |M|^2 of q qbar -> t tbar at the same CM-frame point
MF_HD double matrix_element_qq(const Params& P, double shat, const double k[][4]) {
  double E = 0.5 * sqrt(shat);
  double p1[4] = {E, 0.0, 0.0, E}, p2[4] = {E, 0.0, 0.0, -E};
  return me2_qq_tt(p1, p2, k[0], k[1], P.m_top, 4.0 * kPi * P.alpha_s);
}

// a10: event weight (R12): w = lum/(2 shat) |M|^2 Phi J_parton K J_vegas.
template <int PROC>
MF_HD double event_weight(const Params& P, const Event<PROC>& ev, double lum, double me2) {
  double f = lum / (2.0 * ev.shat) * me2 * ev.phi * ev.jac_parton * P.gev2_to_pb;
  return f * ev.jac_vegas;
}

}  // namespace mf
