// mf_me_coop.cuh — steps a7-a9 for g g -> t tbar g g as a COOPERATIVE program: one event per team of 64
// threads (2 warps), all intermediate currents in a per-team shared-memory scratch (the
// matrix element loops over helicities and sums; DESIGN.md "Kernels" explains why not one thread per event).
//
//   S0   hand written: momentum sums, propagator denominators, polarisation vectors, external spinors
//   S1-3 table driven (csrc/gen_coop.py): one task = one off-shell current for one polarisation assignment of
//        the gluons it contains ("helicity recycling"); a warp executes rounds of 32 equal-shaped tasks
//   S4   generated straight-line code: thread (pols, h, hb) forms its 24 colour-ordered amplitudes and
//        contracts them with the colour matrix; the 64 partial sums are added in a fixed order
//
// Every function is MF_HD and takes the team-thread index explicitly, so tests/host_shim can run the same
// program on the host (looping over the 64 "threads" stage by stage) and compare it with the oracle.
#pragma once
#include "mf_me_prims.cuh"
#include "mf_me_ttgg_coop_generated.cuh"

namespace mf {

constexpr int kCoopTeam = 64;                     // threads per event
constexpr int kCoopInDoubles = 18;                // input area: k[4][4] (t, tbar, g, g; CM frame), shat, pad
constexpr int kCoopRedDoubles = 2;                // one partial per warp
// per-team shared memory (doubles): scratch | input | reduction | pass masks (2 x 2 x u32)
constexpr int kCoopOffIn = (kCoopScratchDoubles + 1) & ~1;
constexpr int kCoopOffRed = kCoopOffIn + kCoopInDoubles;
constexpr int kCoopOffMask = kCoopOffRed + kCoopRedDoubles;
constexpr int kCoopTeamDoubles = kCoopOffMask + 2;

MF_HD double* coop_V(double* scr) { return scr; }
MF_HD double* coop_S(double* scr) { return scr + 4 * kCoopNV; }
MF_HD double* coop_C(double* scr) { return scr + 4 * kCoopNV + 8 * kCoopNS; }
MF_HD double* coop_X(double* scr) { return scr + 4 * kCoopNV + 8 * kCoopNS + 8 * kCoopNC; }

// ---- S0: per-event constants --------------------------------------------------------------------------------
// in[0..15] = k[4][4] (t, tbar, g2, g3 in the partonic CM frame), in[16] = shat.  Gluon labels: 0, 1 = the beams
// (+z, -z, energy sqrt(shat)/2), 2, 3 = the final gluons entering with -k (all gluon momenta incoming).
MF_HD rvec coop_gluon_momentum(const double* in, int g) {
  const double E = 0.5 * sqrt(in[16]);
  rvec p;
  if (g == 0) p = {{E, 0.0, 0.0, E}};
  else if (g == 1) p = {{E, 0.0, 0.0, -E}};
  else p = {{-in[4 * g + 0], -in[4 * g + 1], -in[4 * g + 2], -in[4 * g + 3]}};
  return p;
}

MF_HD void coop_s0(double* scr, const double* in, int tid, double mt) {
  double* V = coop_V(scr);
  double* S = coop_S(scr);
  double* X = coop_X(scr);
  if (tid >= 1 && tid <= 15) {
    const int m = tid;
    rvec P = {{0.0, 0.0, 0.0, 0.0}};
    int n = 0;
#pragma unroll
    for (int g = 0; g < 4; ++g)
      if ((m >> g) & 1) { P = radd(P, coop_gluon_momentum(in, g)); ++n; }
    coop_st_vec(V, kCoopP0 + m - 1, P);
    if (n >= 2) X[kCoopIP2ofMask[m - 1]] = 1.0 / rdot(P, P);
    const double mt2 = mt * mt;
    const int ix = kCoopQXofMask[m - 1], iy = kCoopQYofMask[m - 1];
    if (ix >= 0) {
      rvec q = {{P.v[0] - in[4], P.v[1] - in[5], P.v[2] - in[6], P.v[3] - in[7]}};   // P - p4
      coop_st_vec(V, ix, q);
      X[kCoopIdXofMask[m - 1]] = 1.0 / (rdot(q, q) - mt2);
    }
    if (iy >= 0) {
      rvec q = {{in[0] - P.v[0], in[1] - P.v[1], in[2] - P.v[2], in[3] - P.v[3]}};   // p3 - P
      coop_st_vec(V, iy, q);
      X[kCoopIdYofMask[m - 1]] = 1.0 / (rdot(q, q) - mt2);
    }
  } else if (tid >= 16 && tid < 24) {
    const int g = (tid - 16) >> 1, p = (tid - 16) & 1;
    rvec e;
    if (g == 0) e = p == 0 ? rvec{{0.0, 1.0, 0.0, 0.0}} : rvec{{0.0, 0.0, 1.0, 0.0}};
    else if (g == 1) e = p == 0 ? rvec{{0.0, 1.0, 0.0, 0.0}} : rvec{{0.0, 0.0, -1.0, 0.0}};
    else {
      rvec e1, e2;
      pol_vectors(in + 4 * g, e1, e2);
      e = p == 0 ? e1 : e2;
    }
    coop_st_vec(V, kCoopEps0 + 2 * g + p, e);
  } else if (tid >= 24 && tid < 28) {
    const int s = tid & 1;
    if (tid < 26) coop_st_spin(S, kCoopUb0 + s, ubar_row(in, mt, s));
    else coop_st_spin(S, kCoopV0 + s, v_col(in + 4, mt, s));
  }
}

// ---- S1-S3: the task interpreter -----------------------------------------------------------------------------
// The operand indices of one task: NVEC 16-byte vectors of 8 shorts (registers).
template <int NVEC> struct CoopFields { uint4 q[NVEC]; };

template <int NVEC>
MF_HD int coop_fld(const CoopFields<NVEC>& F, int j) {   // j is a compile-time constant after unrolling
  const uint4& v = F.q[j >> 3];
  const int k = (j >> 1) & 3;
  const unsigned w = k == 0 ? v.x : k == 1 ? v.y : k == 2 ? v.z : v.w;
  return (int)(short)((j & 1) ? (w >> 16) : (w & 0xFFFFu));
}

// `tab` is the operand table (kCoopTable; a shared-memory copy on the device), t the lane's task slot
template <int NVEC>
MF_HD CoopFields<NVEC> coop_load_fields(const uint4* tab, const CoopRound& R, int t, int lane) {
  CoopFields<NVEC> F;
#pragma unroll
  for (int v = 0; v < NVEC; ++v) F.q[v] = tab[R.offset + (t * NVEC + v) * 32 + lane];
  return F;
}

// One task type = how many operand vectors it needs, how its result is computed from the scratch (calc: loads
// and arithmetic only) and where the result goes (store).  Keeping calc free of stores lets the compiler
// interleave the instruction streams of the tasks a lane runs in one round.
template <int NV3, int NV4>
struct CoopTaskJ {   // gluon current: [out, iP2, (J1, P1, J2, P2) x NV3, (J1, J2, J3) x NV4, signs]
  static constexpr int NVEC = (3 + 4 * NV3 + 3 * NV4 + 7) / 8 == 3 ? 4 : (3 + 4 * NV3 + 3 * NV4 + 7) / 8;
  typedef rvec Out;
  MF_HD static rvec calc(const double* scr_c, const CoopFields<NVEC>& F, double) {
    double* scr = const_cast<double*>(scr_c);
    const double* V = coop_V(scr);
    const int signs = coop_fld(F, 2 + 4 * NV3 + 3 * NV4);
    rvec acc = {{0.0, 0.0, 0.0, 0.0}};
#pragma unroll
    for (int t = 0; t < NV3; ++t) {
      const int g = 2 + 4 * t;
      const rvec J1 = coop_ld_vec(V, coop_fld(F, g)), P1 = coop_ld_vec(V, coop_fld(F, g + 1));
      const rvec J2 = coop_ld_vec(V, coop_fld(F, g + 2)), P2 = coop_ld_vec(V, coop_fld(F, g + 3));
      v3_acc(acc, ((signs >> t) & 1) ? -1.0 : 1.0, J1, P1, J2, P2);
    }
#pragma unroll
    for (int t = 0; t < NV4; ++t) {
      const int g = 2 + 4 * NV3 + 3 * t;
      const rvec J1 = coop_ld_vec(V, coop_fld(F, g)), J2 = coop_ld_vec(V, coop_fld(F, g + 1));
      const rvec J3 = coop_ld_vec(V, coop_fld(F, g + 2));
      v4_acc(acc, ((signs >> (NV3 + t)) & 1) ? -1.0 : 1.0, J1, J2, J3);
    }
    return rscale(acc, coop_X(scr)[coop_fld(F, 1)]);
  }
  MF_HD static void store(double* scr, int out, const rvec& r) { coop_st_vec(coop_V(scr), out, r); }
};

template <int NT>
struct CoopTaskX {   // propagated column quark current: [out, qX, idX, (J, X) x NT, signs]
  static constexpr int NVEC = 1;
  typedef spin Out;
  MF_HD static spin calc(const double* scr_c, const CoopFields<NVEC>& F, double mt) {
    double* scr = const_cast<double*>(scr_c);
    const double* V = coop_V(scr);
    const double* S = coop_S(scr);
    const int signs = coop_fld(F, 3 + 2 * NT);
    spin t;
#pragma unroll
    for (int i = 0; i < NT; ++i) {
      const int g = 3 + 2 * i;
      const rvec J = rscale(coop_ld_vec(V, coop_fld(F, g)), ((signs >> i) & 1) ? -1.0 : 1.0);
      const spin x = coop_ld_spin(S, coop_fld(F, g + 1));
      if (i == 0) t = slash_col(J, x);
      else slash_col_acc(t, J, x);
    }
    return prop_col(coop_ld_vec(V, coop_fld(F, 1)), mt, coop_X(scr)[coop_fld(F, 2)], t);
  }
  MF_HD static void store(double* scr, int out, const spin& r) { coop_st_spin(coop_S(scr), out, r); }
};

template <int NT, bool PROP>
struct CoopTaskY {   // row quark current, propagated or not: [out, qY, idY, (Y, J) x NT, signs]
  static constexpr int NVEC = 1;
  typedef spin Out;
  MF_HD static spin calc(const double* scr_c, const CoopFields<NVEC>& F, double mt) {
    double* scr = const_cast<double*>(scr_c);
    const double* V = coop_V(scr);
    const double* S = coop_S(scr);
    const int signs = coop_fld(F, 3 + 2 * NT);
    spin t;
#pragma unroll
    for (int i = 0; i < NT; ++i) {
      const int g = 3 + 2 * i;
      const spin y = coop_ld_spin(S, coop_fld(F, g));
      const rvec J = rscale(coop_ld_vec(V, coop_fld(F, g + 1)), ((signs >> i) & 1) ? -1.0 : 1.0);
      if (i == 0) t = slash_row(y, J);
      else slash_row_acc(t, y, J);
    }
    if (PROP) t = prop_row(t, coop_ld_vec(V, coop_fld(F, 1)), mt, coop_X(scr)[coop_fld(F, 2)]);
    return t;
  }
  MF_HD static void store(double* scr, int out, const spin& r) { coop_st_spin(coop_S(scr), out, r); }
};

struct CoopTaskBil {   // fermion bilinear row gamma^mu col: [out, row, col]
  static constexpr int NVEC = 1;
  typedef cvec Out;
  MF_HD static cvec calc(const double* scr_c, const CoopFields<NVEC>& F, double) {
    const double* S = coop_S(const_cast<double*>(scr_c));
    return bilinear(coop_ld_spin(S, coop_fld(F, 1)), coop_ld_spin(S, coop_fld(F, 2)));
  }
  MF_HD static void store(double* scr, int out, const cvec& r) { coop_st_cvec(coop_C(scr), out, r); }
};

// One round for one lane: M tasks of type Task, all computed before any result is stored.  Idle slots (output
// index < 0, operand indices 0) compute on valid but meaningless operands and store nothing.
template <int M, class Task>
MF_HD void coop_run_tasks(double* scr, const uint4* tab, const CoopRound& R, int lane, double mt) {
  typename Task::Out res[M];
  int out[M];
#pragma unroll
  for (int t = 0; t < M; ++t) {
    const CoopFields<Task::NVEC> F = coop_load_fields<Task::NVEC>(tab, R, t, lane);
    out[t] = coop_fld(F, 0);
    res[t] = Task::calc(scr, F, mt);
  }
#pragma unroll
  for (int t = 0; t < M; ++t)
    if (out[t] >= 0) Task::store(scr, out[t], res[t]);
}

#define MF_COMMA ,
MF_HD void coop_exec_round(double* scr, const uint4* tab, const CoopRound& R, int lane, double mt) {
  switch (R.variant) {
#define MF_COOP_CASE(ID, M, TASK) case ID: coop_run_tasks<M, TASK>(scr, tab, R, lane, mt); break;
    MF_COOP_VARIANTS(MF_COOP_CASE)
#undef MF_COOP_CASE
    default: break;
  }
}

// Host emulation helper (tests/host_shim): all rounds of `stage` for one (warp, lane).
MF_HD void coop_run_stage(double* scr, const uint4* tab, int stage, int warp, int lane, double mt) {
  for (int r = 0; r < kCoopNumRounds[warp]; ++r) {
    const CoopRound R = kCoopRounds[warp][r];
    if (R.stage == stage) coop_exec_round(scr, tab, R, lane, mt);
  }
}

// S4 for team thread tid = pols | h << 4 | hb << 5: colour-contracted |Ahat|^2 of its helicity combination
// (colour-matrix numerators; divide the team sum by kCoopCden).
MF_HD double coop_s4_thread(double* scr, int tid) {
  return coop_s4(coop_V(scr), coop_S(scr), coop_C(scr), tid & 15, (tid >> 4) & 1, (tid >> 5) & 1);
}

#if defined(__CUDACC__)
// ---- device-side driver ---------------------------------------------------------------------------------
// Called by EVERY thread of the block (all teams run in lock-step so that the SM fetches one instruction stream:
// the per-event program is larger than the instruction cache) after the owners have written the input areas
// and the block has synchronised.  Teams with `active` false only keep the barriers.  Leaves
// sum_{helicities} Ahat^dagger C Ahat * kCoopCden (no couplings, no averaging) in the team's reduction slots.
__device__ __forceinline__ void coop_me2_lockstep(double* tm, const uint4* tab, int tid, bool active, double mt) {
  double* scr = tm;
  const int warp = tid >> 5, lane = tid & 31;
  if (active) coop_s0(scr, tm + kCoopOffIn, tid, mt);
  __syncthreads();
  const int nr = kCoopNumRounds[warp];
#pragma unroll 1
  for (int r = 0; r < nr; ++r) {
    const CoopRound R = kCoopRounds[warp][r];
    if (active) coop_exec_round(scr, tab, R, lane, mt);
    if (R.sync) __syncthreads();
  }
  if (active) {
    double acc = coop_s4_thread(scr, tid);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
    if (lane == 0) tm[kCoopOffRed + warp] = acc;
  }
  __syncthreads();
}
#endif

}  // namespace mf
