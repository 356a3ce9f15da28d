// mf_common.cuh — shared definitions of the CUDA path (product code; shares nothing with oracle/).
#pragma once
#include <stdint.h>
#include <math.h>

#if defined(__CUDACC__)
#define MF_HD __host__ __device__ __forceinline__
#define MF_D __device__ __forceinline__
#else
#define MF_HD inline
#define MF_D inline
#endif

namespace mf {

#if !defined(__CUDACC__)
// host builds (tests/host_shim) have no CUDA vector types
struct double2 { double x, y; };
inline double2 make_double2(double x, double y) { return double2{x, y}; }
struct alignas(16) uint4 { unsigned x, y, z, w; };
#endif

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kTwoPi = 6.28318530717958647692528676655900577;

// Static description of the processes (0..3: BASELINE.json configs[0..3]).
//   D      VEGAS dimensions           NF  final-state particles
//   NG     gluons incl. the two beams NGF final-state gluons (the ones the cuts act on)
template <int PROC> struct Traits;
template <> struct Traits<0> { static constexpr int D = 2, NF = 2, NG = 0, NGF = 0; };
template <> struct Traits<1> { static constexpr int D = 4, NF = 2, NG = 2, NGF = 0; };
template <> struct Traits<2> { static constexpr int D = 14, NF = 3, NG = 3, NGF = 1; };
template <> struct Traits<3> { static constexpr int D = 18, NF = 4, NG = 4, NGF = 2; };
// 4: gg -> ttbar + q qbar -> ttbar (flavour summed): the kinematics and alpha_s power of process 1
template <> struct Traits<4> { static constexpr int D = 4, NF = 2, NG = 2, NGF = 0; };
// 5: gg -> ttbar g + the q qbar, q g, qbar g channels (R19): kinematics and cuts of process 2
template <> struct Traits<5> { static constexpr int D = 14, NF = 3, NG = 3, NGF = 1; };
// 6: gg -> ttbar ggg: RAMBO n = 5, 22 dimensions, cuts on three gluons
template <> struct Traits<6> { static constexpr int D = 22, NF = 5, NG = 5, NGF = 3; };
// 7: gg -> ttbar gg + q qbar -> ttbar gg (R22): kinematics and cuts of process 3
template <> struct Traits<7> { static constexpr int D = 18, NF = 4, NG = 4, NGF = 2; };
constexpr int kMaxPartonTables = 11;   // gluon + up to 5 quark/antiquark pairs

// Scalars every kernel needs (passed by value in the launch).
struct Params {
  double s;            // (sqrt_s)^2
  double alpha_em, alpha_s, m_top, mu2;
  double ptmin, etamax, drmin;
  double gev2_to_pb;
  double tau_min, ln_tau_min;
  double me_norm;      // coupling^n / (spin, colour, identical-particle averaging)
  int n_bins;
  int pdf_nx, pdf_nq;
  int pdf_nfl;         // parton tables: 1 (gluon) or 1 + 2 n_f (process 4)
  int pdf_jq;          // Q^2 cell of mu2 (clamped), fixed per process
  double pdf_uq;       // (ln mu2 - lnq2[jq]) / (lnq2[jq+1]-lnq2[jq])
  int dyn_scale;       // 1: mu^2 = m_t^2 + pT(top)^2 per event, running alpha_s (mf_set_dynamic_scale; R16)
};

}  // namespace mf
