// mf_me_coop.cuh — steps a7-a9 for g g -> t tbar g g and g g -> t tbar g as COOPERATIVE programs: one event per
// team of 64 threads (2 warps) resp. 32 threads (1 warp), all intermediate currents in a per-team shared-memory
// scratch (the matrix element loops over helicities and sums; DESIGN.md "Kernels" explains why
// not one thread per event).
//
//   owner  the thread that generated the event evaluates polarisation vectors, external spinors and c0 = ubar gamma v
//          and queues them with the momenta (event record); the team's lanes copy the record into the scratch
//   S0     hand written: momentum sums, propagator momenta and inverse denominators (one reciprocal per lane)
//   S1/A/B table driven (csrc/gen_coop.py, gen_coop3.py): one lane-task = M "polarisation sibling" off-shell currents
//          that share their operands; a warp executes rounds of <= 32 equal-shaped lane-tasks
//   S4     generated straight-line code: thread (pols, hb, k) forms the real / imaginary parts of its colour-ordered
//          amplitudes and contracts them with the colour matrix; the partial sums are added in a fixed order.  Only
//          the top spin state 0 is evaluated (spin-flip symmetry, gen_coop.py): the caller doubles the sum.
//
// The two programs share the task templates (mf_me_coop_tasks.inc, compiled once per process inside namespaces
// mf::g4 / mf::g3 after the process' generated fragment).  Every function is MF_HD and takes the team-thread index
// explicitly, so tests/host_shim can run the same programs on the host (looping over the team's "threads" stage by
// stage) and compare them with the oracle.
#pragma once
#include "mf_me_prims.cuh"

#if defined(__CUDA_ARCH__)
#define MF_TABLE static __device__ const
#define MF_CONST static __constant__ const
#else
#define MF_TABLE static const
#define MF_CONST static const
#endif
#if !defined(__CUDACC__)
#define __align__(n) alignas(n)
#endif

namespace mf {

// ---- S1 / A / B: the task interpreter -----------------------------------------------------------------------
// The operand indices of one lane-task: NVEC 16-byte vectors of 8 shorts (registers).
template <int NVEC> struct CoopFields { uint4 q[NVEC]; };

template <int NVEC>
MF_HD int coop_fld(const CoopFields<NVEC>& F, int j) {   // j is a compile-time constant after unrolling
  const uint4& v = F.q[j >> 3];
  const int k = (j >> 1) & 3;
  const unsigned w = k == 0 ? v.x : k == 1 ? v.y : k == 2 ? v.z : v.w;
  return (int)(short)((j & 1) ? (w >> 16) : (w & 0xFFFFu));
}

// `tab` is the operand table (kCoopTable; a shared-memory copy on the device), `offset` the round's first vector
template <int NVEC>
MF_HD CoopFields<NVEC> coop_load_fields(const uint4* tab, int offset, int lane) {
  CoopFields<NVEC> F;
#pragma unroll
  for (int v = 0; v < NVEC; ++v) F.q[v] = tab[offset + v * 32 + lane];
  return F;
}

}  // namespace mf

// g g -> t tbar g g: teams of 64 threads (csrc/gen_coop.py)
namespace mf { namespace g4 {
#define MF_COOP_WARP0 MF_COOP4_WARP0
#define MF_COOP_WARP1 MF_COOP4_WARP1
#include "mf_me_ttgg_coop_generated.cuh"
#include "mf_me_coop_tasks.inc"
#undef MF_COOP_WARP0
#undef MF_COOP_WARP1
}}  // namespace mf::g4

// g g -> t tbar g: teams of one warp (csrc/gen_coop3.py)
namespace mf { namespace g3 {
#define MF_COOP_WARP0 MF_COOP3_WARP0
#define MF_COOP_WARP1 MF_COOP3_WARP1
#include "mf_me_ttg_coop_generated.cuh"
#include "mf_me_coop_tasks.inc"
#undef MF_COOP_WARP0
#undef MF_COOP_WARP1
}}  // namespace mf::g3
