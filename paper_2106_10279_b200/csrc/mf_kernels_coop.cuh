// mf_kernels_coop.cuh — the fused pass for g g -> t tbar g and g g -> t tbar g g (BASELINE.json configs[2..4]):
// steps a1-a6 and a10-a14 one thread per event exactly as in mf_kernels.cuh, steps a7-a9 (the matrix element,
// >95 % of the arithmetic) by TEAMS of threads per event over a shared-memory scratch
// (mf_me_coop.cuh): 64 threads (2 warps) for g g -> t tbar g g, 32 threads (1 warp) for g g -> t tbar g.
//
// Block = T teams (g g -> t tbar g g: T = 6, 6 x 31.6 kB of scratch + operand table + grid + histogram + PDF row
// fill the 227 kB of one SM; 12 warps = 3 per scheduler, <= 168 registers.  g g -> t tbar g: T = 16 warps).
// Per round every thread generates its own event; the events of the block that passed the cuts are ranked and
// their momenta queued (a per-block slice of a small L2-resident buffer); team t then works through ranks t,
// t + T, ... on its own, synchronising only its own warps (named barriers / __syncwarp), and leaves |M|^2 in a
// per-rank result slot that the owner reads after the round's closing block barrier.  Teams therefore sit in
// different stages of the program at any time, so the latency-bound stages of one team (S0, barriers, table
// fetches) overlap the FP64-bound stages of the others.
#pragma once
#include "mf_kernels.cuh"
#include "mf_me_coop.cuh"

namespace mf {

// the cooperative program of a process and its launch shape
template <int PROC> struct CoopOf { typedef g4::Prog PG; static constexpr int MaxTeams = 6; };   // PROC = 3
template <> struct CoopOf<2> { typedef g3::Prog PG; static constexpr int MaxTeams = 16; };
// pp -> ttbar j: the gg -> ttbar g program for the gluon channel; the owner threads evaluate the quark-channel classes
// (register hungry): 12 teams x 168 registers measured best (8 x 255: 39.9 ms, 12: 36.9 ms, 16 x 128: 38.1 ms per 2^22 events).
// Measured and rejected (profiles/r2_c8.md): the quark classes in a thread-per-event kernel of their own ahead of this pass
// (quark_prepass_kernel, 255 registers) with 16 teams x 128 registers here: 35.3-42.2 ms against 31.1 ms.
template <> struct CoopOf<5> { typedef g3::Prog PG; static constexpr int MaxTeams = 12; };
// pp -> ttbar gg: the g g -> t tbar g g program; the quark channel (q qbar -> t tbar g g, two beam assignments: 155 kflop and
// 4.4 kB of thread-local state per event) comes from quark_prepass_kernel through PassArgs::quark_terms: on the owner threads of
// this kernel (231 kB of shared memory, so almost no L1) it took 350 ms per 2^22 events, ahead of it 195 ms.
template <> struct CoopOf<7> { typedef g4::Prog PG; static constexpr int MaxTeams = 6; };

// queue entry = the event record of mf_me_coop_tasks.inc (momenta, shat, polarisation vectors, spinors, c0): PG::Queue doubles

// shared-memory carve-up of a coop block (doubles; every region starts 16-byte aligned)
template <class PG>
struct CoopSmem {
  int grid, hist, lnx, row, red, cnt, res, tab, teams, total;
  __host__ __device__ CoopSmem(int D, int nb, int nx, int nrow, int n_teams) {   // nrow = nx x parton tables
    auto even = [](int v) { return (v + 1) & ~1; };
    grid = 0;
    hist = grid + even(D * (nb + 1));
    lnx = hist + even(D * nb);
    row = lnx + even(nx);
    red = row + even(nrow);
    cnt = red + 5 * 32;
    res = cnt + 32;
    tab = res + PG::Warps * n_teams * PG::Team;
    teams = tab + 2 * PG::TableVecs;
    total = teams + n_teams * PG::TeamDoubles;
  }
};

// the debug kernels run 64 threads per block (one or two teams)
constexpr int kCoopDebugThreads = 64;
// their shared memory: teams | rank counters | results | queue | operand table
template <class PG>
constexpr int coop_debug_smem_bytes() {
  return ((kCoopDebugThreads / PG::Team) * PG::TeamDoubles + 32 + PG::Warps * kCoopDebugThreads +
          kCoopDebugThreads * PG::Queue + 2 * PG::TableVecs) * 8;
}

// copies the operand table into shared memory (all threads of the block; the caller synchronises)
template <class PG>
__device__ __forceinline__ void coop_load_table(uint4* s_tab) {
  const uint4* g = reinterpret_cast<const uint4*>(PG::table());
  for (int i = threadIdx.x; i < PG::TableVecs; i += blockDim.x) s_tab[i] = g[i];
}

// Teams are tied into groups of G that run the matrix-element program in lock-step (one named barrier per group:
// 1 + group; barrier 0 is __syncthreads).  G = 1 = every team on its own: least barrier wait, but one instruction
// stream per team: the straight-line round programs are executed once per event, so the instruction cache holds
// nothing for a warp unless another warp runs the same code at the same time (ncu: 11 % of the stall samples were
// "no instruction" with G = 1).  Measured on B200, 2^22 events of g g -> t tbar g g (profiles/r2_c3.md): G = 1
// 38.7 ms, G = 2 38.0 ms, G = 3 35.5 ms, G = 6 37.0 ms, G = 3 with the groups interleaved over the teams 36.0 ms.
// One-warp teams need only __syncwarp.
#ifndef MF_COOP_GROUP
#define MF_COOP_GROUP 3
#endif
#ifndef MF_COOP_INTERLEAVE
#define MF_COOP_INTERLEAVE 0
#endif
#ifndef MF_COOP_GROUP_WARP
#define MF_COOP_GROUP_WARP 1
#endif
// MF_COOP_DECOUPLE = 1: group-level rounds (every lock-step group generates, ranks and queues its own threads' events; no block
// barrier in the round).  Measured and rejected (profiles/r2_c3.md): g g -> t tbar g g 35.7 -> 41.9 ms, g g -> t tbar g 9.6 -> 11.4 ms,
// pp -> t tbar j 30.8 -> 44.8 ms: with the groups in different phases the event-generation code and the matrix-element programs
// compete for the instruction cache all the time.
#ifndef MF_COOP_DECOUPLE
#define MF_COOP_DECOUPLE 0
#endif
constexpr int kCoopGroup = MF_COOP_GROUP;            // teams of two warps (g g -> t tbar g g)
constexpr int kCoopGroupWarp = MF_COOP_GROUP_WARP;   // teams of one warp (g g -> t tbar g, pp -> t tbar j)
template <int THREADS>
__device__ __forceinline__ void coop_group_sync(int group) {
  if (THREADS == 32) __syncwarp();
  else asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "n"(THREADS) : "memory");
}

// The teams' share of a round: team t of group g works through ranks g G + t, g G + t + n_teams, ... of the queue;
// the G teams of a group step together (a team whose rank is beyond `total` only keeps the barriers).
template <class PG, int G>
__device__ __forceinline__ void coop_team_loop(double* teams, int n_teams, const uint4* tab, double* s_res,
                                               const double* queue, int total, double mt) {
  (void)n_teams;
  const int team = threadIdx.x / PG::Team, tid = threadIdx.x % PG::Team, warp = tid >> 5, lane = tid & 31;
#if MF_COOP_DECOUPLE
  // every group owns its part of the round (its own events, queue slice and ranks): the teams of a group take ranks
  // member, member + G, ... of the GROUP's queue
  const int group = team / G, member = team - group * G;
  n_teams = G;
  queue += group * (G * PG::Team);
  s_res += PG::Warps * group * (G * PG::Team);
  const int first = 0;
#elif MF_COOP_INTERLEAVE
  const int n_groups = n_teams / G, group = team % n_groups, member = team / n_groups;   // groups {g, g + n_groups, ...}
  const int first = group * G;
#else
  const int group = team / G, member = team - group * G;
  const int first = group * G;
#endif
  double* tm = teams + team * PG::TeamDoubles;
  double* in = tm + PG::OffIn;
  auto sync = [group]() { coop_group_sync<PG::Team * G>(group); };
  // lane `tid` moves doubles tid, tid + Team, ... of the event record from the queue to their places in the scratch
  // (registers in between: the next record is fetched while the current event is being computed)
  constexpr int QPT = (PG::Queue + PG::Team - 1) / PG::Team;
  const int qcap = blockDim.x;                   // the queue is stored [double][rank]
  int dst[QPT];
  double nxt[QPT];
#pragma unroll
  for (int i = 0; i < QPT; ++i) {
    const int j = tid + i * PG::Team;
    dst[i] = j < PG::Queue ? PG::qdest(j) : -1;
    nxt[i] = 0.0;
    if (first + member < total && dst[i] >= 0) nxt[i] = queue[j * qcap + first + member];
  }
#pragma unroll 1
  for (int r0 = first; r0 < total; r0 += n_teams) {
    const int r = r0 + member;
    const bool active = r < total;
#pragma unroll
    for (int i = 0; i < QPT; ++i)
      if (dst[i] >= 0) tm[dst[i]] = nxt[i];
    sync();
    if (r + n_teams < total) {
#pragma unroll
      for (int i = 0; i < QPT; ++i)
        if (dst[i] >= 0) nxt[i] = queue[(tid + i * PG::Team) * qcap + r + n_teams];   // next turn
    }
    if (active) PG::s0(tm, in, tid, mt);
    sync();
    PG::run(tm, tab, warp, lane, mt, active, sync);
    if (active) {
      double acc = PG::s4_thread(tm, tid);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
      if (lane == 0) s_res[PG::Warps * r + warp] = acc;
    }
  }
}

// |M|^2 (with couplings and averaging) of this thread's own event.  EVERY thread of the block must call it (it
// contains block barriers).  The events of the block that passed the cuts are ranked (ballot + prefix over the
// warps) and queued; team t computes ranks t, t + n_teams, ...  `queue` holds blockDim.x entries (global memory
// in the fused pass, shared memory in the debug kernels), s_res PG::Warps doubles per thread of the block, s_cnt
// 2 x 32 unsigned (double-buffered by `round`).  k = the NF final-state momenta.  Returns 0 for threads whose event
// did not pass.
template <class PG, int G>
__device__ __forceinline__ double coop_block_me2(double* teams, int n_teams, const uint4* tab, unsigned* s_cnt,
                                                 double* s_res, double* queue, unsigned round, bool pass,
                                                 const double (*k)[4], double shat, const Params& P) {
#if MF_COOP_DECOUPLE
  // group-level rounds: the G teams of a lock-step group rank, queue and work through THEIR threads' events on their own
  // (named barrier of the group; one-warp teams with G = 1: __syncwarp only), so the groups of a block drift into different
  // phases: event generation (latency bound, special-function sequences) of one overlaps the matrix elements of the others,
  // and no warp waits at a block barrier for another group's tail.
  constexpr int GT = G * PG::Team;
  const int grp = threadIdx.x / GT, gtid = threadIdx.x % GT, bwarp = gtid >> 5, lane = threadIdx.x & 31;
  constexpr int n_warps = GT / 32;
  unsigned* cnt = s_cnt + 32 * (round & 1u) + grp * n_warps;
  auto gsync = [grp]() { coop_group_sync<GT>(grp); };
  const int goff = grp * GT;
#else
  const int bwarp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  unsigned* cnt = s_cnt + 32 * (round & 1u);
  auto gsync = []() { __syncthreads(); };
  const int goff = 0;
#endif
  const unsigned bal = __ballot_sync(0xFFFFFFFFu, pass);
  if (lane == 0) cnt[bwarp] = __popc(bal);
  gsync();
  int base = 0, total = 0;
  for (int w = 0; w < n_warps; ++w) {
    const int c = (int)cnt[w];
    if (w < bwarp) base += c;
    total += c;
  }
  const int rank = base + __popc(bal & ((1u << lane) - 1u));
  if (pass) PG::owner_fill(queue + goff + rank, blockDim.x, k, shat, P.m_top);
  gsync();
  coop_team_loop<PG, G>(teams, n_teams, tab, s_res, queue, total, P.m_top);   // n_teams is a multiple of G
  gsync();
  // top spin state 0 only: the other one gives the same sum (spin-flip symmetry), hence the factor 2
  double sum = 0.0;
  if (pass) {
#pragma unroll
    for (int w = 0; w < PG::Warps; ++w) sum += s_res[PG::Warps * (goff + rank) + w];
  }
  return sum * (2.0 * P.me_norm / PG::Cden);
}

template <int PROC, bool UNW>
__global__ void __launch_bounds__(CoopOf<PROC>::MaxTeams * CoopOf<PROC>::PG::Team, 1)
    fused_pass_coop_kernel(const Params P, const PassArgs A) {
  typedef typename CoopOf<PROC>::PG PG;
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  constexpr int G = PG::Team == 32 ? kCoopGroupWarp : kCoopGroup;
  extern __shared__ double2 smem2[];
  double* smem = reinterpret_cast<double*>(smem2);
  const int nb = P.n_bins, nx = P.pdf_nx, nrow = PROC == 5 ? nx * P.pdf_nfl : nx;   // pp -> ttbar gg: the gluon's row only (the quark rows are the prepass's business)
  const int n_teams = blockDim.x / PG::Team;
  const CoopSmem<PG> L(D, nb, nx, nrow, n_teams);
  double* s_grid = smem + L.grid;
  double* s_hist = smem + L.hist;
  double* s_lnx = smem + L.lnx;
  double* s_row = smem + L.row;
  double* s_red = smem + L.red;
  unsigned* s_cnt = reinterpret_cast<unsigned*>(smem + L.cnt);
  double* s_res = smem + L.res;
  double* s_teams = smem + L.teams;
  uint4* s_tab = reinterpret_cast<uint4*>(smem + L.tab);
  double* queue = A.coop_queue + (size_t)blockIdx.x * blockDim.x * PG::Queue;
  coop_load_table<PG>(s_tab);
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
    const bool valid = idx < A.n_events;
    const uint64_t event = A.first_event + idx;
    Bins<PROC> bins;
    bins.clear();
    Event<PROC> ev;
    ev.pass = false;
    double lum = 0.0, asf = 1.0, quark_sum = 0.0;   // quark_sum: the owner's own channels (pp -> ttbar j), else 0
    if (valid) {
      DebugRow dbg = {nullptr, D, NF};
      generate_event<PROC>(P, s_grid, A.seed, A.iteration, event, ev, bins, dbg);
      if (ev.pass) {
        if constexpr (PROC == 5) lum = pp_ttj_terms(P, A, s_lnx, s_row, ev, asf, quark_sum, nullptr);
        else lum = luminosity<PROC>(P, A, s_lnx, s_row, ev, asf);
        if constexpr (PROC == 7) quark_sum = A.quark_terms[idx];
      }
    }
    const bool pass = valid && ev.pass;
    const int obs_bins = (pass && A.obs != nullptr) ? observable_bins<PROC>(A, ev) : 0;
    const double me2 =
        coop_block_me2<PG, G>(s_teams, n_teams, s_tab, s_cnt, s_res, queue, (unsigned)rd, pass, ev.k, ev.shat, P);
    double w = 0.0;
    if (pass) {
      ++acc.n_pass;
      if (PROC == 5 || PROC == 7) w = event_weight<PROC>(P, ev, 1.0, fma(lum, me2 * asf, quark_sum));
      else w = event_weight<PROC>(P, ev, lum, me2 * asf);
    }
    accumulate_event<PROC, UNW>(P, A, s_grid, s_hist, valid, event, w, bins, acc, obs_bins);
  }
  block_finish(A, acc, s_red, s_hist, D * nb);
}

// carve-up of the debug kernels' shared memory
template <class PG>
struct CoopDebugSmem {
  double *teams, *s_res, *queue;
  unsigned* s_cnt;
  uint4* s_tab;
  __device__ explicit CoopDebugSmem(double* base) {
    constexpr int n_teams = kCoopDebugThreads / PG::Team;
    teams = base;
    s_cnt = reinterpret_cast<unsigned*>(base + n_teams * PG::TeamDoubles);
    s_res = base + n_teams * PG::TeamDoubles + 32;
    queue = s_res + PG::Warps * kCoopDebugThreads;
    s_tab = reinterpret_cast<uint4*>(queue + kCoopDebugThreads * PG::Queue);
  }
};

// Per-event dump through the same team program: block = 64 threads (one or two teams), thread = event.
template <int PROC>
__global__ void __launch_bounds__(kCoopDebugThreads) debug_eval_coop_kernel(const Params P, const PassArgs A, double* out) {
  typedef typename CoopOf<PROC>::PG PG;
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  extern __shared__ double2 smem2[];
  const CoopDebugSmem<PG> L(reinterpret_cast<double*>(smem2));
  coop_load_table<PG>(L.s_tab);
  __syncthreads();
  const int row_len = 3 * D + 4 * (NF + 2) + 9 + (PROC == 7 ? 2 : 0);
  const uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = idx < A.n_events;
  const uint64_t event = A.first_event + idx;
  double* row = out + idx * row_len;
  Event<PROC> ev;
  ev.pass = false;
  Bins<PROC> bins;
  if (valid) {
    DebugRow dbg = {row, D, NF};
    generate_event<PROC>(P, A.grid, A.seed, A.iteration, event, ev, bins, dbg);
  }
  const bool pass = valid && ev.pass;
  double me2 = coop_block_me2<PG, 1>(L.teams, kCoopDebugThreads / PG::Team, L.s_tab, L.s_cnt, L.s_res, L.queue, 0u,
                                     pass, ev.k, ev.shat, P);
  if (!valid) return;
  double mom[NF + 2][4];
  lab_momenta<PROC>(ev, mom);
  double* q = row + D;
  for (int i = 0; i < NF + 2; ++i)
    for (int c = 0; c < 4; ++c) *q++ = mom[i][c];
  double lum = 0.0, w = 0.0;
  if (pass) {
    double asf;
    if constexpr (PROC == 7) {
      double quark_sum, parts[2];
      lum = pp_ttgg_terms(P, A, A.pdf_lnx, A.pdf_row, ev, asf, quark_sum, parts);
      me2 *= asf;
      w = event_weight<PROC>(P, ev, 1.0, fma(lum, me2, quark_sum));
      row[3 * D + 4 * (NF + 2) + 9] = parts[0];
      row[3 * D + 4 * (NF + 2) + 10] = parts[1];
    } else {
      lum = luminosity<PROC>(P, A, A.pdf_lnx, A.pdf_row, ev, asf);
      me2 *= asf;
      w = event_weight<PROC>(P, ev, lum, me2);
    }
  } else if (PROC == 7) {
    row[3 * D + 4 * (NF + 2) + 9] = 0.0;
    row[3 * D + 4 * (NF + 2) + 10] = 0.0;
  }
  q[0] = ev.x1; q[1] = ev.x2; q[2] = lum; q[3] = me2; q[4] = ev.phi; q[5] = ev.jac_vegas; q[6] = w;
  q[7] = pass ? 1.0 : 0.0;
  q[8] = accept_draw(A.seed, A.iteration, event);
}

// |M|^2 at caller-supplied CM-frame momenta mom[n][NF + 2][4] (beams first): block = 64 threads, thread = event.
template <int PROC>
__global__ void __launch_bounds__(kCoopDebugThreads) debug_me2_coop_kernel(const Params P, const double* mom, uint64_t n,
                                                                           double* out) {
  typedef typename CoopOf<PROC>::PG PG;
  constexpr int NF = Traits<PROC>::NF;
  extern __shared__ double2 smem2[];
  const CoopDebugSmem<PG> L(reinterpret_cast<double*>(smem2));
  coop_load_table<PG>(L.s_tab);
  __syncthreads();
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = i < n;
  double k[NF][4];
  double shat = 0.0;
  if (valid) {
    const double* m = mom + i * (NF + 2) * 4;
    for (int f = 0; f < NF; ++f)
      for (int c = 0; c < 4; ++c) k[f][c] = m[(2 + f) * 4 + c];
    shat = 4.0 * m[0] * m[0];
  }
  const double me2 = coop_block_me2<PG, 1>(L.teams, kCoopDebugThreads / PG::Team, L.s_tab, L.s_cnt, L.s_res, L.queue, 0u,
                                           valid, k, shat, P);
  if (valid) out[i] = me2;
}

}  // namespace mf
