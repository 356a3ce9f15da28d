// mf_kernels_coop.cuh — the fused pass for g g -> t tbar g g (BASELINE.json configs[3], [4]): steps a1-a6 and
// a10-a14 one thread per event exactly as in mf_kernels.cuh, steps a7-a9 (the matrix element, >99 % of the
// arithmetic) by teams of 64 threads per event over a shared-memory scratch
// (mf_me_coop.cuh).
//
// Block = T teams of 64 threads (T = 6 for 50 bins: 6 x 30.8 kB of scratch + operand table + grid + histogram +
// PDF row fill the 227 kB of one SM; one block per SM, 12 warps = 3 per scheduler, <= 168 registers).  Per round
// every thread generates its own event; the events of the block that passed the cuts are ranked and in step s
// team t computes the event of rank s T + t: the owner publishes the four final-state momenta, the team computes
// |M|^2, the owner reads the result.  All teams execute the matrix-element program in lock-step (block barriers
// between its stages): the SM then fetches ONE instruction stream, which matters because the program is larger
// than the instruction caches.
#pragma once
#include "mf_kernels.cuh"
#include "mf_me_coop.cuh"

namespace mf {

constexpr int kCoopMaxTeams = 6;

// shared-memory carve-up of a coop block (doubles; every region starts 16-byte aligned)
struct CoopSmem {
  int grid, hist, lnx, row, red, cnt, tab, teams, total;
  __host__ __device__ CoopSmem(int D, int nb, int nx, int n_teams) {
    auto even = [](int v) { return (v + 1) & ~1; };
    grid = 0;
    hist = grid + even(D * (nb + 1));
    lnx = hist + even(D * nb);
    row = lnx + even(nx);
    red = row + even(nx);
    cnt = red + 5 * 32;
    tab = cnt + 32;
    teams = tab + 2 * kCoopTableVecs;
    total = teams + n_teams * kCoopTeamDoubles;
  }
};

// shared memory of the single-team debug kernels: team | rank counters | operand table
constexpr int kCoopDebugSmemBytes = (kCoopTeamDoubles + 32 + 2 * kCoopTableVecs) * 8;

// copies the operand table into shared memory (all threads of the block; the caller synchronises)
__device__ __forceinline__ void coop_load_table(uint4* s_tab) {
  const uint4* g = reinterpret_cast<const uint4*>(kCoopTable);
  for (int i = threadIdx.x; i < kCoopTableVecs; i += blockDim.x) s_tab[i] = g[i];
}

// |M|^2 (with couplings and averaging) of this thread's own event.  EVERY thread of the block must call it (it
// contains block barriers).  The events of the block that passed the cuts are ranked (ballot + prefix over the
// warps); in step s team t computes the event of rank s * n_teams + t: its owner (any thread of the block)
// writes the momenta into that team's input area and reads the result from the team's reduction slots.
// s_cnt: 2 x 32 unsigned (double-buffered by `round`).  Returns 0 for threads whose event did not pass.
__device__ __forceinline__ double coop_block_me2(double* teams, int n_teams, const uint4* tab, unsigned* s_cnt,
                                                 unsigned round, bool pass, const double (*k)[4], double shat,
                                                 const Params& P) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  unsigned* cnt = s_cnt + 32 * (round & 1u);
  const unsigned bal = __ballot_sync(0xFFFFFFFFu, pass);
  if (lane == 0) cnt[warp] = __popc(bal);
  __syncthreads();
  int base = 0, total = 0;
  for (int w = 0; w < n_warps; ++w) {
    const int c = (int)cnt[w];
    if (w < warp) base += c;
    total += c;
  }
  const int rank = base + __popc(bal & ((1u << lane) - 1u));
  const int my_step = pass ? rank / n_teams : -2, my_team = rank - (rank / n_teams) * n_teams;
  const int team = threadIdx.x / kCoopTeam, tid = threadIdx.x % kCoopTeam;
  double* tm = teams + team * kCoopTeamDoubles;
  double* mine = teams + my_team * kCoopTeamDoubles;
  const int n_steps = (total + n_teams - 1) / n_teams;
  double me2 = 0.0;
  // The owner of step s + 1 publishes its momenta while the teams finish step s (the input area is read only by S0,
  // which lies at least one barrier back), so one barrier per step separates "results written / inputs written"
  // from "results read / S0 starts".
  auto publish = [&]() {
    double* in = mine + kCoopOffIn;
#pragma unroll
    for (int f = 0; f < 4; ++f)
#pragma unroll
      for (int c = 0; c < 4; ++c) in[4 * f + c] = k[f][c];
    in[16] = shat;
  };
  if (my_step == 0) publish();
  __syncthreads();
  for (int s = 0; s < n_steps; ++s) {
    coop_me2_lockstep(tm, tab, tid, s * n_teams + team < total, P.m_top);
    if (my_step == s + 1) publish();
    __syncthreads();
    // top spin state 0 only: the other one gives the same sum (spin-flip symmetry), hence the factor 2
    if (s == my_step) me2 = (mine[kCoopOffRed] + mine[kCoopOffRed + 1]) * (2.0 * P.me_norm / kCoopCden);
  }
  return me2;
}

template <bool UNW>
__global__ void __launch_bounds__(kCoopMaxTeams * kCoopTeam, 1) fused_pass_coop_kernel(const Params P, const PassArgs A) {
  constexpr int PROC = 3, D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  extern __shared__ double2 smem2[];
  double* smem = reinterpret_cast<double*>(smem2);
  const int nb = P.n_bins, nx = P.pdf_nx;
  const int n_teams = blockDim.x / kCoopTeam;
  const CoopSmem L(D, nb, nx, n_teams);
  double* s_grid = smem + L.grid;
  double* s_hist = smem + L.hist;
  double* s_lnx = smem + L.lnx;
  double* s_row = smem + L.row;
  double* s_red = smem + L.red;
  unsigned* s_cnt = reinterpret_cast<unsigned*>(smem + L.cnt);
  double* s_teams = smem + L.teams;
  uint4* s_tab = reinterpret_cast<uint4*>(smem + L.tab);
  coop_load_table(s_tab);
  for (int i = threadIdx.x; i < D * (nb + 1); i += blockDim.x) s_grid[i] = A.grid[i];
  for (int i = threadIdx.x; i < D * nb; i += blockDim.x) s_hist[i] = 0.0;
  for (int i = threadIdx.x; i < nx; i += blockDim.x) { s_lnx[i] = A.pdf_lnx[i]; s_row[i] = A.pdf_row[i]; }
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
    double lum = 0.0;
    if (valid) {
      DebugRow dbg = {nullptr, D, NF};
      generate_event<PROC>(P, s_grid, A.seed, A.iteration, event, ev, bins, dbg);
      if (ev.pass) lum = luminosity<PROC>(P, s_lnx, s_row, ev.x1, ev.x2);
    }
    const bool pass = valid && ev.pass;
    const double me2 = coop_block_me2(s_teams, n_teams, s_tab, s_cnt, (unsigned)rd, pass, ev.k, ev.shat, P);
    double w = 0.0;
    if (pass) {
      ++acc.n_pass;
      w = event_weight<PROC>(P, ev, lum, me2);
    }
    accumulate_event<PROC, UNW>(P, A, s_grid, s_hist, valid, event, w, bins, acc);
  }
  block_finish(A, acc, s_red, s_hist, D * nb);
}

// Per-event dump for g g -> t tbar g g through the same team program: block = one team, thread = event.
__global__ void __launch_bounds__(kCoopTeam) debug_eval_coop_kernel(const Params P, const PassArgs A, double* out) {
  constexpr int PROC = 3, D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  extern __shared__ double2 smem2[];
  double* tm = reinterpret_cast<double*>(smem2);
  unsigned* s_cnt = reinterpret_cast<unsigned*>(tm + kCoopTeamDoubles);
  uint4* s_tab = reinterpret_cast<uint4*>(tm + kCoopTeamDoubles + 32);
  coop_load_table(s_tab);
  __syncthreads();
  const int row_len = 3 * D + 4 * (NF + 2) + 9;
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
  const double me2 = coop_block_me2(tm, 1, s_tab, s_cnt, 0u, pass, ev.k, ev.shat, P);
  if (!valid) return;
  double mom[NF + 2][4];
  lab_momenta<PROC>(ev, mom);
  double* q = row + D;
  for (int i = 0; i < NF + 2; ++i)
    for (int c = 0; c < 4; ++c) *q++ = mom[i][c];
  double lum = 0.0, w = 0.0;
  if (pass) {
    lum = luminosity<PROC>(P, A.pdf_lnx, A.pdf_row, ev.x1, ev.x2);
    w = event_weight<PROC>(P, ev, lum, me2);
  }
  q[0] = ev.x1; q[1] = ev.x2; q[2] = lum; q[3] = me2; q[4] = ev.phi; q[5] = ev.jac_vegas; q[6] = w;
  q[7] = pass ? 1.0 : 0.0;
  q[8] = accept_draw(A.seed, A.iteration, event);
}

// |M|^2 at caller-supplied CM-frame momenta mom[n][6][4] (beams first): block = one team, thread = event.
__global__ void __launch_bounds__(kCoopTeam) debug_me2_coop_kernel(const Params P, const double* mom, uint64_t n,
                                                                    double* out) {
  extern __shared__ double2 smem2[];
  double* tm = reinterpret_cast<double*>(smem2);
  unsigned* s_cnt = reinterpret_cast<unsigned*>(tm + kCoopTeamDoubles);
  uint4* s_tab = reinterpret_cast<uint4*>(tm + kCoopTeamDoubles + 32);
  coop_load_table(s_tab);
  __syncthreads();
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = i < n;
  double k[4][4];
  double shat = 0.0;
  if (valid) {
    const double* m = mom + i * 24;
    for (int f = 0; f < 4; ++f)
      for (int c = 0; c < 4; ++c) k[f][c] = m[(2 + f) * 4 + c];
    shat = 4.0 * m[0] * m[0];
  }
  const double me2 = coop_block_me2(tm, 1, s_tab, s_cnt, 0u, valid, k, shat, P);
  if (valid) out[i] = me2;
}

}  // namespace mf
