// mf_kernels_cta.cuh — the fused pass for g g -> t tbar g g g (process 6): steps a1-a6
// and a10-a14 one thread per event exactly as in mf_kernels.cuh; steps a7-a9 (the matrix element: 7.6 Mflop per event, 122 kB
// of off-shell currents) by the WHOLE BLOCK per event (mf_me_cta5.cuh).  Per round every thread generates its own event;
// the events of the block that passed the cuts are ranked and their momenta queued (a per-block slice of a small
// L2-resident buffer, [double][rank]); the block then works through the ranks one after the other and leaves |M|^2 in a
// per-rank result slot that the owner thread reads after the round.
#pragma once
#include "mf_kernels.cuh"
#include "mf_me_cta5.cuh"

namespace mf {

constexpr int kCtaThreads = 512;            // 16 warps, <= 128 registers; one block per SM (shared memory)
constexpr int kCtaQueue = 21;               // k[5][4], shat

// shared-memory carve-up (doubles; every region 16-byte aligned)
struct CtaSmem {
  int grid, hist, lnx, row, red, cnt, res, me, total;
  __host__ __device__ CtaSmem(int D, int nb, int nx, int threads) {
    auto even = [](int v) { return (v + 1) & ~1; };
    grid = 0;
    hist = grid + even(D * (nb + 1));
    lnx = hist + even(D * nb);
    row = lnx + even(nx);
    red = row + even(nx);
    cnt = red + 5 * 32;
    res = cnt + 32;
    me = res + even(threads);
    total = me + g5::kScratchDoubles;
  }
};

// |M|^2 (with couplings and averaging) of this thread's own event.  EVERY thread of the block must call it.  `queue` holds
// kCtaQueue x blockDim.x doubles ([double][rank]); s_cnt 2 x 32 unsigned (double-buffered by `round`); s_res one double per thread.
__device__ __forceinline__ double cta_block_me2(double* S, unsigned* s_cnt, double* s_res, double* s_red, double* queue,
                                                unsigned round, bool pass, const double (*k)[4], double shat, const Params& P) {
  const int bwarp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5, qs = blockDim.x;
  unsigned* cnt = s_cnt + 32 * (round & 1u);
  const unsigned bal = __ballot_sync(0xFFFFFFFFu, pass);
  if (lane == 0) cnt[bwarp] = __popc(bal);
  __syncthreads();
  int base = 0, total = 0;
  for (int w = 0; w < n_warps; ++w) {
    const int c = (int)cnt[w];
    if (w < bwarp) base += c;
    total += c;
  }
  const int rank = base + __popc(bal & ((1u << lane) - 1u));
  if (pass) {
#pragma unroll
    for (int f = 0; f < 5; ++f)
#pragma unroll
      for (int c = 0; c < 4; ++c) queue[(4 * f + c) * qs + rank] = k[f][c];
    queue[20 * qs + rank] = shat;
  }
  __syncthreads();
#pragma unroll 1
  for (int r = 0; r < total; ++r) {
    if (threadIdx.x < kCtaQueue) S[g5::kOffIn + threadIdx.x] = queue[threadIdx.x * qs + r];
    __syncthreads();
    const double sum = g5::cta_me2(S, s_red, P.m_top);
    if (threadIdx.x == 0) s_res[r] = sum;
  }
  __syncthreads();
  // top spin state 0 only: the other one gives the same sum (spin-flip symmetry), hence the factor 2
  return pass ? s_res[rank] * (2.0 * P.me_norm / g5::kCden) : 0.0;
}

template <bool UNW>
__global__ void __launch_bounds__(kCtaThreads, 1) fused_pass_cta_kernel(const Params P, const PassArgs A) {
  constexpr int PROC = 6, D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  extern __shared__ double2 smem2[];
  double* smem = reinterpret_cast<double*>(smem2);
  const int nb = P.n_bins, nx = P.pdf_nx;
  const CtaSmem L(D, nb, nx, blockDim.x);
  double* s_grid = smem + L.grid;
  double* s_hist = smem + L.hist;
  double* s_lnx = smem + L.lnx;
  double* s_row = smem + L.row;
  double* s_red = smem + L.red;
  unsigned* s_cnt = reinterpret_cast<unsigned*>(smem + L.cnt);
  double* s_res = smem + L.res;
  double* S = smem + L.me;
  double* queue = A.coop_queue + (size_t)blockIdx.x * blockDim.x * kCtaQueue;
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
    double lum = 0.0, asf = 1.0;
    if (valid) {
      DebugRow dbg = {nullptr, D, NF};
      generate_event<PROC>(P, s_grid, A.seed, A.iteration, event, ev, bins, dbg);
      if (ev.pass) lum = luminosity<PROC>(P, A, s_lnx, s_row, ev, asf);
    }
    const bool pass = valid && ev.pass;
    const int obs_bins = (pass && A.obs != nullptr) ? observable_bins<PROC>(A, ev) : 0;
    const double me2 = cta_block_me2(S, s_cnt, s_res, s_red, queue, (unsigned)rd, pass, ev.k, ev.shat, P);
    double w = 0.0;
    if (pass) {
      ++acc.n_pass;
      w = event_weight<PROC>(P, ev, lum, me2 * asf);
    }
    accumulate_event<PROC, UNW>(P, A, s_grid, s_hist, valid, event, w, bins, acc, obs_bins);
  }
  block_finish(A, acc, s_red, s_hist, D * nb);
}

// shared memory of the debug kernels: the matrix-element scratch | rank counters | results | reduction | queue
constexpr int kCtaDebugThreads = 128;       // thread = event; the queue of a 512-thread block would not fit beside the scratch
constexpr int cta_debug_smem_bytes() {
  return (g5::kScratchDoubles + 32 + kCtaDebugThreads + 32 + kCtaQueue * kCtaDebugThreads) * 8;
}
struct CtaDebugSmem {
  double *S, *s_res, *s_red, *queue;
  unsigned* s_cnt;
  __device__ explicit CtaDebugSmem(double* base) {
    S = base;
    s_cnt = reinterpret_cast<unsigned*>(base + g5::kScratchDoubles);
    s_res = base + g5::kScratchDoubles + 32;
    s_red = s_res + kCtaDebugThreads;
    queue = s_red + 32;
  }
};

// Per-event dump through the same block program: thread = event.
__global__ void __launch_bounds__(kCtaDebugThreads, 1) debug_eval_cta_kernel(const Params P, const PassArgs A, double* out) {
  constexpr int PROC = 6, D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  extern __shared__ double2 smem2[];
  const CtaDebugSmem L(reinterpret_cast<double*>(smem2));
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
  double me2 = cta_block_me2(L.S, L.s_cnt, L.s_res, L.s_red, L.queue, 0u, pass, ev.k, ev.shat, P);
  if (!valid) return;
  double mom[NF + 2][4];
  lab_momenta<PROC>(ev, mom);
  double* q = row + D;
  for (int i = 0; i < NF + 2; ++i)
    for (int c = 0; c < 4; ++c) *q++ = mom[i][c];
  double lum = 0.0, w = 0.0;
  if (pass) {
    double asf;
    lum = luminosity<PROC>(P, A, A.pdf_lnx, A.pdf_row, ev, asf);
    me2 *= asf;
    w = event_weight<PROC>(P, ev, lum, me2);
  }
  q[0] = ev.x1; q[1] = ev.x2; q[2] = lum; q[3] = me2; q[4] = ev.phi; q[5] = ev.jac_vegas; q[6] = w;
  q[7] = pass ? 1.0 : 0.0;
  q[8] = accept_draw(A.seed, A.iteration, event);
}

// |M|^2 at caller-supplied CM-frame momenta mom[n][7][4] (beams first): thread = event.
__global__ void __launch_bounds__(kCtaDebugThreads, 1) debug_me2_cta_kernel(const Params P, const double* mom, uint64_t n,
                                                                            double* out) {
  extern __shared__ double2 smem2[];
  const CtaDebugSmem L(reinterpret_cast<double*>(smem2));
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const bool valid = i < n;
  double k[5][4];
  double shat = 0.0;
  if (valid) {
    const double* m = mom + i * 7 * 4;
    for (int f = 0; f < 5; ++f)
      for (int c = 0; c < 4; ++c) k[f][c] = m[(2 + f) * 4 + c];
    shat = 4.0 * m[0] * m[0];
  }
  const double me2 = cta_block_me2(L.S, L.s_cnt, L.s_res, L.s_red, L.queue, 0u, valid, k, shat, P);
  if (valid) out[i] = me2;
}

}  // namespace mf
