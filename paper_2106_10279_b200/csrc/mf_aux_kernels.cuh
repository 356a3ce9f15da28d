// mf_aux_kernels.cuh — grid refinement (step a13), the per-event debug dump and the small diagnostic
// kernels behind mf_debug_* / mf_measure_fp64_peak.
#pragma once
#include "mf_kernels.cuh"

namespace mf {

constexpr int kMaxBins = 128;  // == MF_MAX_BINS

// a13. VEGAS grid refinement (Lepage; R14), one warp per dimension:
//   s_i = smoothed histogram / its sum;  r_i = ((s_i - 1)/ln s_i)^alpha (0 for s_i = 0, 1 for s_i >= 1);
//   new edges cut the piecewise-constant density r into nb bins of equal content delta = sum r / nb.
// The smoothing and the damping run across the lanes; the sums and the rebinning walk are sequential in
// lane 0, in bin order.
__global__ void __launch_bounds__(32) refine_grid_kernel(double* grid, const double* hist, int nb, double alpha) {
  __shared__ double s[kMaxBins], r[kMaxBins], e_old[kMaxBins + 1], e_new[kMaxBins + 1];
  const int d = blockIdx.x, lane = threadIdx.x;
  const double* h = hist + (size_t)d * nb;
  double* e = grid + (size_t)d * (nb + 1);
  for (int i = lane; i <= nb; i += 32) e_old[i] = e[i];
  for (int i = lane; i < nb; i += 32) {
    double v;
    if (i == 0) v = (h[0] + h[1]) / 2.0;
    else if (i == nb - 1) v = (h[nb - 2] + h[nb - 1]) / 2.0;
    else v = (h[i - 1] + h[i] + h[i + 1]) / 3.0;
    s[i] = v;
  }
  __syncwarp();
  double S = 0.0;
  for (int i = 0; i < nb; ++i) S += s[i];  // every lane, same order
  if (!(S > 0.0)) return;                  // empty histogram: leave this dimension alone
  for (int i = lane; i < nb; i += 32) {
    double si = s[i] / S, ri;
    if (!(si > 0.0)) ri = 0.0;
    else if (!(si < 1.0)) ri = 1.0;
    else ri = pow((si - 1.0) / log(si), alpha);
    r[i] = ri;
  }
  __syncwarp();
  if (lane == 0) {
    double rsum = 0.0;
    for (int i = 0; i < nb; ++i) rsum += r[i];
    const double delta = rsum / (double)nb;
    double acc = 0.0;
    int j = 0;
    e_new[0] = 0.0;
    e_new[nb] = 1.0;
    for (int i = 1; i < nb; ++i) {
      while (acc < delta && j < nb) { acc += r[j]; ++j; }
      acc -= delta;
      e_new[i] = e_old[j] - (acc / r[j - 1]) * (e_old[j] - e_old[j - 1]);
    }
  }
  __syncwarp();
  for (int i = lane; i <= nb; i += 32) e[i] = e_new[i];
}

// Per-event dump: one thread per event, row layout of include/mf.h.
template <int PROC>
__global__ void __launch_bounds__(kThreads) debug_eval_kernel(const Params P, const PassArgs A, double* out) {
  constexpr int D = Traits<PROC>::D, NF = Traits<PROC>::NF;
  const int row_len = 3 * D + 4 * (NF + 2) + 9 + (PROC == 4 ? 2 : PROC == 5 ? 6 : 0);
  uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= A.n_events) return;
  const uint64_t event = A.first_event + idx;
  double* row = out + idx * row_len;
  Event<PROC> ev;
  Bins<PROC> bins;
  DebugRow dbg = {row, D, NF};
  generate_event<PROC>(P, A.grid, A.seed, A.iteration, event, ev, bins, dbg);
  double mom[NF + 2][4];
  lab_momenta<PROC>(ev, mom);
  double* q = row + D;
  for (int i = 0; i < NF + 2; ++i)
    for (int c = 0; c < 4; ++c) *q++ = mom[i][c];
  double parts[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0}, w = 0.0;
  if (ev.pass) w = weigh_event<PROC>(P, A, A.pdf_lnx, A.pdf_row, ev, parts);
  const double lum = parts[0], me2 = parts[1];
  if (PROC == 4) { row[row_len - 2] = parts[2]; row[row_len - 1] = parts[3]; }
  if (PROC == 5)
    for (int c = 0; c < 6; ++c) row[row_len - 6 + c] = parts[2 + c];
  q[0] = ev.x1; q[1] = ev.x2; q[2] = lum; q[3] = me2; q[4] = ev.phi; q[5] = ev.jac_vegas; q[6] = w;
  q[7] = ev.pass ? 1.0 : 0.0;
  q[8] = accept_draw(A.seed, A.iteration, event);
}

// |M|^2 at caller-supplied CM-frame momenta mom[n][NF+2][4], beams first.
template <int PROC>
__global__ void __launch_bounds__(kThreads) debug_me2_kernel(const Params P, const double* mom, uint64_t n,
                                                             double* out) {
  constexpr int NF = Traits<PROC>::NF;
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double* m = mom + i * (NF + 2) * 4;
  double k[NF][4];
  for (int f = 0; f < NF; ++f)
    for (int c = 0; c < 4; ++c) k[f][c] = m[(2 + f) * 4 + c];
  double shat = 4.0 * m[0] * m[0];
  if (PROC == 4) {   // two channels per point: (gg, q qbar)
    out[2 * i] = me2_call<PROC>(P, shat, k);
    out[2 * i + 1] = matrix_element_qq(P, shat, k);
  } else {
    out[i] = me2_call<PROC>(P, shat, k);
  }
}

// quark channels of pp -> ttbar g at caller-supplied momenta mom[n][5][4] (the two incoming first), kinds of include/mf.h
__global__ void __launch_bounds__(kThreads) debug_me2_quark_gluon_kernel(int kind, double m_top, double g2,
                                                                         const double* mom, uint64_t n, double* out) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  if (kind == 3) {                      // q qbar -> t tbar g g: mom[n][6][4]
    const double* m6 = mom + i * 24;
    out[i] = me2_qq_ttgg(m6, m6 + 4, m6 + 8, m6 + 12, m6 + 16, m6 + 20, m_top, g2);
    return;
  }
  const double* m = mom + i * 20;
  if (kind == 0) out[i] = me2_light_line_ttg(0, m, m + 4, m + 8, m + 12, m + 16, m_top, g2);
  else if (kind == 1) out[i] = me2_light_line_ttg(1, m, m + 16, m + 8, m + 12, m + 4, m_top, g2);
  else out[i] = me2_light_line_ttg(1, m, m + 16, m + 12, m + 8, m + 4, m_top, g2);   // charge conjugate of kind 1
}

__global__ void debug_philox_kernel(uint64_t seed, uint32_t iteration, uint64_t first, uint64_t n, uint32_t n_blocks,
                                    uint32_t* out) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n * n_blocks) return;
  uint64_t k = i / n_blocks;
  uint32_t b = (uint32_t)(i % n_blocks);
  U4 r = philox_block(seed, iteration, first + k, b);
  out[4 * i + 0] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

__global__ void debug_pdf_kernel(const double* lnx, const double* lnq2, const double* xf, int nx, int nq,
                                 const double* x, const double* q2, uint64_t n, double* out) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = pdf_xf_2d(lnx, lnq2, xf, nx, nq, x[i], q2[i]);
}

// collapses every parton table at the process' fixed mu2 (one thread per table and x knot: the tables are contiguous
// [n_tables][nx][nq], so (table, knot) is one flat row index)
__global__ void pdf_collapse_kernel(const double* xf, const double* lnq2, int n_rows, int nq, int jq, double uq,
                                    double* row) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n_rows) row[i] = pdf_collapse_q2(xf, lnq2, nq, i, jq, uq);
}

// FP64 peak probe: 8 independent DFMA chains per thread, enough warps to fill the FP64 pipe.
__global__ void __launch_bounds__(256) dfma_peak_kernel(long long iters, double seed, double* sink) {
  double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6,
         a7 = seed + 7;
  const double m = 0.999999, c = 1e-9 * (double)threadIdx.x;
  for (long long i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == 123456.789) sink[0] = s;
}

// FP64 tensor-path probe: 4 independent DMMA.884 (mma.sync m8n8k4 f64, 256 multiply-adds each) accumulators per warp.
__global__ void __launch_bounds__(256) dmma_peak_kernel(long long iters, double seed, double* sink) {
  double c[4][2];
  for (int i = 0; i < 4; ++i) { c[i][0] = seed + i; c[i][1] = seed - i; }
  const double a = 0.999999, b = 1.0 + 1e-9 * (double)threadIdx.x;
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 4; ++i)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                   : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
  for (int i = 0; i < 4; ++i) s += c[i][0] + c[i][1];
  if (s == 123456.789) sink[0] = s;
}

}  // namespace mf
