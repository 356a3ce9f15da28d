// mf_me_cta5.cuh — steps a7-a9 for g g -> t tbar g g g (the paper's heaviest process,
// 1240 diagrams, 128 helicity states, 120 colour orderings): ONE EVENT PER THREAD BLOCK.  All off-shell currents of the
// event (3266 real 4-vectors, 273 spinors: 122 kB) live in the block's shared memory; the block works through the
// colour-ordered recursion level by level, every thread taking work items of the current level (index tables:
// csrc/gen_cta5.py), and contracts the amplitudes with the 120 x 120 colour matrix on the FP64 tensor path (DMMA).
//
//   stage 0   momentum sums P[mask], propagator momenta and inverse denominators, polarisation vectors, external spinors
//   stage 1   J2 (40 items), Y1 (10), X1 (20)          stage 2   J3 (240), Y2 (80), X2 (160)
//   stage 3   J4 (960)                                  stage 4   J5 (1920)
//   stage 5/6 for each half of the polarisation words (pol of gluon 0): amplitudes of the 120 orderings x 16 words x 2
//             antitop spins x (re, im) -> the 120 x 64 matrix XM;  colour: sum_n XM[.][n]^T C XM[.][n]
//
// Conventions as in mf_me_prims.cuh (real polarisations, hatted currents, top spin 0 only and the sum doubled).
// Every stage function is MF_HD and takes the work-item index, so tests/host_shim can run the same code on the host.
#pragma once
#include "mf_me_prims.cuh"

#if !defined(MF_TABLE)
#if defined(__CUDA_ARCH__)
#define MF_TABLE static __device__ const
#else
#define MF_TABLE static const
#endif
#endif

// tables every lane of a (half) warp reads at the same index: constant memory on the device
#if defined(__CUDA_ARCH__)
#define MF_CTABLE static __constant__ const
#else
#define MF_CTABLE static const
#endif

namespace mf { namespace g5 {

#include "mf_me_ttggg_tables_generated.cuh"

// ---- scratch (doubles): VEC | SPIN | scalars (1/P^2, 1/(qX^2 - m^2), 1/(qY^2 - m^2) by mask) | input | XM ----------------
constexpr int kOffSpin = 4 * kNVec, kOffScal = kOffSpin + 8 * kNSpin, kOffIn = kOffScal + 96;
constexpr int kInDoubles = 22;                        // k[5][4] (t, tbar, g2, g3, g4; partonic CM frame), shat, pad
constexpr int kOffXm = kOffIn + kInDoubles;
constexpr int kScratchDoubles = kOffXm + kNPerm * kXmStride;
constexpr int kStage0Items = 38, kStage1Items = 4 * kNSeq2 + 10 + 20, kStage2Items = 8 * kNSeq3 + 80 + 160;
constexpr int kStage3Items = 16 * kNSeq4, kStage4Items = 32 * kNSeq5, kAmpItems = 16 * kNPerm;

// VEC items as two planes of double2 (components (0, 1) | (2, 3)), SPIN items as four planes of (re, im): lanes that
// touch consecutive items issue conflict-free 128-bit accesses
MF_HD rvec ld_vec(const double* S, int i) {
  const double2* q = reinterpret_cast<const double2*>(S);
  const double2 a = q[i], b = q[kNVec + i];
  return rvec{{a.x, a.y, b.x, b.y}};
}
MF_HD void st_vec(double* S, int i, const rvec& r) {
  double2* q = reinterpret_cast<double2*>(S);
  q[i] = make_double2(r.v[0], r.v[1]);
  q[kNVec + i] = make_double2(r.v[2], r.v[3]);
}
MF_HD spin ld_spin(const double* S, int i) {
  const double2* q = reinterpret_cast<const double2*>(S + kOffSpin);
  spin r;
#pragma unroll
  for (int c = 0; c < 4; ++c) { const double2 t = q[c * kNSpin + i]; r.re[c] = t.x; r.im[c] = t.y; }
  return r;
}
MF_HD void st_spin(double* S, int i, const spin& r) {
  double2* q = reinterpret_cast<double2*>(S + kOffSpin);
#pragma unroll
  for (int c = 0; c < 4; ++c) q[c * kNSpin + i] = make_double2(r.re[c], r.im[c]);
}
MF_HD rvec rsigned(const rvec& a, int sgn) { return sgn < 0 ? rvec{{-a.v[0], -a.v[1], -a.v[2], -a.v[3]}} : a; }
// Jhat of the sub-sequence (base, mask) for the polarisation word pw
MF_HD rvec ld_cur(const double* S, int base, int mask, int pw) { return ld_vec(S, base + kPext[mask][pw]); }
MF_HD int pair_index(int a, int b) { return a * 4 + (b < a ? b : b - 1); }      // position in the ordered-pair list

// ---- stage 0 ------------------------------------------------------------------------------------------------------------
// in[0..19] = k[5][4], in[20] = shat.  Gluon labels 0, 1 = beams (+z, -z; momenta incoming), 2..4 = final gluons (enter with -k).
MF_HD void stage0_item(double* S, int item, double mt) {
  const double* in = S + kOffIn;
  double* X = S + kOffScal;
  if (item < 31) {
    const int m = item + 1;
    const double E = 0.5 * sqrt(in[20]);
    rvec P = {{0.0, 0.0, 0.0, 0.0}};
    if (m & 1) { P.v[0] += E; P.v[3] += E; }
    if (m & 2) { P.v[0] += E; P.v[3] -= E; }
#pragma unroll
    for (int g = 2; g < 5; ++g)
      if (m & (1 << g)) {
#pragma unroll
        for (int c = 0; c < 4; ++c) P.v[c] -= in[4 * g + c];
      }
    st_vec(S, kVP + m, P);
    const int bits = (m & 1) + ((m >> 1) & 1) + ((m >> 2) & 1) + ((m >> 3) & 1) + ((m >> 4) & 1);
    if (bits >= 2) X[m] = 1.0 / rdot(P, P);
    if (bits <= 2) {
      rvec qx, qy;
#pragma unroll
      for (int c = 0; c < 4; ++c) { qx.v[c] = P.v[c] - in[4 + c]; qy.v[c] = in[c] - P.v[c]; }
      st_vec(S, kVQX + m, qx);
      st_vec(S, kVQY + m, qy);
      X[32 + m] = 1.0 / (rdot(qx, qx) - mt * mt);
      X[64 + m] = 1.0 / (rdot(qy, qy) - mt * mt);
    }
  } else if (item < 34) {
    const int g = item - 29;                 // 2, 3, 4
    rvec e1, e2;
    pol_vectors(in + 4 * g, e1, e2);
    st_vec(S, kVEps + 2 * g, e1);
    st_vec(S, kVEps + 2 * g + 1, e2);
  } else if (item == 34) {
    st_vec(S, kVEps + 0, rvec{{0.0, 1.0, 0.0, 0.0}});
    st_vec(S, kVEps + 1, rvec{{0.0, 0.0, 1.0, 0.0}});
    st_vec(S, kVEps + 2, rvec{{0.0, 1.0, 0.0, 0.0}});
    st_vec(S, kVEps + 3, rvec{{0.0, 0.0, -1.0, 0.0}});
  } else if (item == 35) {
    st_spin(S, kSUb, ubar_row(in, mt, 0));
  } else if (item < 38) {
    st_spin(S, kSV + item - 36, v_col(in + 4, mt, item - 36));
  }
}

// ---- gluon currents: item = (sequence c, compressed polarisation v) of level k ------------------------------------------
MF_HD void gluon_item(double* S, int k, int item) {
  const int c = item >> k, v = item & ((1 << k) - 1);
  const short* d = kSeqDesc[k - 2][c];
  const int mask = d[0], n3 = d[3] & 255, n4 = d[3] >> 8;
  const int pw = kPdep[mask][v];
  const short* sp = kSplit + d[2];
  rvec acc = {{0.0, 0.0, 0.0, 0.0}};
  for (int s = 0; s < n3; ++s, sp += 5)
    v3_acc(acc, (double)sp[4], ld_cur(S, sp[0], sp[1], pw), ld_vec(S, kVP + sp[1]), ld_cur(S, sp[2], sp[3], pw),
           ld_vec(S, kVP + sp[3]));
  for (int s = 0; s < n4; ++s, sp += 7)
    v4_acc(acc, (double)sp[6], ld_cur(S, sp[0], sp[1], pw), ld_cur(S, sp[2], sp[3], pw), ld_cur(S, sp[4], sp[5], pw));
  st_vec(S, d[1] + v, rscale(acc, S[kOffScal + mask]));
}

// ---- quark currents with one and two gluons -----------------------------------------------------------------------------
MF_HD void y1_item(double* S, int item, double mt) {          // item = a * 2 + pa
  const int a = item >> 1, m = 1 << a;
  const spin t = slash_row(ld_spin(S, kSUb), ld_vec(S, kVEps + item));
  st_spin(S, kSY1 + item, prop_row(t, ld_vec(S, kVQY + m), mt, S[kOffScal + 64 + m]));
}
MF_HD void x1_item(double* S, int item, double mt) {          // item = (d * 2 + hb) * 2 + pd
  const int d = item >> 2, hb = (item >> 1) & 1, pd = item & 1, m = 1 << d;
  const spin t = slash_col(ld_vec(S, kVEps + 2 * d + pd), ld_spin(S, kSV + hb));
  st_spin(S, kSX1 + item, prop_col(ld_vec(S, kVQX + m), mt, S[kOffScal + 32 + m], t));
}
MF_HD rvec ld_j2(const double* S, int a, int b, int pa, int pb) {   // Jhat(ab) for the polarisations of a and b
  const int lo = a < b ? a : b;
  const rvec j = ld_vec(S, kVJ2 + 4 * kJ2Idx[a][b] + (a == lo ? pa | (pb << 1) : pb | (pa << 1)));
  return rsigned(j, a == lo ? 1 : -1);
}
MF_HD void y2_item(double* S, int item, double mt) {          // item = pair(a, b) * 4 + (pa | pb << 1)
  const int pr = item >> 2, a = pr >> 2, r = pr & 3, b = r < a ? r : r + 1, pa = item & 1, pb = (item >> 1) & 1;
  const int m = (1 << a) | (1 << b);
  spin t = slash_row(ld_spin(S, kSUb), ld_j2(S, a, b, pa, pb));
  slash_row_acc(t, ld_spin(S, kSY1 + 2 * a + pa), ld_vec(S, kVEps + 2 * b + pb));
  st_spin(S, kSY2 + item, prop_row(t, ld_vec(S, kVQY + m), mt, S[kOffScal + 64 + m]));
}
MF_HD void x2_item(double* S, int item, double mt) {          // item = (pair(c, d) * 2 + hb) * 4 + (pc | pd << 1)
  const int pr = item >> 3, c = pr >> 2, r = pr & 3, d = r < c ? r : r + 1, hb = (item >> 2) & 1, pc = item & 1,
            pd = (item >> 1) & 1;
  const int m = (1 << c) | (1 << d);
  spin t = slash_col(ld_vec(S, kVEps + 2 * c + pc), ld_spin(S, kSX1 + (d * 2 + hb) * 2 + pd));
  slash_col_acc(t, ld_j2(S, c, d, pc, pd), ld_spin(S, kSV + hb));
  st_spin(S, kSX2 + item, prop_col(ld_vec(S, kVQX + m), mt, S[kOffScal + 32 + m], t));
}
MF_HD void stage1_item(double* S, int item, double mt) {
  if (item < 4 * kNSeq2) gluon_item(S, 2, item);
  else if (item < 4 * kNSeq2 + 10) y1_item(S, item - 4 * kNSeq2, mt);
  else x1_item(S, item - 4 * kNSeq2 - 10, mt);
}
MF_HD void stage2_item(double* S, int item, double mt) {
  if (item < 8 * kNSeq3) gluon_item(S, 3, item);
  else if (item < 8 * kNSeq3 + 80) y2_item(S, item - 8 * kNSeq3, mt);
  else x2_item(S, item - 8 * kNSeq3 - 80, mt);
}

// ---- amplitudes: item = ordering s (lexicographic) x 16 polarisation words of the half (pol of gluon 0 = half) --------------
// Ahat(sigma) = sum_{i <= 3 <= j} Y(sigma_1..sigma_{i-1}) Jslash(sigma_i..sigma_j) X(sigma_{j+1}..sigma_5); both antitop spins.
// XM[s][part * 32 + hb * 16 + v] = real (part 0) / imaginary (part 1) part.
MF_HD void amp_item(double* S, int half, int item) {
  const int s = item >> 4, v = item & 15, pw = half | (v << 1);
  const short* t = kAmp[s];
  const int s1 = t[27], s2 = t[28], s4 = t[30], s5 = t[31];
  const int p1 = (pw >> s1) & 1, p2 = (pw >> s2) & 1, p4 = (pw >> s4) & 1, p5 = (pw >> s5) & 1;
  spin Y[3];
  Y[0] = ld_spin(S, kSUb);
  Y[1] = ld_spin(S, kSY1 + 2 * s1 + p1);
  Y[2] = ld_spin(S, kSY2 + 4 * pair_index(s1, s2) + (p1 | (p2 << 1)));
  cplx A[2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
  for (int jj = 0; jj < 3; ++jj) {
    spin T;
#pragma unroll
    for (int c = 0; c < 4; ++c) { T.re[c] = 0.0; T.im[c] = 0.0; }
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      const short* e = t + 3 * (3 * jj + i);
      slash_row_acc(T, Y[i], rsigned(ld_cur(S, e[0], e[1], pw), e[2]));
    }
#pragma unroll
    for (int hb = 0; hb < 2; ++hb) {
      const int xi = jj == 0 ? kSX2 + (pair_index(s4, s5) * 2 + hb) * 4 + (p4 | (p5 << 1))
                             : jj == 1 ? kSX1 + (s5 * 2 + hb) * 2 + p5 : kSV + hb;
      const cplx z = sdot(T, ld_spin(S, xi));
      A[hb].re += z.re;
      A[hb].im += z.im;
    }
  }
  double* xm = S + kOffXm + s * kXmStride + v;
#pragma unroll
  for (int hb = 0; hb < 2; ++hb) { xm[hb * 16] = A[hb].re; xm[32 + hb * 16] = A[hb].im; }
}

// ---- colour contraction of one half: sum over the 64 columns n of XM[.][n]^T Cnum XM[.][n] -----------------------------------
// Host (tests/host_shim): the plain double loop, "thread" tid of nthreads takes rows tid, tid + nthreads, ...
MF_HD double colour_rows_plain(const double* S, int tid, int nthreads) {
  const double* xm = S + kOffXm;
  double acc = 0.0;
  for (int s = tid; s < kNPerm; s += nthreads)
    for (int n = 0; n < 64; ++n) {
      double y = 0.0;
      for (int u = s; u < kNPerm; ++u) y = fma(kColour[s * kNPerm + u], xm[u * kXmStride + n], y);
      acc = fma(xm[s * kXmStride + n], y, acc);
    }
  return acc;
}
#if defined(__CUDACC__)
// Device: Y = kColour XM (upper triangle of 120 x 120 times 120 x 64) as DMMA.884 tiles: row tile m (8 orderings) needs the
// k-steps 2 m .. 29 only; the 15 row tiles are paired {p, 14 - p} (32 k-steps per pair) and split over the two halves of
// the 64 columns: 16 equal tasks for 16 warps.  One C fragment per k-step is reused for 4 column tiles; the warp then
// multiplies its Y fragments with the XM entries at the same positions.  The colour matrix is read from global memory
// (115 kB, the same for every block: L2).
__device__ __forceinline__ double colour_half_dmma(const double* S, int warp, int n_warps, int lane) {
  const double* xm = S + kOffXm;
  const int g = lane >> 2, t = lane & 3;
  double acc = 0.0;
  // task = (pair of row tiles {p, 14 - p}: 30 - 2 p and 2 + 2 p k-steps = 32 in all; tile 7 alone: 16) x half of the columns
#pragma unroll 1
  for (int task = warp; task < 16; task += n_warps) {
    const int p = task >> 1, nh = task & 1;
#pragma unroll 1
    for (int which = 0; which < (p == 7 ? 1 : 2); ++which) {
      const int mt = which == 0 ? p : 14 - p;
      double c[4][2];
#pragma unroll
      for (int n = 0; n < 4; ++n) c[n][0] = c[n][1] = 0.0;
      const double* crow = kColour + (8 * mt + g) * kNPerm + t;
      const double* xcol = xm + t * kXmStride + g + 32 * nh;
#pragma unroll 4
      for (int ks = 2 * mt; ks < kNPerm / 4; ++ks) {
        const double a = crow[4 * ks];
        const double* xr = xcol + 4 * ks * kXmStride;
#pragma unroll
        for (int n = 0; n < 4; ++n) {
          const double b = xr[8 * n];
#if defined(__CUDA_ARCH__)
          asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
              : "+d"(c[n][0]), "+d"(c[n][1]) : "d"(a), "d"(b));
#else
          (void)a; (void)b;      // host pass of nvcc: never executed
#endif
        }
      }
      const double* xo = xm + (8 * mt + g) * kXmStride + 2 * t + 32 * nh;
#pragma unroll
      for (int n = 0; n < 4; ++n) {
        const double2 x = *reinterpret_cast<const double2*>(xo + 8 * n);
        acc = fma(x.x, c[n][0], acc);
        acc = fma(x.y, c[n][1], acc);
      }
    }
  }
  return acc;
}
#endif

// ---- the whole matrix element by one thread block (device) ------------------------------------------------------------------
// Every thread of the block calls it; the event must already be in S + kOffIn and visible (a barrier before the call).
// Returns, in EVERY thread, sum_{hb, pols} Ahat^dagger Cnum Ahat for top spin 0 (the caller multiplies by 2 me_norm / kCden).
// s_red: 32 doubles of shared memory for the block reduction.
#if defined(__CUDACC__)
__device__ __forceinline__ double cta_me2(double* S, double* s_red, double mt) {
  const int tid = threadIdx.x, nt = blockDim.x, warp = tid >> 5, lane = tid & 31;
  for (int i = tid; i < kStage0Items; i += nt) stage0_item(S, i, mt);
  __syncthreads();
  for (int i = tid; i < kStage1Items; i += nt) stage1_item(S, i, mt);
  __syncthreads();
  for (int i = tid; i < kStage2Items; i += nt) stage2_item(S, i, mt);
  __syncthreads();
  for (int i = tid; i < kStage3Items; i += nt) gluon_item(S, 4, i);
  __syncthreads();
  for (int i = tid; i < kStage4Items; i += nt) gluon_item(S, 5, i);
  __syncthreads();
  double acc = 0.0;
#pragma unroll 1
  for (int half = 0; half < 2; ++half) {
    for (int i = tid; i < kAmpItems; i += nt) amp_item(S, half, i);
    __syncthreads();
    acc += colour_half_dmma(S, warp, nt >> 5, lane);
    __syncthreads();
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, o);
  if (lane == 0) s_red[warp] = acc;
  __syncthreads();
  double tot = 0.0;
  for (int w = 0; w < (nt >> 5); ++w) tot += s_red[w];
  __syncthreads();
  return tot;
}
#endif

}}  // namespace mf::g5
