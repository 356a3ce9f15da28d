// madflow_b200.cu — the C ABI of include/mf.h over the sm_100a kernels.  Host side only does argument
// checking, launch geometry and kernel launches; every step of the hot path runs on the device.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/mf.h"
#include "mf_aux_kernels.cuh"
#include "mf_kernels_coop.cuh"
#include "mf_kernels_cta.cuh"

// Scratch of mf_vegas_iterate_static (include/mf.h): per-block partial sums and histogram slices of ONE fused-pass launch.
// File scope, so every GPU that loads the library holds these MF_STATIC_SCRATCH_BYTES until exit.  In host code this name is a
// host-side stand-in, NOT a device address: the address kernels may use comes from cudaGetSymbolAddress (mf_create_process,
// once per handle, with the handle's device current).
static __device__ __align__(256) unsigned char mf_static_scratch[MF_STATIC_SCRATCH_BYTES];

static_assert(sizeof(mf::IterResult) == sizeof(mf_iter_result), "result layouts must agree");
static_assert(mf::kMaxBins == MF_MAX_BINS, "bin limits must agree");

struct mf_process {
  int process = 0, D = 0, NF = 0, device = 0;
  mf::Params P;
  double *d_lnx = nullptr, *d_lnq2 = nullptr, *d_xf = nullptr, *d_row = nullptr;  // PDF table + collapsed row
  mf::BlockPartial* d_partials = nullptr;
  double* d_queue = nullptr;          // cooperative pass: per-block momenta queue
  unsigned char* d_static = nullptr;  // device address of mf_static_scratch on the handle's device (cudaGetSymbolAddress)
  double* d_quark = nullptr;          // MF_PP_TTGG: quark-channel term per event of the current piece (kQuarkChunk events, made at create)
  uint64_t quark_cap = 0;
  unsigned long long* d_start = nullptr;   // cooperative / block processes: the record cursor before the current mf_unweight call
  double* d_obs = nullptr;            // caller-owned observable histograms (mf_set_observables) or NULL
  int obs_nb = 0;
  double obs_ptmax = 0.0, obs_etamax = 0.0;
  double* d_hist_part = nullptr;
  int blocks = 0, threads = mf::kThreads;
  int blocks_unw = 0;
  int prepass_blocks = 0;             // quark_prepass_kernel: resident blocks of the device
  size_t smem = 0;
  char err[256] = {0};
};

namespace {

constexpr uint64_t kQuarkChunk = 1ull << 22;     // events per piece of an MF_PP_TTGG call (32 MB of quark terms)

const char* kNullHandle = "null handle";

int fail(mf_process* p, int code, const char* what, cudaError_t e = cudaSuccess) {
  if (p) {
    if (e != cudaSuccess) snprintf(p->err, sizeof(p->err), "%s: %s", what, cudaGetErrorString(e));
    else snprintf(p->err, sizeof(p->err), "%s", what);
  }
  return code;
}

template <int PROC, bool UNW> const void* pass_fn() { return (const void*)mf::fused_pass_kernel<PROC, UNW>; }
const void* pass_fn(int proc, bool unw) {
  switch (proc) {
    case 0: return unw ? pass_fn<0, true>() : pass_fn<0, false>();
    case 1: return unw ? pass_fn<1, true>() : pass_fn<1, false>();
    case 4: return unw ? pass_fn<4, true>() : pass_fn<4, false>();
    case 5: return unw ? (const void*)mf::fused_pass_coop_kernel<5, true> : (const void*)mf::fused_pass_coop_kernel<5, false>;
    case 6: return unw ? (const void*)mf::fused_pass_cta_kernel<true> : (const void*)mf::fused_pass_cta_kernel<false>;
    case 2: return unw ? (const void*)mf::fused_pass_coop_kernel<2, true> : (const void*)mf::fused_pass_coop_kernel<2, false>;
    case 7: return unw ? (const void*)mf::fused_pass_coop_kernel<7, true> : (const void*)mf::fused_pass_coop_kernel<7, false>;
    default: return unw ? (const void*)mf::fused_pass_coop_kernel<3, true> : (const void*)mf::fused_pass_coop_kernel<3, false>;
  }
}

// launch shape, shared-memory sizes and kernel attributes of the cooperative pass of process PROC
template <int PROC>
cudaError_t coop_setup(mf_process* p, const cudaDeviceProp& prop) {
  typedef typename mf::CoopOf<PROC>::PG PG;
  const mf::Params& P = p->P;
  const int group = PG::Team == 32 ? mf::kCoopGroupWarp : mf::kCoopGroup;      // teams run in lock-step groups
  int n_teams = mf::CoopOf<PROC>::MaxTeams;
  while (n_teams > 0 &&
         (size_t)mf::CoopSmem<PG>(p->D, P.n_bins, P.pdf_nx, PROC == 5 ? P.pdf_nx * P.pdf_nfl : P.pdf_nx, n_teams).total * 8 > (size_t)prop.sharedMemPerBlockOptin)
    --n_teams;
  n_teams -= n_teams % group;
  if (n_teams < 1) return cudaErrorInvalidConfiguration;
  p->threads = n_teams * PG::Team;
  p->smem = (size_t)mf::CoopSmem<PG>(p->D, P.n_bins, P.pdf_nx, PROC == 5 ? P.pdf_nx * P.pdf_nfl : P.pdf_nx, n_teams).total * 8;
  cudaError_t e;
  for (int u = 0; u < 2; ++u)
    // the attribute belongs to the kernel, not to the handle: always ask for the device maximum, so that handles with
    // different bin counts (different shared-memory needs) can coexist
    if ((e = cudaFuncSetAttribute(pass_fn(PROC, u != 0), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  (int)prop.sharedMemPerBlockOptin)) != cudaSuccess) return e;
  if constexpr (PROC == 5) return cudaSuccess;   // its debug entry points are the thread-per-event kernels
  else if ((e = cudaFuncSetAttribute((const void*)mf::debug_eval_coop_kernel<PROC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                mf::coop_debug_smem_bytes<PG>())) != cudaSuccess) return e;
  else return cudaFuncSetAttribute((const void*)mf::debug_me2_coop_kernel<PROC>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              mf::coop_debug_smem_bytes<PG>());
}

void free_all(mf_process* p) {
  cudaFree(p->d_lnx); cudaFree(p->d_lnq2); cudaFree(p->d_xf); cudaFree(p->d_row);
  cudaFree(p->d_partials); cudaFree(p->d_hist_part); cudaFree(p->d_queue); cudaFree(p->d_quark); cudaFree(p->d_start);
}

// launches the fused pass + finalize on `stream`
int run_pass(mf_process* p, bool unw, const double* d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
             uint64_t n_events, double w_max, void* d_records, uint64_t capacity, uint64_t* d_count, double* d_hist,
             mf_iter_result* d_result, void* stream) {
  if (!p) return MF_EINVAL;
  if (!d_grid || !d_result) return fail(p, MF_EINVAL, "d_grid and d_result must not be NULL");
  if (unw && (!d_count || !(w_max > 0.0))) return fail(p, MF_EINVAL, "mf_unweight needs d_count and w_max > 0");
  if (unw && capacity > 0 && !d_records) return fail(p, MF_EINVAL, "capacity > 0 with d_records == NULL");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
    return fail(p, MF_EINVAL, "the handle belongs to another device than the current one");
  mf::PassArgs A;
  A.grid = d_grid; A.pdf_lnx = p->d_lnx; A.pdf_row = p->d_row; A.pdf_lnq2 = p->d_lnq2; A.pdf_xf = p->d_xf;
  A.seed = seed; A.first_event = first_event; A.n_events = n_events; A.iteration = iteration;
  A.w_max = w_max; A.records = (char*)d_records; A.capacity = capacity; A.count = (unsigned long long*)d_count;
  A.partials = p->d_partials; A.hist_part = d_hist ? p->d_hist_part : nullptr;
  A.coop_queue = p->d_queue;
  A.obs = p->d_obs; A.obs_nb = p->obs_nb; A.obs_ptmax = p->obs_ptmax; A.obs_etamax = p->obs_etamax;
  cudaStream_t st = (cudaStream_t)stream;
  A.quark_terms = nullptr;
  const int blocks = unw ? p->blocks_unw : p->blocks;
  const int n_hist = p->D * p->P.n_bins;
  const int fin_blocks = (n_hist + 255) / 256 + 1;
  // cooperative / block processes: the records of this call are completed by record_kernel after the pass (momenta, partonic
  // channel); it needs the cursor as it was before
  const bool draw_channels = unw && d_records && capacity > 0 && n_events > 0 && mf::defers_record(p->process);
  cudaError_t e;
  if (draw_channels && (e = cudaMemcpyAsync(p->d_start, d_count, sizeof(unsigned long long), cudaMemcpyDeviceToDevice, st)) != cudaSuccess)
    return fail(p, MF_ECUDA, "record cursor snapshot", e);
  // MF_PP_TTGG keeps one double per event between its two kernels, in a buffer of kQuarkChunk events made at create: a larger
  // call runs as consecutive pieces whose results finalize_kernel adds up (in piece order: deterministic)
  const uint64_t piece_max = p->process == MF_PP_TTGG ? p->quark_cap : n_events;
  uint64_t done = 0;
  int piece = 0;
  do {
    const uint64_t m = n_events - done < piece_max ? n_events - done : piece_max;
    A.first_event = first_event + done;
    A.n_events = m;
    if (p->process == MF_PP_TTGG && m > 0) {
      // the quark channel of every event of this piece, ahead of the cooperative pass on the same stream
      const size_t smem = (size_t)mf::prepass_smem_doubles(p->D, p->P.n_bins, p->P.pdf_nx, p->P.pdf_nfl) * sizeof(double);
      const uint64_t want = (m + mf::kPrepassThreads - 1) / mf::kPrepassThreads;
      const unsigned pre_blocks = (unsigned)(want < (uint64_t)p->prepass_blocks ? want : (uint64_t)p->prepass_blocks);
      mf::quark_prepass_kernel<7><<<pre_blocks, mf::kPrepassThreads, smem, st>>>(p->P, A, p->d_quark);
      if ((e = cudaGetLastError()) != cudaSuccess) return fail(p, MF_ECUDA, "quark prepass launch", e);
      A.quark_terms = p->d_quark;
    }
    void* args[2] = {(void*)&p->P, (void*)&A};
    e = cudaLaunchKernel(pass_fn(p->process, unw), dim3(blocks), dim3(p->threads), args, p->smem, st);
    if (e != cudaSuccess) return fail(p, MF_ECUDA, "fused pass launch", e);
    mf::finalize_kernel<<<fin_blocks, 256, 0, st>>>(p->d_partials, p->d_hist_part, blocks, n_hist, d_hist,
                                                    (mf::IterResult*)d_result, piece > 0 ? 1 : 0);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(p, MF_ECUDA, "finalize launch", e);
    done += m;
    ++piece;
  } while (done < n_events);
  if (draw_channels) {
    A.first_event = first_event;
    A.n_events = n_events;
    const int cb = p->prepass_blocks;       // one block per SM: accepted events are few
    switch (p->process) {
      case 2: mf::record_kernel<2><<<cb, mf::kThreads, 0, st>>>(p->P, A, p->d_start); break;
      case 5: mf::record_kernel<5><<<cb, mf::kThreads, 0, st>>>(p->P, A, p->d_start); break;
      default: mf::record_kernel<7><<<cb, mf::kThreads, 0, st>>>(p->P, A, p->d_start); break;
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(p, MF_ECUDA, "record kernel launch", e);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "finalize launch", e);
  return MF_OK;
}

}  // namespace

extern "C" {

int mf_create_process(const mf_process_desc* d, mf_process** out) {
  if (out) *out = nullptr;
  if (!d || !out) return MF_EINVAL;
  if (d->process < 0 || d->process > 7 || d->n_bins < 2 || d->n_bins > MF_MAX_BINS || !(d->sqrt_s > 0.0) ||
      !(d->gev2_to_pb > 0.0))
    return MF_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return MF_ECUDA; }
  mf_process* p = new (std::nothrow) mf_process;
  if (!p) return MF_ENOMEM;
  static const int Dtab[8] = {2, 4, 14, 18, 4, 14, 22, 18}, nftab[8] = {2, 2, 3, 4, 2, 3, 5, 4};
  p->process = d->process; p->D = Dtab[d->process]; p->NF = nftab[d->process];
  mf::Params& P = p->P;
  std::memset(&P, 0, sizeof(P));
  P.s = d->sqrt_s * d->sqrt_s;
  P.alpha_em = d->alpha_em; P.alpha_s = d->alpha_s; P.m_top = d->m_top; P.mu2 = d->mu2;
  P.ptmin = d->ptmin; P.etamax = d->etamax; P.drmin = d->drmin; P.gev2_to_pb = d->gev2_to_pb;
  P.n_bins = d->n_bins;
  const double gs2 = 4.0 * mf::kPi * d->alpha_s;
  // |M|^2 normalisation: g_s^{2 n_g} / (4 helicity x 64 colour averages x (n_g - 2)! identical gluons)
  if (d->process == 0) {
    if (!(d->alpha_em > 0.0)) { delete p; return MF_EINVAL; }
    P.me_norm = 1.0;
  } else {
    if (!(d->alpha_s > 0.0) || !(d->m_top > 0.0) || !(d->mu2 > 0.0)) { delete p; return MF_EINVAL; }
    if (d->pdf_nx < 4 || d->pdf_nq < 4 || d->pdf_nx > 512 || !d->pdf_lnx || !d->pdf_lnq2 || !d->pdf_xf) {
      delete p; return MF_EINVAL;
    }
    for (int i = 1; i < d->pdf_nx; ++i) if (!(d->pdf_lnx[i] > d->pdf_lnx[i - 1])) { delete p; return MF_EINVAL; }
    for (int i = 1; i < d->pdf_nq; ++i) if (!(d->pdf_lnq2[i] > d->pdf_lnq2[i - 1])) { delete p; return MF_EINVAL; }
    const bool flavoured = d->process == MF_PP_TT || d->process == MF_PP_TTG || d->process == MF_PP_TTGG;
    const int ng = d->process == MF_PP_TT ? 2 : d->process == MF_PP_TTG ? 3 : d->process == MF_GG_TTGGG ? 5 : d->process == MF_PP_TTGG ? 4 : d->process + 1;
    const int nfl = flavoured ? d->pdf_nfl : 1;
    if (flavoured && (nfl < 3 || nfl % 2 == 0 || nfl > mf::kMaxPartonTables)) { delete p; return MF_EINVAL; }
    P.pdf_nfl = nfl;
    P.me_norm = std::pow(gs2, ng) / (256.0 * (ng == 4 ? 2.0 : ng == 5 ? 6.0 : 1.0));
    const int ncut = p->NF - 2;
    const double thr = 2.0 * d->m_top + ncut * (d->ptmin > 0.0 ? d->ptmin : 0.0);
    P.tau_min = thr * thr / P.s;
    P.ln_tau_min = std::log(P.tau_min);
    const double lq = std::log(d->mu2);
    if (!(lq >= d->pdf_lnq2[0] && lq <= d->pdf_lnq2[d->pdf_nq - 1])) { delete p; return MF_ERANGE; }
    if (!(P.tau_min < 1.0) || !(P.ln_tau_min >= d->pdf_lnx[0])) { delete p; return MF_ERANGE; }
    P.pdf_nx = d->pdf_nx; P.pdf_nq = d->pdf_nq;
    P.pdf_jq = mf::find_cell(d->pdf_lnq2, d->pdf_nq, lq);
    P.pdf_uq = (lq - d->pdf_lnq2[P.pdf_jq]) / (d->pdf_lnq2[P.pdf_jq + 1] - d->pdf_lnq2[P.pdf_jq]);
  }
  // device-side constants
  cudaError_t e = cudaSuccess;
  if (d->process != 0) {
    const size_t nx = d->pdf_nx, nq = d->pdf_nq, nt = (size_t)P.pdf_nfl;
    if ((e = cudaMalloc(&p->d_lnx, nx * 8)) != cudaSuccess || (e = cudaMalloc(&p->d_lnq2, nq * 8)) != cudaSuccess ||
        (e = cudaMalloc(&p->d_xf, nt * nx * nq * 8)) != cudaSuccess || (e = cudaMalloc(&p->d_row, nt * nx * 8)) != cudaSuccess) {
      free_all(p); delete p; cudaGetLastError(); return MF_ENOMEM;
    }
    if ((e = cudaMemcpy(p->d_lnx, d->pdf_lnx, nx * 8, cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(p->d_lnq2, d->pdf_lnq2, nq * 8, cudaMemcpyHostToDevice)) != cudaSuccess ||
        (e = cudaMemcpy(p->d_xf, d->pdf_xf, nt * nx * nq * 8, cudaMemcpyHostToDevice)) != cudaSuccess) {
      free_all(p); delete p; cudaGetLastError(); return MF_ECUDA;
    }
    mf::pdf_collapse_kernel<<<(int)((nt * nx + 127) / 128), 128>>>(p->d_xf, p->d_lnq2, (int)(nt * nx), (int)nq, P.pdf_jq,
                                                                  P.pdf_uq, p->d_row);
    if ((e = cudaGetLastError()) != cudaSuccess || (e = cudaDeviceSynchronize()) != cudaSuccess) {
      free_all(p); delete p; cudaGetLastError(); return MF_ECUDA;
    }
  }
  // launch geometry: fill every SM with as many blocks as fit
  cudaDeviceProp prop;
  int dev = 0;
  if ((e = cudaGetDevice(&dev)) != cudaSuccess || (e = cudaGetDeviceProperties(&prop, dev)) != cudaSuccess) {
    free_all(p); delete p; cudaGetLastError(); return MF_ECUDA;
  }
  p->device = dev;
  if ((e = cudaGetSymbolAddress((void**)&p->d_static, mf_static_scratch)) != cudaSuccess || p->d_static == nullptr) {
    free_all(p); delete p; cudaGetLastError(); return MF_ECUDA;
  }
  const bool coop = p->process == 2 || p->process == 3 || p->process == 5 || p->process == 7;
  if (coop) {
    // cooperative pass: as many teams per block as the SM's shared memory holds, one block per SM
    e = p->process == 3 ? coop_setup<3>(p, prop) : p->process == 5 ? coop_setup<5>(p, prop) : p->process == 7 ? coop_setup<7>(p, prop) : coop_setup<2>(p, prop);
    if (e != cudaSuccess) { free_all(p); delete p; cudaGetLastError(); return MF_ECUDA; }
  } else if (p->process == MF_GG_TTGGG) {
    // one event per block: the whole block's shared memory is the scratch of the matrix element
    p->threads = mf::kCtaThreads;
    p->smem = (size_t)mf::CtaSmem(p->D, P.n_bins, P.pdf_nx, p->threads).total * 8;
    if (p->smem > (size_t)prop.sharedMemPerBlockOptin) { free_all(p); delete p; return MF_EINVAL; }   // n_bins too large
    e = cudaSuccess;
    for (int u = 0; u < 2 && e == cudaSuccess; ++u)
      e = cudaFuncSetAttribute(pass_fn(6, u != 0), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin);
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute((const void*)mf::debug_eval_cta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               mf::cta_debug_smem_bytes());
    if (e == cudaSuccess)
      e = cudaFuncSetAttribute((const void*)mf::debug_me2_cta_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               mf::cta_debug_smem_bytes());
    if (e != cudaSuccess) { free_all(p); delete p; cudaGetLastError(); return MF_ECUDA; }
  } else {
    p->smem = (size_t)(p->D * (2 * P.n_bins + 1) + (1 + P.pdf_nfl) * P.pdf_nx + 5 * 32) * sizeof(double);
  }
  int per_sm = 0, per_sm_unw = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pass_fn(p->process, false), p->threads, p->smem);
  if (e == cudaSuccess)
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm_unw, pass_fn(p->process, true), p->threads, p->smem);
  if (e != cudaSuccess || per_sm < 1 || per_sm_unw < 1) { free_all(p); delete p; cudaGetLastError(); return MF_ECUDA; }
  p->blocks = prop.multiProcessorCount * per_sm;
  p->blocks_unw = prop.multiProcessorCount * per_sm_unw;
  p->prepass_blocks = prop.multiProcessorCount;
  if (p->process == MF_PP_TTGG) {
    const int need = mf::prepass_smem_doubles(p->D, P.n_bins, P.pdf_nx, P.pdf_nfl) * (int)sizeof(double);
    if (need > (int)prop.sharedMemPerBlockOptin) { free_all(p); delete p; return MF_EINVAL; }
    if (cudaFuncSetAttribute((const void*)mf::quark_prepass_kernel<7>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)prop.sharedMemPerBlockOptin) != cudaSuccess) {
      free_all(p); delete p; cudaGetLastError(); return MF_ECUDA;
    }
  }
  const int max_blocks = p->blocks > p->blocks_unw ? p->blocks : p->blocks_unw;
  if ((e = cudaMalloc(&p->d_partials, (size_t)max_blocks * sizeof(mf::BlockPartial))) != cudaSuccess ||
      (e = cudaMalloc(&p->d_hist_part, (size_t)max_blocks * p->D * P.n_bins * 8)) != cudaSuccess) {
    free_all(p); delete p; cudaGetLastError(); return MF_ENOMEM;
  }
  const int queue_doubles = p->process == MF_GG_TTGGG ? mf::kCtaQueue : (p->process == 3 || p->process == 7) ? mf::g4::Prog::Queue : mf::g3::Prog::Queue;
  if ((coop || p->process == MF_GG_TTGGG) &&
      (e = cudaMalloc(&p->d_queue, (size_t)max_blocks * p->threads * queue_doubles * 8)) != cudaSuccess) {
    free_all(p); delete p; cudaGetLastError(); return MF_ENOMEM;
  }
  if (p->process == MF_PP_TTGG) {
    if ((e = cudaMalloc(&p->d_quark, kQuarkChunk * sizeof(double))) != cudaSuccess) { free_all(p); delete p; cudaGetLastError(); return MF_ENOMEM; }
    p->quark_cap = kQuarkChunk;
  }
  if (mf::defers_record(p->process) && (e = cudaMalloc(&p->d_start, sizeof(unsigned long long))) != cudaSuccess) {
    free_all(p); delete p; cudaGetLastError(); return MF_ENOMEM;
  }
  snprintf(p->err, sizeof(p->err), "ok");
  *out = p;
  return MF_OK;
}

int mf_destroy_process(mf_process* p) {
  if (!p) return MF_EINVAL;
  free_all(p);
  delete p;
  return MF_OK;
}

int mf_n_dims(const mf_process* p, int32_t* D) { if (!p || !D) return MF_EINVAL; *D = p->D; return MF_OK; }
int mf_n_final(const mf_process* p, int32_t* n) { if (!p || !n) return MF_EINVAL; *n = p->NF; return MF_OK; }
int mf_record_size(const mf_process* p, int32_t* b) {
  if (!p || !b) return MF_EINVAL;
  *b = (p->NF + 2) * 32 + 16 + ((p->process == MF_PP_TT || p->process == MF_PP_TTG || p->process == MF_PP_TTGG) ? 8 : 0);
  return MF_OK;
}
int mf_debug_row_len(const mf_process* p, int32_t* n) {
  if (!p || !n) return MF_EINVAL;
  *n = 3 * p->D + 4 * (p->NF + 2) + 9 + ((p->process == MF_PP_TT || p->process == MF_PP_TTGG) ? 2 : p->process == MF_PP_TTG ? 6 : 0);
  return MF_OK;
}
const char* mf_last_error(const mf_process* p) { return p ? p->err : kNullHandle; }
int mf_launch_config(const mf_process* p, int32_t* blocks, int32_t* threads) {
  if (!p || !blocks || !threads) return MF_EINVAL;
  *blocks = p->blocks; *threads = p->threads;
  return MF_OK;
}

int mf_set_dynamic_scale(mf_process* p, int32_t on) {
  if (!p) return MF_EINVAL;
  if (p->process == 0) return fail(p, MF_EINVAL, "mf_set_dynamic_scale: the leptonic process has no scale");
  p->P.dyn_scale = on ? 1 : 0;
  return MF_OK;
}

int mf_set_observables(mf_process* p, double* d_obs, int32_t n_bins, double pt_max, double eta_max) {
  if (!p) return MF_EINVAL;
  if (!d_obs) { p->d_obs = nullptr; p->obs_nb = 0; return MF_OK; }
  if (n_bins < 1 || n_bins > 4096 || !(pt_max > 0.0) || !(eta_max > 0.0)) return fail(p, MF_EINVAL, "mf_set_observables: bad argument");
  p->d_obs = d_obs; p->obs_nb = n_bins; p->obs_ptmax = pt_max; p->obs_etamax = eta_max;
  return MF_OK;
}

int mf_vegas_iterate(mf_process* p, const double* d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                     uint64_t n_events, double* d_hist, mf_iter_result* d_result, void* stream) {
  return run_pass(p, false, d_grid, seed, iteration, first_event, n_events, 0.0, nullptr, 0, nullptr, d_hist, d_result,
                  stream);
}

int mf_vegas_iterate_static(mf_process* p, const double* d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                            uint64_t n_events, double* d_hist, mf_iter_result* d_result, void* stream) {
  if (!p) return MF_EINVAL;
  if (!d_grid || !d_result) return fail(p, MF_EINVAL, "d_grid and d_result must not be NULL");
  if (p->process != MF_EE_MUMU && p->process != MF_GG_TT && p->process != MF_PP_TT)
    return fail(p, MF_EINVAL, "mf_vegas_iterate_static: thread-per-event processes only (MF_EE_MUMU, MF_GG_TT, MF_PP_TT); "
                              "the others queue events in tens of MB of scratch");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != p->device)
    return fail(p, MF_EINVAL, "the handle belongs to another device than the current one");
  const int blocks = p->blocks, n_hist = p->D * p->P.n_bins;
  const size_t off_hist = ((size_t)blocks * sizeof(mf::BlockPartial) + 255) & ~(size_t)255;
  const size_t need = off_hist + (size_t)blocks * n_hist * sizeof(double);
  if (need > (size_t)MF_STATIC_SCRATCH_BYTES) {
    snprintf(p->err, sizeof(p->err), "mf_vegas_iterate_static: %d blocks x %d histogram bins need %zu bytes of scratch, the static "
             "array holds %d (use fewer bins, or mf_vegas_iterate)", blocks, n_hist, need, (int)MF_STATIC_SCRATCH_BYTES);
    return MF_EINVAL;
  }
  mf::PassArgs A;
  std::memset(&A, 0, sizeof(A));
  A.grid = d_grid; A.pdf_lnx = p->d_lnx; A.pdf_row = p->d_row; A.pdf_lnq2 = p->d_lnq2; A.pdf_xf = p->d_xf;
  A.seed = seed; A.first_event = first_event; A.n_events = n_events; A.iteration = iteration;
  // nothing in the scratch has to start at zero: every block of the pass overwrites its partial and its whole histogram slice
  // before finalize_kernel (next on the stream) reads them, so the previous call's contents are never seen
  A.partials = reinterpret_cast<mf::BlockPartial*>(p->d_static);
  A.hist_part = d_hist ? reinterpret_cast<double*>(p->d_static + off_hist) : nullptr;
  A.obs = p->d_obs; A.obs_nb = p->obs_nb; A.obs_ptmax = p->obs_ptmax; A.obs_etamax = p->obs_etamax;
  cudaStream_t st = (cudaStream_t)stream;
  void* args[2] = {(void*)&p->P, (void*)&A};
  cudaError_t e = cudaLaunchKernel(pass_fn(p->process, false), dim3(blocks), dim3(p->threads), args, p->smem, st);
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "fused pass launch", e);
  mf::finalize_kernel<<<(n_hist + 255) / 256 + 1, 256, 0, st>>>(A.partials, A.hist_part, blocks, n_hist, d_hist,
                                                               (mf::IterResult*)d_result, 0);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "finalize launch", e);
  return MF_OK;
}

int mf_unweight(mf_process* p, const double* d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                uint64_t n_events, double w_max, void* d_records, uint64_t capacity, uint64_t* d_count, double* d_hist,
                mf_iter_result* d_result, void* stream) {
  return run_pass(p, true, d_grid, seed, iteration, first_event, n_events, w_max, d_records, capacity, d_count, d_hist,
                  d_result, stream);
}

int mf_refine_grid(mf_process* p, double* d_grid, const double* d_hist, double alpha, void* stream) {
  if (!p) return MF_EINVAL;
  if (!d_grid || !d_hist || !(alpha >= 0.0)) return fail(p, MF_EINVAL, "mf_refine_grid: bad argument");
  mf::refine_grid_kernel<<<p->D, 32, 0, (cudaStream_t)stream>>>(d_grid, d_hist, p->P.n_bins, alpha);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "refine launch", e);
  return MF_OK;
}

int mf_debug_eval(mf_process* p, const double* d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                  uint64_t n_events, double* d_out, void* stream) {
  if (!p) return MF_EINVAL;
  if (!d_grid || (!d_out && n_events)) return fail(p, MF_EINVAL, "mf_debug_eval: NULL argument");
  if (n_events == 0) return MF_OK;
  mf::PassArgs A;
  std::memset(&A, 0, sizeof(A));
  A.grid = d_grid; A.pdf_lnx = p->d_lnx; A.pdf_row = p->d_row; A.pdf_lnq2 = p->d_lnq2; A.pdf_xf = p->d_xf;
  A.seed = seed; A.first_event = first_event; A.n_events = n_events; A.iteration = iteration;
  cudaStream_t st = (cudaStream_t)stream;
  const unsigned blocks = (unsigned)((n_events + mf::kThreads - 1) / mf::kThreads);
  switch (p->process) {
    case 0: mf::debug_eval_kernel<0><<<blocks, mf::kThreads, 0, st>>>(p->P, A, d_out); break;
    case 1: mf::debug_eval_kernel<1><<<blocks, mf::kThreads, 0, st>>>(p->P, A, d_out); break;
    case 4: mf::debug_eval_kernel<4><<<blocks, mf::kThreads, 0, st>>>(p->P, A, d_out); break;
    case 5: mf::debug_eval_kernel<5><<<blocks, mf::kThreads, 0, st>>>(p->P, A, d_out); break;
    case 6:
      mf::debug_eval_cta_kernel<<<(unsigned)((n_events + mf::kCtaDebugThreads - 1) / mf::kCtaDebugThreads), mf::kCtaDebugThreads,
                                  mf::cta_debug_smem_bytes(), st>>>(p->P, A, d_out);
      break;
    case 2:
      mf::debug_eval_coop_kernel<2><<<(unsigned)((n_events + mf::kCoopDebugThreads - 1) / mf::kCoopDebugThreads),
                                      mf::kCoopDebugThreads, mf::coop_debug_smem_bytes<mf::g3::Prog>(), st>>>(p->P, A, d_out);
      break;
    case 7:
      mf::debug_eval_coop_kernel<7><<<(unsigned)((n_events + mf::kCoopDebugThreads - 1) / mf::kCoopDebugThreads),
                                      mf::kCoopDebugThreads, mf::coop_debug_smem_bytes<mf::g4::Prog>(), st>>>(p->P, A, d_out);
      break;
    default:
      mf::debug_eval_coop_kernel<3><<<(unsigned)((n_events + mf::kCoopDebugThreads - 1) / mf::kCoopDebugThreads),
                                      mf::kCoopDebugThreads, mf::coop_debug_smem_bytes<mf::g4::Prog>(), st>>>(p->P, A, d_out);
      break;
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "debug_eval launch", e);
  return MF_OK;
}

int mf_debug_philox(uint64_t seed, uint32_t iteration, uint64_t first_event, uint64_t n_events, uint32_t n_blocks,
                    uint32_t* d_out, void* stream) {
  if (n_blocks != 0 && n_events > UINT64_MAX / n_blocks) return MF_EINVAL;      // n_events * n_blocks must not wrap
  if (!d_out && n_events * n_blocks) return MF_EINVAL;
  uint64_t total = n_events * n_blocks;
  if (total == 0) return MF_OK;
  mf::debug_philox_kernel<<<(unsigned)((total + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      seed, iteration, first_event, n_events, n_blocks, d_out);
  return cudaGetLastError() == cudaSuccess ? MF_OK : MF_ECUDA;
}

int mf_debug_pdf(mf_process* p, const double* d_x, const double* d_q2, uint64_t n, double* d_out, void* stream) {
  if (!p) return MF_EINVAL;
  if (p->process == 0) return fail(p, MF_EINVAL, "process has no PDF");
  if (n == 0) return MF_OK;
  if (!d_x || !d_q2 || !d_out) return fail(p, MF_EINVAL, "mf_debug_pdf: NULL argument");
  mf::debug_pdf_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(
      p->d_lnx, p->d_lnq2, p->d_xf, p->P.pdf_nx, p->P.pdf_nq, d_x, d_q2, n, d_out);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "debug_pdf launch", e);
  return MF_OK;
}

int mf_debug_me2(mf_process* p, const double* d_mom, uint64_t n, double* d_out, void* stream) {
  if (!p) return MF_EINVAL;
  if (n == 0) return MF_OK;
  if (!d_mom || !d_out) return fail(p, MF_EINVAL, "mf_debug_me2: NULL argument");
  cudaStream_t st = (cudaStream_t)stream;
  const unsigned blocks = (unsigned)((n + mf::kThreads - 1) / mf::kThreads);
  switch (p->process) {
    case 0: mf::debug_me2_kernel<0><<<blocks, mf::kThreads, 0, st>>>(p->P, d_mom, n, d_out); break;
    case 1: mf::debug_me2_kernel<1><<<blocks, mf::kThreads, 0, st>>>(p->P, d_mom, n, d_out); break;
    case 4: mf::debug_me2_kernel<4><<<blocks, mf::kThreads, 0, st>>>(p->P, d_mom, n, d_out); break;
    case 5: mf::debug_me2_kernel<5><<<blocks, mf::kThreads, 0, st>>>(p->P, d_mom, n, d_out); break;
    case 6:
      mf::debug_me2_cta_kernel<<<(unsigned)((n + mf::kCtaDebugThreads - 1) / mf::kCtaDebugThreads), mf::kCtaDebugThreads,
                                 mf::cta_debug_smem_bytes(), st>>>(p->P, d_mom, n, d_out);
      break;
    case 2:
      mf::debug_me2_coop_kernel<2><<<(unsigned)((n + mf::kCoopDebugThreads - 1) / mf::kCoopDebugThreads),
                                     mf::kCoopDebugThreads, mf::coop_debug_smem_bytes<mf::g3::Prog>(), st>>>(p->P, d_mom, n, d_out);
      break;
    case 7:
      mf::debug_me2_coop_kernel<7><<<(unsigned)((n + mf::kCoopDebugThreads - 1) / mf::kCoopDebugThreads),
                                     mf::kCoopDebugThreads, mf::coop_debug_smem_bytes<mf::g4::Prog>(), st>>>(p->P, d_mom, n, d_out);
      break;
    default:
      mf::debug_me2_coop_kernel<3><<<(unsigned)((n + mf::kCoopDebugThreads - 1) / mf::kCoopDebugThreads),
                                     mf::kCoopDebugThreads, mf::coop_debug_smem_bytes<mf::g4::Prog>(), st>>>(p->P, d_mom, n, d_out);
      break;
  }
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, MF_ECUDA, "debug_me2 launch", e);
  return MF_OK;
}

int mf_debug_me2_quark_gluon(int32_t kind, double m_top, double alpha_s, const double* d_mom, uint64_t n, double* d_out,
                             void* stream) {
  if (kind < 0 || kind > 3 || !(m_top > 0.0) || !(alpha_s > 0.0)) return MF_EINVAL;
  if (n == 0) return MF_OK;
  if (!d_mom || !d_out) return MF_EINVAL;
  mf::debug_me2_quark_gluon_kernel<<<(unsigned)((n + mf::kThreads - 1) / mf::kThreads), mf::kThreads, 0,
                                     (cudaStream_t)stream>>>(kind, m_top, 4.0 * mf::kPi * alpha_s, d_mom, n, d_out);
  return cudaGetLastError() == cudaSuccess ? MF_OK : MF_ECUDA;
}

int mf_measure_fp64_peak(int64_t iters, double* h_flops, double* h_ms) {
  if (iters <= 0 || !h_flops) return MF_EINVAL;
  cudaDeviceProp prop;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return MF_ECUDA;
  double* sink = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess) return MF_ENOMEM;
  const int blocks = prop.multiProcessorCount * 4, threads = 256;
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  mf::dfma_peak_kernel<<<blocks, threads>>>(iters / 8 + 1, 1.0, sink);  // warm-up
  cudaEventRecord(a);
  mf::dfma_peak_kernel<<<blocks, threads>>>(iters, 1.0, sink);
  cudaEventRecord(b);
  cudaError_t e = cudaEventSynchronize(b);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, a, b);
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
  if (e != cudaSuccess) return MF_ECUDA;
  *h_flops = 2.0 * 8.0 * (double)iters * (double)blocks * (double)threads / ((double)ms * 1e-3);
  if (h_ms) *h_ms = ms;
  return MF_OK;
}

int mf_measure_dmma_peak(int64_t iters, double* h_flops, double* h_ms) {
  if (iters <= 0 || !h_flops) return MF_EINVAL;
  cudaDeviceProp prop;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return MF_ECUDA;
  double* sink = nullptr;
  if (cudaMalloc(&sink, 8) != cudaSuccess) return MF_ENOMEM;
  const int blocks = prop.multiProcessorCount * 2, threads = 256;
  cudaEvent_t a, b;
  cudaEventCreate(&a); cudaEventCreate(&b);
  mf::dmma_peak_kernel<<<blocks, threads>>>(iters / 8 + 1, 1.0, sink);  // warm-up
  cudaEventRecord(a);
  mf::dmma_peak_kernel<<<blocks, threads>>>(iters, 1.0, sink);
  cudaEventRecord(b);
  cudaError_t e = cudaEventSynchronize(b);
  float ms = 0.f;
  cudaEventElapsedTime(&ms, a, b);
  cudaEventDestroy(a); cudaEventDestroy(b); cudaFree(sink);
  if (e != cudaSuccess) return MF_ECUDA;
  // 4 DMMA per iteration and warp, 2 x 8 x 8 x 4 flop each
  *h_flops = 4.0 * 512.0 * (double)iters * (double)blocks * (double)(threads / 32) / ((double)ms * 1e-3);
  if (h_ms) *h_ms = ms;
  return MF_OK;
}

}  // extern "C"
