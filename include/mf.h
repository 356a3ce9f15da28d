/* mf.h — C ABI of the B200-native MadFlow leading-order integrand hot path.
 *
 * What the library computes ("generation of random numbers, computation of the phase space
 * kinematics, matrix element evaluation and histogram accumulation"; L27 VEGAS + PDF interpolation;
 * L65-67 helicity-summed matrix elements from HELAS-style routines; L71-75 RAMBO; L81-83 unweighting;
 * BASELINE.json north_star fixes the rest): for every event index k in [first_event, first_event+n_events)
 *
 *   Philox4x32-10(seed, iteration, k) -> uniforms -> VEGAS map -> (x1, x2) -> phase space (2-body / RAMBO)
 *   -> lab boost + cuts -> PDF -> |M|^2 (helicity and colour summed) -> weight w
 *
 * in ONE fused CUDA pass, then reduces sum w, sum w^2, max|w|, n_pass and the per-dimension VEGAS
 * histograms of w^2.  Nothing per event touches HBM except the records mf_unweight accepts.
 * DESIGN.md states every reading of the paper (R1..R19) the arithmetic follows.
 *
 * Conventions
 *  - All functions return int: MF_OK (0) or a negative error code.  No exceptions, no aborts, no printing.
 *  - Pointers named d_* are DEVICE pointers owned by the caller (e.g. torch tensors); pointers named h_* and
 *    the mf_process_desc fields are HOST pointers.  `stream` is a cudaStream_t passed as void* (NULL = the
 *    legacy default stream).
 *  - The library allocates device memory only in mf_create_process and frees it only in
 *    mf_destroy_process.  The hot calls never allocate, never synchronise the stream and never touch host
 *    memory: they are asynchronous, results are valid after the caller synchronises `stream`.  (MF_PP_TTGG keeps one
 *    double per event between its two kernels in a buffer of 2^22 events made at create; a larger call runs as
 *    consecutive pieces on the stream whose sums are added in piece order.)
 *  - A handle is used from one stream at a time (it owns per-block partial-sum scratch).
 *  - There is no CPU fallback: without a CUDA device mf_create_process returns MF_ECUDA.
 */
#ifndef MF_H
#define MF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mf_process mf_process; /* opaque; owns its device-side constants and scratch */

/* process ids: 0..3 are BASELINE.json configs[0..3]; MF_PP_TT ("pp -> ttbar (7 diagrams)")
 * adds to g g -> t tbar, at the same phase-space point and in the same pass, the q qbar -> t tbar channel of every
 * quark flavour of a multi-flavour PDF table, the quark taken from either beam:
 *   w ~ L_gg |M_gg|^2 + sum_i [ q_i(x1) qbar_i(x2) + qbar_i(x1) q_i(x2) ] / (x1 x2) |M_qq|^2                                */
enum { MF_EE_MUMU = 0, MF_GG_TT = 1, MF_GG_TTG = 2, MF_GG_TTGG = 3, MF_PP_TT = 4, MF_PP_TTG = 5, MF_GG_TTGGG = 6, MF_PP_TTGG = 7 };
/* MF_GG_TTGGG ("pp -> ttbar ggg", the paper's heaviest process): g g -> t tbar g g g, 1240 diagrams,
 * 128 helicity states, 120 x 120 colour matrix; RAMBO with five final-state particles, D = 22; the cuts act on the three gluons.
 * One event per thread block (csrc/mf_me_cta5.cuh); its shared-memory scratch leaves room for n_bins <= 64 (else MF_EINVAL). */
/* MF_PP_TTG ("pp -> ttbar g (36 diagrams)"; R19): at the phase-space point, cuts and stream of MF_GG_TTG the
 * weight sums g g -> t tbar g and the flavour-summed q qbar -> t tbar g, q g -> t tbar q, qbar g -> t tbar qbar channels (either
 * beam assignment); the light final-state parton is a jet whatever its flavour.  Same multi-flavour table as MF_PP_TT. */
/* MF_PP_TTGG (P:L101 and Table 1, "pp -> ttbar gg (267 diagrams)" = 123 + 4 x 36; R22): at the phase-space point,
 * cuts and stream of MF_GG_TTGG the weight sums g g -> t tbar g g and q qbar -> t tbar g g of every flavour of the multi-flavour
 * table, the quark from either beam (the two assignments have different matrix elements: the charge asymmetry).  Accepted
 * events carry the channel code of MF_PP_TT (0 gg; 1 + 2 i quark i from beam 1; 2 + 2 i from beam 2). */
enum { MF_OK = 0, MF_EINVAL = -1, MF_ECUDA = -2, MF_EOVERFLOW = -3, MF_ERANGE = -4, MF_ENOMEM = -5 };

/* Process descriptor (host memory; copied at create).  Same field order as the oracle's mfo_process_desc. */
typedef struct {
  int32_t process;            /* enum above; fixes n_final, D (2/4/14/18/4/14/22/18), helicities, colour matrix */
  double sqrt_s;              /* GeV; hadronic (pp) for processes 1-3, leptonic for 0                   */
  double alpha_em, alpha_s;   /* couplings: e^2 = 4 pi alpha_em, g_s^2 = 4 pi alpha_s                   */
  double m_top;               /* GeV; width 0                                                           */
  double mu2;                 /* mu_F^2 = mu_R^2 in GeV^2 (fixed scale)                                  */
  double ptmin, etamax, drmin;/* cuts on the final-state gluons; <= 0 disables each                     */
  double gev2_to_pb;          /* 0.3894e9                                                               */
  int32_t n_bins;             /* VEGAS bins per dimension, 2..MF_MAX_BINS                               */
  int32_t pdf_nx, pdf_nq;     /* knots of the PDF table (0, 0 for MF_EE_MUMU)                           */
  const double *pdf_lnx;      /* [pdf_nx] ln x knots, increasing, last = 0                              */
  const double *pdf_lnq2;     /* [pdf_nq] ln Q^2 knots, increasing                                      */
  const double *pdf_xf;       /* [pdf_nx][pdf_nq] x*g(x,Q^2), row-major xf[ix*nq+iq]; MF_PP_TT:         */
                              /* [pdf_nfl][pdf_nx][pdf_nq], table 0 gluon, 1+2i quark i, 2+2i antiquark i */
  int32_t pdf_nfl;            /* parton tables; read for MF_PP_TT / _TTG / _TTGG: 1 + 2 n_f, n_f = 1..5    */
} mf_process_desc;
#define MF_MAX_BINS 128

/* Per-iteration sums (device memory, written by the finalize kernel of each hot call). */
typedef struct {
  double sum_w, sum_w2, max_abs_w; /* signed sum of w, sum of w^2, max |w| over the events of the call  */
  uint64_t n_pass, n_accept;       /* events passing the cuts; events accepted (mf_unweight only)      */
} mf_iter_result;

/* Creates a handle for one process of the problem of PAPER.md L25 (i)-(v): (i) the parton-level process and its
 * couplings, (ii) the parton densities (the table is copied to the device and collapsed at mu2), (iii) the fiducial cuts,
 * (iv)-(v) the integration set-up (n_bins) the hot calls of PAPER.md L61 then run with.  Errors: NULL / bad enum / n_bins out of range / bad table or table count -> MF_EINVAL;
 * mu2 outside the Q^2 knots or tau_min below the x knots -> MF_ERANGE; no device or CUDA failure ->
 * MF_ECUDA; device allocation failure -> MF_ENOMEM.  On error *out is set to NULL. */
int mf_create_process(const mf_process_desc *desc, mf_process **out);
/* Frees everything mf_create_process allocated (the handle is the process definition, nothing else lives in
 * it).  The handle must be destroyed on the device it was created on, after the streams using it have drained. */
int mf_destroy_process(mf_process *p);
int mf_n_dims(const mf_process *p, int32_t *D);              /* VEGAS dimensions: 2, 4, 14, 18, 4, 14, 22 */
int mf_n_final(const mf_process *p, int32_t *n);             /* final-state particles: 2, 2, 3, 4, 2, 3, 5 */
int mf_record_size(const mf_process *p, int32_t *bytes);     /* (n_final+2)*32 + 16 (+8: MF_PP_TT, _TTG, _TTGG) */
int mf_debug_row_len(const mf_process *p, int32_t *n_doubles);/* 3*D + 4*(n_final+2) + 9 (+2 / +6: MF_PP_TT / _TTG) */
const char *mf_last_error(const mf_process *p);              /* static or handle-owned string           */
/* launch geometry of the fused pass (blocks, threads per block), for reporting */
int mf_launch_config(const mf_process *p, int32_t *blocks, int32_t *threads);

/* One VEGAS iteration (steps a1-a12 of SURVEY.md 8(a)): events
 * [first_event, first_event+n_events) of Philox stream (seed, iteration), mapped through
 * d_grid[D][n_bins+1] (edges, row-major).  Writes d_hist[D][n_bins] = sum of w^2 per bin (overwritten) and
 * *d_result.  d_hist may be NULL.  n_events may be 0 (all outputs zero). */
int mf_vegas_iterate(mf_process *p, const double *d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                     uint64_t n_events, double *d_hist, mf_iter_result *d_result, void *stream);

/* mf_vegas_iterate for callers that must not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * same arguments, same kernels, same results; the per-block partial sums and histogram slices of the launch live in a file-scope
 * `static __device__` array of MF_STATIC_SCRATCH_BYTES inside the library (held by every GPU that loads it, until exit) instead of
 * the handle's buffers.  The call itself calls no cudaMalloc / cudaFree or allocating library routine (the handle was created,
 * and the array's device address looked up, at set-up in mf_create_process).
 * Limits: MF_EE_MUMU, MF_GG_TT and MF_PP_TT handles only (the cooperative kernels queue events in tens of MB), and
 *   launch blocks x (40 + 8 D n_bins) bytes <= MF_STATIC_SCRATCH_BYTES  (e.g. MF_GG_TT, 444 blocks on a B200: 0.73 MB with 50 bins; refused with 128 bins);
 * anything else returns MF_EINVAL with the reason in mf_last_error.
 * Every call on a device shares the one array, from every handle and stream: two calls that overlap on the GPU race (keep
 * them on one stream, or order them with events).  The array keeps the last call's contents; nothing in it has to start at
 * zero, every block overwrites its part before it is read. */
#define MF_STATIC_SCRATCH_BYTES (1024 * 1024)
int mf_vegas_iterate_static(mf_process *p, const double *d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                            uint64_t n_events, double *d_hist, mf_iter_result *d_result, void *stream);

/* VEGAS grid refinement (step a13; the integration is VEGAS importance sampling, whose grid adapts between
 * iterations; Lepage's smoothing + damping r = ((s-1)/ln s)^alpha + rebinning), in
 * place on d_grid from d_hist.  A dimension whose histogram is all zero is left unchanged. */
int mf_refine_grid(mf_process *p, double *d_grid, const double *d_hist, double alpha, void *stream);

/* Same pass plus hit-or-miss unweighting (step a14): event k is accepted iff
 * r_k * w_max < |w_k| with r_k the Philox accept draw; accepted events are appended to d_records
 * (array of structs of mf_record_size bytes: (n_final+2) lab-frame four-momenta (E,px,py,pz), beams first,
 * as doubles; signed w as double; event id as uint64).  *d_count is an in/out cursor: every accepted event
 * advances it, only slots < capacity are written, so *d_count > capacity after synchronising IS the
 * overflow signal.  Record order is unspecified (sort by event id).  d_hist may be NULL.
 * MF_PP_TT appends one more uint64 to each record: the partonic channel of the event (0 = g g; 1 + 2 i = quark i from
 * beam 1 and its antiquark from beam 2; 2 + 2 i = the other way round), drawn in proportion to |luminosity x |M|^2| of
 * the channels, in that order, with the second uniform of the accept block (R18).
 * MF_PP_TTG likewise (R20; the LHE writer needs the partons of every event): 0 = g g; 1 + 6 i + c = flavour i in
 * class c (0 q qbar, 1 qbar q, 2 q g, 3 g q, 4 qbar g, 5 g qbar; first parton from beam 1): records of 5 x 32 + 16 + 8 bytes.
 * For MF_GG_TTG, MF_PP_TTG and MF_PP_TTGG the momenta (and channel) of the new records are filled in by a second kernel that
 * follows the pass on the same stream (complete when the stream has reached the end of the call, like everything else the call
 * writes). */
int mf_unweight(mf_process *p, const double *d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                uint64_t n_events, double w_max, void *d_records, uint64_t capacity, uint64_t *d_count,
                double *d_hist, mf_iter_result *d_result, void *stream);

/* Dynamic scale (R16).  on != 0: every later pass uses, event by event,
 * mu_F^2 = mu_R^2 = m_t^2 + pT(top)^2, the general 2-D log-bicubic PDF lookup at that scale, and the strong coupling
 * running at one loop (n_f = 5) from the descriptor's alpha_s at the descriptor's mu2:
 * alpha_s(mu^2) = alpha_s / (1 + alpha_s (23 / 12 pi) ln(mu^2 / mu2)); |M|^2 is rescaled by (alpha_s(mu^2)/alpha_s)^n_g.
 * on == 0 restores the fixed scale.  MF_EINVAL for MF_EE_MUMU. */
int mf_set_dynamic_scale(mf_process *p, int32_t on);

/* Observable histograms accumulated in the same pass ("histogram accumulation"; L109-119, Fig. 2:
 * d sigma / d pT,top and d sigma / d eta,top).  Attaches a caller-owned DEVICE buffer d_obs[2][n_bins + 1] of doubles
 * to the handle; from then on every mf_vegas_iterate / mf_unweight call ADDS (never overwrites; the caller zeroes)
 * the weights w of its events (pb per event: divide by the number of events for a cross section per bin) into
 *   d_obs[0][i]  lab-frame pT of the FIRST final-state particle (the top quark; mu- for MF_EE_MUMU) in
 *                [i, i+1) * pt_max / n_bins;            i = n_bins: pT >= pt_max
 *   d_obs[1][i]  its pseudorapidity asinh(pz / pT) in -eta_max + [i, i+1) * 2 eta_max / n_bins;  i = n_bins: outside
 * Events failing the cuts (w = 0) are not entered.  The additions are L2 atomics: per-bin sums are reproducible up
 * to the rounding of the summation order.  d_obs = NULL detaches.  Errors: n_bins outside 1..4096 or a non-positive
 * range -> MF_EINVAL.  The buffer must stay valid while attached. */
int mf_set_observables(mf_process *p, double *d_obs, int32_t n_bins, double pt_max, double eta_max);

/* Test/diagnostic: per-event rows of mf_debug_row_len doubles, identical to the oracle's layout:
 * x[D] | (n+2)x(E,px,py,pz) lab, beams first | x1 x2 | lum | me2 | phi | jvegas | w | pass | r | u[D] | bin[D]
 * MF_PP_TT and MF_PP_TTGG append | lum_qq | me2_qq  (lum, me2 are then the gg channel's; w is the sum of both channels;
 * for MF_PP_TTGG me2_qq is the luminosity-weighted mean of the two beam assignments);
 * MF_PP_TTG appends luminosity x |M|^2 of its six quark-channel classes: q qbar, qbar q, q g, g q, qbar g, g qbar */
int mf_debug_eval(mf_process *p, const double *d_grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                  uint64_t n_events, double *d_out, void *stream);

/* Test/diagnostic: raw Philox4x32-10 words for blocks (event, iteration, block) of stream `seed`:
 * d_out[4*n] uint32, block index b of event first_event+k at d_out[4*(k*n_blocks+b)..]. */
int mf_debug_philox(uint64_t seed, uint32_t iteration, uint64_t first_event, uint64_t n_events, uint32_t n_blocks,
                    uint32_t *d_out, void *stream);
/* Test/diagnostic: general 2-D log-bicubic PDF lookup x*g(x, q2) (parton table 0) for n points (device arrays). */
int mf_debug_pdf(mf_process *p, const double *d_x, const double *d_q2, uint64_t n, double *d_out, void *stream);
/* Test/diagnostic: averaged |M|^2 at n sets of CM-frame momenta d_mom[n][n_final+2][4] (beams first) -> d_out[n];
 * MF_PP_TT: d_out[n][2] = (g g -> t tbar, q qbar -> t tbar). */
int mf_debug_me2(mf_process *p, const double *d_mom, uint64_t n, double *d_out, void *stream);

/* Test/diagnostic: averaged |M|^2 of the quark channels of pp -> ttbar g at n sets of momenta d_mom[n][5][4] (the two
 * incoming first) -> d_out[n].  kind 0: q qbar -> t tbar g; 1: q g -> t tbar q; 2: qbar g -> t tbar qbar.
 * kind 3: q qbar -> t tbar g g, the quark channel of MF_PP_TTGG, at d_mom[n][6][4]. */
int mf_debug_me2_quark_gluon(int32_t kind, double m_top, double alpha_s, const double *d_mom, uint64_t n, double *d_out,
                             void *stream);

/* Measurement helper: runs a dependent-free DFMA chain on every SM for `iters` iterations and returns the
 * achieved FP64 rate in flop/s (2 flop per DFMA) in *h_flops.  Synchronous.  Used by bench.py for the
 * "alu" roofline denominator (FP64 peak is not in MEASURED_PEAKS.json). */
int mf_measure_fp64_peak(int64_t iters, double *h_flops, double *h_ms);
/* The same for the FP64 tensor path: independent DMMA.884 (mma.sync m8n8k4 f64) accumulators, 2 x 256 flop per instruction and
 * warp.  BASELINE.json north_star allows DMMA only on evidence: this probe and profiles/r2_dmma_probe.md are the evidence
 * (37.0 TFLOP/s on B200, the full FP64 rate, at a sixteenth of the issue slots of a DFMA stream). */
int mf_measure_dmma_peak(int64_t iters, double *h_flops, double *h_ms);

#ifdef __cplusplus
}
#endif
#endif
