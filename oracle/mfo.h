/* ORACLE — TEST INFRASTRUCTURE ONLY.  C ABI of the CPU oracle (prefix mfo_), mirroring include/mf.h
 * so that tests can call both with identical arguments.  All pointers are HOST pointers.
 * Shares no code with the CUDA path.  `prec` selects the real type the arithmetic runs in:
 * 0 = double (the oracle proper), 1 = long double, 2 = __float128 (referees).               */
#ifndef MFO_H
#define MFO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct mfo_process mfo_process;

/* same field order and meaning as mf_process_desc (include/mf.h) */
typedef struct {
  int32_t process; /* 0 ee->mumu, 1 gg->tt, 2 gg->ttg, 3 gg->ttgg, 4 pp->tt (gg + q qbar, flavour summed), 5 pp->ttg (gg + q qbar, q g, qbar g), 6 gg->ttggg */
  double sqrt_s;
  double alpha_em, alpha_s;
  double m_top;
  double mu2;
  double ptmin, etamax, drmin;
  double gev2_to_pb;
  int32_t n_bins;
  int32_t pdf_nx, pdf_nq;
  const double *pdf_lnx, *pdf_lnq2, *pdf_xf; /* pdf_xf[max(pdf_nfl,1)][pdf_nx][pdf_nq]: table 0 gluon, 1+2i quark i, 2+2i antiquark i */
  int32_t pdf_nfl;                           /* parton tables: 0 or 1 = gluon only; process 4 needs 1 + 2 n_f (odd, >= 3)          */
} mfo_process_desc;

typedef struct {
  double sum_w, sum_w2, max_abs_w;
  uint64_t n_pass, n_accept;
} mfo_iter_result;

int mfo_create_process(const mfo_process_desc*, mfo_process** out);
int mfo_destroy_process(mfo_process*);
/* R16: on != 0 switches to the dynamic scale mu_F^2 = mu_R^2 = m_t^2 + pT(top)^2 with one-loop running alpha_s
 * (n_f = 5) from the descriptor's alpha_s at its mu2; not for process 0 (-1) */
int mfo_set_dynamic_scale(mfo_process*, int32_t on);
int mfo_n_dims(const mfo_process*, int32_t* D);
int mfo_n_final(const mfo_process*, int32_t* n);
int mfo_record_size(const mfo_process*, int32_t* bytes);
int mfo_debug_row_len(const mfo_process*, int32_t* n_doubles);

/* O1-O13: one VEGAS iteration over events [first_event, first_event+n_events) */
int mfo_vegas_iterate(mfo_process*, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                      uint64_t n_events, double* hist, mfo_iter_result* result, int prec);
/* O14 */
int mfo_refine_grid(mfo_process*, double* grid, const double* hist, double alpha, int prec);
/* O15: accepted events appended in event order at records[*count]; *count advances for every accepted event.
 * Record: (n+2) lab four-momenta, w, u64 event id; process 4 appends the u64 channel code of R18
 * (0 gg; 1+2i quark i from beam 1; 2+2i quark i from beam 2), drawn with the second uniform of the accept block;
 * process 5 likewise (R20): 0 gg; 1 + 6 i + c = flavour i in class c (q qbar, qbar q, q g, g q, qbar g, g qbar) */
int mfo_unweight(mfo_process*, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                 uint64_t n_events, double w_max, void* records, uint64_t capacity, uint64_t* count, double* hist,
                 mfo_iter_result* result, int prec);
/* per-event rows:  x[D] | (n+2)x(E,px,py,pz) lab | x1 x2 | lum | me2 | phi | jvegas | w | pass | r | u[D] | bin[D]
 * process 4 appends | lum_qq | me2_qq (lum, me2 = the gg channel; w = the sum of both channels);
 * process 5 appends luminosity x |M|^2 of the six quark-channel classes q qbar, qbar q, q g, g q, qbar g, g qbar */
int mfo_debug_eval(mfo_process*, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                   uint64_t n_events, double* out, int prec);

/* ---- component entry points for the pins --------------------------------------------------- */
/* averaged |M|^2 of q(mom[0]) qbar(mom[1]) -> t(mom[2]) tbar(mom[3]) (process 4 only) */
double mfo_me2_qq(const mfo_process*, const double* mom, int basis, int prec);
/* Quark channels of pp -> ttbar g (R19): averaged |M|^2 from the five Feynman diagrams with explicit colour.  kind 0: q(mom0) qbar(mom1) -> t(mom2) tbar(mom3) g(mom4); kind 1: q(mom0) g(mom1) -> t(mom2) tbar(mom3) q(mom4);
 * kind 2: qbar(mom0) g(mom1) -> t(mom2) tbar(mom3) qbar(mom4).  subst != 0: gluon polarisation -> its momentum (Ward identity: 0). */
double mfo_me2_light_line_ttbar_g(int kind, const double* mom, double mt, double alpha_s, int basis, int subst, int prec);
/* q(mom0) qbar(mom1) -> t(mom2) tbar(mom3) g(mom4) g(mom5): averaged |M|^2 from the 36 tree
 * diagrams with explicit colour tensors.  subst = 0 / 1: that gluon's polarisation -> its momentum (Ward identity: 0), -1: none. */
double mfo_me2_qq_ttbar_gg(const double* mom, double mt, double alpha_s, int basis, int subst, int prec);
/* the same amplitude iM for explicit helicities lam[6] in {-1,+1} (q, qbar, t, tbar, g, g) and colours col[6] = (antiquark, quark,
 * top, antitop in 0..2; gluons in 0..7): out[0..1] = sum over the diagrams, out[2..3] = colour-dressed subset recursion */
void mfo_qq_ttbar_gg_amplitude(const double* mom, double mt, double gs, const int32_t* lam, int basis, const int32_t* col,
                               double out[4]);
/* x f(x, q2) of parton table `table` (0 gluon, 1+2i quark i, 2+2i antiquark i) */
double mfo_pdf_xf_table(const mfo_process*, int table, double x, double q2, int prec);
void mfo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void mfo_philox_block(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t block, uint32_t out[4]);
double mfo_uniform_from_words(uint32_t hi, uint32_t lo);
double mfo_vegas_map(const double* grid, int D, int nb, const double* u, double* x, int32_t* bin);
/* out = tau, y, x1, x2, shat, jac */
void mfo_parton_fractions(double x0, double x1, double tau_min, double s, double out[6]);
/* mom[4][4]; returns the weight per unit (xc, xphi) */
double mfo_two_body(double shat, double m, double xc, double xphi, double* mom);
/* k[n][4]; returns the volume V */
double mfo_rambo(int n, const double* mass, double w, const double* rho, double* k, int prec);
/* (2 pi)^(4 - 3 n): dPhi_n = (2 pi)^(4 - 3 n) V (O6 step 6) */
double mfo_two_pi_power(int n);
/* returns 1 if the gluons pass; obs[ng][3] = pt, eta, phi */
int mfo_cuts(int ng, const double* gluons_lab, double ptmin, double etamax, double drmin, double* obs);
void mfo_boost_z(double y, const double in[4], double out[4]);
double mfo_pdf_xf(const mfo_process*, double x, double q2, int prec);
/* n! x n! doubles, permutations in lexicographic order */
int mfo_colour_matrix(int n, double* out);
/* one entry straight from the definition: sum over all 8^n colour assignments of Tr(T^{a_sigma(0)} .. T^{a_sigma(n-1)} (T^{a_tau(0)} .. )^dagger) */
double mfo_colour_matrix_entry(int n, const int32_t* sigma, const int32_t* tau);
/* averaged |M|^2 for the process' particle content at the given momenta [(n+2)][4] (beams first).
 * basis bit0: spinor basis, bit1: polarisation basis; subst_gluon: -1 or the gluon whose polarisation
 * is replaced by its momentum; amps (may be NULL): [n_hel][n_perm][2] ordered amplitudes;
 * per_hel (may be NULL, C0 only): 16 values. */
double mfo_me2(const mfo_process*, const double* mom, int basis, int subst_gluon, double* amps, double* per_hel,
               int prec);
/* colour-dressed amplitude iM_ij for fixed helicities hel[ng+2] = (t, tbar, g0..) in {-1,+1} and gluon
 * colours col[ng] in 0..7, quark colours icol, jcol in 0..2; out = (re, im) */
int mfo_dressed_amplitude(const mfo_process*, const double* mom, const int32_t* hel, const int32_t* col,
                          int icol, int jcol, double out[2]);
/* the same helicity's ordered amplitudes contracted with the colour factors (T..T)_ij: out = (re, im) */
int mfo_ordered_amplitude_coloured(const mfo_process*, const double* mom, const int32_t* hel, const int32_t* col,
                                   int icol, int jcol, double out[2]);
/* wavefunction checks: spinor u (kind 0) or v (kind 1), 4 complex = 8 doubles */
void mfo_spinor(const double p[4], double m, int lambda, int basis, int kind, double out[8]);
void mfo_polarisation(const double p[4], int lambda, int basis, double out[8]);
/* flops of one |M|^2 evaluation with the operation-counting scalar: out = add, mul, div, sqrt, trans, cmp */
int mfo_count_ops_me2(const mfo_process*, const double* mom, uint64_t out[6]);
/* same for a whole event (debug row path) */
int mfo_count_ops_event(mfo_process*, const double* grid, uint64_t seed, uint32_t iteration, uint64_t event,
                        uint64_t out[6]);

#ifdef __cplusplus
}
#endif
#endif
