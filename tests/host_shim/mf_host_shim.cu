// Test-only shim: compiles the PRODUCT's __host__ __device__ per-event code for the host so that the
// `-m "not gpu"` tests can compare its arithmetic with the oracle without a GPU.  It is not part of the
// product library (libmadflow_b200.so has no host evaluation path) and is loaded only by tests/.
#include <cstring>
#include "../../paper_2106_10279_b200/csrc/mf_event.cuh"
#include "../../paper_2106_10279_b200/csrc/mf_me_qttg.cuh"
#include "../../paper_2106_10279_b200/csrc/mf_me_coop.cuh"
#include "../../paper_2106_10279_b200/csrc/mf_me_cta5.cuh"
#include "../../paper_2106_10279_b200/csrc/mf_me_qqttgg.cuh"
#include <vector>

using namespace mf;

// PG = mf::g4::Prog / mf::g3::Prog; mom[(n+2)][4] beams first; norm = couplings / averaging (top spin 0 only is
// evaluated and doubled: spin-flip symmetry)
template <class PG>
static double coop_host_me2(const double* mom, double m_top, double norm) {
  std::vector<double> tm(PG::TeamDoubles, 0.0), q(PG::Queue, 0.0);
  double k[4][4] = {};
  for (int i = 0; i < PG::NFinal; ++i) for (int m = 0; m < 4; ++m) k[i][m] = mom[(2 + i) * 4 + m];
  PG::owner_fill(q.data(), 1, k, 4.0 * mom[0] * mom[0], m_top);        // what the event's owner thread does
  for (int j = 0; j < PG::Queue; ++j) tm[PG::qdest(j)] = q[j];      // what the team's lanes do with the record
  double* in = tm.data() + PG::OffIn;
  for (int t = 0; t < PG::Team; ++t) PG::s0(tm.data(), in, t, m_top);
  for (int s = 0; s < PG::Phases; ++s)
    for (int w = 0; w < PG::Warps; ++w)
      for (int l = 0; l < 32; ++l) PG::run_phase(tm.data(), reinterpret_cast<const uint4*>(PG::table()), s, w, l, m_top);
  double sum = 0.0;
  for (int t = 0; t < PG::Team; ++t) sum += PG::s4_thread(tm.data(), t);
  return 2.0 * sum / PG::Cden * norm;
}

extern "C" {

// averaged |M|^2 at CM-frame momenta mom[(n+2)][4], beams first (oracle layout)
double mfh_me2(int process, const double* mom, double m_top, double alpha_s, double alpha_em) {
  Params P;
  std::memset(&P, 0, sizeof(P));
  P.alpha_em = alpha_em; P.alpha_s = alpha_s; P.m_top = m_top;
  double shat = 4.0 * mom[0] * mom[0];
  double gs2 = 4.0 * kPi * alpha_s;
  double k[4][4];
  int nf = (process <= 1 || process == 4) ? 2 : process + 1;
  for (int i = 0; i < nf; ++i) for (int m = 0; m < 4; ++m) k[i][m] = mom[(2 + i) * 4 + m];
  switch (process) {
    case 0: return matrix_element<0>(P, shat, k);
    case 1: P.me_norm = gs2 * gs2 / 256.0; return matrix_element<1>(P, shat, k);
    case 2: P.me_norm = gs2 * gs2 * gs2 / 256.0; return matrix_element<2>(P, shat, k);
    case 3: P.me_norm = gs2 * gs2 * gs2 * gs2 / 512.0; return matrix_element<3>(P, shat, k);
    case 4: return matrix_element_qq(P, shat, k);      // the quark channel of MF_PP_TT
  }
  return -1.0;
}

// The cooperative matrix-element programs of the fused pass (mf_me_coop.cuh), emulated on the host: the team
// threads are looped over stage by stage (a barrier separates the stages on the device).
double mfh_me2_coop(const double* mom, double m_top, double alpha_s) {   // g g -> t tbar g g
  double gs2 = 4.0 * kPi * alpha_s;
  return coop_host_me2<g4::Prog>(mom, m_top, gs2 * gs2 * gs2 * gs2 / 512.0);
}
double mfh_me2_coop3(const double* mom, double m_top, double alpha_s) {  // g g -> t tbar g
  double gs2 = 4.0 * kPi * alpha_s;
  return coop_host_me2<g3::Prog>(mom, m_top, gs2 * gs2 * gs2 / 256.0);
}

// g g -> t tbar g g g (mf_me_cta5.cuh): the block's work items looped over stage by stage; mom[7][4] beams first
double mfh_me2_cta5(const double* mom, double m_top, double alpha_s) {
  using namespace mf::g5;
  std::vector<double> S(kScratchDoubles, 0.0);
  for (int i = 0; i < 5; ++i) for (int m = 0; m < 4; ++m) S[kOffIn + 4 * i + m] = mom[(2 + i) * 4 + m];
  S[kOffIn + 20] = 4.0 * mom[0] * mom[0];
  for (int i = 0; i < kStage0Items; ++i) stage0_item(S.data(), i, m_top);
  for (int i = 0; i < kStage1Items; ++i) stage1_item(S.data(), i, m_top);
  for (int i = 0; i < kStage2Items; ++i) stage2_item(S.data(), i, m_top);
  for (int i = 0; i < kStage3Items; ++i) gluon_item(S.data(), 4, i);
  for (int i = 0; i < kStage4Items; ++i) gluon_item(S.data(), 5, i);
  double tot = 0.0;
  for (int half = 0; half < 2; ++half) {
    for (int i = 0; i < kAmpItems; ++i) amp_item(S.data(), half, i);
    tot += colour_rows_plain(S.data(), 0, 1);
  }
  const double gs2 = 4.0 * kPi * alpha_s;
  return 2.0 * tot / kCden * (gs2 * gs2 * gs2 * gs2 * gs2 / (256.0 * 6.0));
}

// quark channels of pp -> ttbar g (component; mf_me_qttg.cuh): mom = p1, p2, p3, p4, p5 as in the oracle's entry point
double mfh_me2_light_line_ttg(int kind, const double* mom, double m_top, double alpha_s) {
  const double* prow = kind == 0 ? mom + 4 : mom + 16;
  const double* pg = kind == 0 ? mom + 16 : mom + 4;
  return me2_light_line_ttg(kind, mom, prow, mom + 8, mom + 12, pg, m_top, 4.0 * kPi * alpha_s);
}

// all six classes at one CM-frame point: mom = b1, b2, t, tbar, parton (mf_me_qttg.cuh: shared top-line currents)
void mfh_me2_ttj_quark_classes(const double* mom, double m_top, double alpha_s, double out[6]) {
  me2_ttj_quark_classes(mom, mom + 4, mom + 8, mom + 12, mom + 16, m_top, 4.0 * kPi * alpha_s, out);
}

// q qbar -> t tbar g g at one CM-frame point: mom = q, qbar, t, tbar, g, g (mf_me_qqttgg.cuh)
double mfh_me2_qq_ttgg(const double* mom, double m_top, double alpha_s) {
  return me2_qq_ttgg(mom, mom + 4, mom + 8, mom + 12, mom + 16, mom + 20, m_top, 4.0 * kPi * alpha_s);
}

double mfh_me2_qq_ttgg_mem(const double* mom, double m_top, double alpha_s) {
  return me2_qq_ttgg_mem(mom, mom + 4, mom + 8, mom + 12, mom + 16, mom + 20, m_top, 4.0 * kPi * alpha_s);
}

void mfh_philox(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t block, uint32_t out[4]) {
  U4 r = philox_block(seed, iteration, event, block);
  out[0] = r.x; out[1] = r.y; out[2] = r.z; out[3] = r.w;
}
double mfh_uniform52(uint32_t hi, uint32_t lo) { return uniform52(hi, lo); }

double mfh_pdf_2d(const double* lnx, const double* lnq2, const double* xf, int nx, int nq, double x, double q2) {
  return pdf_xf_2d(lnx, lnq2, xf, nx, nq, x, q2);
}
// collapsed-row path used by the fused pass
double mfh_pdf_row(const double* lnx, const double* lnq2, const double* xf, int nx, int nq, double x, double q2) {
  double lq = log(q2);
  int jq = find_cell(lnq2, nq, lq);
  double uq = (lq - lnq2[jq]) / (lnq2[jq + 1] - lnq2[jq]);
  double row[512];
  for (int i = 0; i < nx; ++i) row[i] = pdf_collapse_q2(xf, lnq2, nq, i, jq, uq);
  return pdf_xf_row(lnx, row, nx, x);
}
// the multi-table variant of it (weights once per x, four FMAs per table)
double mfh_pdf_row_weights(const double* lnx, const double* lnq2, const double* xf, int nx, int nq, double x, double q2) {
  double lq = log(q2);
  int jq = find_cell(lnq2, nq, lq);
  double uq = (lq - lnq2[jq]) / (lnq2[jq + 1] - lnq2[jq]);
  double row[512];
  for (int i = 0; i < nx; ++i) row[i] = pdf_collapse_q2(xf, lnq2, nq, i, jq, uq);
  HermiteWeights W = hermite_weights(lnx, nx, x);
  return hermite_apply(W, row, nx);
}

}  // extern "C"

// full per-event chain on the host: writes x1, x2, phi, jac_vegas, jac_parton, pass, me2(if pass), momenta(lab)
template <int PROC>
static void event_host(const Params& P, const double* grid, uint64_t seed, uint32_t it, uint64_t e, double* out) {
  Event<PROC> ev;
  Bins<PROC> bins;
  DebugRow dbg = {nullptr, Traits<PROC>::D, Traits<PROC>::NF};
  generate_event<PROC>(P, grid, seed, it, e, ev, bins, dbg);
  out[0] = ev.x1; out[1] = ev.x2; out[2] = ev.phi; out[3] = ev.jac_vegas; out[4] = ev.jac_parton;
  out[5] = ev.pass ? 1.0 : 0.0;
  out[6] = ev.pass ? matrix_element<PROC>(P, ev.shat, ev.k) : 0.0;
  out[7] = ev.shat;
  for (int i = 0; i < Traits<PROC>::NF; ++i) for (int m = 0; m < 4; ++m) out[8 + 4 * i + m] = ev.k[i][m];
  for (int d = 0; d < Traits<PROC>::D; ++d) out[8 + 16 + d] = (double)bins.get(d);
}
extern "C" {

void mfh_event(int process, const double* grid, int n_bins, double sqrt_s, double m_top, double alpha_s,
               double alpha_em, double ptmin, double etamax, double drmin, double tau_min, uint64_t seed,
               uint32_t it, uint64_t e, double* out) {
  Params P;
  std::memset(&P, 0, sizeof(P));
  P.s = sqrt_s * sqrt_s; P.alpha_em = alpha_em; P.alpha_s = alpha_s; P.m_top = m_top;
  P.ptmin = ptmin; P.etamax = etamax; P.drmin = drmin; P.n_bins = n_bins;
  P.tau_min = tau_min; P.ln_tau_min = tau_min > 0 ? log(tau_min) : 0.0;
  double gs2 = 4.0 * kPi * alpha_s;
  switch (process) {
    case 0: event_host<0>(P, grid, seed, it, e, out); break;
    case 1: P.me_norm = gs2 * gs2 / 256.0; event_host<1>(P, grid, seed, it, e, out); break;
    case 2: P.me_norm = gs2 * gs2 * gs2 / 256.0; event_host<2>(P, grid, seed, it, e, out); break;
    case 3: P.me_norm = gs2 * gs2 * gs2 * gs2 / 512.0; event_host<3>(P, grid, seed, it, e, out); break;
  }
}

}  // extern "C"
