// ORACLE — TEST INFRASTRUCTURE ONLY (see real.hpp, mfo.h).
//
// mfo.cpp: the per-event chain O1..O12 put together in the paper's order (random numbers
// -> phase-space kinematics -> matrix element -> accumulation), the iteration sums O13, unweighting O15,
// and the C ABI.  One event at a time, one thread, no SIMD, no blocking.
#include "mfo.h"
#include <cstring>
#include <memory>
#include <type_traits>
#include "amplitude.hpp"
#include "amplitude_qq.hpp"
#include "method.hpp"

using namespace mfo;

struct mfo_process {
  mfo_process_desc d;
  PdfTable pdf;                   // the gluon (table 0)
  std::vector<PdfTable> pdfq;     // process 4: quark and antiquark tables, [2 i] quark i, [2 i + 1] antiquark i
  int D = 0, nfinal = 0, ng = 0;  // ng = gluons including the two beams (0 for ee->mumu)
  int dyn_scale = 0;              // mfo_set_dynamic_scale (R16)
  double tau_min = 0;
  std::vector<double> C_d;
  std::vector<long double> C_l;
  std::vector<__float128> C_q;
  std::vector<Counted> C_c;
};

namespace {

template <class R> const std::vector<R>& colour_of(mfo_process& P);
template <> const std::vector<double>& colour_of<double>(mfo_process& P) { return P.C_d; }
template <> const std::vector<long double>& colour_of<long double>(mfo_process& P) {
  if (P.C_l.empty() && P.ng) P.C_l = colour_matrix<long double>(P.ng);
  return P.C_l;
}
template <> const std::vector<__float128>& colour_of<__float128>(mfo_process& P) {
  if (P.C_q.empty() && P.ng) P.C_q = colour_matrix<__float128>(P.ng);
  return P.C_q;
}
template <> const std::vector<Counted>& colour_of<Counted>(mfo_process& P) {
  if (P.C_c.empty() && P.ng) {
    for (double c : P.C_d) P.C_c.push_back(Counted(c));
  }
  return P.C_c;
}

template <class R> struct EventOut {
  double u[24];
  int bin[24];
  R x[24];
  R mom[7][4];  // lab frame, beams first
  R x1, x2, lum, me2, phi, jac, w;
  R lum_qq, me2_qq;  // process 4: the flavour-summed q qbar luminosity and the q qbar matrix element
  R chan[32];        // process 4: luminosity x |M|^2 of every partonic channel (0 gg; 1+2i q_i from beam 1; 2+2i from beam 2)
                     // process 5 (R20): 0 gg; 1 + 6 i + c: flavour i in class c (q qbar, qbar q, q g, g q, qbar g, g qbar)
  int n_chan;
  R chq[6];          // process 5: luminosity x |M|^2 of the six flavour-summed quark-channel classes
  int pass;
};

// averaged |M|^2 at CM-frame momenta
template <class R> R matrix_element(mfo_process& P, const R mom[][4], int basis, int subst, R* amps, R* per_hel) {
  if (P.d.process == 0) {
    R m4[4][4];
    for (int i = 0; i < 4; ++i)
      for (int m = 0; m < 4; ++m) m4[i][m] = mom[i][m];
    return me2_ee_mumu<R>(m4, R(P.d.alpha_em), basis & 1, per_hel);
  }
  return me2_gg_ttbar_ng<R>(P.ng, mom, R(P.d.m_top), R(P.d.alpha_s), basis, subst, colour_of<R>(P), amps);
}

// O1..O12 for one event
template <class R>
void eval_event(mfo_process& P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t event, EventOut<R>& o) {
  const int D = P.D, nb = P.d.n_bins, n = P.nfinal;
  uniforms_for_event(seed, iteration, event, D, o.u);           // O1, O2
  o.jac = vegas_map<R>(grid, D, nb, o.u, o.x, o.bin);           // O3
  const R s = R(P.d.sqrt_s) * R(P.d.sqrt_s);
  R cm[7][4];
  R y = R(0), shat = s, jac_parton = R(1);
  o.x1 = R(1);
  o.x2 = R(1);
  if (P.d.process == 0) {
    R m4[4][4];
    o.phi = two_body<R>(s, R(0), o.x[0], o.x[1], m4);            // O5
    for (int i = 0; i < 4; ++i)
      for (int m = 0; m < 4; ++m) cm[i][m] = m4[i][m];
  } else {
    PartonKin<R> k = parton_fractions<R>(o.x[0], o.x[1], R(P.tau_min), s);  // O4
    y = k.y; shat = k.shat; jac_parton = k.jac; o.x1 = k.x1; o.x2 = k.x2;
    if (P.d.process == 1 || P.d.process == 4) {
      R m4[4][4];
      o.phi = two_body<R>(shat, R(P.d.m_top), o.x[2], o.x[3], m4);  // O5
      for (int i = 0; i < 4; ++i)
        for (int m = 0; m < 4; ++m) cm[i][m] = m4[i][m];
    } else {
      R w = r_sqrt(shat);
      R mass[5] = {R(P.d.m_top), R(P.d.m_top), R(0), R(0), R(0)};
      R kf[8][4];
      R V = rambo<R>(n, mass, w, o.x + 2, kf);                  // O6
      o.phi = two_pi_power<R>(n) * V;
      R E = w / R(2);
      cm[0][0] = E; cm[0][1] = R(0); cm[0][2] = R(0); cm[0][3] = E;
      cm[1][0] = E; cm[1][1] = R(0); cm[1][2] = R(0); cm[1][3] = -E;
      for (int i = 0; i < n; ++i)
        for (int m = 0; m < 4; ++m) cm[2 + i][m] = kf[i][m];
    }
  }
  for (int i = 0; i < n + 2; ++i) boost_z<R>(y, cm[i], o.mom[i]);  // O7
  int nglu = n - 2;
  o.pass = 1;
  if (P.d.process >= 2) {
    R gl[4][4];
    for (int g = 0; g < nglu; ++g)
      for (int m = 0; m < 4; ++m) gl[g][m] = o.mom[4 + g][m];
    o.pass = pass_cuts<R>(nglu, gl, R(P.d.ptmin), R(P.d.etamax), R(P.d.drmin)) ? 1 : 0;
  }
  o.lum = R(0);
  o.me2 = R(0);
  o.w = R(0);
  o.lum_qq = R(0);
  o.me2_qq = R(0);
  o.n_chan = 0;
  for (int c = 0; c < 6; ++c) o.chq[c] = R(0);
  if (!o.pass) return;
  o.lum = R(1);
  R mu2 = R(P.d.mu2), as_factor = R(1);
  if (P.d.process != 0 && P.dyn_scale) {
    // R16 (dynamic scale): mu_F^2 = mu_R^2 = m_t^2 + pT(top)^2, event by event; the strong coupling
    // runs at one loop from its value alpha_s at the reference scale mu2 of the descriptor:
    //   alpha_s(mu^2) = alpha_s / (1 + alpha_s b0 ln(mu^2 / mu2)),  b0 = (33 - 2 n_f) / (12 pi),  n_f = 5;
    // |M|^2 ~ alpha_s^{n_g}, so it is rescaled by (alpha_s(mu^2) / alpha_s)^{n_g}.
    R pt2 = cm[2][1] * cm[2][1] + cm[2][2] * cm[2][2];
    mu2 = R(P.d.m_top) * R(P.d.m_top) + pt2;
    R b0 = R(23) / (R(12) * r_pi<R>());
    R ratio = R(1) / (R(1) + R(P.d.alpha_s) * b0 * r_log(mu2 / R(P.d.mu2)));
    for (int g = 0; g < P.ng; ++g) as_factor = as_factor * ratio;
  }
  if (P.d.process != 0) {
    R f1 = pdf_xf<R>(P.pdf, o.x1, mu2), f2 = pdf_xf<R>(P.pdf, o.x2, mu2);  // O8
    o.lum = f1 * f2 / (o.x1 * o.x2);
  }
  o.me2 = matrix_element<R>(P, cm, 0, -1, nullptr, nullptr) * as_factor;     // O9-O11 (x R16 factor)
  // O12: f = lum/(2 shat) |M|^2 Phi J_tau J_y K ; w = f * J_vegas
  R f = o.lum / (R(2) * shat) * o.me2 * o.phi * jac_parton * R(P.d.gev2_to_pb);
  if (P.d.process == 4 || P.d.process == 7) {
    // quark channels: for every flavour the quark may come from either beam,
    //   sum_i [ q_i(x1) qbar_i(x2) |M|^2(q along +z) + qbar_i(x1) q_i(x2) |M|^2(q along -z) ] / (x1 x2),
    // added to the gg term at the same phase-space point.  Both are of the same order in alpha_s: the same R16 factor.
    // Process 4: q qbar -> ttbar; process 7 (R22): q qbar -> ttbar g g, the 36 diagrams of amplitude_qq.hpp.
    R ma[6][4], mb[6][4];
    for (int i = 0; i < n + 2; ++i)
      for (int m = 0; m < 4; ++m) { ma[i][m] = cm[i][m]; mb[i][m] = cm[i][m]; }
    for (int m = 0; m < 4; ++m) { mb[0][m] = cm[1][m]; mb[1][m] = cm[0][m]; }   // quark from beam 2
    R Ma, Mb;
    if (P.d.process == 4) {
      Ma = me2_qq_ttbar<R>(ma, R(P.d.m_top), R(P.d.alpha_s), 0) * as_factor;
      Mb = me2_qq_ttbar<R>(mb, R(P.d.m_top), R(P.d.alpha_s), 0) * as_factor;
    } else {
      Ma = me2_qq_ttbar_gg<R>(ma, R(P.d.m_top), R(P.d.alpha_s), 0, -1) * as_factor;
      Mb = me2_qq_ttbar_gg<R>(mb, R(P.d.m_top), R(P.d.alpha_s), 0, -1) * as_factor;
    }
    R La = R(0), Lb = R(0);
    for (size_t i = 0; i + 1 < P.pdfq.size(); i += 2) {
      R q1 = pdf_xf<R>(P.pdfq[i], o.x1, mu2), qb1 = pdf_xf<R>(P.pdfq[i + 1], o.x1, mu2);
      R q2 = pdf_xf<R>(P.pdfq[i], o.x2, mu2), qb2 = pdf_xf<R>(P.pdfq[i + 1], o.x2, mu2);
      La = La + q1 * qb2;
      Lb = Lb + qb1 * q2;
      o.chan[1 + i] = q1 * qb2 / (o.x1 * o.x2) * Ma;
      o.chan[2 + i] = qb1 * q2 / (o.x1 * o.x2) * Mb;
    }
    o.chan[0] = o.lum * o.me2;
    o.n_chan = 1 + (int)P.pdfq.size();
    La = La / (o.x1 * o.x2);
    Lb = Lb / (o.x1 * o.x2);
    o.lum_qq = La + Lb;
    R both = La * Ma + Lb * Mb;
    o.me2_qq = (o.lum_qq != R(0)) ? both / o.lum_qq : Ma;     // the luminosity-weighted mean of the two orientations
    f = (o.lum * o.me2 + both) / (R(2) * shat) * o.phi * jac_parton * R(P.d.gev2_to_pb);
  }
  if (P.d.process == 5) {
    // quark channels of pp -> ttbar g (R19), flavour summed (the quarks are massless, so the
    // matrix elements do not depend on the flavour), the light parton of the final state being whatever the channel
    // makes it (the cuts act on it alike):
    //   q qbar, qbar q -> ttbar g;   q g, g q -> ttbar q;   qbar g, g qbar -> ttbar qbar
    R Q1 = R(0), Qb1 = R(0), Q2 = R(0), Qb2 = R(0), D12 = R(0), D21 = R(0);
    R g1 = pdf_xf<R>(P.pdf, o.x1, mu2), g2 = pdf_xf<R>(P.pdf, o.x2, mu2);
    R lumf[5][6];   // per flavour and class (R20: the partonic channel of an accepted event)
    int nfl = 0;
    for (size_t i = 0; i + 1 < P.pdfq.size(); i += 2, ++nfl) {
      R q1 = pdf_xf<R>(P.pdfq[i], o.x1, mu2), qb1 = pdf_xf<R>(P.pdfq[i + 1], o.x1, mu2);
      R q2 = pdf_xf<R>(P.pdfq[i], o.x2, mu2), qb2 = pdf_xf<R>(P.pdfq[i + 1], o.x2, mu2);
      Q1 = Q1 + q1; Qb1 = Qb1 + qb1; Q2 = Q2 + q2; Qb2 = Qb2 + qb2;
      D12 = D12 + q1 * qb2;
      D21 = D21 + qb1 * q2;
      lumf[nfl][0] = q1 * qb2; lumf[nfl][1] = qb1 * q2; lumf[nfl][2] = q1 * g2; lumf[nfl][3] = g1 * q2;
      lumf[nfl][4] = qb1 * g2; lumf[nfl][5] = g1 * qb2;
    }
    R lumc[6] = {D12, D21, Q1 * g2, g1 * Q2, Qb1 * g2, g1 * Qb2};
    const int kind[6] = {0, 0, 1, 1, 2, 2};
    R both = R(0);
    o.chan[0] = o.lum * o.me2;
    o.n_chan = 1 + 6 * nfl;
    for (int c = 0; c < 6; ++c) {
      R m5[5][4];
      for (int i = 0; i < 5; ++i)
        for (int m = 0; m < 4; ++m) m5[i][m] = cm[i][m];
      if (c & 1)                                     // the (anti)quark comes from beam 2
        for (int m = 0; m < 4; ++m) { m5[0][m] = cm[1][m]; m5[1][m] = cm[0][m]; }
      R M = me2_light_line_ttbar_g<R>(kind[c], m5, R(P.d.m_top), R(P.d.alpha_s), 0, 0) * as_factor;
      o.chq[c] = lumc[c] / (o.x1 * o.x2) * M;
      both = both + o.chq[c];
      for (int i = 0; i < nfl; ++i) o.chan[1 + 6 * i + c] = lumf[i][c] / (o.x1 * o.x2) * M;
    }
    f = (o.lum * o.me2 + both) / (R(2) * shat) * o.phi * jac_parton * R(P.d.gev2_to_pb);
  }
  o.w = f * o.jac;
}

template <class R> struct SumType { typedef long double type; };
template <> struct SumType<__float128> { typedef __float128 type; };
template <> struct SumType<Counted> { typedef double type; };

struct Record { /* layout only: (n+2)*4 doubles, double w, uint64 id */ };

// O13 (+O15 if records != nullptr or w_max > 0)
template <class R>
int iterate(mfo_process& P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first, uint64_t n_events,
            double* hist, mfo_iter_result* res, bool unweight, double w_max, char* records, uint64_t capacity,
            uint64_t* count) {
  typedef typename SumType<R>::type S;
  const int D = P.D, nb = P.d.n_bins;
  std::vector<S> h((size_t)D * nb, S(0));
  S sw = S(0), sw2 = S(0);
  double maxw = 0;
  uint64_t npass = 0, nacc = 0;
  const bool has_channel = P.d.process == 4 || P.d.process == 5 || P.d.process == 7;
  int recsize = (P.nfinal + 2) * 32 + 16 + (has_channel ? 8 : 0);
  EventOut<R> o;
  for (uint64_t e = first; e < first + n_events; ++e) {
    eval_event<R>(P, grid, seed, iteration, e, o);
    double w = r_to_double(o.w);
    S ws = S(w);
    sw = sw + ws;
    sw2 = sw2 + ws * ws;
    if (o.pass) ++npass;
    if (std::fabs(w) > maxw) maxw = std::fabs(w);
    if (w != 0.0)
      for (int d = 0; d < D; ++d) h[(size_t)d * nb + o.bin[d]] = h[(size_t)d * nb + o.bin[d]] + ws * ws;
    if (unweight) {
      double r = accept_draw(seed, iteration, e);
      if (r * w_max < std::fabs(w)) {  // O15: accept iff r * w_max < |w|
        ++nacc;
        uint64_t slot = (*count)++;
        if (records && slot < capacity) {
          char* rec = records + slot * (uint64_t)recsize;
          double buf[7 * 4 + 1];
          for (int i = 0; i < P.nfinal + 2; ++i)
            for (int m = 0; m < 4; ++m) buf[i * 4 + m] = r_to_double(o.mom[i][m]);
          buf[(P.nfinal + 2) * 4] = w;
          std::memcpy(rec, buf, ((P.nfinal + 2) * 4 + 1) * sizeof(double));
          std::memcpy(rec + ((P.nfinal + 2) * 4 + 1) * sizeof(double), &e, sizeof(uint64_t));
          if (has_channel) {
            // R18 / R20: the partonic channel of an accepted event is drawn in proportion to |luminosity x |M|^2| of the
            // channels, in channel order: the first c with  sum_{c' <= c} |a_c'| > v * sum |a|,  v the channel draw
            double a[32], total = 0.0;
            for (int c = 0; c < o.n_chan; ++c) { a[c] = std::fabs(r_to_double(o.chan[c])); total += a[c]; }
            double v = channel_draw(seed, iteration, e) * total, cum = 0.0;
            uint64_t pick = (uint64_t)(o.n_chan - 1);
            for (int c = 0; c < o.n_chan; ++c) {
              cum += a[c];
              if (cum > v) { pick = (uint64_t)c; break; }
            }
            std::memcpy(rec + ((P.nfinal + 2) * 4 + 2) * sizeof(double), &pick, sizeof(uint64_t));
          }
        }
      }
    }
  }
  if (hist)
    for (size_t i = 0; i < h.size(); ++i) hist[i] = (double)h[i];
  if (res) {
    res->sum_w = (double)sw;
    res->sum_w2 = (double)sw2;
    res->max_abs_w = maxw;
    res->n_pass = npass;
    res->n_accept = nacc;
  }
  return 0;
}

template <class R>
int debug_eval(mfo_process& P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first, uint64_t n_events,
               double* out) {
  const int D = P.D, n = P.nfinal;
  const int rowlen = 3 * D + 4 * (n + 2) + 9 + ((P.d.process == 4 || P.d.process == 7) ? 2 : P.d.process == 5 ? 6 : 0);
  EventOut<R> o;
  for (uint64_t k = 0; k < n_events; ++k) {
    uint64_t e = first + k;
    eval_event<R>(P, grid, seed, iteration, e, o);
    double* row = out + k * rowlen;
    int c = 0;
    for (int d = 0; d < D; ++d) row[c++] = r_to_double(o.x[d]);
    for (int i = 0; i < n + 2; ++i)
      for (int m = 0; m < 4; ++m) row[c++] = r_to_double(o.mom[i][m]);
    row[c++] = r_to_double(o.x1);
    row[c++] = r_to_double(o.x2);
    row[c++] = r_to_double(o.lum);
    row[c++] = r_to_double(o.me2);
    row[c++] = r_to_double(o.phi);
    row[c++] = r_to_double(o.jac);
    row[c++] = r_to_double(o.w);
    row[c++] = (double)o.pass;
    row[c++] = accept_draw(seed, iteration, e);
    for (int d = 0; d < D; ++d) row[c++] = o.u[d];
    for (int d = 0; d < D; ++d) row[c++] = (double)o.bin[d];
    if (P.d.process == 4 || P.d.process == 7) {
      row[c++] = r_to_double(o.lum_qq);
      row[c++] = r_to_double(o.me2_qq);
    }
    if (P.d.process == 5)
      for (int q = 0; q < 6; ++q) row[c++] = r_to_double(o.chq[q]);
  }
  return 0;
}

template <class R> void load_momenta(const mfo_process& P, const double* mom, R out[][4]) {
  for (int i = 0; i < P.nfinal + 2; ++i)
    for (int m = 0; m < 4; ++m) out[i][m] = R(mom[i * 4 + m]);
}

template <class R>
double me2_entry(mfo_process& P, const double* mom, int basis, int subst, double* amps, double* per_hel) {
  R m[7][4];
  load_momenta<R>(P, mom, m);
  std::vector<R> a, ph(16);
  if (amps && P.ng) {
    int np = 1;
    for (int j = 2; j <= P.ng; ++j) np *= j;
    a.resize((size_t)(4 << P.ng) * np * 2);
  }
  R v = matrix_element<R>(P, m, basis, subst, a.empty() ? nullptr : a.data(), per_hel ? ph.data() : nullptr);
  for (size_t i = 0; i < a.size(); ++i) amps[i] = r_to_double(a[i]);
  if (per_hel && P.d.process == 0)
    for (int i = 0; i < 16; ++i) per_hel[i] = r_to_double(ph[i]);
  return r_to_double(v);
}

void load_helicities(DressedContext<long double>& d, mfo_process& P, const long double mom[][4], const int32_t* hel) {
  typedef long double R;
  AmpContext<R>& c = d.base;
  R gs = r_sqrt(R(4) * r_pi<R>() * R(P.d.alpha_s));
  setup_context<R>(c, P.ng, mom, R(P.d.m_top), gs);
  c.ubar3 = bar(u_spinor<R>(c.p3, c.mt, hel[0], 0));
  c.v4 = v_spinor<R>(c.p4, c.mt, hel[1], 0);
  for (int g = 0; g < P.ng; ++g) {
    if (g < 2) c.eps[g] = polarisation<R>(c.P[g], hel[2 + g], 0);
    else c.eps[g] = cconj(polarisation<R>(mom[2 + g], hel[2 + g], 0));
  }
}

}  // namespace

#define DISPATCH(prec, CALL)                         \
  switch (prec) {                                    \
    case 0: { typedef double R; return CALL; }       \
    case 1: { typedef long double R; return CALL; }  \
    case 2: { typedef __float128 R; return CALL; }   \
    default: return -1;                              \
  }

extern "C" {

int mfo_create_process(const mfo_process_desc* d, mfo_process** out) {
  if (!d || !out) return -1;
  if (d->process < 0 || d->process > 7 || d->n_bins < 2 || !(d->sqrt_s > 0)) return -1;
  std::unique_ptr<mfo_process> P(new mfo_process);
  P->d = *d;
  static const int Dtab[8] = {2, 4, 14, 18, 4, 14, 22, 18}, ntab[8] = {2, 2, 3, 4, 2, 3, 5, 4}, ngtab[8] = {0, 2, 3, 4, 2, 3, 5, 4};
  P->D = Dtab[d->process];
  P->nfinal = ntab[d->process];
  P->ng = ngtab[d->process];
  if (d->process != 0) {
    if (d->pdf_nx < 4 || d->pdf_nq < 4 || !d->pdf_lnx || !d->pdf_lnq2 || !d->pdf_xf) return -1;
    P->pdf.nx = d->pdf_nx;
    P->pdf.nq = d->pdf_nq;
    P->pdf.lnx.assign(d->pdf_lnx, d->pdf_lnx + d->pdf_nx);
    P->pdf.lnq2.assign(d->pdf_lnq2, d->pdf_lnq2 + d->pdf_nq);
    P->pdf.xf.assign(d->pdf_xf, d->pdf_xf + (size_t)d->pdf_nx * d->pdf_nq);
    if (d->process == 4 || d->process == 5 || d->process == 7) {
      if (d->pdf_nfl < 3 || d->pdf_nfl % 2 == 0) return -1;
      for (int t = 1; t < d->pdf_nfl; ++t) {
        PdfTable T = P->pdf;
        const double* src = d->pdf_xf + (size_t)t * d->pdf_nx * d->pdf_nq;
        T.xf.assign(src, src + (size_t)d->pdf_nx * d->pdf_nq);
        P->pdfq.push_back(T);
      }
    }
    double lq = std::log(d->mu2);
    if (!(lq >= P->pdf.lnq2.front() && lq <= P->pdf.lnq2.back())) return -4;
    int ncut = P->nfinal - 2;
    double thr = 2 * d->m_top + ncut * (d->ptmin > 0 ? d->ptmin : 0.0);
    P->tau_min = thr * thr / (d->sqrt_s * d->sqrt_s);  // O4
    if (!(std::log(P->tau_min) >= P->pdf.lnx.front())) return -4;
    P->C_d = colour_matrix<double>(P->ng);
  }
  P->d.pdf_lnx = P->d.pdf_lnq2 = P->d.pdf_xf = nullptr;
  *out = P.release();
  return 0;
}
int mfo_destroy_process(mfo_process* P) { delete P; return 0; }
int mfo_set_dynamic_scale(mfo_process* P, int32_t on) {
  if (!P || P->d.process == 0) return -1;
  P->dyn_scale = on ? 1 : 0;
  return 0;
}
int mfo_n_dims(const mfo_process* P, int32_t* D) { if (!P || !D) return -1; *D = P->D; return 0; }
int mfo_n_final(const mfo_process* P, int32_t* n) { if (!P || !n) return -1; *n = P->nfinal; return 0; }
int mfo_record_size(const mfo_process* P, int32_t* b) {
  if (!P || !b) return -1;
  *b = (P->nfinal + 2) * 32 + 16 + ((P->d.process == 4 || P->d.process == 5 || P->d.process == 7) ? 8 : 0);   // processes 4, 5, 7 append the u64 channel code
  return 0;
}
int mfo_debug_row_len(const mfo_process* P, int32_t* n) {
  if (!P || !n) return -1;
  *n = 3 * P->D + 4 * (P->nfinal + 2) + 9 + ((P->d.process == 4 || P->d.process == 7) ? 2 : P->d.process == 5 ? 6 : 0);
  return 0;
}

int mfo_vegas_iterate(mfo_process* P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                      uint64_t n_events, double* hist, mfo_iter_result* result, int prec) {
  if (!P || !grid) return -1;
  DISPATCH(prec, iterate<R>(*P, grid, seed, iteration, first_event, n_events, hist, result, false, 0.0, nullptr, 0, nullptr));
}
int mfo_refine_grid(mfo_process* P, double* grid, const double* hist, double alpha, int prec) {
  if (!P || !grid || !hist) return -1;
  switch (prec) {
    case 0: refine_grid<double>(grid, hist, P->D, P->d.n_bins, alpha); return 0;
    case 1: refine_grid<long double>(grid, hist, P->D, P->d.n_bins, (long double)alpha); return 0;
    case 2: refine_grid<__float128>(grid, hist, P->D, P->d.n_bins, (__float128)alpha); return 0;
  }
  return -1;
}
int mfo_unweight(mfo_process* P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                 uint64_t n_events, double w_max, void* records, uint64_t capacity, uint64_t* count, double* hist,
                 mfo_iter_result* result, int prec) {
  if (!P || !grid || !count) return -1;
  DISPATCH(prec, iterate<R>(*P, grid, seed, iteration, first_event, n_events, hist, result, true, w_max, (char*)records,
                            capacity, count));
}
int mfo_debug_eval(mfo_process* P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t first_event,
                   uint64_t n_events, double* out, int prec) {
  if (!P || !grid || !out) return -1;
  DISPATCH(prec, debug_eval<R>(*P, grid, seed, iteration, first_event, n_events, out));
}

void mfo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) { philox4x32_10(ctr, key, out); }
void mfo_philox_block(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t block, uint32_t out[4]) {
  philox_block(seed, iteration, event, block, out);
}
double mfo_uniform_from_words(uint32_t hi, uint32_t lo) { return uniform_from_words(hi, lo); }
double mfo_vegas_map(const double* grid, int D, int nb, const double* u, double* x, int32_t* bin) {
  std::vector<int> b(D);
  double j = vegas_map<double>(grid, D, nb, u, x, b.data());
  for (int d = 0; d < D; ++d) bin[d] = b[d];
  return j;
}
void mfo_parton_fractions(double x0, double x1, double tau_min, double s, double out[6]) {
  PartonKin<double> k = parton_fractions<double>(x0, x1, tau_min, s);
  out[0] = k.tau; out[1] = k.y; out[2] = k.x1; out[3] = k.x2; out[4] = k.shat; out[5] = k.jac;
}
double mfo_two_body(double shat, double m, double xc, double xphi, double* mom) {
  double m4[4][4];
  double w = two_body<double>(shat, m, xc, xphi, m4);
  std::memcpy(mom, m4, sizeof(m4));
  return w;
}
double mfo_rambo(int n, const double* mass, double w, const double* rho, double* k, int prec) {
  if (n < 2 || n > 8) return -1;
  if (prec == 0) {
    double kk[8][4];
    double V = rambo<double>(n, mass, w, rho, kk);
    std::memcpy(k, kk, sizeof(double) * 4 * n);
    return V;
  }
  typedef __float128 Q;
  Q m[8], r[32], kk[8][4];
  for (int i = 0; i < n; ++i) m[i] = mass[i];
  for (int i = 0; i < 4 * n; ++i) r[i] = rho[i];
  Q V = rambo<Q>(n, m, Q(w), r, kk);
  for (int i = 0; i < n; ++i)
    for (int c = 0; c < 4; ++c) k[i * 4 + c] = (double)kk[i][c];
  return (double)V;
}
double mfo_two_pi_power(int n) { return two_pi_power<double>(n); }
int mfo_cuts(int ng, const double* gl, double ptmin, double etamax, double drmin, double* obs) {
  double g[4][4];
  for (int i = 0; i < ng; ++i)
    for (int m = 0; m < 4; ++m) g[i][m] = gl[i * 4 + m];
  if (obs)
    for (int i = 0; i < ng; ++i) {
      CutObs<double> o = cut_observables<double>(g[i]);
      obs[3 * i] = o.pt; obs[3 * i + 1] = o.eta; obs[3 * i + 2] = o.phi;
    }
  return pass_cuts<double>(ng, g, ptmin, etamax, drmin) ? 1 : 0;
}
void mfo_boost_z(double y, const double in[4], double out[4]) { boost_z<double>(y, in, out); }
double mfo_pdf_xf(const mfo_process* P, double x, double q2, int prec) {
  if (prec == 2) return (double)pdf_xf<__float128>(P->pdf, x, q2);
  if (prec == 1) return (double)pdf_xf<long double>(P->pdf, x, q2);
  return pdf_xf<double>(P->pdf, x, q2);
}
double mfo_pdf_xf_table(const mfo_process* P, int table, double x, double q2, int prec) {
  if (table == 0) return mfo_pdf_xf(P, x, q2, prec);
  if (table < 0 || (size_t)table > P->pdfq.size()) return 0.0;
  const PdfTable& T = P->pdfq[table - 1];
  if (prec == 2) return (double)pdf_xf<__float128>(T, x, q2);
  if (prec == 1) return (double)pdf_xf<long double>(T, x, q2);
  return pdf_xf<double>(T, x, q2);
}
double mfo_me2_qq(const mfo_process* P, const double* mom, int basis, int prec) {
  if (!P || P->d.process != 4 || !mom) return -1.0;
  if (prec == 1) {
    long double m[4][4];
    for (int i = 0; i < 4; ++i)
      for (int c = 0; c < 4; ++c) m[i][c] = mom[4 * i + c];
    return (double)me2_qq_ttbar<long double>(m, P->d.m_top, P->d.alpha_s, basis);
  }
  double m[4][4];
  for (int i = 0; i < 4; ++i)
    for (int c = 0; c < 4; ++c) m[i][c] = mom[4 * i + c];
  return me2_qq_ttbar<double>(m, P->d.m_top, P->d.alpha_s, basis);
}
double mfo_me2_qq_ttbar_gg(const double* mom, double mt, double alpha_s, int basis, int subst, int prec) {
  if (prec == 1) {
    long double m[6][4];
    for (int i = 0; i < 6; ++i)
      for (int k = 0; k < 4; ++k) m[i][k] = mom[4 * i + k];
    return (double)me2_qq_ttbar_gg<long double>(m, mt, alpha_s, basis, subst);
  }
  double m[6][4];
  for (int i = 0; i < 6; ++i)
    for (int k = 0; k < 4; ++k) m[i][k] = mom[4 * i + k];
  return me2_qq_ttbar_gg<double>(m, mt, alpha_s, basis, subst);
}
void mfo_qq_ttbar_gg_amplitude(const double* mom, double mt, double gs, const int32_t* lam, int basis, const int32_t* col,
                               double out[4]) {
  double m[6][4];
  for (int i = 0; i < 6; ++i)
    for (int k = 0; k < 4; ++k) m[i][k] = mom[4 * i + k];
  int l[6];
  for (int i = 0; i < 6; ++i) l[i] = lam[i];
  const Cx<double> a = qq_diagram_sum<double>(m, mt, gs, l, basis, col[0], col[1], col[2], col[3], col[4], col[5]);
  const Cx<double> b = qq_dressed_amplitude<double>(m, mt, gs, l, basis, col[0], col[1], col[2], col[3], col[4], col[5]);
  out[0] = a.re; out[1] = a.im; out[2] = b.re; out[3] = b.im;
}
double mfo_me2_light_line_ttbar_g(int kind, const double* mom, double mt, double alpha_s, int basis, int subst,
                                  int prec) {
  if (!mom || kind < 0 || kind > 2) return -1.0;
  if (prec == 1) {
    long double m[5][4];
    for (int i = 0; i < 5; ++i)
      for (int c = 0; c < 4; ++c) m[i][c] = mom[4 * i + c];
    return (double)me2_light_line_ttbar_g<long double>(kind, m, mt, alpha_s, basis, subst);
  }
  double m[5][4];
  for (int i = 0; i < 5; ++i)
    for (int c = 0; c < 4; ++c) m[i][c] = mom[4 * i + c];
  return me2_light_line_ttbar_g<double>(kind, m, mt, alpha_s, basis, subst);
}
double mfo_colour_matrix_entry(int n, const int32_t* sigma, const int32_t* tau) {
  if (n < 1 || n > 5) return 0.0;
  int s[5], t[5];
  for (int i = 0; i < n; ++i) { s[i] = sigma[i]; t[i] = tau[i]; }
  return colour_matrix_entry<double>(n, s, t);
}
int mfo_colour_matrix(int n, double* out) {
  if (n < 1 || n > 5) return -1;
  std::vector<double> C = colour_matrix<double>(n);
  std::memcpy(out, C.data(), C.size() * sizeof(double));
  return 0;
}
double mfo_me2(const mfo_process* Pc, const double* mom, int basis, int subst_gluon, double* amps, double* per_hel,
               int prec) {
  mfo_process& P = *const_cast<mfo_process*>(Pc);
  DISPATCH(prec, me2_entry<R>(P, mom, basis, subst_gluon, amps, per_hel));
}
int mfo_dressed_amplitude(const mfo_process* Pc, const double* mom, const int32_t* hel, const int32_t* col, int icol,
                          int jcol, double out[2]) {
  mfo_process& P = *const_cast<mfo_process*>(Pc);
  if (!P.ng) return -1;
  typedef long double R;
  static DressedContext<R> d;
  static bool init = false;
  if (!init) { dressed_init(d); init = true; }
  R m[7][4];
  load_momenta<R>(P, mom, m);
  load_helicities(d, P, m, hel);
  for (int g = 0; g < P.ng; ++g) d.col[g] = col[g];
  Cx<R> M = dressed_amplitude(d, icol, jcol);
  out[0] = (double)M.re;
  out[1] = (double)M.im;
  return 0;
}
int mfo_ordered_amplitude_coloured(const mfo_process* Pc, const double* mom, const int32_t* hel, const int32_t* col,
                                   int icol, int jcol, double out[2]) {
  mfo_process& P = *const_cast<mfo_process*>(Pc);
  if (!P.ng) return -1;
  typedef long double R;
  DressedContext<R> d;  // only its AmpContext is used
  R m[7][4];
  load_momenta<R>(P, mom, m);
  load_helicities(d, P, m, hel);
  auto perms = permutations(P.ng);
  Cx<R> M;
  for (auto& s : perms) {
    Mat3<R> prod = su3_generator<R>(col[s[0]]);
    for (int i = 1; i < P.ng; ++i) prod = mat3_mul(prod, su3_generator<R>(col[s[i]]));
    M += prod.m[icol][jcol] * ordered_amplitude(d.base, s.data());
  }
  out[0] = (double)M.re;
  out[1] = (double)M.im;
  return 0;
}
void mfo_spinor(const double p[4], double m, int lambda, int basis, int kind, double out[8]) {
  Spinor<double> s = kind == 0 ? u_spinor<double>(p, m, lambda, basis) : v_spinor<double>(p, m, lambda, basis);
  for (int i = 0; i < 4; ++i) { out[2 * i] = s.c[i].re; out[2 * i + 1] = s.c[i].im; }
}
void mfo_polarisation(const double p[4], int lambda, int basis, double out[8]) {
  CVec4<double> e = polarisation<double>(p, lambda, basis);
  for (int i = 0; i < 4; ++i) { out[2 * i] = e.c[i].re; out[2 * i + 1] = e.c[i].im; }
}
static void export_counts(uint64_t out[6]) {
  OpCounts& c = op_counts();
  out[0] = c.add; out[1] = c.mul; out[2] = c.div; out[3] = c.sqrt; out[4] = c.trans; out[5] = c.cmp;
}
int mfo_count_ops_me2(const mfo_process* Pc, const double* mom, uint64_t out[6]) {
  mfo_process& P = *const_cast<mfo_process*>(Pc);
  colour_of<Counted>(P);
  Counted m[7][4];
  load_momenta<Counted>(P, mom, m);
  op_counts() = OpCounts();
  matrix_element<Counted>(P, m, 0, -1, nullptr, nullptr);
  export_counts(out);
  return 0;
}
int mfo_count_ops_event(mfo_process* P, const double* grid, uint64_t seed, uint32_t iteration, uint64_t event,
                        uint64_t out[6]) {
  colour_of<Counted>(*P);
  EventOut<Counted> o;
  op_counts() = OpCounts();
  eval_event<Counted>(*P, grid, seed, iteration, event, o);
  export_counts(out);
  return 0;
}

}  // extern "C"
