// ORACLE — TEST INFRASTRUCTURE ONLY.  Memory-safety driver for the oracle: built by
// tests/test_oracle_sanitizers.py together with mfo.cpp under -fsanitize=address,undefined and run once in the CPU
// test tier.  It walks every C-ABI entry point of mfo.h for every process on a few events (fp64, and the long double /
// __float128 referees on fewer), including the edge sizes (0 and 1 events, a record buffer that overflows).
// It checks nothing numerically: the pins in tests/ do that.  Exit code 0 and an empty sanitizer log is the result.
//
//   sanitize_main <table.bin>     table.bin = int32 nfl, nx, nq; then lnx[nx], lnq2[nq], xf[nfl][nx][nq] as doubles
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include "mfo.h"

static void die(const char* what) {
  std::fprintf(stderr, "sanitize_main: %s\n", what);
  std::exit(2);
}

int main(int argc, char** argv) {
  if (argc < 2) die("usage: sanitize_main table.bin");
  FILE* f = std::fopen(argv[1], "rb");
  if (!f) die("cannot open the table");
  int32_t hdr[3];
  if (std::fread(hdr, sizeof(int32_t), 3, f) != 3) die("short header");
  const int nfl = hdr[0], nx = hdr[1], nq = hdr[2];
  std::vector<double> lnx(nx), lnq2(nq), xf((size_t)nfl * nx * nq);
  if (std::fread(lnx.data(), 8, nx, f) != (size_t)nx || std::fread(lnq2.data(), 8, nq, f) != (size_t)nq ||
      std::fread(xf.data(), 8, xf.size(), f) != xf.size())
    die("short table");
  std::fclose(f);

  const int n_proc = 8;
  const int nfinal[n_proc] = {2, 2, 3, 4, 2, 3, 5, 4};
  const int n_events[n_proc] = {200, 100, 30, 6, 80, 16, 1, 1};
  for (int proc = 0; proc < n_proc; ++proc) {
    mfo_process_desc d;
    std::memset(&d, 0, sizeof d);
    d.process = proc;
    d.sqrt_s = proc == 0 ? 100.0 : 13000.0;
    d.alpha_em = 1.0 / 132.507;
    d.alpha_s = 0.118;
    d.m_top = 173.0;
    d.mu2 = 173.0 * 173.0;
    if (nfinal[proc] > 2) { d.ptmin = 30.0; d.etamax = 2.5; }
    if (nfinal[proc] > 3) d.drmin = 0.4;
    d.gev2_to_pb = 0.3894e9;
    d.n_bins = 50;
    if (proc != 0) {
      d.pdf_nx = nx; d.pdf_nq = nq;
      d.pdf_lnx = lnx.data(); d.pdf_lnq2 = lnq2.data(); d.pdf_xf = xf.data();
      d.pdf_nfl = (proc == 4 || proc == 5 || proc == 7) ? nfl : 1;
    }
    mfo_process* P = nullptr;
    int rc = mfo_create_process(&d, &P);
    if (rc != 0) {
      if (proc == 6) continue;          // a build of the oracle without g g -> t tbar g g g
      die("mfo_create_process failed");
    }
    int32_t D = 0, nf = 0, rs = 0, rl = 0;
    mfo_n_dims(P, &D); mfo_n_final(P, &nf); mfo_record_size(P, &rs); mfo_debug_row_len(P, &rl);
    const int nb = d.n_bins, n = n_events[proc];
    std::vector<double> grid((size_t)D * (nb + 1)), hist((size_t)D * nb);
    for (int dd = 0; dd < D; ++dd)
      for (int i = 0; i <= nb; ++i) grid[(size_t)dd * (nb + 1) + i] = (double)i / nb;
    mfo_iter_result res;
    // two adapting iterations, then edge sizes, then unweighting with a buffer that is too small
    for (int it = 0; it < 2; ++it) {
      if (mfo_vegas_iterate(P, grid.data(), 5, it, 0, n, hist.data(), &res, 0) != 0) die("vegas_iterate");
      if (mfo_refine_grid(P, grid.data(), hist.data(), 1.5, 0) != 0) die("refine_grid");
    }
    mfo_vegas_iterate(P, grid.data(), 5, 2, 0, 0, hist.data(), &res, 0);
    mfo_vegas_iterate(P, grid.data(), 5, 2, ~0ull - 3, 1, hist.data(), &res, 0);
    mfo_vegas_iterate(P, grid.data(), 5, 2, 0, 1, nullptr, nullptr, 0);
    const double w_max = res.max_abs_w > 0 ? 0.01 * res.max_abs_w : 1.0;
    const uint64_t cap = 3;
    std::vector<char> rec((size_t)cap * rs);
    uint64_t count = 1;
    if (mfo_unweight(P, grid.data(), 5, 3, 0, n, w_max, rec.data(), cap, &count, hist.data(), &res, 0) != 0) die("unweight");
    count = 0;
    mfo_unweight(P, grid.data(), 5, 3, 0, n, w_max, nullptr, 0, &count, nullptr, &res, 0);
    std::vector<double> rows((size_t)rl * 4);
    for (int prec = 0; prec < 3; ++prec) {
      const int m = ((prec == 0 && proc != 7) || proc < 3) ? 4 : 1;
      if ((proc >= 6 && prec != 0) || ((proc == 3 || proc == 5) && prec == 2)) continue;   // minutes under the sanitizers
      if (mfo_debug_eval(P, grid.data(), 5, 1, 7, m, rows.data(), prec) != 0) die("debug_eval");
      mfo_vegas_iterate(P, grid.data(), 5, 1, 7, m, hist.data(), &res, prec);
      mfo_refine_grid(P, grid.data(), hist.data(), 1.5, prec);
    }
    if (proc != 0) {
      mfo_set_dynamic_scale(P, 1);
      mfo_debug_eval(P, grid.data(), 5, 1, 7, 2, rows.data(), 0);
      mfo_set_dynamic_scale(P, 0);
      for (double x : {1e-9, 3e-4, 0.5, 0.9, 1.0}) {
        mfo_pdf_xf(P, x, 2.72, 0);
        mfo_pdf_xf(P, x, 1e10, 2);
        if (d.pdf_nfl > 1) mfo_pdf_xf_table(P, d.pdf_nfl - 1, x, 3e4, 0);
      }
    }
    // the matrix element at the momenta of the last row, with every gluon substituted in turn, amplitudes exported
    if (proc >= 1 && proc <= 3) {
      const int ng = nf;     // gluons including the beams
      int nperm = 1;
      for (int j = 2; j <= ng; ++j) nperm *= j;
      std::vector<double> amps((size_t)(4 << ng) * nperm * 2);
      const double* mom = rows.data() + D;   // lab momenta: |M|^2 is Lorentz invariant, any frame is a valid input
      for (int g = -1; g < ng; ++g) mfo_me2(P, mom, g & 3, g, amps.data(), nullptr, 0);
      uint64_t ops[6];
      mfo_count_ops_me2(P, mom, ops);
      mfo_count_ops_event(P, grid.data(), 5, 1, 7, ops);
      int32_t hel[8] = {1, -1, 1, 1, -1, 1, 1, 1}, col[6] = {0, 3, 7, 4, 1, 2};
      double out[2];
      mfo_dressed_amplitude(P, mom, hel, col, 0, 2, out);
      mfo_ordered_amplitude_coloured(P, mom, hel, col, 1, 1, out);
    }
    if (proc == 4) {
      mfo_me2_qq(P, rows.data() + D, 0, 0);
      mfo_me2_qq(P, rows.data() + D, 1, 1);
    }
    if (proc == 0) {
      double per[16];
      mfo_me2(P, rows.data() + D, 1, -1, nullptr, per, 0);
    }
    mfo_destroy_process(P);
  }
  // component calls
  {
    uint32_t ctr[4] = {1, 2, 3, 4}, key[2] = {5, 6}, out[4];
    mfo_philox4x32_10(ctr, key, out);
    mfo_philox_block(~0ull, ~0u, ~0ull, ~0u, out);
    mfo_uniform_from_words(~0u, ~0u);
    double grid[2 * 9], u[2] = {1.0 - 0x1.0p-53, 0x1.0p-53}, x[2];
    int32_t bin[2];
    for (int dd = 0; dd < 2; ++dd)
      for (int i = 0; i <= 8; ++i) grid[dd * 9 + i] = i / 8.0;
    mfo_vegas_map(grid, 2, 8, u, x, bin);
    double pf[6], mom[4 * 4];
    mfo_parton_fractions(0.3, 0.7, 1e-3, 1.69e8, pf);
    mfo_two_body(1e6, 173.0, 0.2, 0.9, mom);
    for (int n = 2; n <= 8; ++n) {
      double mass[8] = {173, 173, 0, 0, 0, 0, 0, 0}, rho[32], k[32];
      for (int i = 0; i < 32; ++i) rho[i] = (i + 0.5) / 32.5;
      mfo_rambo(n, mass, 2000.0, rho, k, 0);
      mfo_rambo(n, mass, 2000.0, rho, k, 2);
      mfo_two_pi_power(n);
    }
    double gl[3 * 4] = {50, 30, 40, 0, 100, -60, 10, 79, 90, 1, -40, 80}, obs[9], o4[4];
    mfo_cuts(3, gl, 30.0, 2.5, 0.4, obs);
    mfo_cuts(1, gl, 0.0, 0.0, 0.0, nullptr);
    mfo_boost_z(-1.3, gl, o4);
    for (int n = 1; n <= 4; ++n) {          // n = 5 (120 x 120 over 8^5 colours) takes minutes under the sanitizers
      int f = 1;
      for (int j = 2; j <= n; ++j) f *= j;
      std::vector<double> C((size_t)f * f);
      mfo_colour_matrix(n, C.data());
    }
    double p[4] = {200, 30, -40, std::sqrt(200.0 * 200 - 2500 - 173.0 * 173)}, sp[8];
    for (int b = 0; b < 2; ++b)
      for (int lam = -1; lam <= 1; lam += 2) {
        mfo_spinor(p, 173.0, lam, b, 0, sp);
        mfo_spinor(p, 173.0, lam, b, 1, sp);
        mfo_polarisation(gl, lam, b, sp);
      }
    double m5[5 * 4] = {500, 0, 0, 500, 500, 0, 0, -500, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    double mass[3] = {173, 173, 0}, rho[12] = {0.15, 0.35, 0.55, 0.25, 0.35, 0.5, 0.45, 0.35, 0.55, 0.65, 0.35, 0.45};
    mfo_rambo(3, mass, 1000.0, rho, m5 + 8, 0);
    for (int kind = 0; kind < 3; ++kind)
      for (int prec = 0; prec < 2; ++prec) mfo_me2_light_line_ttbar_g(kind, m5, 173.0, 0.118, prec, prec, prec);
    double m6[6 * 4] = {500, 0, 0, 500, 500, 0, 0, -500};
    double mass4[4] = {173, 173, 0, 0}, rho4[16] = {0.15, 0.35, 0.55, 0.25, 0.35, 0.5, 0.45, 0.35, 0.55, 0.65, 0.35, 0.45, 0.2, 0.7, 0.4, 0.6};
    mfo_rambo(4, mass4, 1000.0, rho4, m6 + 8, 0);
    mfo_me2_qq_ttbar_gg(m6, 173.0, 0.118, 3, 1, 0);
    const int32_t lam[6] = {1, -1, 1, 1, -1, 1}, col[6] = {2, 2, 0, 0, 3, 3};
    double amp[4];
    mfo_qq_ttbar_gg_amplitude(m6, 173.0, 1.2, lam, 2, col, amp);
  }
  std::puts("sanitize_main: ok");
  return 0;
}
