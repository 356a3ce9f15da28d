// mf_pdf.cuh — step a6: PDF lookup by log-bicubic interpolation of x*g on an (ln x, ln Q^2) grid
// (PAPER.md L27 PDFFlow by citation; table and meaning from BASELINE.json configs[1]; rule = DESIGN.md R8:
// LHAPDF-style cubic Hermite in ln x, then in ln Q^2, of the value x*g; knot derivative = one-sided
// difference at the table ends, mean of the two one-sided differences inside; no clamping to >= 0).
//
// Two entry points.  pdf_xf_2d is the general per-point 2-D lookup.  The fused pass uses the fact that
// mu_F^2 is fixed per process: both interpolations are linear in the table, so the ln Q^2 Hermite step is
// applied ONCE per block to every x-knot (pdf_collapse_q2, run by the block while it stages its tables)
// and the per-event work is the 1-D Hermite in ln x on that collapsed row held in shared memory.
#pragma once
#include "mf_common.cuh"

namespace mf {

MF_HD double hermite(double t, double f0, double d0, double f1, double d1, double h) {
  double t2 = t * t, t3 = t2 * t;
  return (2.0 * t3 - 3.0 * t2 + 1.0) * f0 + (t3 - 2.0 * t2 + t) * h * d0 + (3.0 * t2 - 2.0 * t3) * f1 +
         (t3 - t2) * h * d1;
}

// cubic Hermite across cell [j, j+1] of a 1-D knot sequence with values g(-1..2 relative to j)
MF_HD double hermite_cell(const double* knots, int n, int j, double u, double gm, double g0, double g1, double g2) {
  double h = knots[j + 1] - knots[j];
  double right0 = (g1 - g0) / h;
  double d0 = right0, d1 = right0;
  if (j > 0) d0 = 0.5 * ((g0 - gm) / (knots[j] - knots[j - 1]) + right0);
  if (j + 2 < n) d1 = 0.5 * (right0 + (g2 - g1) / (knots[j + 2] - knots[j + 1]));
  return hermite(u, g0, d0, g1, d1, h);
}

// cell index with knots[i] <= v < knots[i+1], clamped to [0, n-2]; starts from the uniform-spacing guess
// and walks, so it is exact for any increasing knot sequence.
MF_HD int find_cell(const double* knots, int n, double v) {
  double guess = (v - knots[0]) / (knots[n - 1] - knots[0]) * (double)(n - 1);
  int i = guess > 0.0 ? (int)guess : 0;
  if (i > n - 2) i = n - 2;
  while (i < n - 2 && !(v < knots[i + 1])) ++i;
  while (i > 0 && v < knots[i]) --i;
  return i;
}

// Collapse the ln Q^2 direction at fixed (jq, uq) for x-knot ix: row[ix] = Hermite_Q(xf[ix][jq-1..jq+2]).
MF_HD double pdf_collapse_q2(const double* xf, const double* lnq2, int nq, int ix, int jq, double uq) {
  const double* r = xf + (size_t)ix * nq;
  double gm = jq > 0 ? r[jq - 1] : 0.0, g2 = jq + 2 < nq ? r[jq + 2] : 0.0;
  return hermite_cell(lnq2, nq, jq, uq, gm, r[jq], r[jq + 1], g2);
}

// 1-D Hermite in ln x on a (collapsed) row.
MF_HD double pdf_xf_row(const double* lnx, const double* row, int nx, double x) {
  double lx = log(x);
  int i = find_cell(lnx, nx, lx);
  double h = lnx[i + 1] - lnx[i];
  double t = (lx - lnx[i]) / h;
  double fm = i > 0 ? row[i - 1] : 0.0, f2 = i + 2 < nx ? row[i + 2] : 0.0;
  return hermite_cell(lnx, nx, i, t, fm, row[i], row[i + 1], f2);
}

// The same on NT collapsed rows rows[t * nx + i] at once (multi-flavour table).  The Hermite interpolant is linear in
// the four knot values f(i-1), f(i), f(i+1), f(i+2) it uses, so the cell search, the logarithm, the basis polynomials
// and the knot-derivative coefficients (all the divisions) are done ONCE per x and every table costs four FMAs:
//   F = h00 f0 + a d0 + h01 f1 + b d1,   a = h10 h,  b = h11 h,
//   d0 = al (f0 - fm) + be0 (f1 - f0),   d1 = be1 (f1 - f0) + ga (f2 - f1)
// with (al, be0) = (1/2hl, 1/2h) inside and (0, 1/h) at the first cell, (be1, ga) = (1/2h, 1/2hr) inside and (1/h, 0)
// at the last cell (the one-sided differences of R8).
struct HermiteWeights { int i; double wm, w0, w1, w2; };
MF_HD HermiteWeights hermite_weights(const double* lnx, int nx, double x) {
  HermiteWeights W;
  const double lx = log(x);
  const int i = find_cell(lnx, nx, lx);
  const double h = lnx[i + 1] - lnx[i], rh = 1.0 / h;
  const double t = (lx - lnx[i]) * rh, t2 = t * t, t3 = t2 * t;
  const double h00 = 2.0 * t3 - 3.0 * t2 + 1.0, h01 = 3.0 * t2 - 2.0 * t3;
  const double a = (t3 - 2.0 * t2 + t) * h, b = (t3 - t2) * h;
  double al = 0.0, be0 = rh, be1 = rh, ga = 0.0;
  if (i > 0) { al = 0.5 / (lnx[i] - lnx[i - 1]); be0 = 0.5 * rh; }
  if (i + 2 < nx) { ga = 0.5 / (lnx[i + 2] - lnx[i + 1]); be1 = 0.5 * rh; }
  W.i = i;
  W.wm = -a * al;
  W.w0 = h00 + a * (al - be0) - b * be1;
  W.w1 = h01 + a * be0 + b * (be1 - ga);
  W.w2 = b * ga;
  return W;
}
MF_HD double hermite_apply(const HermiteWeights& W, const double* row, int nx) {
  const int i = W.i;
  const double fm = i > 0 ? row[i - 1] : 0.0, f2 = i + 2 < nx ? row[i + 2] : 0.0;
  return fma(W.wm, fm, fma(W.w2, f2, fma(W.w0, row[i], W.w1 * row[i + 1])));
}

// General 2-D lookup: Hermite in ln x on the rows jq-1..jq+2 that exist, then Hermite in ln Q^2.
MF_HD double pdf_xf_2d(const double* lnx, const double* lnq2, const double* xf, int nx, int nq, double x, double q2) {
  double lx = log(x), lq = log(q2);
  int i = find_cell(lnx, nx, lx), j = find_cell(lnq2, nq, lq);
  double h = lnx[i + 1] - lnx[i];
  double t = (lx - lnx[i]) / h;
  double g[4];
#pragma unroll
  for (int r = 0; r < 4; ++r) {
    int jj = j - 1 + r;
    g[r] = 0.0;
    if (jj >= 0 && jj < nq) {
      double fm = i > 0 ? xf[(size_t)(i - 1) * nq + jj] : 0.0;
      double f2 = i + 2 < nx ? xf[(size_t)(i + 2) * nq + jj] : 0.0;
      g[r] = hermite_cell(lnx, nx, i, t, fm, xf[(size_t)i * nq + jj], xf[(size_t)(i + 1) * nq + jj], f2);
    }
  }
  double u = (lq - lnq2[j]) / (lnq2[j + 1] - lnq2[j]);
  return hermite_cell(lnq2, nq, j, u, g[0], g[1], g[2], g[3]);
}

}  // namespace mf
