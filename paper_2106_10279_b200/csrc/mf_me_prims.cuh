// mf_me_prims.cuh — steps a7/a8: HELAS-style wavefunction, vertex and propagator routines
// (matrix elements are built from ALOHA/HELAS wavefunction and vertex routines and
// summed over helicities; the paper prints no formula — DESIGN.md R9/R10 state the conventions).
//
// Conventions of the CUDA path (deliberately unlike the oracle's Dirac-representation 4x4 matrices):
//  * metric (+,-,-,-); chiral representation gamma^mu = [[0, sigma^mu], [sigmabar^mu, 0]]; a Dirac spinor
//    is (psi_L; psi_R), two complex components each; every gamma-matrix product is written out on the
//    2x2 blocks, no matrix is ever formed.
//  * fermion spin states: the two z-axis spin states xi = (1,0), (0,1) in
//    u = ((p.sigma + m) xi; (p.sigmabar + m) xi) / sqrt(2(E+m)),  v = ((p.sigma + m) xi; -(p.sigmabar + m) xi)/sqrt(2(E+m)).
//    Branch free, no pT -> 0 singularity; the spin-summed |M|^2 is basis independent.
//  * gluon polarisation states: the two REAL linear polarisation vectors e1, e2 transverse to k.  The
//    polarisation sum equals the helicity sum (same 2-dimensional transverse space, unitary change of
//    basis), and with real polarisations every pure-gluon off-shell current is REAL, which halves the
//    storage and roughly quarters the arithmetic of the gluon currents.
//  * "hatted" currents: all factors of i and g_s are pulled out of the recursion (R10):
//      J(1..k) = g_s^{k-1} Jhat,   Jhat(seq) = [ -sum_splits V3 + sum_splits V4 ] / P^2
//      X(seq)  = g_s^{k}  Xhat,    Xhat(seq) = -(qslash + m)/(q^2 - m^2) sum_j Jhat-slash(head_j) Xhat(tail_j)
//      A(sigma) = i g_s^n Ahat(sigma)
//    so the recursion has real coefficients only and |A|^2 = g_s^{2n} |Ahat|^2.
#pragma once
#include "mf_common.cuh"

namespace mf {

struct rvec { double v[4]; };                 // real Lorentz vector, upper index (t, x, y, z)
struct cvec { double re[4], im[4]; };         // complex Lorentz vector
struct spin { double re[4], im[4]; };         // Dirac spinor (column or row), components (L0, L1, R0, R1)
struct cplx { double re, im; };

MF_HD double rdot(const rvec& a, const rvec& b) {
  return a.v[0] * b.v[0] - a.v[1] * b.v[1] - a.v[2] * b.v[2] - a.v[3] * b.v[3];
}
MF_HD rvec radd(const rvec& a, const rvec& b) {
  rvec o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.v[m] = a.v[m] + b.v[m];
  return o;
}
MF_HD rvec rsub(const rvec& a, const rvec& b) {
  rvec o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.v[m] = a.v[m] - b.v[m];
  return o;
}

// ---- gluon vertices (colour-ordered Feynman rules, all momenta incoming) -----------------------------
// V3^r(J1,P1; J2,P2) = (J1.J2)(P1-P2)^r + J2^r ((P2-Q).J1) + J1^r ((Q-P1).J2),  Q = -(P1+P2)
//                    = (J1.J2)(P1-P2)^r + J2^r ((P1+2P2).J1) - J1^r ((2P1+P2).J2)
//                    = (J1.J2)(P1-P2)^r + 2 (P2.J1) J2^r - 2 (P1.J2) J1^r
// the last line by current conservation, P.J(P) = 0, which holds for the polarisation vectors (k.eps = 0) and
// for every off-shell current built from them by this recursion (Berends-Giele).  acc += sgn * V3, sgn = +-1.
MF_HD void v3_acc(rvec& acc, double sgn, const rvec& J1, const rvec& P1, const rvec& J2, const rvec& P2) {
  const double s12 = sgn * rdot(J1, J2);
  const double sgn2 = sgn + sgn;
  const double s1 = sgn2 * rdot(P2, J1), s2 = -sgn2 * rdot(P1, J2);
#pragma unroll
  for (int m = 0; m < 4; ++m)
    acc.v[m] = fma(s2, J1.v[m], fma(s1, J2.v[m], fma(s12, P1.v[m] - P2.v[m], acc.v[m])));
}
// V4^r(J1,J2,J3) = 2 (J1.J3) J2^r - (J2.J3) J1^r - (J1.J2) J3^r ;  acc += sgn * V4, sgn = +-1
MF_HD void v4_acc(rvec& acc, double sgn, const rvec& J1, const rvec& J2, const rvec& J3) {
  const double a2 = (sgn + sgn) * rdot(J1, J3), a1 = -sgn * rdot(J2, J3), a3 = -sgn * rdot(J1, J2);
#pragma unroll
  for (int m = 0; m < 4; ++m) acc.v[m] = fma(a3, J3.v[m], fma(a1, J1.v[m], fma(a2, J2.v[m], acc.v[m])));
}
MF_HD rvec rscale(const rvec& a, double s) {
  rvec o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.v[m] = a.v[m] * s;
  return o;
}

// ---- fermion line ------------------------------------------------------------------------------------
// a-slash = [[0, a0 - a.sigma], [a0 + a.sigma, 0]] for a real vector a (upper index).
// column:  (a-slash psi)
MF_HD spin slash_col(const rvec& a, const spin& c) {
  double am = a.v[0] - a.v[3], ap = a.v[0] + a.v[3], a1 = a.v[1], a2 = a.v[2];
  spin o;
  // out0 = am c2 + (-a1 + i a2) c3
  o.re[0] = am * c.re[2] - a1 * c.re[3] - a2 * c.im[3];
  o.im[0] = am * c.im[2] - a1 * c.im[3] + a2 * c.re[3];
  // out1 = (-a1 - i a2) c2 + ap c3
  o.re[1] = -a1 * c.re[2] + a2 * c.im[2] + ap * c.re[3];
  o.im[1] = -a1 * c.im[2] - a2 * c.re[2] + ap * c.im[3];
  // out2 = ap c0 + (a1 - i a2) c1
  o.re[2] = ap * c.re[0] + a1 * c.re[1] + a2 * c.im[1];
  o.im[2] = ap * c.im[0] + a1 * c.im[1] - a2 * c.re[1];
  // out3 = (a1 + i a2) c0 + am c1
  o.re[3] = a1 * c.re[0] - a2 * c.im[0] + am * c.re[1];
  o.im[3] = a1 * c.im[0] + a2 * c.re[0] + am * c.im[1];
  return o;
}
// row:  (psibar a-slash)
MF_HD spin slash_row(const spin& r, const rvec& a) {
  double am = a.v[0] - a.v[3], ap = a.v[0] + a.v[3], a1 = a.v[1], a2 = a.v[2];
  spin o;
  // out0 = r2 ap + r3 (a1 + i a2)
  o.re[0] = ap * r.re[2] + a1 * r.re[3] - a2 * r.im[3];
  o.im[0] = ap * r.im[2] + a1 * r.im[3] + a2 * r.re[3];
  // out1 = r2 (a1 - i a2) + r3 am
  o.re[1] = a1 * r.re[2] + a2 * r.im[2] + am * r.re[3];
  o.im[1] = a1 * r.im[2] - a2 * r.re[2] + am * r.im[3];
  // out2 = r0 am + r1 (-a1 - i a2)
  o.re[2] = am * r.re[0] - a1 * r.re[1] + a2 * r.im[1];
  o.im[2] = am * r.im[0] - a1 * r.im[1] - a2 * r.re[1];
  // out3 = r0 (-a1 + i a2) + r1 ap
  o.re[3] = -a1 * r.re[0] - a2 * r.im[0] + ap * r.re[1];
  o.im[3] = -a1 * r.im[0] + a2 * r.re[0] + ap * r.im[1];
  return o;
}
// acc += a-slash c  (column) and acc += r a-slash (row), every component as one FMA chain onto acc
MF_HD void slash_col_acc(spin& o, const rvec& a, const spin& c) {
  const double am = a.v[0] - a.v[3], ap = a.v[0] + a.v[3], a1 = a.v[1], a2 = a.v[2];
  o.re[0] = fma(-a2, c.im[3], fma(-a1, c.re[3], fma(am, c.re[2], o.re[0])));
  o.im[0] = fma(a2, c.re[3], fma(-a1, c.im[3], fma(am, c.im[2], o.im[0])));
  o.re[1] = fma(ap, c.re[3], fma(a2, c.im[2], fma(-a1, c.re[2], o.re[1])));
  o.im[1] = fma(ap, c.im[3], fma(-a2, c.re[2], fma(-a1, c.im[2], o.im[1])));
  o.re[2] = fma(a2, c.im[1], fma(a1, c.re[1], fma(ap, c.re[0], o.re[2])));
  o.im[2] = fma(-a2, c.re[1], fma(a1, c.im[1], fma(ap, c.im[0], o.im[2])));
  o.re[3] = fma(am, c.re[1], fma(-a2, c.im[0], fma(a1, c.re[0], o.re[3])));
  o.im[3] = fma(am, c.im[1], fma(a2, c.re[0], fma(a1, c.im[0], o.im[3])));
}
MF_HD void slash_row_acc(spin& o, const spin& r, const rvec& a) {
  const double am = a.v[0] - a.v[3], ap = a.v[0] + a.v[3], a1 = a.v[1], a2 = a.v[2];
  o.re[0] = fma(-a2, r.im[3], fma(a1, r.re[3], fma(ap, r.re[2], o.re[0])));
  o.im[0] = fma(a2, r.re[3], fma(a1, r.im[3], fma(ap, r.im[2], o.im[0])));
  o.re[1] = fma(am, r.re[3], fma(a2, r.im[2], fma(a1, r.re[2], o.re[1])));
  o.im[1] = fma(am, r.im[3], fma(-a2, r.re[2], fma(a1, r.im[2], o.im[1])));
  o.re[2] = fma(a2, r.im[1], fma(-a1, r.re[1], fma(am, r.re[0], o.re[2])));
  o.im[2] = fma(-a2, r.re[1], fma(-a1, r.im[1], fma(am, r.im[0], o.im[2])));
  o.re[3] = fma(ap, r.re[1], fma(-a2, r.im[0], fma(-a1, r.re[0], o.re[3])));
  o.im[3] = fma(ap, r.im[1], fma(a2, r.re[0], fma(-a1, r.im[0], o.im[3])));
}
MF_HD void spin_acc(spin& acc, const spin& a) {
#pragma unroll
  for (int m = 0; m < 4; ++m) { acc.re[m] += a.re[m]; acc.im[m] += a.im[m]; }
}
// hatted propagators:  -(q-slash + m) psi / (q^2 - m^2)   with idn = 1/(q^2 - m^2) precomputed
MF_HD spin prop_col(const rvec& q, double m, double idn, const spin& c) {
  spin t = slash_col(q, c), o;
#pragma unroll
  for (int k = 0; k < 4; ++k) { o.re[k] = -(t.re[k] + m * c.re[k]) * idn; o.im[k] = -(t.im[k] + m * c.im[k]) * idn; }
  return o;
}
MF_HD spin prop_row(const spin& r, const rvec& q, double m, double idn) {
  spin t = slash_row(r, q), o;
#pragma unroll
  for (int k = 0; k < 4; ++k) { o.re[k] = -(t.re[k] + m * r.re[k]) * idn; o.im[k] = -(t.im[k] + m * r.im[k]) * idn; }
  return o;
}
// row . column (two FMA chains)
MF_HD cplx sdot(const spin& r, const spin& c) {
  cplx o;
  o.re = r.re[0] * c.re[0];
  o.im = r.re[0] * c.im[0];
  o.re = fma(-r.im[0], c.im[0], o.re);
  o.im = fma(r.im[0], c.re[0], o.im);
#pragma unroll
  for (int k = 1; k < 4; ++k) {
    o.re = fma(r.re[k], c.re[k], o.re);
    o.im = fma(r.re[k], c.im[k], o.im);
    o.re = fma(-r.im[k], c.im[k], o.re);
    o.im = fma(r.im[k], c.re[k], o.im);
  }
  return o;
}
// fermion bilinear  c^mu = row gamma^mu col
MF_HD cvec bilinear(const spin& r, const spin& c) {
#define MF_CMUL(RE, IM, a, b)                                   \
  double RE = r.re[a] * c.re[b] - r.im[a] * c.im[b];            \
  double IM = r.re[a] * c.im[b] + r.im[a] * c.re[b];
  MF_CMUL(p02r, p02i, 0, 2) MF_CMUL(p13r, p13i, 1, 3) MF_CMUL(p03r, p03i, 0, 3) MF_CMUL(p12r, p12i, 1, 2)
  MF_CMUL(p20r, p20i, 2, 0) MF_CMUL(p31r, p31i, 3, 1) MF_CMUL(p21r, p21i, 2, 1) MF_CMUL(p30r, p30i, 3, 0)
#undef MF_CMUL
  cvec o;
  o.re[0] = (p02r + p13r) + (p20r + p31r);
  o.im[0] = (p02i + p13i) + (p20i + p31i);
  o.re[1] = (p03r + p12r) - (p21r + p30r);
  o.im[1] = (p03i + p12i) - (p21i + p30i);
  // c^2 = i [ (r1c2 - r0c3) + (r2c1 - r3c0) ]
  double tr = (p12r - p03r) + (p21r - p30r), ti = (p12i - p03i) + (p21i - p30i);
  o.re[2] = -ti;
  o.im[2] = tr;
  o.re[3] = (p02r - p13r) - (p20r - p31r);
  o.im[3] = (p02i - p13i) - (p20i - p31i);
  return o;
}
// Minkowski contraction of a complex with a real vector
MF_HD cplx cdot_r(const cvec& c, const rvec& j) {
  cplx o;
  o.re = c.re[0] * j.v[0] - c.re[1] * j.v[1] - c.re[2] * j.v[2] - c.re[3] * j.v[3];
  o.im = c.im[0] * j.v[0] - c.im[1] * j.v[1] - c.im[2] * j.v[2] - c.im[3] * j.v[3];
  return o;
}
MF_HD cplx cdot_c(const cvec& a, const cvec& b) {
  cplx o = {0.0, 0.0};
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    double sg = m == 0 ? 1.0 : -1.0;
    o.re += sg * (a.re[m] * b.re[m] - a.im[m] * b.im[m]);
    o.im += sg * (a.re[m] * b.im[m] + a.im[m] * b.re[m]);
  }
  return o;
}

// ---- external wavefunctions (a7) ---------------------------------------------------------------------
// u(p, s) column and the row ubar = u^dagger gamma^0; s = 0: xi = (1,0), s = 1: xi = (0,1).
MF_HD spin u_col(const double p[4], double m, int s) {
  double em = p[0] + m, n = 1.0 / sqrt(2.0 * em);
  spin u;
  if (s == 0) {
    // (E+m - p.sigma) xi = (em - pz, -(px + i py));  (E+m + p.sigma) xi = (em + pz, px + i py)
    u.re[0] = n * (em - p[3]); u.im[0] = 0.0;   u.re[1] = -n * p[1]; u.im[1] = -n * p[2];
    u.re[2] = n * (em + p[3]); u.im[2] = 0.0;   u.re[3] = n * p[1];  u.im[3] = n * p[2];
  } else {
    // (E+m - p.sigma) xi = (-(px - i py), em + pz);  (E+m + p.sigma) xi = (px - i py, em - pz)
    u.re[0] = -n * p[1]; u.im[0] = n * p[2];    u.re[1] = n * (em + p[3]); u.im[1] = 0.0;
    u.re[2] = n * p[1];  u.im[2] = -n * p[2];   u.re[3] = n * (em - p[3]); u.im[3] = 0.0;
  }
  return u;
}
MF_HD spin bar_of(const spin& u) {  // psi^dagger gamma^0 = (conj psi_R, conj psi_L)
  spin r;
  r.re[0] = u.re[2]; r.im[0] = -u.im[2]; r.re[1] = u.re[3]; r.im[1] = -u.im[3];
  r.re[2] = u.re[0]; r.im[2] = -u.im[0]; r.re[3] = u.re[1]; r.im[3] = -u.im[1];
  return r;
}
MF_HD spin ubar_row(const double p[4], double m, int s) { return bar_of(u_col(p, m, s)); }
// v(p, s) = ((p.sigma + m) xi; -(p.sigmabar + m) xi) / sqrt(2(E+m))
MF_HD spin v_col(const double p[4], double m, int s) {
  spin v = u_col(p, m, s);
  v.re[2] = -v.re[2]; v.im[2] = -v.im[2]; v.re[3] = -v.re[3]; v.im[3] = -v.im[3];
  return v;
}
// Real transverse polarisation vectors of a massless momentum k (pT > 0 guaranteed by the cuts; the pT = 0
// limit is taken towards the x axis): e1 = (0; kx kz/(|k| pT), ky kz/(|k| pT), -pT/|k|), e2 = (0; -ky/pT, kx/pT, 0).
MF_HD void pol_vectors(const double k[4], rvec& e1, rvec& e2) {
  double pt2 = k[1] * k[1] + k[2] * k[2];
  double pt = sqrt(pt2), pabs = k[0];   // massless: |k| = E
  if (pt > 0.0) {
    double ipt = 1.0 / pt, ip = 1.0 / pabs;
    double cx = k[1] * ipt, cy = k[2] * ipt, cz = k[3] * ip, sz = pt * ip;
    e1.v[0] = 0.0; e1.v[1] = cx * cz; e1.v[2] = cy * cz; e1.v[3] = -sz;
    e2.v[0] = 0.0; e2.v[1] = -cy; e2.v[2] = cx; e2.v[3] = 0.0;
  } else {
    double sg = k[3] >= 0.0 ? 1.0 : -1.0;
    e1.v[0] = 0.0; e1.v[1] = 1.0; e1.v[2] = 0.0; e1.v[3] = 0.0;
    e2.v[0] = 0.0; e2.v[1] = 0.0; e2.v[2] = sg; e2.v[3] = 0.0;
  }
}

}  // namespace mf
