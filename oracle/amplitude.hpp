// ORACLE — TEST INFRASTRUCTURE ONLY (see real.hpp).
//
// amplitude.hpp: steps O9–O11 of SURVEY.md §8(c): external wavefunctions, tree amplitudes and the
// colour sum.  PAPER.md L49, L65-67: matrix elements are built from ALOHA/HELAS wavefunction and vertex
// routines [Murayama, Watanabe, Hagiwara, ref. 22]; "smatrix ... loops over initial and final state
// particle helicities and aggregates their contribution to the final squared amplitude".
// The paper prints no formula; what follows is the textbook QCD/QED Feynman rules written out.
//
// Deliberately different from the CUDA path: DIRAC representation with explicit 4x4 gamma matrices
// (the kernels use two-component chiral spinors), explicit matrix products, amplitudes evaluated by
// the colour-ordered recursion at run time with one memo table per helicity configuration, optional
// linear polarisations and z-axis spin states (the helicity sum is basis independent: a pin), and a
// second, colour-DRESSED brute-force evaluation used as referee.
#pragma once
#include <algorithm>
#include <map>
#include <vector>
#include "real.hpp"

namespace mfo {

template <class R> struct Spinor { Cx<R> c[4]; };
template <class R> struct CVec4 { Cx<R> c[4]; };  // complex Lorentz vector, upper index, (t,x,y,z)
template <class R> struct Mat4 { Cx<R> m[4][4]; };

// Minkowski product, metric (+,-,-,-), no complex conjugation
template <class R> inline Cx<R> mdot(const CVec4<R>& a, const CVec4<R>& b) {
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}
template <class R> inline R mdot_rr(const R a[4], const R b[4]) {
  return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
}
template <class R> inline CVec4<R> cvec_from_real(const R p[4]) {
  CVec4<R> v;
  for (int m = 0; m < 4; ++m) v.c[m] = Cx<R>(p[m]);
  return v;
}

// Dirac representation: gamma^0 = diag(1,1,-1,-1), gamma^i = [[0, sigma^i], [-sigma^i, 0]].
template <class R> inline Mat4<R> gamma_matrix(int mu) {
  Mat4<R> g;
  const Cx<R> one(R(1)), I(R(0), R(1));
  if (mu == 0) {
    g.m[0][0] = one; g.m[1][1] = one; g.m[2][2] = -one; g.m[3][3] = -one;
    return g;
  }
  Cx<R> s[2][2];
  if (mu == 1) { s[0][1] = one; s[1][0] = one; }
  if (mu == 2) { s[0][1] = -I; s[1][0] = I; }
  if (mu == 3) { s[0][0] = one; s[1][1] = -one; }
  for (int a = 0; a < 2; ++a)
    for (int b = 0; b < 2; ++b) { g.m[a][2 + b] = s[a][b]; g.m[2 + a][b] = -s[a][b]; }
  return g;
}
// a-slash = a_mu gamma^mu = a^0 gamma^0 - a^1 gamma^1 - a^2 gamma^2 - a^3 gamma^3
template <class R> inline Mat4<R> slash(const CVec4<R>& a) {
  Mat4<R> out;
  for (int mu = 0; mu < 4; ++mu) {
    Mat4<R> g = gamma_matrix<R>(mu);
    Cx<R> coeff = (mu == 0) ? a.c[0] : -a.c[mu];
    for (int i = 0; i < 4; ++i)
      for (int j = 0; j < 4; ++j) out.m[i][j] += coeff * g.m[i][j];
  }
  return out;
}
template <class R> inline Spinor<R> mat_vec(const Mat4<R>& M, const Spinor<R>& s) {
  Spinor<R> o;
  for (int i = 0; i < 4; ++i)
    for (int j = 0; j < 4; ++j) o.c[i] += M.m[i][j] * s.c[j];
  return o;
}
template <class R> inline Cx<R> row_times_col(const Spinor<R>& row, const Spinor<R>& col) {
  Cx<R> o;
  for (int i = 0; i < 4; ++i) o += row.c[i] * col.c[i];
  return o;
}
// psi-bar = psi^dagger gamma^0 (a row)
template <class R> inline Spinor<R> bar(const Spinor<R>& s) {
  Spinor<R> o;
  o.c[0] = conj(s.c[0]); o.c[1] = conj(s.c[1]); o.c[2] = -conj(s.c[2]); o.c[3] = -conj(s.c[3]);
  return o;
}

// ---------------------------------------------------------------------------------------------
// O9. External wavefunctions.
// Two-spinors: basis 0 = helicity eigenstates chi_lambda(p-hat) (lambda = +1/-1), basis 1 = spin up/down
// along the fixed z axis (then "lambda" just labels the two states).  Both are orthonormal bases, so
// sum_lambda u u-bar = p-slash + m and sum_lambda v v-bar = p-slash - m hold for either.
template <class R> inline void two_spinor(const R p[4], int lambda, int basis, Cx<R> chi[2]) {
  if (basis == 1) {
    chi[0] = Cx<R>(lambda > 0 ? R(1) : R(0));
    chi[1] = Cx<R>(lambda > 0 ? R(0) : R(1));
    return;
  }
  R pabs = r_sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  if (pabs == R(0)) {  // at rest: quantise along z
    chi[0] = Cx<R>(lambda > 0 ? R(1) : R(0));
    chi[1] = Cx<R>(lambda > 0 ? R(0) : R(1));
    return;
  }
  R ppz = pabs + p[3];
  if (p[1] == R(0) && p[2] == R(0) && p[3] < R(0)) {  // along -z
    if (lambda > 0) { chi[0] = Cx<R>(R(0)); chi[1] = Cx<R>(R(1)); }
    else { chi[0] = Cx<R>(R(-1)); chi[1] = Cx<R>(R(0)); }
    return;
  }
  R nrm = R(1) / r_sqrt(R(2) * pabs * ppz);
  if (lambda > 0) { chi[0] = Cx<R>(nrm * ppz); chi[1] = Cx<R>(nrm * p[1], nrm * p[2]); }
  else { chi[0] = Cx<R>(-nrm * p[1], nrm * p[2]); chi[1] = Cx<R>(nrm * ppz); }
}
template <class R> inline void sigma_dot_p(const R p[4], const Cx<R> in[2], Cx<R> out[2]) {
  // sigma.p = [[pz, px - i py], [px + i py, -pz]]
  out[0] = p[3] * in[0] + Cx<R>(p[1], -p[2]) * in[1];
  out[1] = Cx<R>(p[1], p[2]) * in[0] - p[3] * in[1];
}
// u(p, lambda) = ( sqrt(E+m) chi ; sigma.p chi / sqrt(E+m) )      [(p-slash - m) u = 0]
template <class R> inline Spinor<R> u_spinor(const R p[4], R m, int lambda, int basis) {
  Cx<R> chi[2], sp[2];
  two_spinor(p, lambda, basis, chi);
  sigma_dot_p(p, chi, sp);
  R n = r_sqrt(p[0] + m);
  Spinor<R> u;
  u.c[0] = n * chi[0]; u.c[1] = n * chi[1]; u.c[2] = sp[0] / n; u.c[3] = sp[1] / n;
  return u;
}
// v(p, lambda) = ( sigma.p eta / sqrt(E+m) ; sqrt(E+m) eta ), eta = chi_{-lambda}   [(p-slash + m) v = 0]
template <class R> inline Spinor<R> v_spinor(const R p[4], R m, int lambda, int basis) {
  Cx<R> eta[2], sp[2];
  two_spinor(p, -lambda, basis, eta);
  sigma_dot_p(p, eta, sp);
  R n = r_sqrt(p[0] + m);
  Spinor<R> v;
  v.c[0] = sp[0] / n; v.c[1] = sp[1] / n; v.c[2] = n * eta[0]; v.c[3] = n * eta[1];
  return v;
}
// Massless polarisation vectors for momentum p.  Two real unit vectors e1, e2 orthogonal to p-vector
// and to each other, built from the coordinate axis least aligned with p (a construction unlike the
// kernels').  basis 0: circular, eps(lambda) = (-lambda e1 - i e2)/sqrt2; basis 1: linear,
// eps(+1) = e1, eps(-1) = e2.  eps.p = 0, eps.eps* = -1, time component 0.
template <class R> inline CVec4<R> polarisation(const R p[4], int lambda, int basis) {
  R pabs = r_sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  R n[3] = {p[1] / pabs, p[2] / pabs, p[3] / pabs};
  int ax = 0;
  for (int a = 1; a < 3; ++a)
    if (r_fabs(n[a]) < r_fabs(n[ax])) ax = a;
  R axis[3] = {R(0), R(0), R(0)};
  axis[ax] = R(1);
  // e1 = normalise(n x axis), e2 = n x e1
  R e1[3] = {n[1] * axis[2] - n[2] * axis[1], n[2] * axis[0] - n[0] * axis[2], n[0] * axis[1] - n[1] * axis[0]};
  R l = r_sqrt(e1[0] * e1[0] + e1[1] * e1[1] + e1[2] * e1[2]);
  for (int a = 0; a < 3; ++a) e1[a] = e1[a] / l;
  R e2[3] = {n[1] * e1[2] - n[2] * e1[1], n[2] * e1[0] - n[0] * e1[2], n[0] * e1[1] - n[1] * e1[0]};
  CVec4<R> eps;
  if (basis == 1) {
    for (int a = 0; a < 3; ++a) eps.c[a + 1] = Cx<R>(lambda > 0 ? e1[a] : e2[a]);
  } else {
    R rs = R(1) / r_sqrt(R(2));
    for (int a = 0; a < 3; ++a) eps.c[a + 1] = Cx<R>(-R(lambda) * e1[a] * rs, -e2[a] * rs);
  }
  return eps;
}
template <class R> inline CVec4<R> cconj(const CVec4<R>& v) {
  CVec4<R> o;
  for (int m = 0; m < 4; ++m) o.c[m] = conj(v.c[m]);
  return o;
}

// ---------------------------------------------------------------------------------------------
// O10 (C0). e-(p1) e+(p2) -> mu-(p3) mu+(p4), s-channel photon only (BASELINE.json configs[0]):
// iM = [v-bar(p2) (i e gamma^mu) u(p1)] (-i g_{mu nu}/s) [u-bar(p3) (i e gamma^nu) v(p4)].
// Returns (1/4) sum over the 16 helicity combinations of |M|^2; per-helicity |M|^2 in out16 if given.
template <class R>
inline R me2_ee_mumu(const R mom[4][4], R alpha_em, int basis, R* out16) {
  R e2 = R(4) * r_pi<R>() * alpha_em;  // e^2
  R P[4];
  for (int m = 0; m < 4; ++m) P[m] = mom[0][m] + mom[1][m];
  R s = mdot_rr(P, P);
  R total = R(0);
  int idx = 0;
  for (int l1 = -1; l1 <= 1; l1 += 2)
    for (int l2 = -1; l2 <= 1; l2 += 2)
      for (int l3 = -1; l3 <= 1; l3 += 2)
        for (int l4 = -1; l4 <= 1; l4 += 2) {
          Spinor<R> u1 = u_spinor(mom[0], R(0), l1, basis), v2b = bar(v_spinor(mom[1], R(0), l2, basis));
          Spinor<R> u3b = bar(u_spinor(mom[2], R(0), l3, basis)), v4 = v_spinor(mom[3], R(0), l4, basis);
          CVec4<R> je, jm;  // the two fermion currents, upper index
          for (int mu = 0; mu < 4; ++mu) {
            Mat4<R> g = gamma_matrix<R>(mu);
            je.c[mu] = row_times_col(v2b, mat_vec(g, u1));
            jm.c[mu] = row_times_col(u3b, mat_vec(g, v4));
          }
          // i e * (-i/s) * i e = i e^2 / s
          Cx<R> M = cx_i<R>() * (mdot(je, jm) * (e2 / s));
          R m2 = norm2(M);
          if (out16) out16[idx] = m2;
          ++idx;
          total = total + m2;
        }
  return total / R(4);
}

// ---------------------------------------------------------------------------------------------
// O10 (C1-C3). g g -> t t-bar + (ng-2) g.  All gluon momenta are taken INCOMING: P[0], P[1] are the
// beams, P[i>=2] = -k_i of the outgoing gluons, whose polarisation enters complex conjugated.
// Colour decomposition: iM_ij = sum_{sigma in S_ng} (T^{a_sigma1} ... T^{a_sigma_ng})_ij A(sigma).
//
// Colour-ordered rules (from the Feynman rules with T^a = lambda^a/2, [T^a,T^b] = i f^{abc} T^c):
//   ordered gluon current   J(i1..ik) = (-i/P^2) [ sum_j (-i gs) V3(J(i1..ij), J(ij+1..ik))
//                                                + sum_{j<l} (i gs^2) V4(J(i1..ij), J(ij+1..il), J(il+1..ik)) ]
//   V3^r(J1,P1;J2,P2) = (J1.J2)(P1-P2)^r + J2^r ((P2-Q).J1) + J1^r ((Q-P1).J2),  Q = -(P1+P2)
//   V4^r(J1,J2,J3)    = 2 (J1.J3) J2^r - (J2.J3) J1^r - (J1.J2) J3^r
//   ordered quark current   X() = v(p4);  X(i1..ik) = i (q-slash + m)/(q^2 - m^2) sum_j (i gs) J-slash(i1..ij) X(ij+1..ik),
//                           q = -p4 + P_{i1..ik}
//   A(sigma) = u-bar(p3) sum_j (i gs) J-slash(sigma1..sigmaj) X(sigmaj+1..sigma_ng)
template <class R> struct AmpContext {
  int ng = 0;
  R P[6][4];         // incoming gluon momenta
  CVec4<R> eps[6];   // external gluon wavefunctions (already conjugated for outgoing gluons)
  R p3[4], p4[4];    // t, t-bar (outgoing)
  Spinor<R> ubar3, v4;
  R mt = R(0), gs = R(0);
  std::map<uint32_t, CVec4<R>> memoJ;
  std::map<uint32_t, Spinor<R>> memoX;
};
inline uint32_t seq_key(const int* seq, int len) {
  uint32_t k = 1;
  for (int i = 0; i < len; ++i) k = k * 8u + (uint32_t)seq[i];
  return k;
}
template <class R> inline void seq_momentum(const AmpContext<R>& c, const int* seq, int len, R out[4]) {
  for (int m = 0; m < 4; ++m) out[m] = R(0);
  for (int i = 0; i < len; ++i)
    for (int m = 0; m < 4; ++m) out[m] = out[m] + c.P[seq[i]][m];
}
template <class R>
inline CVec4<R> vertex3(const CVec4<R>& J1, const R P1[4], const CVec4<R>& J2, const R P2[4]) {
  R Q[4], d12[4], d2q[4], dq1[4];
  for (int m = 0; m < 4; ++m) {
    Q[m] = -(P1[m] + P2[m]);
    d12[m] = P1[m] - P2[m];
    d2q[m] = P2[m] - Q[m];
    dq1[m] = Q[m] - P1[m];
  }
  Cx<R> j12 = mdot(J1, J2), a = mdot(cvec_from_real(d2q), J1), b = mdot(cvec_from_real(dq1), J2);
  CVec4<R> o;
  for (int m = 0; m < 4; ++m) o.c[m] = j12 * d12[m] + J2.c[m] * a + J1.c[m] * b;
  return o;
}
template <class R> inline CVec4<R> vertex4(const CVec4<R>& J1, const CVec4<R>& J2, const CVec4<R>& J3) {
  Cx<R> j13 = mdot(J1, J3), j23 = mdot(J2, J3), j12 = mdot(J1, J2);
  CVec4<R> o;
  for (int m = 0; m < 4; ++m) o.c[m] = R(2) * (j13 * J2.c[m]) - j23 * J1.c[m] - j12 * J3.c[m];
  return o;
}
template <class R> CVec4<R> gluon_current(AmpContext<R>& c, const int* seq, int len) {
  if (len == 1) return c.eps[seq[0]];
  uint32_t key = seq_key(seq, len);
  auto it = c.memoJ.find(key);
  if (it != c.memoJ.end()) return it->second;
  CVec4<R> sum;
  const Cx<R> I = cx_i<R>();
  for (int j = 1; j < len; ++j) {  // three-gluon vertex: split seq = [0,j) + [j,len)
    R P1[4], P2[4];
    seq_momentum(c, seq, j, P1);
    seq_momentum(c, seq + j, len - j, P2);
    CVec4<R> v = vertex3(gluon_current(c, seq, j), P1, gluon_current(c, seq + j, len - j), P2);
    Cx<R> f = -(I * c.gs);
    for (int m = 0; m < 4; ++m) sum.c[m] += f * v.c[m];
  }
  for (int j = 1; j < len; ++j)  // four-gluon vertex: [0,j) + [j,l) + [l,len)
    for (int l = j + 1; l < len; ++l) {
      CVec4<R> v = vertex4(gluon_current(c, seq, j), gluon_current(c, seq + j, l - j), gluon_current(c, seq + l, len - l));
      Cx<R> f = I * (c.gs * c.gs);
      for (int m = 0; m < 4; ++m) sum.c[m] += f * v.c[m];
    }
  R P[4];
  seq_momentum(c, seq, len, P);
  R P2 = mdot_rr(P, P);
  CVec4<R> out;
  for (int m = 0; m < 4; ++m) out.c[m] = (-I) * (sum.c[m] / P2);
  c.memoJ[key] = out;
  return out;
}
template <class R> Spinor<R> quark_current(AmpContext<R>& c, const int* seq, int len) {
  if (len == 0) return c.v4;
  uint32_t key = seq_key(seq, len);
  auto it = c.memoX.find(key);
  if (it != c.memoX.end()) return it->second;
  const Cx<R> I = cx_i<R>();
  Spinor<R> sum;
  for (int j = 1; j <= len; ++j) {
    Spinor<R> t = mat_vec(slash(gluon_current(c, seq, j)), quark_current(c, seq + j, len - j));
    for (int a = 0; a < 4; ++a) sum.c[a] += (I * c.gs) * t.c[a];
  }
  R q[4], Pq[4];
  seq_momentum(c, seq, len, Pq);
  for (int m = 0; m < 4; ++m) q[m] = Pq[m] - c.p4[m];
  R den = mdot_rr(q, q) - c.mt * c.mt;
  Mat4<R> num = slash(cvec_from_real(q));
  for (int a = 0; a < 4; ++a) num.m[a][a] += Cx<R>(c.mt);
  Spinor<R> t = mat_vec(num, sum), out;
  for (int a = 0; a < 4; ++a) out.c[a] = I * (t.c[a] / den);
  c.memoX[key] = out;
  return out;
}
template <class R> Cx<R> ordered_amplitude(AmpContext<R>& c, const int* sigma) {
  const Cx<R> I = cx_i<R>();
  Cx<R> A;
  for (int j = 1; j <= c.ng; ++j) {
    Spinor<R> t = mat_vec(slash(gluon_current(c, sigma, j)), quark_current(c, sigma + j, c.ng - j));
    A += (I * c.gs) * row_times_col(c.ubar3, t);
  }
  return A;
}

// Permutations of 0..n-1 in lexicographic order; this fixes the row/column order of the colour matrix.
inline std::vector<std::vector<int>> permutations(int n) {
  std::vector<int> p(n);
  for (int i = 0; i < n; ++i) p[i] = i;
  std::vector<std::vector<int>> out;
  do out.push_back(p); while (std::next_permutation(p.begin(), p.end()));
  return out;
}

// ---------------------------------------------------------------------------------------------
// O11. Colour matrix  C_{sigma sigma'} = sum_{a_1..a_n} Tr( T^{a_sigma1}..T^{a_sigman} T^{a_sigma'n}..T^{a_sigma'1} )
// by brute force from the Gell-Mann matrices: for every colour assignment build M_sigma = prod T and add
// Tr(M_sigma M_sigma'^dagger) (T hermitian).
template <class R> struct Mat3 { Cx<R> m[3][3]; };
template <class R> inline Mat3<R> mat3_mul(const Mat3<R>& a, const Mat3<R>& b) {
  Mat3<R> o;
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      for (int k = 0; k < 3; ++k) o.m[i][j] += a.m[i][k] * b.m[k][j];
  return o;
}
template <class R> inline Mat3<R> su3_generator(int a) {  // T^a = lambda^a / 2, a = 0..7
  Mat3<R> t;
  const R h = R(0.5);
  const Cx<R> I(R(0), R(1));
  switch (a) {
    case 0: t.m[0][1] = h; t.m[1][0] = h; break;
    case 1: t.m[0][1] = -(I * h); t.m[1][0] = I * h; break;
    case 2: t.m[0][0] = h; t.m[1][1] = -h; break;
    case 3: t.m[0][2] = h; t.m[2][0] = h; break;
    case 4: t.m[0][2] = -(I * h); t.m[2][0] = I * h; break;
    case 5: t.m[1][2] = h; t.m[2][1] = h; break;
    case 6: t.m[1][2] = -(I * h); t.m[2][1] = I * h; break;
    case 7: {
      R s = R(1) / (R(2) * r_sqrt(R(3)));
      t.m[0][0] = s; t.m[1][1] = s; t.m[2][2] = -(R(2) * s);
      break;
    }
  }
  return t;
}
// M(a) = T^{a_0} T^{a_1} .. T^{a_{n-1}} for all 8^n colour assignments a (code = sum_i a_i 8^i)
template <class R> inline std::vector<Mat3<R>> colour_product_table(int n) {
  Mat3<R> T[8];
  for (int a = 0; a < 8; ++a) T[a] = su3_generator<R>(a);
  int ncol = 1;
  for (int i = 0; i < n; ++i) ncol *= 8;
  std::vector<Mat3<R>> M(ncol);
  for (int code = 0; code < ncol; ++code) {
    int a[6] = {0, 0, 0, 0, 0, 0}, cc = code;
    for (int i = 0; i < n; ++i) { a[i] = cc % 8; cc /= 8; }
    Mat3<R> prod = T[a[0]];
    for (int i = 1; i < n; ++i) prod = mat3_mul(prod, T[a[i]]);
    M[code] = prod;
  }
  return M;
}
// sum_a Tr( M(a o sigma) M(a o tau)^dagger ), (a o sigma)_i = a_{sigma(i)}: the DEFINITION of C_{sigma tau}, with the matrix
// products looked up in the table (M_sigma(a) = T^{a_sigma(0)} .. T^{a_sigma(n-1)} = M(a o sigma))
template <class R> inline R colour_sum_with_table(int n, const std::vector<Mat3<R>>& M, const int* sigma, const int* tau) {
  int ncol = (int)M.size();
  R total = R(0);
  for (int code = 0; code < ncol; ++code) {
    int a[6], cc = code;
    for (int i = 0; i < n; ++i) { a[i] = cc % 8; cc /= 8; }
    int cs = 0, ct = 0, pw = 1;
    for (int i = 0; i < n; ++i) { cs += a[sigma[i]] * pw; ct += a[tau[i]] * pw; pw *= 8; }
    const Mat3<R>&A = M[cs], &B = M[ct];
    Cx<R> tr;
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) tr += A.m[i][j] * conj(B.m[i][j]);
    total = total + tr.re;
  }
  return total;
}
template <class R> inline R colour_matrix_entry(int n, const int* sigma, const int* tau) {
  std::vector<Mat3<R>> M = colour_product_table<R>(n);
  return colour_sum_with_table<R>(n, M, sigma, tau);
}
template <class R> inline std::vector<R> colour_matrix(int n) {
  auto perms = permutations(n);
  int np = (int)perms.size();
  std::vector<R> C(np * np, R(0));
  if (n >= 5) {
    // 120 x 120 entries over 8^5 colour assignments: the sum over all colour assignments is invariant under relabelling
    // the summation indices, a -> a o sigma^-1, hence C_{sigma tau} = C_{id, sigma^-1 o tau}: one row from the definition
    // (colour_sum_with_table), the others by lookup.  tests/ pins this against the definition entry by entry (n <= 4: all
    // entries against the plain loop below; n = 5: sampled entries against colour_matrix_entry).
    std::vector<Mat3<R>> M = colour_product_table<R>(n);
    std::map<std::vector<int>, int> index;
    for (int s = 0; s < np; ++s) index[perms[s]] = s;
    std::vector<R> row(np);
    for (int t = 0; t < np; ++t) row[t] = colour_sum_with_table<R>(n, M, perms[0].data(), perms[t].data());
    for (int s = 0; s < np; ++s) {
      std::vector<int> inv(n);
      for (int i = 0; i < n; ++i) inv[perms[s][i]] = i;
      for (int t = 0; t < np; ++t) {
        std::vector<int> rho(n);
        for (int i = 0; i < n; ++i) rho[i] = inv[perms[t][i]];
        C[s * np + t] = row[index[rho]];
      }
    }
    return C;
  }
  Mat3<R> T[8];
  for (int a = 0; a < 8; ++a) T[a] = su3_generator<R>(a);
  int ncol = 1;
  for (int i = 0; i < n; ++i) ncol *= 8;
  std::vector<Mat3<R>> M(np);
  for (int code = 0; code < ncol; ++code) {
    int a[6], cc = code;
    for (int i = 0; i < n; ++i) { a[i] = cc % 8; cc /= 8; }
    for (int s = 0; s < np; ++s) {
      Mat3<R> prod = T[a[perms[s][0]]];
      for (int i = 1; i < n; ++i) prod = mat3_mul(prod, T[a[perms[s][i]]]);
      M[s] = prod;
    }
    for (int s = 0; s < np; ++s)
      for (int t = 0; t < np; ++t) {
        Cx<R> tr;
        for (int i = 0; i < 3; ++i)
          for (int j = 0; j < 3; ++j) tr += M[s].m[i][j] * conj(M[t].m[i][j]);
        C[s * np + t] = C[s * np + t] + tr.re;
      }
  }
  return C;
}

// ---------------------------------------------------------------------------------------------
// O10 (quark channel, "pp -> ttbar": the q qbar diagram beside the three gg ones).
// q(p1, colour i) qbar(p2, colour j) -> t(p3, colour k) tbar(p4, colour l), massless q, s-channel gluon only:
//   iM = [v-bar(p2) (i g T^a_{ji} gamma^mu) u(p1)] (-i g_{mu nu} delta^{ab} / s) [u-bar(p3) (i g T^b_{kl} gamma^nu) v(p4)]
// Returns (1/4)(1/9) sum over helicities and colours of |M|^2.  The colour sum
//   sum_{ijkl} | sum_a T^a_{ji} T^a_{kl} |^2
// is evaluated from the explicit generators, not typed in.
template <class R>
inline R me2_qq_ttbar(const R mom[4][4], R mt, R alpha_s, int basis) {
  R g2 = R(4) * r_pi<R>() * alpha_s;
  R P[4];
  for (int m = 0; m < 4; ++m) P[m] = mom[0][m] + mom[1][m];
  R s = mdot_rr(P, P);
  R colour = R(0);
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j)
      for (int k = 0; k < 3; ++k)
        for (int l = 0; l < 3; ++l) {
          Cx<R> c;
          for (int a = 0; a < 8; ++a) {
            Mat3<R> T = su3_generator<R>(a);
            c += T.m[j][i] * T.m[k][l];
          }
          colour = colour + norm2(c);
        }
  R total = R(0);
  for (int l1 = -1; l1 <= 1; l1 += 2)
    for (int l2 = -1; l2 <= 1; l2 += 2)
      for (int l3 = -1; l3 <= 1; l3 += 2)
        for (int l4 = -1; l4 <= 1; l4 += 2) {
          Spinor<R> u1 = u_spinor(mom[0], R(0), l1, basis), v2b = bar(v_spinor(mom[1], R(0), l2, basis));
          Spinor<R> u3b = bar(u_spinor(mom[2], mt, l3, basis)), v4 = v_spinor(mom[3], mt, l4, basis);
          CVec4<R> jq, jt;
          for (int mu = 0; mu < 4; ++mu) {
            Mat4<R> g = gamma_matrix<R>(mu);
            jq.c[mu] = row_times_col(v2b, mat_vec(g, u1));
            jt.c[mu] = row_times_col(u3b, mat_vec(g, v4));
          }
          Cx<R> M = cx_i<R>() * (mdot(jq, jt) * (g2 / s));   // i g * (-i / s) * i g, colour factor apart
          total = total + norm2(M);
        }
  return total * colour / R(36);
}

// ---------------------------------------------------------------------------------------------
// Helicity-summed, colour-summed, averaged |M|^2 for g g -> t tbar (ng-2) g   (O10 + O11).
// mom = [g_a, g_b, t, tbar, g_1.., ] physical momenta (beams incoming, the rest outgoing).
// |M|^2_avg = 1/(4 * 64 * (ng-2)!) sum_h A_h^dagger C A_h.
// basis: bit 0 = spinor basis (0 helicity, 1 z-spin), bit 1 = polarisation basis (0 circular, 1 linear).
// subst_gluon >= 0 replaces that gluon's polarisation by its momentum (gauge-invariance pin).
// If amps_out != nullptr it receives A(sigma) for every helicity: [hel][perm][re,im], hel index =
// bits (lt, ltbar, l_g0.. l_g{ng-1}) with bit set meaning lambda = +1, lt the MOST significant.
template <class R> inline void setup_context(AmpContext<R>& c, int ng, const R mom[][4], R mt, R gs) {
  c.ng = ng;
  c.mt = mt;
  c.gs = gs;
  for (int m = 0; m < 4; ++m) {
    c.P[0][m] = mom[0][m];
    c.P[1][m] = mom[1][m];
    c.p3[m] = mom[2][m];
    c.p4[m] = mom[3][m];
    for (int g = 2; g < ng; ++g) c.P[g][m] = -mom[2 + g][m];
  }
}
template <class R>
inline R me2_gg_ttbar_ng(int ng, const R mom[][4], R mt, R alpha_s, int basis, int subst_gluon,
                         const std::vector<R>& C, R* amps_out) {
  AmpContext<R> c;
  R gs = r_sqrt(R(4) * r_pi<R>() * alpha_s);
  setup_context(c, ng, mom, mt, gs);
  auto perms = permutations(ng);
  int np = (int)perms.size();
  int sb = basis & 1, pb = (basis >> 1) & 1;
  R total = R(0);
  int nhel = 4 << ng;
  for (int h = 0; h < nhel; ++h) {
    int lt = ((h >> (ng + 1)) & 1) ? 1 : -1, ltb = ((h >> ng) & 1) ? 1 : -1;
    c.ubar3 = bar(u_spinor(c.p3, mt, lt, sb));
    c.v4 = v_spinor(c.p4, mt, ltb, sb);
    for (int g = 0; g < ng; ++g) {
      int lg = ((h >> (ng - 1 - g)) & 1) ? 1 : -1;
      if (g < 2) c.eps[g] = polarisation(c.P[g], lg, pb);
      else c.eps[g] = cconj(polarisation(mom[2 + g], lg, pb));
      if (g == subst_gluon) c.eps[g] = cvec_from_real(c.P[g]);
    }
    c.memoJ.clear();
    c.memoX.clear();
    std::vector<Cx<R>> A(np);
    for (int s = 0; s < np; ++s) {
      A[s] = ordered_amplitude(c, perms[s].data());
      if (amps_out) { amps_out[(h * np + s) * 2] = A[s].re; amps_out[(h * np + s) * 2 + 1] = A[s].im; }
    }
    for (int s = 0; s < np; ++s)
      for (int t = 0; t < np; ++t) total = total + C[s * np + t] * (conj(A[s]) * A[t]).re;
  }
  R ident = R(1);
  for (int j = 2; j <= ng - 2; ++j) ident = ident * R(j);
  return total / (R(4) * R(64) * ident);
}

// ---------------------------------------------------------------------------------------------
// Referee: colour-DRESSED recursion with explicit adjoint and fundamental indices (O10, first bullet).
// External gluon g carries colour col[g]; quark colour i (row), antiquark colour j.  Returns iM_ij.
template <class R> struct DressedCurrent { CVec4<R> a[8]; };  // J^{a mu}
template <class R> struct DressedQuark { Spinor<R> c[3]; };    // fundamental index x spinor
template <class R> inline R structure_constant(int a, int b, int c) {
  // f^{abc} = -2i Tr([T^a,T^b] T^c)
  Mat3<R> A = su3_generator<R>(a), B = su3_generator<R>(b), Cc = su3_generator<R>(c);
  Mat3<R> AB = mat3_mul(A, B), BA = mat3_mul(B, A);
  Cx<R> tr;
  for (int i = 0; i < 3; ++i)
    for (int k = 0; k < 3; ++k) tr += (AB.m[i][k] - BA.m[i][k]) * Cc.m[k][i];
  Cx<R> f = Cx<R>(R(0), R(-2)) * tr;
  return f.re;
}
template <class R> struct DressedContext {
  AmpContext<R> base;
  int col[6];
  R f[8][8][8];
  Mat3<R> T[8];
  std::map<uint32_t, DressedCurrent<R>> memoJ;
  std::map<uint32_t, DressedQuark<R>> memoX;
};
template <class R> inline void subset_momentum(const AmpContext<R>& c, uint32_t S, R out[4]) {
  for (int m = 0; m < 4; ++m) out[m] = R(0);
  for (int g = 0; g < c.ng; ++g)
    if (S & (1u << g))
      for (int m = 0; m < 4; ++m) out[m] = out[m] + c.P[g][m];
}
template <class R> DressedCurrent<R> dressed_gluon(DressedContext<R>& d, uint32_t S) {
  auto it = d.memoJ.find(S);
  if (it != d.memoJ.end()) return it->second;
  DressedCurrent<R> out;
  if ((S & (S - 1)) == 0) {  // single gluon
    int g = 0;
    while (!(S & (1u << g))) ++g;
    out.a[d.col[g]] = d.base.eps[g];
    d.memoJ[S] = out;
    return out;
  }
  const Cx<R> I = cx_i<R>();
  R gs = d.base.gs;
  DressedCurrent<R> sum;
  // three-gluon vertices: unordered pairs {S1, S2}, S1 contains the lowest set bit
  uint32_t low = S & (~S + 1);
  for (uint32_t S1 = (S - 1) & S; S1; S1 = (S1 - 1) & S) {
    if (!(S1 & low)) continue;
    uint32_t S2 = S ^ S1;
    if (!S2) continue;
    DressedCurrent<R> J1 = dressed_gluon(d, S1), J2 = dressed_gluon(d, S2);
    R P1[4], P2[4];
    subset_momentum(d.base, S1, P1);
    subset_momentum(d.base, S2, P2);
    for (int a = 0; a < 8; ++a)
      for (int b = 0; b < 8; ++b) {
        CVec4<R> v = vertex3(J1.a[a], P1, J2.a[b], P2);
        for (int cidx = 0; cidx < 8; ++cidx) {
          R fabc = d.f[a][b][cidx];
          if (fabc == R(0)) continue;
          for (int m = 0; m < 4; ++m) sum.a[cidx].c[m] += (gs * fabc) * v.c[m];
        }
      }
  }
  // four-gluon vertices: unordered triples {S1, S2, S3}
  for (uint32_t S1 = (S - 1) & S; S1; S1 = (S1 - 1) & S) {
    if (!(S1 & low)) continue;
    uint32_t rest = S ^ S1;
    uint32_t low2 = rest & (~rest + 1);
    for (uint32_t S2 = (rest - 1) & rest; S2; S2 = (S2 - 1) & rest) {
      if (!(S2 & low2)) continue;
      uint32_t S3 = rest ^ S2;
      if (!S3) continue;
      DressedCurrent<R> J1 = dressed_gluon(d, S1), J2 = dressed_gluon(d, S2), J3 = dressed_gluon(d, S3);
      for (int a = 0; a < 8; ++a)
        for (int b = 0; b < 8; ++b)
          for (int cc = 0; cc < 8; ++cc) {
            Cx<R> j12 = mdot(J1.a[a], J2.a[b]), j13 = mdot(J1.a[a], J3.a[cc]), j23 = mdot(J2.a[b], J3.a[cc]);
            for (int dd = 0; dd < 8; ++dd) {
              R c1 = R(0), c2 = R(0), c3 = R(0);  // f^{abe}f^{cde}, f^{ace}f^{bde}, f^{ade}f^{bce}
              for (int e = 0; e < 8; ++e) {
                c1 = c1 + d.f[a][b][e] * d.f[cc][dd][e];
                c2 = c2 + d.f[a][cc][e] * d.f[b][dd][e];
                c3 = c3 + d.f[a][dd][e] * d.f[b][cc][e];
              }
              if (c1 == R(0) && c2 == R(0) && c3 == R(0)) continue;
              for (int m = 0; m < 4; ++m) {
                Cx<R> t = c1 * (j13 * J2.a[b].c[m] - j23 * J1.a[a].c[m]) +
                          c2 * (j12 * J3.a[cc].c[m] - j23 * J1.a[a].c[m]) +
                          c3 * (j12 * J3.a[cc].c[m] - j13 * J2.a[b].c[m]);
                sum.a[dd].c[m] += (-(I * (gs * gs))) * t;
              }
            }
          }
    }
  }
  R P[4];
  subset_momentum(d.base, S, P);
  R P2 = mdot_rr(P, P);
  for (int a = 0; a < 8; ++a)
    for (int m = 0; m < 4; ++m) out.a[a].c[m] = (-I) * (sum.a[a].c[m] / P2);
  d.memoJ[S] = out;
  return out;
}
// sum over non-empty S1 subset of S of (i gs gamma_mu T^a) J_{S1}^{a mu} X_{S \ S1}
template <class R> DressedQuark<R> dressed_quark(DressedContext<R>& d, uint32_t S, int jcol);
template <class R> DressedQuark<R> dressed_attach(DressedContext<R>& d, uint32_t S, int jcol) {
  const Cx<R> I = cx_i<R>();
  DressedQuark<R> sum;
  for (uint32_t S1 = S; S1; S1 = (S1 - 1) & S) {
    DressedCurrent<R> J = dressed_gluon(d, S1);
    DressedQuark<R> X = dressed_quark(d, S ^ S1, jcol);
    for (int a = 0; a < 8; ++a) {
      Mat4<R> Js = slash(J.a[a]);
      for (int i2 = 0; i2 < 3; ++i2) {
        Spinor<R> t = mat_vec(Js, X.c[i2]);
        for (int i1 = 0; i1 < 3; ++i1) {
          Cx<R> tc = d.T[a].m[i1][i2];
          if (tc.re == R(0) && tc.im == R(0)) continue;
          for (int s = 0; s < 4; ++s) sum.c[i1].c[s] += (I * d.base.gs) * (tc * t.c[s]);
        }
      }
    }
  }
  return sum;
}
template <class R> DressedQuark<R> dressed_quark(DressedContext<R>& d, uint32_t S, int jcol) {
  if (S == 0) {
    DressedQuark<R> x;
    x.c[jcol] = d.base.v4;
    return x;
  }
  auto it = d.memoX.find(S);
  if (it != d.memoX.end()) return it->second;
  const Cx<R> I = cx_i<R>();
  DressedQuark<R> sum = dressed_attach(d, S, jcol), out;
  R q[4], Pq[4];
  subset_momentum(d.base, S, Pq);
  for (int m = 0; m < 4; ++m) q[m] = Pq[m] - d.base.p4[m];
  R den = mdot_rr(q, q) - d.base.mt * d.base.mt;
  Mat4<R> num = slash(cvec_from_real(q));
  for (int a = 0; a < 4; ++a) num.m[a][a] += Cx<R>(d.base.mt);
  for (int i = 0; i < 3; ++i) {
    Spinor<R> t = mat_vec(num, sum.c[i]);
    for (int s = 0; s < 4; ++s) out.c[i].c[s] = I * (t.c[s] / den);
  }
  d.memoX[S] = out;
  return out;
}
// iM_{icol jcol} for the helicities and colours loaded in d
template <class R> Cx<R> dressed_amplitude(DressedContext<R>& d, int icol, int jcol) {
  d.memoJ.clear();
  d.memoX.clear();
  uint32_t all = (1u << d.base.ng) - 1u;
  DressedQuark<R> s = dressed_attach(d, all, jcol);
  return row_times_col(d.base.ubar3, s.c[icol]);
}
template <class R> inline void dressed_init(DressedContext<R>& d) {
  for (int a = 0; a < 8; ++a) d.T[a] = su3_generator<R>(a);
  for (int a = 0; a < 8; ++a)
    for (int b = 0; b < 8; ++b)
      for (int c = 0; c < 8; ++c) {
        R f = structure_constant<R>(a, b, c);
        if (r_fabs(f) < R(1e-14)) f = R(0);
        d.f[a][b][c] = f;
      }
}

// ---------------------------------------------------------------------------------------------
// O10 (quark channels with one gluon, "pp -> ttbar g (36 diagrams)": 16 gg + 5 for each
// of q qbar -> ttbar g, q g -> ttbar q, ...; R19).
//
// One massless quark line, the top line and one external gluon; the five tree diagrams written out from the Feynman
// rules (quark-gluon vertex i g gamma^mu T^a, fermion propagator i (pslash + m)/(p^2 - m^2), gluon propagator
// -i g_{mu nu} delta^{ab}/q^2, three-gluon vertex g f^{abc} [g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu +
// g^{rho mu}(k3-k1)^nu], all momenta incoming), for explicit colours.
// The light line is given by its column spinor C with fermion-flow momentum pc INTO the line and its row spinor Rw with
// flow momentum pr OUT of it; the gluon by its wavefunction E and OUTGOING momentum kg:
//   q(p1) qbar(p2) -> t tbar g(k5):  C = u(p1), pc = p1;  Rw = vbar(p2), pr = -p2;  E = eps*(k5), kg = k5
//   q(p1) g(p2) -> t tbar q(p5):     C = u(p1), pc = p1;  Rw = ubar(p5), pr = p5;   E = eps(p2),   kg = -p2
// kin[0..4] = the colour-stripped amplitudes of the diagrams (gluon from the light line before / after the virtual
// gluon, from the top, from the antitop, three-gluon vertex), with all factors of i and g included.
template <class R> inline Mat4<R> slash_plus_mass(const R p[4], R m) {
  Mat4<R> M = slash(cvec_from_real(p));
  for (int i = 0; i < 4; ++i) M.m[i][i] += Cx<R>(m);
  return M;
}
template <class R> inline Spinor<R> row_times_mat(const Spinor<R>& row, const Mat4<R>& M) {
  Spinor<R> o;
  for (int j = 0; j < 4; ++j)
    for (int i = 0; i < 4; ++i) o.c[j] += row.c[i] * M.m[i][j];
  return o;
}
template <class R>
inline void light_line_ttbar_g_diagrams(const Spinor<R>& Rw, const R pr[4], const Spinor<R>& C, const R pc[4],
                                        const Spinor<R>& ub3, const R p3[4], const Spinor<R>& v4, const R p4[4],
                                        const CVec4<R>& E, const R kg[4], R mt, R g, Cx<R> kin[5]) {
  const Cx<R> I = cx_i<R>();
  R ql[4], qt[4], a1[4], a2[4], t1[4], t2[4];
  for (int m = 0; m < 4; ++m) {
    ql[m] = pc[m] - pr[m];            // virtual gluon leaving the light line when the gluon is not emitted from it
    qt[m] = p3[m] + p4[m];            // virtual gluon entering the top line when the gluon is not emitted from it
    a1[m] = pc[m] - kg[m];            // light-line propagator, emission on the incoming side
    a2[m] = pr[m] + kg[m];            // light-line propagator, emission on the outgoing side
    t1[m] = p3[m] + kg[m];            // top propagator, emission from the top
    t2[m] = -p4[m] - kg[m];           // top propagator, emission from the antitop
  }
  const R sl = mdot_rr(ql, ql), st = mdot_rr(qt, qt);
  const Mat4<R> Es = slash(E);
  const Cx<R> vert3 = (I * g) * (I * g) * (I * g);      // three quark-gluon vertices
  const Cx<R> fprop = I, gprop = -I;
  // currents with an open Lorentz index
  CVec4<R> jl, jt, jlA, jlB, jtC, jtD;
  const Spinor<R> lineA = mat_vec(slash_plus_mass(a1, R(0)), mat_vec(Es, C));        // (a1-slash) E-slash C
  const Spinor<R> rowB = row_times_mat(row_times_mat(Rw, Es), slash_plus_mass(a2, R(0)));
  const Spinor<R> rowC = row_times_mat(row_times_mat(ub3, Es), slash_plus_mass(t1, mt));
  const Spinor<R> colD = mat_vec(slash_plus_mass(t2, mt), mat_vec(Es, v4));
  for (int mu = 0; mu < 4; ++mu) {
    const Mat4<R> gm = gamma_matrix<R>(mu);
    jl.c[mu] = row_times_col(Rw, mat_vec(gm, C));
    jt.c[mu] = row_times_col(ub3, mat_vec(gm, v4));
    jlA.c[mu] = row_times_col(Rw, mat_vec(gm, lineA));
    jlB.c[mu] = row_times_col(rowB, mat_vec(gm, C));
    jtC.c[mu] = row_times_col(rowC, mat_vec(gm, v4));
    jtD.c[mu] = row_times_col(ub3, mat_vec(gm, colD));
  }
  const R dA = mdot_rr(a1, a1), dB = mdot_rr(a2, a2), dC = mdot_rr(t1, t1) - mt * mt, dD = mdot_rr(t2, t2) - mt * mt;
  kin[0] = vert3 * fprop * gprop * mdot(jlA, jt) / (dA * st);
  kin[1] = vert3 * fprop * gprop * mdot(jlB, jt) / (dB * st);
  kin[2] = vert3 * fprop * gprop * mdot(jl, jtC) / (dC * sl);
  kin[3] = vert3 * fprop * gprop * mdot(jl, jtD) / (dD * sl);
  // three-gluon vertex with incoming momenta k1 = ql (index mu, from the light line), k2 = -qt (index nu, to the top
  // line), k3 = -kg (index rho, the external gluon):  jl_mu jt_nu E_rho V^{mu nu rho}
  CVec4<R> k12, k23, k31;
  for (int m = 0; m < 4; ++m) {
    k12.c[m] = Cx<R>(ql[m] + qt[m]);
    k23.c[m] = Cx<R>(-qt[m] + kg[m]);
    k31.c[m] = Cx<R>(-kg[m] - ql[m]);
  }
  const Cx<R> V = mdot(jl, jt) * mdot(k12, E) + mdot(jt, E) * mdot(k23, jl) + mdot(E, jl) * mdot(k31, jt);
  kin[4] = (I * g) * (I * g) * Cx<R>(g) * gprop * gprop * V / (sl * st);
}

// colour tensors of the five diagrams, contracted over all colours: CC[d][e] = sum_{i j k l a} conj(C_d) C_e with
//   C_0 = (T^b T^a)_{ji} T^b_{kl},  C_1 = (T^a T^b)_{ji} T^b_{kl},  C_2 = T^b_{ji} (T^a T^b)_{kl},
//   C_3 = T^b_{ji} (T^b T^a)_{kl},  C_4 = f^{bca} T^b_{ji} T^c_{kl}
// (j, i = colours of the light line's row and column spinor, k, l = of the top's; a = the external gluon), brute force.
template <class R> inline void light_line_colour_matrix(Cx<R> CC[5][5]) {
  Mat3<R> T[8];
  for (int a = 0; a < 8; ++a) T[a] = su3_generator<R>(a);
  for (int d = 0; d < 5; ++d)
    for (int e = 0; e < 5; ++e) CC[d][e] = Cx<R>();
  for (int a = 0; a < 8; ++a) {
    Mat3<R> TbTa[8], TaTb[8];
    for (int b = 0; b < 8; ++b) { TbTa[b] = mat3_mul(T[b], T[a]); TaTb[b] = mat3_mul(T[a], T[b]); }
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j)
        for (int k = 0; k < 3; ++k)
          for (int l = 0; l < 3; ++l) {
            Cx<R> c[5];
            for (int b = 0; b < 8; ++b) {
              c[0] += TbTa[b].m[j][i] * T[b].m[k][l];
              c[1] += TaTb[b].m[j][i] * T[b].m[k][l];
              c[2] += T[b].m[j][i] * TaTb[b].m[k][l];
              c[3] += T[b].m[j][i] * TbTa[b].m[k][l];
              for (int cc = 0; cc < 8; ++cc) {
                R f = structure_constant<R>(b, cc, a);
                if (f != R(0)) c[4] += (T[b].m[j][i] * T[cc].m[k][l]) * f;
              }
            }
            for (int d = 0; d < 5; ++d)
              for (int e = 0; e < 5; ++e) CC[d][e] += conj(c[d]) * c[e];
          }
  }
}
// Averaged |M|^2.  kind 0: q(mom0) qbar(mom1) -> t(mom2) tbar(mom3) g(mom4), average 1/(4 x 9);
// kind 1: q(mom0) g(mom1) -> t(mom2) tbar(mom3) q(mom4), average 1/(4 x 24);
// kind 2: qbar(mom0) g(mom1) -> t(mom2) tbar(mom3) qbar(mom4), average 1/(4 x 24): the light line runs from the outgoing
// antiquark (column v(mom4), flow momentum -mom4 into the line) to the incoming one (row vbar(mom0), flow -mom0 out).
// subst != 0 replaces the gluon's
// polarisation vector by its momentum (the Ward identity: the result must vanish).
template <class R>
inline R me2_light_line_ttbar_g(int kind, const R mom[5][4], R mt, R alpha_s, int basis, int subst) {
  const R g = r_sqrt(R(4) * r_pi<R>() * alpha_s);
  const int sb = basis & 1, pb = (basis >> 1) & 1;
  static Cx<R> CC[5][5];          // computed once per real type (the oracle is single-threaded)
  static bool have_cc = false;
  if (!have_cc) { light_line_colour_matrix<R>(CC); have_cc = true; }
  R pr[4], pc[4], kg[4];
  const R* pg = kind == 0 ? mom[4] : mom[1];                       // the gluon's physical momentum
  const R* prow = kind == 0 ? mom[1] : kind == 1 ? mom[4] : mom[0]; // the particle behind the light line's row spinor
  const R* pcol = kind == 2 ? mom[4] : mom[0];                     // ... and behind its column spinor
  for (int m = 0; m < 4; ++m) {
    pr[m] = kind == 1 ? prow[m] : -prow[m];
    pc[m] = kind == 2 ? -pcol[m] : pcol[m];
    kg[m] = kind == 0 ? pg[m] : -pg[m];
  }
  R total = R(0);
  for (int l1 = -1; l1 <= 1; l1 += 2)
    for (int l2 = -1; l2 <= 1; l2 += 2)
      for (int l3 = -1; l3 <= 1; l3 += 2)
        for (int l4 = -1; l4 <= 1; l4 += 2)
          for (int lg = -1; lg <= 1; lg += 2) {
            const Spinor<R> C = kind == 2 ? v_spinor(pcol, R(0), l1, sb) : u_spinor(pcol, R(0), l1, sb);
            const Spinor<R> Rw = kind == 1 ? bar(u_spinor(prow, R(0), l2, sb)) : bar(v_spinor(prow, R(0), l2, sb));
            const Spinor<R> ub3 = bar(u_spinor(mom[2], mt, l3, sb)), v4 = v_spinor(mom[3], mt, l4, sb);
            CVec4<R> E = polarisation(pg, lg, pb);
            if (kind == 0) E = cconj(E);
            if (subst) E = cvec_from_real(pg);
            Cx<R> kin[5];
            light_line_ttbar_g_diagrams<R>(Rw, pr, C, pc, ub3, mom[2], v4, mom[3], E, kg, mt, g, kin);
            Cx<R> acc;
            for (int d = 0; d < 5; ++d)
              for (int e = 0; e < 5; ++e) acc += conj(kin[d]) * CC[d][e] * kin[e];
            total = total + acc.re;
          }
  return total / (kind == 0 ? R(36) : R(96));
}

}  // namespace mfo
