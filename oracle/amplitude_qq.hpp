// ORACLE — TEST INFRASTRUCTURE ONLY (see real.hpp).
//
// amplitude_qq.hpp: step O10 for  q(p1) qbar(p2) -> t(p3) tbar(p4) g(k5) g(k6)  (PAPER.md L101 and Table 1,
// L140: "pp -> ttbar gg (267 diagrams)" = 123 of g g -> ttbar g g + 36 for each of the four massless flavours).
// The paper prints no formula (the matrix elements are HELAS-style wavefunction and vertex calls); what follows
// is the 36 tree diagrams written out from the Feynman rules already used in amplitude.hpp:
//   quark-gluon vertex  i gs gamma^mu T^a;   quark propagator  i (q-slash + m)/(q^2 - m^2);   gluon propagator  -i g_{mu nu}/P^2;
//   three-gluon vertex  gs f^{abc} V3 (vertex3, all momenta incoming);
//   four-gluon vertex   -i gs^2 [ f^{abe}f^{cde}(g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho}) + f^{ace}f^{bde}(g^{mu nu}g^{rho sigma}
//                        - g^{mu sigma}g^{nu rho}) + f^{ade}f^{bce}(g^{mu nu}g^{rho sigma} - g^{mu rho}g^{nu sigma}) ].
// Every diagram is the top line  ubar(p3) [ ... ] v(p4)  with an ordered list of gluon-like currents attached to it; the
// currents are the two external gluons, their merger through a three-gluon vertex, and everything that contains the light
// quark line: the light line with zero, one or two of the gluons attached before / after the vertex where the virtual gluon
// leaves it, and those currents joined with external gluons by three- and four-gluon vertices.  Colour is carried along as
// explicit tensors built from the Gell-Mann matrices (no colour algebra is typed in); the colour-summed square is
//   sum_{d e} conj(kin_d) CC[d][e] kin_e,   CC[d][e] = sum over all external colours of conj(c_d) c_e.
// Second method (referee): a colour-dressed recursion over subsets for explicit colours (qq_dressed_amplitude).
// Different from the CUDA path: Dirac 4x4 matrices, diagram by diagram, colour tensors by brute force.
#pragma once
#include <vector>

#include "amplitude.hpp"

namespace mfo {

// A gluon-like current: wavefunction J^mu (propagator included), INCOMING momentum P, and its colour, either a vector w[c]
// over the adjoint index (pure-gluon currents) or, when it contains the light quark line, a 3x3 matrix K[c] over the light
// line's (row = antiquark, column = quark) colours for every adjoint index c.
template <class R> struct QQCurrent {
  CVec4<R> J;
  R P[4];
  bool light = false;
  R w[8];
  Mat3<R> K[8];
};

template <class R> struct QQContext {
  Spinor<R> u1, vbar2, ubar3, v4;   // light line: column u(p1), row vbar(p2); top line: row ubar(p3), column v(p4)
  R p1[4], p2[4], p3[4], p4[4];
  CVec4<R> eps[2];                  // wavefunctions of the outgoing gluons (conjugated polarisation vectors)
  R Pg[2][4];                       // their incoming momenta (-k5, -k6)
  R mt, gs;
  bool colour = false;              // build the colour tensors as well (for the external gluon colours a[0], a[1])
  int a[2] = {0, 0};
  Mat3<R> T[8];
  R f[8][8][8];
};

template <class R> inline void qq_colour_tables(QQContext<R>& c) {
  for (int a = 0; a < 8; ++a) c.T[a] = su3_generator<R>(a);
  for (int a = 0; a < 8; ++a)
    for (int b = 0; b < 8; ++b)
      for (int d = 0; d < 8; ++d) {
        R f = structure_constant<R>(a, b, d);
        c.f[a][b][d] = (r_fabs(f) < R(1e-14)) ? R(0) : f;
      }
}

template <class R> inline Mat3<R> mat3_zero() { return Mat3<R>(); }
template <class R> inline Mat3<R> mat3_identity() {
  Mat3<R> o;
  for (int i = 0; i < 3; ++i) o.m[i][i] = Cx<R>(R(1));
  return o;
}
template <class R> inline void mat3_add_scaled(Mat3<R>& o, const Mat3<R>& a, R s) {
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) o.m[i][j] += s * a.m[i][j];
}
// sum_c w[c] T^c of a pure-gluon current
template <class R> inline Mat3<R> qq_generator_of(const QQContext<R>& c, const QQCurrent<R>& g) {
  Mat3<R> o;
  for (int a = 0; a < 8; ++a)
    if (g.w[a] != R(0)) mat3_add_scaled(o, c.T[a], g.w[a]);
  return o;
}

template <class R> inline QQCurrent<R> qq_external_gluon(const QQContext<R>& c, int g) {
  QQCurrent<R> o;
  o.J = c.eps[g];
  for (int m = 0; m < 4; ++m) o.P[m] = c.Pg[g][m];
  for (int a = 0; a < 8; ++a) o.w[a] = (c.colour && a == c.a[g]) ? R(1) : R(0);
  return o;
}

// two currents joined by a three-gluon vertex:  J^{c} = (-i/P^2) gs f^{abc} V3(A^a, P_A; B^b, P_B).  B is a pure-gluon current.
template <class R> inline QQCurrent<R> qq_join3(const QQContext<R>& c, const QQCurrent<R>& A, const QQCurrent<R>& B) {
  const Cx<R> I = cx_i<R>();
  QQCurrent<R> o;
  for (int m = 0; m < 4; ++m) o.P[m] = A.P[m] + B.P[m];
  const R P2 = mdot_rr(o.P, o.P);
  const CVec4<R> v = vertex3(A.J, A.P, B.J, B.P);
  for (int m = 0; m < 4; ++m) o.J.c[m] = (-I) * ((c.gs * v.c[m]) / P2);
  o.light = A.light;
  for (int d = 0; d < 8; ++d) o.w[d] = R(0);
  if (c.colour)
    for (int a = 0; a < 8; ++a)
      for (int b = 0; b < 8; ++b)
        for (int d = 0; d < 8; ++d) {
          const R fabd = c.f[a][b][d];
          if (fabd == R(0) || B.w[b] == R(0)) continue;
          if (A.light) mat3_add_scaled(o.K[d], A.K[a], fabd * B.w[b]);
          else o.w[d] = o.w[d] + fabd * A.w[a] * B.w[b];
        }
  return o;
}

// three currents joined by the four-gluon vertex: one term per colour structure (f^{abe}f^{cde}, f^{ace}f^{bde}, f^{ade}f^{bce}).
// A contains the light line, B and C are pure-gluon currents.
template <class R>
inline void qq_join4(const QQContext<R>& c, const QQCurrent<R>& A, const QQCurrent<R>& B, const QQCurrent<R>& C, QQCurrent<R> out[3]) {
  const Cx<R> I = cx_i<R>();
  R P[4];
  for (int m = 0; m < 4; ++m) P[m] = A.P[m] + B.P[m] + C.P[m];
  const R P2 = mdot_rr(P, P);
  const Cx<R> jab = mdot(A.J, B.J), jac = mdot(A.J, C.J), jbc = mdot(B.J, C.J);
  for (int t = 0; t < 3; ++t) {
    QQCurrent<R>& o = out[t];
    o = QQCurrent<R>();
    o.light = true;
    for (int d = 0; d < 8; ++d) o.w[d] = R(0);
    for (int m = 0; m < 4; ++m) {
      o.P[m] = P[m];
      Cx<R> v;
      if (t == 0) v = jac * B.J.c[m] - jbc * A.J.c[m];
      if (t == 1) v = jab * C.J.c[m] - jbc * A.J.c[m];
      if (t == 2) v = jab * C.J.c[m] - jac * B.J.c[m];
      o.J.c[m] = (-I) * (((-I) * (c.gs * c.gs)) * v / P2);
    }
    if (!c.colour) continue;
    for (int a = 0; a < 8; ++a)
      for (int b = 0; b < 8; ++b)
        for (int g = 0; g < 8; ++g) {
          if (B.w[b] == R(0) || C.w[g] == R(0)) continue;
          for (int d = 0; d < 8; ++d) {
            R cf = R(0);
            for (int e = 0; e < 8; ++e) {
              if (t == 0) cf = cf + c.f[a][b][e] * c.f[g][d][e];
              if (t == 1) cf = cf + c.f[a][g][e] * c.f[b][d][e];
              if (t == 2) cf = cf + c.f[a][d][e] * c.f[b][g][e];
            }
            if (cf != R(0)) mat3_add_scaled(o.K[d], A.K[a], cf * B.w[b] * C.w[g]);
          }
        }
  }
}

// The light line with pure-gluon currents attached: `before` in the order they are met going from the column spinor u(p1)
// towards the vertex where the virtual gluon leaves, `after` from the row spinor vbar(p2) backwards towards that vertex.
//   J^{c mu} = (-i/P^2)  chi (i gs gamma^mu T^c) psi,   P = p1 + p2 + sum of the attached currents' momenta,
//   psi = [ i q-slash/q^2 (i gs B-slash) ] ... u(p1),      q = p1 + momenta absorbed so far (fermion flow from u to vbar),
//   chi = vbar(p2) ... [ (i gs A-slash) i q'-slash/q'^2 ], q' = -p2 - momenta attached on the row side so far.
template <class R>
inline QQCurrent<R> qq_light_line(const QQContext<R>& c, const std::vector<const QQCurrent<R>*>& after,
                                  const std::vector<const QQCurrent<R>*>& before) {
  const Cx<R> I = cx_i<R>();
  Spinor<R> psi = c.u1, chi = c.vbar2;
  R q[4], qp[4];
  for (int m = 0; m < 4; ++m) { q[m] = c.p1[m]; qp[m] = -c.p2[m]; }
  Mat3<R> col_side = mat3_identity<R>(), row_side = mat3_identity<R>();
  for (const QQCurrent<R>* g : before) {
    Spinor<R> t = mat_vec(slash(g->J), psi);
    for (int m = 0; m < 4; ++m) q[m] = q[m] + g->P[m];
    t = mat_vec(slash_plus_mass(q, R(0)), t);
    const R den = mdot_rr(q, q);
    for (int s = 0; s < 4; ++s) psi.c[s] = I * ((I * c.gs) * t.c[s] / den);
    if (c.colour) col_side = mat3_mul(qq_generator_of(c, *g), col_side);
  }
  for (const QQCurrent<R>* g : after) {
    Spinor<R> t = row_times_mat(chi, slash(g->J));
    for (int m = 0; m < 4; ++m) qp[m] = qp[m] - g->P[m];
    t = row_times_mat(t, slash_plus_mass(qp, R(0)));
    const R den = mdot_rr(qp, qp);
    for (int s = 0; s < 4; ++s) chi.c[s] = I * ((I * c.gs) * t.c[s] / den);
    if (c.colour) row_side = mat3_mul(row_side, qq_generator_of(c, *g));
  }
  QQCurrent<R> o;
  o.light = true;
  for (int m = 0; m < 4; ++m) o.P[m] = q[m] - qp[m];
  const R P2 = mdot_rr(o.P, o.P);
  for (int mu = 0; mu < 4; ++mu) {
    const Cx<R> v = row_times_col(chi, mat_vec(gamma_matrix<R>(mu), psi));
    o.J.c[mu] = (-I) * ((I * c.gs) * v / P2);
  }
  for (int d = 0; d < 8; ++d) o.w[d] = R(0);
  if (c.colour)
    for (int d = 0; d < 8; ++d) o.K[d] = mat3_mul(row_side, mat3_mul(c.T[d], col_side));
  return o;
}

// One diagram: ubar(p3) (i gs J1-slash) i(q-slash + m)/(q^2 - m^2) (i gs J2-slash) ... v(p4), the currents listed from the row
// spinor's side; q = -p4 + momenta of the currents between the propagator and v(p4).  Exactly one current of the list contains
// the light line.  kin = the colour-stripped amplitude; ctens[j][i][k][l] (if c.colour) = its colour tensor for the external
// gluon colours c.a[]: light-line colours (row j, column i), top-line colours (row k = top, column l = antitop).
template <class R> struct QQEntry {
  Cx<R> kin;
  Cx<R> ctens[81];
};
template <class R>
inline QQEntry<R> qq_top_line(const QQContext<R>& c, const std::vector<const QQCurrent<R>*>& list) {
  const Cx<R> I = cx_i<R>();
  QQEntry<R> e;
  Spinor<R> X = c.v4;
  R q[4];
  for (int m = 0; m < 4; ++m) q[m] = -c.p4[m];
  for (int k = (int)list.size() - 1; k >= 0; --k) {
    Spinor<R> t = mat_vec(slash(list[k]->J), X);
    for (int s = 0; s < 4; ++s) X.c[s] = (I * c.gs) * t.c[s];
    if (k > 0) {
      for (int m = 0; m < 4; ++m) q[m] = q[m] + list[k]->P[m];
      t = mat_vec(slash_plus_mass(q, c.mt), X);
      const R den = mdot_rr(q, q) - c.mt * c.mt;
      for (int s = 0; s < 4; ++s) X.c[s] = I * (t.c[s] / den);
    }
  }
  e.kin = row_times_col(c.ubar3, X);
  if (c.colour) {
    Mat3<R> pre = mat3_identity<R>(), post = mat3_identity<R>();
    const QQCurrent<R>* L = nullptr;
    for (const QQCurrent<R>* g : list) {
      if (g->light) { L = g; continue; }
      if (!L) pre = mat3_mul(pre, qq_generator_of(c, *g));
      else post = mat3_mul(post, qq_generator_of(c, *g));
    }
    for (int d = 0; d < 8; ++d) {
      const Mat3<R> M = mat3_mul(pre, mat3_mul(c.T[d], post));
      for (int j = 0; j < 3; ++j)
        for (int i = 0; i < 3; ++i)
          for (int k = 0; k < 3; ++k)
            for (int l = 0; l < 3; ++l) e.ctens[((j * 3 + i) * 3 + k) * 3 + l] += L->K[d].m[j][i] * M.m[k][l];
    }
  }
  return e;
}

// The 36 diagrams (38 entries: the four-gluon vertex has three colour structures).
constexpr int kQQEntries = 38;
template <class R> inline std::vector<QQEntry<R>> qq_diagrams(const QQContext<R>& c) {
  typedef QQCurrent<R> Cur;
  typedef std::vector<const Cur*> List;
  std::vector<QQEntry<R>> out;
  const Cur g[2] = {qq_external_gluon(c, 0), qq_external_gluon(c, 1)};
  const Cur G = qq_join3(c, g[0], g[1]);                       // the two gluons merged
  const Cur L0 = qq_light_line(c, List{}, List{});             // the bare light line
  // (1) nothing attached to the light line or to the virtual gluon: 6 + 2 diagrams
  const Cur* three[3] = {&L0, &g[0], &g[1]};
  const int perm3[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
  for (const auto& p : perm3) out.push_back(qq_top_line(c, List{three[p[0]], three[p[1]], three[p[2]]}));
  out.push_back(qq_top_line(c, List{&L0, &G}));
  out.push_back(qq_top_line(c, List{&G, &L0}));
  // (2) one gluon on the virtual gluon, the other on the top line: 4 diagrams
  for (int a = 0; a < 2; ++a) {
    const Cur La = qq_join3(c, L0, g[a]);
    out.push_back(qq_top_line(c, List{&La, &g[1 - a]}));
    out.push_back(qq_top_line(c, List{&g[1 - a], &La}));
    // (3) both on the virtual gluon, one after the other: 2 diagrams
    const Cur Lab = qq_join3(c, La, g[1 - a]);
    out.push_back(qq_top_line(c, List{&Lab}));
  }
  // (3') the merged pair on the virtual gluon, and the four-gluon vertex: 2 diagrams (4 entries)
  const Cur LG = qq_join3(c, L0, G);
  out.push_back(qq_top_line(c, List{&LG}));
  Cur L4[3];
  qq_join4(c, L0, g[0], g[1], L4);
  for (int t = 0; t < 3; ++t) out.push_back(qq_top_line(c, List{&L4[t]}));
  // (4) one gluon on the light line (before / after the virtual gluon's vertex); the other on the top line (2 places) or on
  //     the virtual gluon: 2 x 2 x 3 = 12 diagrams
  for (int a = 0; a < 2; ++a)
    for (int side = 0; side < 2; ++side) {
      const Cur La = side == 0 ? qq_light_line(c, List{}, List{&g[a]}) : qq_light_line(c, List{&g[a]}, List{});
      out.push_back(qq_top_line(c, List{&La, &g[1 - a]}));
      out.push_back(qq_top_line(c, List{&g[1 - a], &La}));
      const Cur Lab = qq_join3(c, La, g[1 - a]);
      out.push_back(qq_top_line(c, List{&Lab}));
    }
  // (5) both gluons on the light line: 6 orderings of (gluon, gluon, virtual gluon) along it + the merged pair on either side
  for (int a = 0; a < 2; ++a) {
    const Cur* x = &g[a];
    const Cur* y = &g[1 - a];
    const Cur bb = qq_light_line(c, List{}, List{x, y});        // both before (x first)
    const Cur ba = qq_light_line(c, List{y}, List{x});          // x before, y after
    const Cur aa = qq_light_line(c, List{x, y}, List{});        // both after (x next to the row spinor)
    out.push_back(qq_top_line(c, List{&bb}));
    out.push_back(qq_top_line(c, List{&ba}));
    out.push_back(qq_top_line(c, List{&aa}));
  }
  const Cur Gb = qq_light_line(c, List{}, List{&G}), Ga = qq_light_line(c, List{&G}, List{});
  out.push_back(qq_top_line(c, List{&Gb}));
  out.push_back(qq_top_line(c, List{&Ga}));
  return out;
}

// CC[d][e] = sum over the 3^4 x 8^2 external colour assignments of conj(c_d) c_e  (kinematics-independent; any momenta do)
template <class R> inline void qq_colour_matrix(std::vector<Cx<R>>& CC) {
  QQContext<R> c;
  qq_colour_tables(c);
  c.colour = true;
  c.mt = R(1); c.gs = R(1);
  const R P[6][4] = {{R(5), R(0), R(0), R(5)}, {R(5), R(0), R(0), R(-5)}, {R(3), R(1), R(2), R(1.5)}, {R(3), R(-1), R(-1), R(-2)},
                     {R(2), R(0.5), R(-1.5), R(1)}, {R(2), R(-0.5), R(0.5), R(-0.5)}};   // placeholders: only the tensors are used
  for (int m = 0; m < 4; ++m) {
    c.p1[m] = P[0][m]; c.p2[m] = P[1][m]; c.p3[m] = P[2][m]; c.p4[m] = P[3][m];
    c.Pg[0][m] = -P[4][m]; c.Pg[1][m] = -P[5][m];
    c.eps[0].c[m] = Cx<R>(R(m == 1)); c.eps[1].c[m] = Cx<R>(R(m == 2));
  }
  c.u1.c[0] = Cx<R>(R(1)); c.vbar2.c[1] = Cx<R>(R(1)); c.ubar3.c[2] = Cx<R>(R(1)); c.v4.c[3] = Cx<R>(R(1));
  CC.assign((size_t)kQQEntries * kQQEntries, Cx<R>());
  for (int a = 0; a < 8; ++a)
    for (int b = 0; b < 8; ++b) {
      c.a[0] = a; c.a[1] = b;
      const std::vector<QQEntry<R>> en = qq_diagrams(c);
      for (int x = 0; x < 81; ++x)
        for (int d = 0; d < kQQEntries; ++d)
          for (int e = 0; e < kQQEntries; ++e) CC[(size_t)d * kQQEntries + e] += conj(en[d].ctens[x]) * en[e].ctens[x];
    }
}

template <class R> inline void qq_load_point(QQContext<R>& c, const R mom[6][4], R mt, R gs) {
  for (int m = 0; m < 4; ++m) {
    c.p1[m] = mom[0][m]; c.p2[m] = mom[1][m]; c.p3[m] = mom[2][m]; c.p4[m] = mom[3][m];
    c.Pg[0][m] = -mom[4][m]; c.Pg[1][m] = -mom[5][m];
  }
  c.mt = mt; c.gs = gs;
}
template <class R> inline void qq_load_helicities(QQContext<R>& c, const R mom[6][4], const int lam[6], int basis, int subst) {
  const int sb = basis & 1, pb = (basis >> 1) & 1;
  c.u1 = u_spinor(mom[0], R(0), lam[0], sb);
  c.vbar2 = bar(v_spinor(mom[1], R(0), lam[1], sb));
  c.ubar3 = bar(u_spinor(mom[2], c.mt, lam[2], sb));
  c.v4 = v_spinor(mom[3], c.mt, lam[3], sb);
  for (int g = 0; g < 2; ++g) {
    c.eps[g] = cconj(polarisation(mom[4 + g], lam[4 + g], pb));
    if (subst == g) c.eps[g] = cvec_from_real(mom[4 + g]);
  }
}

// Averaged |M|^2 of q(mom0) qbar(mom1) -> t(mom2) tbar(mom3) g(mom4) g(mom5): 1/(4 x 9) for the initial state, 1/2! for the
// identical gluons.  basis as in me2_gg_ttbar_ng; subst = 0 / 1 replaces that gluon's polarisation by its momentum (Ward identity).
template <class R> inline R me2_qq_ttbar_gg(const R mom[6][4], R mt, R alpha_s, int basis, int subst) {
  static std::vector<Cx<R>> CC;              // once per real type (the oracle is single-threaded)
  if (CC.empty()) qq_colour_matrix<R>(CC);
  QQContext<R> c;
  qq_load_point(c, mom, mt, r_sqrt(R(4) * r_pi<R>() * alpha_s));
  R total = R(0);
  for (int h = 0; h < 64; ++h) {
    int lam[6];
    for (int k = 0; k < 6; ++k) lam[k] = ((h >> k) & 1) ? 1 : -1;
    qq_load_helicities(c, mom, lam, basis, subst);
    const std::vector<QQEntry<R>> en = qq_diagrams(c);
    Cx<R> acc;
    for (int d = 0; d < kQQEntries; ++d)
      for (int e = 0; e < kQQEntries; ++e) acc += conj(en[d].kin) * CC[(size_t)d * kQQEntries + e] * en[e].kin;
    total = total + acc.re;
  }
  return total / R(72);
}

// The full amplitude iM for explicit colours (light line: antiquark jq, quark iq; top k, antitop l; gluons a5, a6) as the sum
// over the diagrams of colour tensor x kinematic factor (for the comparison with the dressed recursion below).
template <class R>
inline Cx<R> qq_diagram_sum(const R mom[6][4], R mt, R gs, const int lam[6], int basis, int jq, int iq, int k, int l, int a5, int a6) {
  QQContext<R> c;
  qq_colour_tables(c);
  c.colour = true;
  c.a[0] = a5; c.a[1] = a6;
  qq_load_point(c, mom, mt, gs);
  qq_load_helicities(c, mom, lam, basis, -1);
  Cx<R> M;
  for (const QQEntry<R>& e : qq_diagrams(c)) M += e.ctens[((jq * 3 + iq) * 3 + k) * 3 + l] * e.kin;
  return M;
}

// ---------------------------------------------------------------------------------------------
// Referee: colour-dressed recursion over subsets of {gluon 5 (bit 0), gluon 6 (bit 1), the light quark pair (bit 2)} for
// explicit external colours; no diagram is enumerated.  J_S^{a mu} = the off-shell gluon leaving the blob that contains the
// particles of S:
//   J_S = (-i/P_S^2) [ sum over {S1, S2} gs f^{abc} V3(J_S1^a, J_S2^b) + sum over {S1, S2, S3} (four-gluon vertex)
//                      + (if the pair is in S) the light line with the pure-gluon currents of S attached to it ]
// quark lines:  X_S = i (q-slash + m)/(q^2 - m^2) sum_{S1} (i gs gamma_mu T^a) J_S1^{a mu} X_{S \ S1}  (column, from u(p1) or v(p4)),
//               Y_S = sum_{S1} Y_{S \ S1} (i gs gamma_mu T^a) J_S1^{a mu} i (q'-slash)/q'^2             (row, from vbar(p2)).
template <class R> struct QQDressed {
  QQContext<R> c;                   // spinors, momenta, tables
  int col_g[2], jq, iq, l;          // external colours: gluons, light antiquark / quark, antitop
  std::map<uint32_t, DressedCurrent<R>> memoJ;
};
template <class R> inline void qq_subset_momentum(const QQDressed<R>& d, uint32_t S, R out[4]) {
  for (int m = 0; m < 4; ++m) {
    out[m] = R(0);
    if (S & 1u) out[m] = out[m] + d.c.Pg[0][m];
    if (S & 2u) out[m] = out[m] + d.c.Pg[1][m];
    if (S & 4u) out[m] = out[m] + d.c.p1[m] + d.c.p2[m];
  }
}
template <class R> DressedCurrent<R> qq_dressed_gluon(QQDressed<R>& d, uint32_t S);

// (i gs gamma_mu T^a) J^{a mu} applied to a coloured column spinor
template <class R> inline DressedQuark<R> qq_vertex_col(const QQDressed<R>& d, const DressedCurrent<R>& J, const DressedQuark<R>& X) {
  const Cx<R> I = cx_i<R>();
  DressedQuark<R> o;
  for (int a = 0; a < 8; ++a) {
    const Mat4<R> Js = slash(J.a[a]);
    for (int i2 = 0; i2 < 3; ++i2) {
      const Spinor<R> t = mat_vec(Js, X.c[i2]);
      for (int i1 = 0; i1 < 3; ++i1)
        for (int s = 0; s < 4; ++s) o.c[i1].c[s] += (I * d.c.gs) * (d.c.T[a].m[i1][i2] * t.c[s]);
    }
  }
  return o;
}
// a coloured row spinor times (i gs gamma_mu T^a) J^{a mu}
template <class R> inline DressedQuark<R> qq_vertex_row(const QQDressed<R>& d, const DressedQuark<R>& Y, const DressedCurrent<R>& J) {
  const Cx<R> I = cx_i<R>();
  DressedQuark<R> o;
  for (int a = 0; a < 8; ++a) {
    const Mat4<R> Js = slash(J.a[a]);
    for (int i1 = 0; i1 < 3; ++i1) {
      const Spinor<R> t = row_times_mat(Y.c[i1], Js);
      for (int i2 = 0; i2 < 3; ++i2)
        for (int s = 0; s < 4; ++s) o.c[i2].c[s] += (I * d.c.gs) * (d.c.T[a].m[i1][i2] * t.c[s]);
    }
  }
  return o;
}
// column current of a quark line that starts from `base` (colour index c0) with flow momentum p0 and absorbs the currents of S
template <class R>
DressedQuark<R> qq_column(QQDressed<R>& d, uint32_t S, const Spinor<R>& base, int c0, const R p0[4], R mass) {
  DressedQuark<R> out;
  if (S == 0) { out.c[c0] = base; return out; }
  const Cx<R> I = cx_i<R>();
  DressedQuark<R> sum;
  for (uint32_t S1 = S; S1; S1 = (S1 - 1) & S) {
    const DressedQuark<R> t = qq_vertex_col(d, qq_dressed_gluon(d, S1), qq_column(d, S ^ S1, base, c0, p0, mass));
    for (int i = 0; i < 3; ++i)
      for (int s = 0; s < 4; ++s) sum.c[i].c[s] += t.c[i].c[s];
  }
  R q[4], PS[4];
  qq_subset_momentum(d, S, PS);
  for (int m = 0; m < 4; ++m) q[m] = p0[m] + PS[m];
  const R den = mdot_rr(q, q) - mass * mass;
  const Mat4<R> num = slash_plus_mass(q, mass);
  for (int i = 0; i < 3; ++i) {
    const Spinor<R> t = mat_vec(num, sum.c[i]);
    for (int s = 0; s < 4; ++s) out.c[i].c[s] = I * (t.c[s] / den);
  }
  return out;
}
// row current of the light line: from vbar(p2) (colour jq) backwards, the pure-gluon currents of S attached
template <class R> DressedQuark<R> qq_light_row(QQDressed<R>& d, uint32_t S) {
  DressedQuark<R> out;
  if (S == 0) { out.c[d.jq] = d.c.vbar2; return out; }
  const Cx<R> I = cx_i<R>();
  DressedQuark<R> sum;
  for (uint32_t S1 = S; S1; S1 = (S1 - 1) & S) {
    const DressedQuark<R> t = qq_vertex_row(d, qq_light_row(d, S ^ S1), qq_dressed_gluon(d, S1));
    for (int i = 0; i < 3; ++i)
      for (int s = 0; s < 4; ++s) sum.c[i].c[s] += t.c[i].c[s];
  }
  R q[4], PS[4];
  qq_subset_momentum(d, S, PS);
  for (int m = 0; m < 4; ++m) q[m] = -d.c.p2[m] - PS[m];
  const R den = mdot_rr(q, q);
  const Mat4<R> num = slash_plus_mass(q, R(0));
  for (int i = 0; i < 3; ++i) {
    const Spinor<R> t = row_times_mat(sum.c[i], num);
    for (int s = 0; s < 4; ++s) out.c[i].c[s] = I * (t.c[s] / den);
  }
  return out;
}
template <class R> DressedCurrent<R> qq_dressed_gluon(QQDressed<R>& d, uint32_t S) {
  auto it = d.memoJ.find(S);
  if (it != d.memoJ.end()) return it->second;
  DressedCurrent<R> out;
  if (S == 1u || S == 2u) {
    out.a[d.col_g[S - 1]] = d.c.eps[S - 1];
    d.memoJ[S] = out;
    return out;
  }
  const Cx<R> I = cx_i<R>();
  const R gs = d.c.gs;
  DressedCurrent<R> sum;
  const uint32_t low = S & (~S + 1);
  for (uint32_t S1 = (S - 1) & S; S1; S1 = (S1 - 1) & S) {        // three-gluon vertices: unordered pairs
    if (!(S1 & low)) continue;
    const uint32_t S2 = S ^ S1;
    const DressedCurrent<R> J1 = qq_dressed_gluon(d, S1), J2 = qq_dressed_gluon(d, S2);
    R P1[4], P2[4];
    qq_subset_momentum(d, S1, P1);
    qq_subset_momentum(d, S2, P2);
    for (int a = 0; a < 8; ++a)
      for (int b = 0; b < 8; ++b) {
        const CVec4<R> v = vertex3(J1.a[a], P1, J2.a[b], P2);
        for (int e = 0; e < 8; ++e)
          if (d.c.f[a][b][e] != R(0))
            for (int m = 0; m < 4; ++m) sum.a[e].c[m] += (gs * d.c.f[a][b][e]) * v.c[m];
      }
  }
  if (S == 7u) {                                                   // the four-gluon vertex joins the three single particles
    const DressedCurrent<R> J1 = qq_dressed_gluon(d, 1u), J2 = qq_dressed_gluon(d, 2u), J3 = qq_dressed_gluon(d, 4u);
    for (int a = 0; a < 8; ++a)
      for (int b = 0; b < 8; ++b)
        for (int g = 0; g < 8; ++g) {
          const Cx<R> j12 = mdot(J1.a[a], J2.a[b]), j13 = mdot(J1.a[a], J3.a[g]), j23 = mdot(J2.a[b], J3.a[g]);
          for (int e = 0; e < 8; ++e) {
            R c1 = R(0), c2 = R(0), c3 = R(0);
            for (int x = 0; x < 8; ++x) {
              c1 = c1 + d.c.f[a][b][x] * d.c.f[g][e][x];
              c2 = c2 + d.c.f[a][g][x] * d.c.f[b][e][x];
              c3 = c3 + d.c.f[a][e][x] * d.c.f[b][g][x];
            }
            if (c1 == R(0) && c2 == R(0) && c3 == R(0)) continue;
            for (int m = 0; m < 4; ++m) {
              const Cx<R> t = c1 * (j13 * J2.a[b].c[m] - j23 * J1.a[a].c[m]) + c2 * (j12 * J3.a[g].c[m] - j23 * J1.a[a].c[m]) +
                              c3 * (j12 * J3.a[g].c[m] - j13 * J2.a[b].c[m]);
              sum.a[e].c[m] += (-(I * (gs * gs))) * t;
            }
          }
        }
  }
  if (S & 4u) {                                                    // the light line itself, the gluons of S attached to it
    const uint32_t G = S & 3u;
    for (uint32_t S1 = G;; S1 = (S1 - 1) & G) {
      const DressedQuark<R> X = qq_column(d, S1, d.c.u1, d.iq, d.c.p1, R(0)), Y = qq_light_row(d, G ^ S1);
      for (int a = 0; a < 8; ++a)
        for (int mu = 0; mu < 4; ++mu) {
          const Mat4<R> gm = gamma_matrix<R>(mu);
          for (int i1 = 0; i1 < 3; ++i1)
            for (int i2 = 0; i2 < 3; ++i2) {
              const Cx<R> tc = d.c.T[a].m[i1][i2];
              if (tc.re == R(0) && tc.im == R(0)) continue;
              sum.a[a].c[mu] += (I * gs) * (tc * row_times_col(Y.c[i1], mat_vec(gm, X.c[i2])));
            }
        }
      if (S1 == 0) break;
    }
  }
  R P[4];
  qq_subset_momentum(d, S, P);
  const R P2 = mdot_rr(P, P);
  for (int a = 0; a < 8; ++a)
    for (int m = 0; m < 4; ++m) out.a[a].c[m] = (-I) * (sum.a[a].c[m] / P2);
  d.memoJ[S] = out;
  return out;
}
template <class R>
inline Cx<R> qq_dressed_amplitude(const R mom[6][4], R mt, R gs, const int lam[6], int basis, int jq, int iq, int k, int l, int a5, int a6) {
  QQDressed<R> d;
  qq_colour_tables(d.c);
  qq_load_point(d.c, mom, mt, gs);
  qq_load_helicities(d.c, mom, lam, basis, -1);
  d.col_g[0] = a5; d.col_g[1] = a6; d.jq = jq; d.iq = iq; d.l = l;
  R mp4[4];
  for (int m = 0; m < 4; ++m) mp4[m] = -mom[3][m];
  // the last vertex on the top line has no propagator after it: sum over the current S1 that attaches there
  DressedQuark<R> sum;
  for (uint32_t S1 = 7u; S1; S1 = (S1 - 1) & 7u) {
    const DressedQuark<R> t = qq_vertex_col(d, qq_dressed_gluon(d, S1), qq_column(d, 7u ^ S1, d.c.v4, l, mp4, mt));
    for (int i = 0; i < 3; ++i)
      for (int s = 0; s < 4; ++s) sum.c[i].c[s] += t.c[i].c[s];
  }
  return row_times_col(d.c.ubar3, sum.c[k]);
}

}  // namespace mfo
