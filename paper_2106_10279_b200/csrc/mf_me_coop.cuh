// mf_me_coop.cuh — steps a7-a9 for g g -> t tbar g g as a COOPERATIVE program: one event per team of 64
// threads (2 warps), all intermediate currents in a per-team shared-memory scratch (the
// matrix element loops over helicities and sums; DESIGN.md "Kernels" explains why not one thread per event).
//
//   S0     hand written: momentum sums, propagator denominators, polarisation vectors, external spinors, c0
//   S1/A/B table driven (csrc/gen_coop.py): one lane-task = M "polarisation sibling" off-shell currents that
//          share their operands; a warp executes rounds of 32 equal-shaped lane-tasks
//   S4     generated straight-line code: thread (pols, hb, k) forms the real / imaginary parts of its 24
//          colour-ordered amplitudes and contracts them with the colour matrix; the 64 partial sums are
//          added in a fixed order.  Only the top spin state 0 is evaluated (spin-flip symmetry, gen_coop.py):
//          the caller doubles the sum.
//
// Every function is MF_HD and takes the team-thread index explicitly, so tests/host_shim can run the same
// program on the host (looping over the 64 "threads" stage by stage) and compare it with the oracle.
#pragma once
#include "mf_me_prims.cuh"
#include "mf_me_ttgg_coop_generated.cuh"

namespace mf {

constexpr int kCoopTeam = 64;                     // threads per event
constexpr int kCoopInDoubles = 18;                // input area: k[4][4] (t, tbar, g, g; CM frame), shat, pad
constexpr int kCoopRedDoubles = 2;                // one partial per warp
// per-team shared memory (doubles): scratch | input | reduction
constexpr int kCoopOffIn = (kCoopScratchDoubles + 1) & ~1;
constexpr int kCoopOffRed = kCoopOffIn + kCoopInDoubles;
constexpr int kCoopTeamDoubles = kCoopOffRed + kCoopRedDoubles;

MF_HD double* coop_V(double* scr) { return scr; }
MF_HD double* coop_S(double* scr) { return scr + 4 * kCoopNV; }
MF_HD double* coop_Z(double* scr) { return scr + 4 * kCoopNV + 8 * kCoopNS; }
MF_HD double* coop_X(double* scr) { return scr + 4 * kCoopNV + 8 * kCoopNS + 2 * kCoopZPlane; }

MF_HD rvec rflip(const rvec& a, int neg) {
  rvec o;
#pragma unroll
  for (int m = 0; m < 4; ++m) o.v[m] = mf_flip(a.v[m], neg);
  return o;
}

// ---- S0: per-event constants --------------------------------------------------------------------------------
// in[0..15] = k[4][4] (t, tbar, g2, g3 in the partonic CM frame), in[16] = shat, in[17] = sqrt(shat) / 2.  Gluon
// labels: 0, 1 = the beams (+z, -z), 2, 3 = the final gluons entering with -k (all gluon momenta incoming).
//
// team threads 0 .. kCoopS0Lanes-1 (warp 0): one momentum sum / propagator momentum and its inverse denominator
// each (uniform code, one reciprocal per lane; table kCoopS0Tab); 30, 31: v(hb), ubar and c0(hb) = ubar gamma v(hb);
// 32, 33 (warp 1): the polarisation vectors of the final gluons; 36..39: the constant beam polarisations
MF_HD void coop_s0(double* scr, const double* in, int tid, double mt) {
  double* V = coop_V(scr);
  double* S = coop_S(scr);
  double* X = coop_X(scr);
  if (tid < kCoopS0Lanes) {
    const int kind = kCoopS0Tab[tid][0], m = kCoopS0Tab[tid][1], iv = kCoopS0Tab[tid][2], ix = kCoopS0Tab[tid][3];
    const double E = in[17];
    // sum of the gluon momenta in the mask (beams: (E, 0, 0, +-E); final gluons enter with -k)
    const double b0 = (m & 1) ? 1.0 : 0.0, b1 = (m & 2) ? 1.0 : 0.0, b2 = (m & 4) ? -1.0 : 0.0, b3 = (m & 8) ? -1.0 : 0.0;
    rvec P;
    P.v[0] = fma(b3, in[12], fma(b2, in[8], (b0 + b1) * E));
    P.v[1] = fma(b3, in[13], b2 * in[9]);
    P.v[2] = fma(b3, in[14], b2 * in[10]);
    P.v[3] = fma(b3, in[15], fma(b2, in[11], (b0 - b1) * E));
    // kind 0: P;  kind 1: P - p4;  kind 2: p3 - P
    const double sp = kind == 2 ? -1.0 : 1.0;
    const double* q = kind == 1 ? in + 4 : in;
    const double sq = kind == 0 ? 0.0 : (kind == 1 ? -1.0 : 1.0);
    rvec v;
#pragma unroll
    for (int c = 0; c < 4; ++c) v.v[c] = fma(sq, q[c], sp * P.v[c]);
    coop_st_vec(V, iv, v);
    if (ix >= 0) X[ix] = 1.0 / (rdot(v, v) - (kind == 0 ? 0.0 : mt * mt));
  } else if (tid >= 30 && tid < 32) {
    const int hb = tid - 30;
    const spin ub = ubar_row(in, mt, 0), v = v_col(in + 4, mt, hb);
    if (hb == 0) coop_st_spin(S, kCoopUb, ub);
    coop_st_spin(S, kCoopV0 + hb, v);
    const cvec c = bilinear(ub, v);
    coop_st_vec(V, kCoopC0 + 2 * hb, rvec{{c.re[0], c.re[1], c.re[2], c.re[3]}});
    coop_st_vec(V, kCoopC0 + 2 * hb + 1, rvec{{c.im[0], c.im[1], c.im[2], c.im[3]}});
  } else if (tid >= 32 && tid < 34) {
    const int g = tid - 30;
    rvec e1, e2;
    pol_vectors(in + 4 * g, e1, e2);
    coop_st_vec(V, kCoopEps0 + 2 * g, e1);
    coop_st_vec(V, kCoopEps0 + 2 * g + 1, e2);
  } else if (tid >= 36 && tid < 40) {
    const int g = (tid - 36) >> 1, p = (tid - 36) & 1;
    const rvec e = p == 0 ? rvec{{0.0, 1.0, 0.0, 0.0}} : rvec{{0.0, 0.0, g == 0 ? 1.0 : -1.0, 0.0}};
    coop_st_vec(V, kCoopEps0 + 2 * g + p, e);
  }
}

// ---- S1 / A / B: the task interpreter -----------------------------------------------------------------------
// The operand indices of one lane-task: NVEC 16-byte vectors of 8 shorts (registers).
template <int NVEC> struct CoopFields { uint4 q[NVEC]; };

template <int NVEC>
MF_HD int coop_fld(const CoopFields<NVEC>& F, int j) {   // j is a compile-time constant after unrolling
  const uint4& v = F.q[j >> 3];
  const int k = (j >> 1) & 3;
  const unsigned w = k == 0 ? v.x : k == 1 ? v.y : k == 2 ? v.z : v.w;
  return (int)(short)((j & 1) ? (w >> 16) : (w & 0xFFFFu));
}

// `tab` is the operand table (kCoopTable; a shared-memory copy on the device), `offset` the round's first vector
template <int NVEC>
MF_HD CoopFields<NVEC> coop_load_fields(const uint4* tab, int offset, int lane) {
  CoopFields<NVEC> F;
#pragma unroll
  for (int v = 0; v < NVEC; ++v) F.q[v] = tab[offset + v * 32 + lane];
  return F;
}

// acc -= V3(J1, P1; J2, P2) for MA x MD sibling pairs (J1[ia], J2[id]); the dot products with the momenta are
// shared between siblings.  V3 = (J1.J2)(P1-P2) + 2 (P2.J1) J2 - 2 (P1.J2) J1  (mf_me_prims.cuh).
template <int MA, int MD>
MF_HD void coop_v3_sub(rvec* acc, const rvec* J1, const rvec& P1, const rvec* J2, const rvec& P2) {
  const rvec dP = rsub(P1, P2);
  double s1[MA], s2[MD];
#pragma unroll
  for (int a = 0; a < MA; ++a) s1[a] = -2.0 * rdot(P2, J1[a]);
#pragma unroll
  for (int d = 0; d < MD; ++d) s2[d] = 2.0 * rdot(P1, J2[d]);
#pragma unroll
  for (int d = 0; d < MD; ++d)
#pragma unroll
    for (int a = 0; a < MA; ++a) {
      const double s12 = -rdot(J1[a], J2[d]);
      rvec& o = acc[a + MA * d];
#pragma unroll
      for (int m = 0; m < 4; ++m) o.v[m] = fma(s2[d], J1[a].v[m], fma(s1[a], J2[d].v[m], fma(s12, dP.v[m], o.v[m])));
    }
}
// acc += V4(J1[ia], J2, J3[id]) with V4 = 2 (J1.J3) J2 - (J2.J3) J1 - (J1.J2) J3: the middle operand is common to the
// siblings, the first varies with ia and the last with id (all three four-gluon vertices of J4 have this shape).
template <int MA, int MD>
MF_HD void coop_v4_add_mid(rvec* acc, const rvec* J1, const rvec& J2, const rvec* J3) {   // V4(J1[a], J2, J3[d])
  double b1[MA], b3[MD];
#pragma unroll
  for (int a = 0; a < MA; ++a) b1[a] = -rdot(J1[a], J2);     // coefficient of J3
#pragma unroll
  for (int d = 0; d < MD; ++d) b3[d] = -rdot(J2, J3[d]);     // coefficient of J1
#pragma unroll
  for (int d = 0; d < MD; ++d)
#pragma unroll
    for (int a = 0; a < MA; ++a) {
      const double a2 = 2.0 * rdot(J1[a], J3[d]);
      rvec& o = acc[a + MA * d];
#pragma unroll
      for (int m = 0; m < 4; ++m) o.v[m] = fma(b1[a], J3[d].v[m], fma(b3[d], J1[a].v[m], fma(a2, J2.v[m], o.v[m])));
    }
}
struct CoopTaskJ2 {   // [out, iP2, eA, PA, eB, PB]:  J2(ab) = -V3(eA, eB) / P_ab^2
  static constexpr int NF = 6, NVEC = 1;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double) {
    double* V = coop_V(scr);
    const rvec J1 = coop_ld_vec(V, coop_fld(F, 2)), P1 = coop_ld_vec(V, coop_fld(F, 3));
    const rvec J2 = coop_ld_vec(V, coop_fld(F, 4)), P2 = coop_ld_vec(V, coop_fld(F, 5));
    rvec acc = {{0.0, 0.0, 0.0, 0.0}};
    coop_v3_sub<1, 1>(&acc, &J1, P1, &J2, P2);
    coop_st_vec(V, coop_fld(F, 0), rscale(acc, coop_X(scr)[coop_fld(F, 1)]));
  }
};

struct CoopTaskX1c {   // [outX, q, idn, eD, v, ub, outCre, outCim]: X1(d) = prop eD-slash v;  cR = ubar gamma X1
  static constexpr int NF = 8, NVEC = 1;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double mt) {
    double* V = coop_V(scr);
    double* S = coop_S(scr);
    const spin t = slash_col(coop_ld_vec(V, coop_fld(F, 3)), coop_ld_spin(S, coop_fld(F, 4)));
    const spin x = prop_col(coop_ld_vec(V, coop_fld(F, 1)), mt, coop_X(scr)[coop_fld(F, 2)], t);
    coop_st_spin(S, coop_fld(F, 0), x);
    const cvec c = bilinear(coop_ld_spin(S, coop_fld(F, 5)), x);
    coop_st_vec(V, coop_fld(F, 6), rvec{{c.re[0], c.re[1], c.re[2], c.re[3]}});
    coop_st_vec(V, coop_fld(F, 7), rvec{{c.im[0], c.im[1], c.im[2], c.im[3]}});
  }
};

struct CoopTaskY1c {   // [outY, q, idn, ub, eA, v0, v1, outC x 4]: Y1(a) = ubar eA-slash prop;  cL(hb) = Y1 gamma v(hb)
  static constexpr int NF = 11, NVEC = 2;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double mt) {
    double* V = coop_V(scr);
    double* S = coop_S(scr);
    const spin t = slash_row(coop_ld_spin(S, coop_fld(F, 3)), coop_ld_vec(V, coop_fld(F, 4)));
    const spin y = prop_row(t, coop_ld_vec(V, coop_fld(F, 1)), mt, coop_X(scr)[coop_fld(F, 2)]);
    coop_st_spin(S, coop_fld(F, 0), y);
    const cvec c0 = bilinear(y, coop_ld_spin(S, coop_fld(F, 5)));
    coop_st_vec(V, coop_fld(F, 7), rvec{{c0.re[0], c0.re[1], c0.re[2], c0.re[3]}});
    coop_st_vec(V, coop_fld(F, 8), rvec{{c0.im[0], c0.im[1], c0.im[2], c0.im[3]}});
    const cvec c1 = bilinear(y, coop_ld_spin(S, coop_fld(F, 6)));
    coop_st_vec(V, coop_fld(F, 9), rvec{{c1.re[0], c1.re[1], c1.re[2], c1.re[3]}});
    coop_st_vec(V, coop_fld(F, 10), rvec{{c1.im[0], c1.im[1], c1.im[2], c1.im[3]}});
  }
};

// J3(abc) = [ -V3(eA, J2bc) - V3(J2ab, eC) + V4(eA, eB, eC) ] / P_abc^2 for M polarisations of c
// [out x M, iP2, eA, PA, J2bc x M, Pbc, J2ab, Pab, eC x M, PC, eB, signs (bit 0: -J2bc, bit 1: -J2ab)]
template <int M> struct CoopTaskJ3 {
  static constexpr int NF = 3 * M + 9, NVEC = (NF + 7) / 8;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double) {
    double* V = coop_V(scr);
    const int sg = coop_fld(F, 3 * M + 8);
    const rvec eA = coop_ld_vec(V, coop_fld(F, M + 1)), PA = coop_ld_vec(V, coop_fld(F, M + 2));
    const rvec Pbc = coop_ld_vec(V, coop_fld(F, 2 * M + 3));
    const rvec J2ab = rflip(coop_ld_vec(V, coop_fld(F, 2 * M + 4)), (sg >> 1) & 1);
    const rvec Pab = coop_ld_vec(V, coop_fld(F, 2 * M + 5)), PC = coop_ld_vec(V, coop_fld(F, 3 * M + 6));
    const rvec eB = coop_ld_vec(V, coop_fld(F, 3 * M + 7));
    rvec J2bc[M], eC[M], acc[M];
#pragma unroll
    for (int m = 0; m < M; ++m) {
      J2bc[m] = rflip(coop_ld_vec(V, coop_fld(F, M + 3 + m)), sg & 1);
      eC[m] = coop_ld_vec(V, coop_fld(F, 2 * M + 6 + m));
      acc[m] = {{0.0, 0.0, 0.0, 0.0}};
    }
    coop_v3_sub<1, M>(acc, &eA, PA, J2bc, Pbc);
    coop_v3_sub<1, M>(acc, &J2ab, Pab, eC, PC);
    coop_v4_add_mid<1, M>(acc, &eA, eB, eC);
    const double ip2 = coop_X(scr)[coop_fld(F, M)];
#pragma unroll
    for (int m = 0; m < M; ++m) coop_st_vec(V, coop_fld(F, m), rscale(acc[m], ip2));
  }
};

// z2 = c0(hb) . J4(abcd), J4 = [ -V3(eA, J3bcd) - V3(J2ab, J2cd) - V3(J3abc, eD) + V4(eA, eB, J2cd) + V4(eA, J2bc, eD)
// + V4(J2ab, eC, eD) ] / P^2 for MA polarisations of a times MD of d
// [out x MA*MD (ia + MA id), iP2, eA x MA, J2ab x MA, J3abc x MA, eD x MD, J2cd x MD, J3bcd x MD, eB, eC, J2bc,
//  Pa, Pbcd, Pab, Pcd, Pabc, Pd, c0, signs (bit 0: -J2ab, 1: -J2cd, 2: -J2bc)]
template <int MA, int MD> struct CoopTaskJ4 {
  static constexpr int MM = MA * MD;
  static constexpr int O_IP2 = MM, O_EA = MM + 1, O_J2AB = O_EA + MA, O_J3ABC = O_J2AB + MA, O_ED = O_J3ABC + MA,
                       O_J2CD = O_ED + MD, O_J3BCD = O_J2CD + MD, O_EB = O_J3BCD + MD, O_EC = O_EB + 1, O_J2BC = O_EB + 2,
                       O_P = O_EB + 3, O_C0 = O_P + 6, O_SG = O_C0 + 1;
  static constexpr int NF = O_SG + 1, NVEC = (NF + 7) / 8;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double) {
    double* V = coop_V(scr);
    const int sg = coop_fld(F, O_SG);
    rvec acc[MM];
#pragma unroll
    for (int m = 0; m < MM; ++m) acc[m] = {{0.0, 0.0, 0.0, 0.0}};
    rvec eA[MA], eD[MD];
#pragma unroll
    for (int a = 0; a < MA; ++a) eA[a] = coop_ld_vec(V, coop_fld(F, O_EA + a));
#pragma unroll
    for (int d = 0; d < MD; ++d) eD[d] = coop_ld_vec(V, coop_fld(F, O_ED + d));
    {
      rvec J3bcd[MD];
#pragma unroll
      for (int d = 0; d < MD; ++d) J3bcd[d] = coop_ld_vec(V, coop_fld(F, O_J3BCD + d));
      coop_v3_sub<MA, MD>(acc, eA, coop_ld_vec(V, coop_fld(F, O_P)), J3bcd, coop_ld_vec(V, coop_fld(F, O_P + 1)));
    }
    {
      rvec J3abc[MA];
#pragma unroll
      for (int a = 0; a < MA; ++a) J3abc[a] = coop_ld_vec(V, coop_fld(F, O_J3ABC + a));
      coop_v3_sub<MA, MD>(acc, J3abc, coop_ld_vec(V, coop_fld(F, O_P + 4)), eD, coop_ld_vec(V, coop_fld(F, O_P + 5)));
    }
    {
      rvec J2ab[MA], J2cd[MD];
#pragma unroll
      for (int a = 0; a < MA; ++a) J2ab[a] = rflip(coop_ld_vec(V, coop_fld(F, O_J2AB + a)), sg & 1);
#pragma unroll
      for (int d = 0; d < MD; ++d) J2cd[d] = rflip(coop_ld_vec(V, coop_fld(F, O_J2CD + d)), (sg >> 1) & 1);
      coop_v3_sub<MA, MD>(acc, J2ab, coop_ld_vec(V, coop_fld(F, O_P + 2)), J2cd, coop_ld_vec(V, coop_fld(F, O_P + 3)));
      coop_v4_add_mid<MA, MD>(acc, eA, coop_ld_vec(V, coop_fld(F, O_EB)), J2cd);
      coop_v4_add_mid<MA, MD>(acc, J2ab, coop_ld_vec(V, coop_fld(F, O_EC)), eD);
    }
    coop_v4_add_mid<MA, MD>(acc, eA, rflip(coop_ld_vec(V, coop_fld(F, O_J2BC)), (sg >> 2) & 1), eD);
    const double ip2 = coop_X(scr)[coop_fld(F, O_IP2)];
    const int ic0 = coop_fld(F, O_C0);
    double* Z = coop_Z(scr);
#pragma unroll
    for (int h = 0; h < 4; ++h) {   // h = 2 hb + k
      const rvec c = rscale(coop_ld_vec(V, ic0 + h), ip2);
#pragma unroll
      for (int m = 0; m < MM; ++m) Z[coop_fld(F, m) + (h >> 1) * kCoopZRow + (h & 1) * kCoopZPlane] = rdot(c, acc[m]);
    }
  }
};

// X2(cd) = prop [ eC-slash X1(d) + J2cd-slash v ] for M polarisations of c
// [out x M, q, idn, X1, v, eC x M, J2 x M, signs (bit 0: -J2)]
template <int M> struct CoopTaskX2 {
  static constexpr int NF = 3 * M + 5, NVEC = (NF + 7) / 8;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double mt) {
    double* V = coop_V(scr);
    double* S = coop_S(scr);
    const int sg = coop_fld(F, 3 * M + 4);
    const spin x1 = coop_ld_spin(S, coop_fld(F, M + 2)), v = coop_ld_spin(S, coop_fld(F, M + 3));
    const rvec q = coop_ld_vec(V, coop_fld(F, M));
    const double idn = coop_X(scr)[coop_fld(F, M + 1)];
#pragma unroll
    for (int m = 0; m < M; ++m) {
      spin t = slash_col(coop_ld_vec(V, coop_fld(F, M + 4 + m)), x1);
      slash_col_acc(t, rflip(coop_ld_vec(V, coop_fld(F, 2 * M + 4 + m)), sg & 1), v);
      coop_st_spin(S, coop_fld(F, m), prop_col(q, mt, idn, t));
    }
  }
};

// Ytilde(ab) = ubar J2ab-slash + Y1(a) eB-slash for M polarisations of b
// [out x M, ub, Y1, J2 x M, eB x M, signs (bit 0: -J2)]
template <int M> struct CoopTaskYt {
  static constexpr int NF = 3 * M + 3, NVEC = (NF + 7) / 8;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double) {
    double* V = coop_V(scr);
    double* S = coop_S(scr);
    const int sg = coop_fld(F, 3 * M + 2);
    const spin ub = coop_ld_spin(S, coop_fld(F, M)), y1 = coop_ld_spin(S, coop_fld(F, M + 1));
#pragma unroll
    for (int m = 0; m < M; ++m) {
      spin t = slash_row(ub, rflip(coop_ld_vec(V, coop_fld(F, M + 2 + m)), sg & 1));
      slash_row_acc(t, y1, coop_ld_vec(V, coop_fld(F, 2 * M + 2 + m)));
      coop_st_spin(S, coop_fld(F, m), t);
    }
  }
};

// z5 = [Y1(a) gamma X1(d)] . J2(bc) for the 4 polarisations of (b, c) and M polarisations of d
// [out x M, bit of pb, bit of pc in the z5 word, Y1, X1 x M, J2bc (variant 0; variants kCoopJ2Stride apart)]
template <int M> struct CoopTaskZ5 {
  static constexpr int NF = 2 * M + 4, NVEC = (NF + 7) / 8;
  MF_HD static void run(double* scr, const CoopFields<NVEC>& F, double) {
    double* V = coop_V(scr);
    double* S = coop_S(scr);
    double* Z = coop_Z(scr);
    const int ob = coop_fld(F, M), oc = coop_fld(F, M + 1), j2 = coop_fld(F, 2 * M + 3);
    const spin y = coop_ld_spin(S, coop_fld(F, M + 2));
    cvec c[M];
#pragma unroll
    for (int m = 0; m < M; ++m) c[m] = bilinear(y, coop_ld_spin(S, coop_fld(F, M + 3 + m)));
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const rvec j = coop_ld_vec(V, j2 + p * kCoopJ2Stride);
      const int off = (p & 1) * ob + (p >> 1) * oc;
#pragma unroll
      for (int m = 0; m < M; ++m) {
        const cplx z = cdot_r(c[m], j);
        Z[coop_fld(F, m) + off] = z.re;
        Z[coop_fld(F, m) + off + kCoopZPlane] = z.im;
      }
    }
  }
};

// One round for one lane: fetch the lane-task's operand indices and run it (idle lanes: field 0 < 0).
template <class Task>
MF_HD void coop_run_task(double* scr, const uint4* tab, int offset, int lane, double mt) {
  const CoopFields<Task::NVEC> F = coop_load_fields<Task::NVEC>(tab, offset, lane);
  if (coop_fld(F, 0) >= 0) Task::run(scr, F, mt);
}

// Host emulation helper (tests/host_shim): all rounds of `phase` of the program of `warp`, for one lane.
MF_HD void coop_run_phase(double* scr, const uint4* tab, int phase, int warp, int lane, double mt) {
  int ph = 0;
#define MF_R(OFF, ...) if (ph == phase) coop_run_task<__VA_ARGS__>(scr, tab, OFF, lane, mt);
#define MF_S() ++ph;
  if (warp == 0) { MF_COOP_WARP0(MF_R, MF_S) } else { MF_COOP_WARP1(MF_R, MF_S) }
#undef MF_R
#undef MF_S
}

// S4 for team thread tid = pols | hb << 4 | k << 5 (k is warp uniform): x^T Cnum x of the real / imaginary parts of
// its helicity combination (colour-matrix numerators; the team sum times 2 / kCoopCden is sum_hel A^dagger C A).
MF_HD double coop_s4_thread(double* scr, int tid) {
  const int pols = tid & 15, hb = (tid >> 4) & 1;
  return coop_s4(coop_V(scr), coop_S(scr), coop_Z(scr), pols, hb, (tid >> 5) & 1);
}

}  // namespace mf
