// no_core.h -- arithmetic of the 3N normal-ordering kernel, written as plain inline functions so
// that the SAME source is compiled into the sm_100a kernel (no_kernel.cuh) and into the host-side
// lane-by-lane emulation that the CPU unit tests drive (tests/host_emu.cpp).  Nothing here is
// shared with oracle/.
//
// Formulation.  With A_123 = (1 - P12)(1 - P13 - P23) (reading R4)
//     M(p,p',P) = G(p,p',P) - P12 G(p,-p',P),      G = T_id - T_13 - T_23,
// and every traced term is expanded in Pauli operators of the two external nucleons.  All k3
// dependence sits in a few scalar "moments"; with k3 = r u (u = unit direction) and the four
// legs x_l = k3 - kappa_l (kappa = k1, k2, k1', k2'), D_l = x_l^2 + mpi^2:
//     first level (one direction, sum over radial nodes, registers):
//        R0 = sum wF,  S_l^k = sum wF r^k / D_l (k=0,1,2),
//        pair (x,y):  g = wF/(D_x D_y), a.b = -x.y = c_xy - (D_x+D_y)/2, h = g (al + be a.b)
//                     HAB = sum h a.b, H0 = sum h, H1 = sum h r
//     second level (sum over directions with angular weight, lane-private shared memory):
//        A0 = sum S^0, A1 = sum S^1 u, A2 = sum S^2 u u^T   (per leg)
//        BS = sum HAB, B0 = sum H0, B1 = sum H1 u           (per pair)
// from which  sum wF x/D = A1 - kappa A0,  sum wF x x^T/D = A2 - sym(A1 kappa^T) + kappa kappa^T A0, ...
// The regulator is evaluated as F = exp(-E0) exp(-dE(d^2)), E0 = (p^2/L^2)^n + (p'^2/L^2)^n the
// k3-independent part of the exponent, dE a degree-n polynomial in d^2 = |k3 - P/2|^2 without a
// constant term: identical to Eq. (13) applied to the in- and outgoing triples (R5), but the
// node-dependent rounding error scales with dE (O(1) where the integrand is large) instead of
// with the full exponent.
#pragma once

#include <math.h>

#ifdef __CUDACC__
#define NO_HD __host__ __device__ __forceinline__
#else
#define NO_HD inline
#endif

namespace no3n {

constexpr int kLanes = 32;
constexpr int kMaxRegPoly = 12;   // largest regulator exponent of the generic path

// kernel-wide constants, all in fm units
struct DevParams {
  const double* tab;      // device tables, see table layout below
  int n_r, n_cos, n_phi;
  int n_pass;             // number of Fermi spheres to integrate (1 or 2)
  int tab_doubles;        // doubles to stage into shared memory (all passes), multiple of 2
  int pass_off[2];        // offset (in doubles) of each pass's tables inside tab
  double nsp[2];          // sum over the species of this pass of 1     (1, or 2 for fused SNM)
  double esum[2];         // sum over the species of this pass of tau_z (+1 proton, -1 neutron, 0 fused)
  double m2;              // mpi^2
  double inv_L2;          // 1/Lambda^2 (0 if unregulated)
  double al, be;          // f(a.b) = al + be a.b:  al = -4 c1 mpi^2/fpi^2, be = 2 c3/fpi^2
  double G2;              // (gA/(2 fpi))^2
  double gD;              // -gA cD/(8 fpi^4 Lchi)
  double gE2;             // cE/(fpi^4 Lchi)
  double g4;              // G2 c4/fpi^2
  int n_reg;              // regulator exponent (generic path)
};

// table layout of one pass: radial nodes as [n_r][4] = (r, r^2, w_r r^2/(2 pi)^3, 0), then
// cos(theta)[n_cos], sin(theta)[n_cos], w_cos[n_cos], cos(phi)[n_phi], sin(phi)[n_phi], w_phi[n_phi]
// (padded to a multiple of 4 doubles so that every pass's radial block stays 32-byte aligned)
NO_HD int tab_pass_doubles(int n_r, int n_cos, int n_phi) { return (4 * n_r + 3 * n_cos + 3 * n_phi + 3) & ~3; }

// second-level accumulator rows
template <bool C4> struct Layout {
  static constexpr int kPairFirst = C4 ? 6 : 3;     // first-level sums per pair
  static constexpr int kPairRows = C4 ? 15 : 5;     // second-level rows per pair
  static constexpr int kRowLeg = 1;                 // row 0 is R0; leg l at 1 + 10 l
  static constexpr int kRowPair = 41;
  static constexpr int kRows = 41 + 4 * kPairRows;  // 61 or 101
};

// legs of the four exchange terms.  pair t uses x-leg kPairX[t] (incoming) and y-leg kPairY[t] (outgoing)
//   t = 0: P13 of G   (a = k3-k1, b = k1'-k3)      t = 1: P23 of G   (a = k3-k2, b = k2'-k3)
//   t = 2: P13 of G~  (a = k3-k1, b = k2'-k3)      t = 3: P23 of G~  (a = k3-k2, b = k1'-k3)
#define NO_PAIR_X(t) ((t) & 1)
#define NO_PAIR_Y(t) (2 + (((t) & 1) ^ ((t) >> 1)))

struct CfgConst {
  double kap[4][3];   // k1, k2, k1', k2'
  double gam[4];      // |kappa_l|^2 + mpi^2
  double hP[3];       // P/2
  double gamd;        // |P/2|^2
  double cpair[4];    // |kappa_x - kappa_y|^2/2 + mpi^2
  double E0;          // k3-independent part of the regulator exponent
  double rc[kMaxRegPoly];  // dE = sum_k rc[k-1] (d^2)^k, k = 1..n
};

template <int NREG>
NO_HD void cfg_setup(const DevParams& P, const double* cfg, CfgConst& c) {
  double p2 = 0, pp2 = 0;
  c.gamd = 0;
  for (int a = 0; a < 3; ++a) {
    const double p = cfg[a], pp = cfg[3 + a], h = 0.5 * cfg[6 + a];
    c.hP[a] = h;
    c.kap[0][a] = h + p;
    c.kap[1][a] = h - p;
    c.kap[2][a] = h + pp;
    c.kap[3][a] = h - pp;
    p2 = fma(p, p, p2);
    pp2 = fma(pp, pp, pp2);
    c.gamd = fma(h, h, c.gamd);
  }
  for (int l = 0; l < 4; ++l)
    c.gam[l] = fma(c.kap[l][0], c.kap[l][0], fma(c.kap[l][1], c.kap[l][1], fma(c.kap[l][2], c.kap[l][2], P.m2)));
  for (int t = 0; t < 4; ++t) {
    const int x = NO_PAIR_X(t), y = NO_PAIR_Y(t);
    double s = 0;
    for (int a = 0; a < 3; ++a) {
      const double d = c.kap[x][a] - c.kap[y][a];
      s = fma(d, d, s);
    }
    c.cpair[t] = fma(0.5, s, P.m2);
  }
  // regulator: (X0 + s3 d2)^n + (X1 + s3 d2)^n = E0 + sum_{k=1..n} C(n,k) (X0^(n-k) + X1^(n-k)) s3^k d2^k
  c.E0 = 0;
  for (int k = 0; k < kMaxRegPoly; ++k) c.rc[k] = 0;
  if (NREG >= 0) {
    const int n = NREG > 0 ? NREG : P.n_reg;
    const double X0 = p2 * P.inv_L2, X1 = pp2 * P.inv_L2, s3 = P.inv_L2 * (1.0 / 3.0);
    double px0[kMaxRegPoly + 1], px1[kMaxRegPoly + 1], ps3[kMaxRegPoly + 1];
    px0[0] = px1[0] = ps3[0] = 1.0;
    for (int j = 1; j <= n; ++j) {
      px0[j] = px0[j - 1] * X0;
      px1[j] = px1[j - 1] * X1;
      ps3[j] = ps3[j - 1] * s3;
    }
    double binom = 1.0;                       // C(n, k), exact in double
    for (int k = 1; k <= n; ++k) {
      binom = binom * (double)(n - k + 1) / (double)k;
      c.rc[k - 1] = binom * (px0[n - k] + px1[n - k]) * ps3[k];
    }
    c.E0 = px0[n] + px1[n];
  }
}

// dE(d2) = d2 (rc0 + d2 (rc1 + ...)), no constant term
template <int NREG>
NO_HD double reg_poly(const DevParams& P, const CfgConst& c, double d2) {
  if (NREG == 1) return d2 * c.rc[0];
  if (NREG == 2) return d2 * fma(d2, c.rc[1], c.rc[0]);
  if (NREG == 3) return d2 * fma(d2, fma(d2, c.rc[2], c.rc[1]), c.rc[0]);
  if (NREG == 4) return d2 * fma(d2, fma(d2, fma(d2, c.rc[3], c.rc[2]), c.rc[1]), c.rc[0]);
  double s = 0;
  for (int k = P.n_reg - 1; k >= 0; --k) s = fma(d2, s, c.rc[k]);
  return d2 * s;
}

// per-direction constants
struct DirConst {
  double u[3];
  double bet[4];   // -2 u.kappa_l
  double betd;     // -2 u.P/2
};

NO_HD void dir_setup(const CfgConst& c, double ux, double uy, double uz, DirConst& d) {
  d.u[0] = ux; d.u[1] = uy; d.u[2] = uz;
  for (int l = 0; l < 4; ++l) d.bet[l] = -2.0 * fma(ux, c.kap[l][0], fma(uy, c.kap[l][1], uz * c.kap[l][2]));
  d.betd = -2.0 * fma(ux, c.hP[0], fma(uy, c.hP[1], uz * c.hP[2]));
}

template <bool C4> struct First {
  double R0;
  double S[4][3];
  double Pr[4][Layout<C4>::kPairFirst];   // !C4: HAB, H0, H1      C4: G0, G1, G2, GA0, GA1, GAA0
};

template <bool C4> NO_HD void first_zero(First<C4>& f) {
  f.R0 = 0;
  for (int l = 0; l < 4; ++l) for (int k = 0; k < 3; ++k) f.S[l][k] = 0;
  for (int t = 0; t < 4; ++t) for (int k = 0; k < Layout<C4>::kPairFirst; ++k) f.Pr[t][k] = 0;
}

NO_HD double no_exp_neg(double e) {   // exp(-e), e >= 0
  return exp(-e);
}

NO_HD double no_rcp(double x) { return 1.0 / x; }

// one k3 node: r, r2 = r^2, wr = w_r r^2/(2 pi)^3   (the HOT loop body)
template <int NREG, bool C4>
NO_HD void node(const DevParams& P, const CfgConst& c, const DirConst& d, double r, double r2, double wr,
                First<C4>& f) {
  double wf = wr;
  if (NREG >= 0) {
    const double d2 = fma(r, r + d.betd, c.gamd);
    wf = wr * no_exp_neg(reg_poly<NREG>(P, c, d2));
  }
  double D[4];
  for (int l = 0; l < 4; ++l) D[l] = fma(r, r + d.bet[l], c.gam[l]);
  // four reciprocals from one division
  const double p01 = D[0] * D[1], p23 = D[2] * D[3];
  const double inv = no_rcp(p01 * p23);
  const double i01 = inv * p23, i23 = inv * p01;
  double iD[4];
  iD[0] = i01 * D[1];
  iD[1] = i01 * D[0];
  iD[2] = i23 * D[3];
  iD[3] = i23 * D[2];
  const double wf1 = wf * r, wf2 = wf * r2;
  f.R0 += wf;
  for (int l = 0; l < 4; ++l) {
    f.S[l][0] = fma(wf, iD[l], f.S[l][0]);
    f.S[l][1] = fma(wf1, iD[l], f.S[l][1]);
    f.S[l][2] = fma(wf2, iD[l], f.S[l][2]);
  }
  const double wi0 = wf * iD[0], wi1 = wf * iD[1];
  for (int t = 0; t < 4; ++t) {
    const int x = NO_PAIR_X(t), y = NO_PAIR_Y(t);
    const double g = (x == 0 ? wi0 : wi1) * iD[y];
    const double ab = fma(-0.5, D[x] + D[y], c.cpair[t]);
    if (!C4) {
      const double h = g * fma(P.be, ab, P.al);
      f.Pr[t][0] = fma(h, ab, f.Pr[t][0]);
      f.Pr[t][1] += h;
      f.Pr[t][2] = fma(h, r, f.Pr[t][2]);
    } else {
      const double ga = g * ab;
      f.Pr[t][0] += g;
      f.Pr[t][1] = fma(g, r, f.Pr[t][1]);
      f.Pr[t][2] = fma(g, r2, f.Pr[t][2]);
      f.Pr[t][3] += ga;
      f.Pr[t][4] = fma(ga, r, f.Pr[t][4]);
      f.Pr[t][5] = fma(ga, ab, f.Pr[t][5]);
    }
  }
}

// second level: acc[row * kLanes + lane] += w_ang * (first-level sum) * (1 | u | u u^T)
template <bool C4>
NO_HD void second_level(const First<C4>& f, const DirConst& d, double w, volatile double* acc /* + lane */) {
  // `volatile`: every row is read, updated and written back in shared memory right here; without it
  // the compiler keeps all rows live in registers across the direction loop and spills them
  const double ux = d.u[0], uy = d.u[1], uz = d.u[2];
  const double wx = w * ux, wy = w * uy, wz = w * uz;
  const double wxx = wx * ux, wxy = wx * uy, wxz = wx * uz, wyy = wy * uy, wyz = wy * uz, wzz = wz * uz;
#define NO_ACCW(row, wgt, val) acc[(row) * kLanes] = fma((wgt), (val), acc[(row) * kLanes])
  NO_ACCW(0, w, f.R0);
  for (int l = 0; l < 4; ++l) {
    const int b = Layout<C4>::kRowLeg + 10 * l;
    NO_ACCW(b + 0, w, f.S[l][0]);
    NO_ACCW(b + 1, wx, f.S[l][1]);
    NO_ACCW(b + 2, wy, f.S[l][1]);
    NO_ACCW(b + 3, wz, f.S[l][1]);
    NO_ACCW(b + 4, wxx, f.S[l][2]);
    NO_ACCW(b + 5, wxy, f.S[l][2]);
    NO_ACCW(b + 6, wxz, f.S[l][2]);
    NO_ACCW(b + 7, wyy, f.S[l][2]);
    NO_ACCW(b + 8, wyz, f.S[l][2]);
    NO_ACCW(b + 9, wzz, f.S[l][2]);
  }
  for (int t = 0; t < 4; ++t) {
    const int b = Layout<C4>::kRowPair + Layout<C4>::kPairRows * t;
    if (!C4) {
      NO_ACCW(b + 0, w, f.Pr[t][0]);    // BS
      NO_ACCW(b + 1, w, f.Pr[t][1]);    // B0
      NO_ACCW(b + 2, wx, f.Pr[t][2]);   // B1
      NO_ACCW(b + 3, wy, f.Pr[t][2]);
      NO_ACCW(b + 4, wz, f.Pr[t][2]);
    } else {
      NO_ACCW(b + 0, w, f.Pr[t][0]);    // G0
      NO_ACCW(b + 1, wx, f.Pr[t][1]);   // G1 u
      NO_ACCW(b + 2, wy, f.Pr[t][1]);
      NO_ACCW(b + 3, wz, f.Pr[t][1]);
      NO_ACCW(b + 4, wxx, f.Pr[t][2]);  // G2 u u^T
      NO_ACCW(b + 5, wxy, f.Pr[t][2]);
      NO_ACCW(b + 6, wxz, f.Pr[t][2]);
      NO_ACCW(b + 7, wyy, f.Pr[t][2]);
      NO_ACCW(b + 8, wyz, f.Pr[t][2]);
      NO_ACCW(b + 9, wzz, f.Pr[t][2]);
      NO_ACCW(b + 10, w, f.Pr[t][3]);   // GA0
      NO_ACCW(b + 11, wx, f.Pr[t][4]);  // GA1 u
      NO_ACCW(b + 12, wy, f.Pr[t][4]);
      NO_ACCW(b + 13, wz, f.Pr[t][4]);
      NO_ACCW(b + 14, w, f.Pr[t][5]);   // GAA0
    }
  }
#undef NO_ACCW
}

// ------------------------------------------------------------------------------------------
// Epilogue, phase 1: from the reduced moments mom[row] of one pass to the Pauli-operator
// records of the four exchange terms (job 0..3) and the two direct terms (job 4, 5).
//   exchange record (kRecX doubles): TA[9] TB[9] sC wC[3] eE | T4[9] n4[3] pad
//   direct   record (kRecD doubles): Dten[9] dE
// ------------------------------------------------------------------------------------------
constexpr int kRecX = 36, kRecD = 10;
constexpr int kRecDoubles = 4 * kRecX + 2 * kRecD;   // 164

// symmetric 3x3 stored as xx,xy,xz,yy,yz,zz
NO_HD void leg_moments(const double* mom, int base, const double* kap, double& A0, double V[3], double T[6]) {
  A0 = mom[base];
  const double a1[3] = {mom[base + 1], mom[base + 2], mom[base + 3]};
  for (int a = 0; a < 3; ++a) V[a] = fma(-kap[a], A0, a1[a]);
  // T = A2 - (A1 kap^T + kap A1^T) + kap kap^T A0  =  A2 - A1 kap^T - kap V^T
  int n = 0;
  for (int a = 0; a < 3; ++a) for (int b = a; b < 3; ++b, ++n)
    T[n] = mom[base + 4 + n] - a1[a] * kap[b] - kap[a] * V[b];
}

NO_HD double sym_at(const double* T, int a, int b) {
  const int lo = a < b ? a : b, hi = a < b ? b : a;
  return T[lo == 0 ? hi : (lo == 1 ? 2 + hi : 5)];
}

NO_HD void cross(const double* a, const double* b, double* c) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

template <bool C4>
NO_HD void phase1_job(const DevParams& P, const CfgConst& c, const double* mom, int job, double* rec) {
  const double R0 = mom[0];
  if (job < 4) {
    const int t = job, x = NO_PAIR_X(t), y = NO_PAIR_Y(t);
    double* o = rec + kRecX * t;
    double kx[3], ky[3];                                   // selects, not indexed loads: c stays in registers
    for (int a = 0; a < 3; ++a) {
      kx[a] = x == 0 ? c.kap[0][a] : c.kap[1][a];
      ky[a] = y == 2 ? c.kap[2][a] : c.kap[3][a];
    }
    double A0x, Va[3], Ta[6], A0y, Vb[3], Tb[6];
    leg_moments(mom, Layout<C4>::kRowLeg + 10 * x, kx, A0x, Va, Ta);
    leg_moments(mom, Layout<C4>::kRowLeg + 10 * y, ky, A0y, Vb, Tb);
    for (int a = 0; a < 3; ++a) Vb[a] = -Vb[a];          // b = -(k3 - kappa_y)
    double Q[3], cv[3];
    for (int a = 0; a < 3; ++a) { Q[a] = ky[a] - kx[a]; cv[a] = -Q[a]; }   // a + b + c = 0
    const double Dc = fma(cv[0], cv[0], fma(cv[1], cv[1], fma(cv[2], cv[2], P.m2)));
    const double iDc = 1.0 / Dc;
    const int pb = Layout<C4>::kRowPair + Layout<C4>::kPairRows * t;
    double BS, B0, B1[3];
    if (!C4) {
      BS = mom[pb]; B0 = mom[pb + 1];
      for (int a = 0; a < 3; ++a) B1[a] = mom[pb + 2 + a];
    } else {
      BS = P.al * mom[pb + 10] + P.be * mom[pb + 14];
      B0 = P.al * mom[pb] + P.be * mom[pb + 10];
      for (int a = 0; a < 3; ++a) B1[a] = P.al * mom[pb + 1 + a] + P.be * mom[pb + 11 + a];
    }
    double hab[3];
    for (int a = 0; a < 3; ++a) hab[a] = fma(-kx[a], B0, B1[a]);
    double va[3], vb[3], Tac[3], Tbc[3];
    for (int a = 0; a < 3; ++a) {
      Tac[a] = sym_at(Ta, a, 0) * cv[0] + sym_at(Ta, a, 1) * cv[1] + sym_at(Ta, a, 2) * cv[2];
      Tbc[a] = sym_at(Tb, a, 0) * cv[0] + sym_at(Tb, a, 1) * cv[1] + sym_at(Tb, a, 2) * cv[2];
      va[a] = P.al * Va[a] + P.be * Tac[a];
      vb[a] = P.al * Vb[a] + P.be * Tbc[a];
    }
    const double trA = Ta[0] + Ta[3] + Ta[5], trB = Tb[0] + Tb[3] + Tb[5];
    const double g2c = P.G2 * iDc, r0c = R0 * iDc;
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
      const double cc = r0c * cv[a] * cv[b];
      o[3 * a + b] = g2c * va[a] * cv[b] + P.gD * (sym_at(Ta, a, b) + cc);       // TA
      o[9 + 3 * a + b] = g2c * vb[a] * cv[b] + P.gD * (sym_at(Tb, a, b) + cc);   // TB
    }
    o[18] = P.G2 * BS + P.gD * (trA + trB);     // sC
    double w[3];
    cross(Q, hab, w);
    for (int a = 0; a < 3; ++a) o[19 + a] = P.G2 * w[a];   // wC
    o[22] = P.gE2 * R0;                          // eE
    for (int a = 0; a < 12; ++a) o[23 + a] = 0;  // T4[9], n4[3] (c4 topology)
    if (C4) {
      // Ga = sum g a, GAa = sum g (a.b) a, Gaa = sum g a a^T   (a = r u - kappa_x)
      double G0, Ga[3], Gaa[6], GA0, GAa[3];
      leg_moments(mom, pb, kx, G0, Ga, Gaa);
      GA0 = mom[pb + 10];
      for (int a = 0; a < 3; ++a) GAa[a] = fma(-kx[a], GA0, mom[pb + 11 + a]);
      (void)G0; (void)Ga;
      double v12[3];
      for (int a = 0; a < 3; ++a) v12[a] = cv[a] * (trA + trB) - (Tac[a] + Tbc[a]);
      // NN = [Q]x Gaa [Q]x^T : columns of CA = Q x (columns of Gaa); rows of NN = Q x (rows of CA)
      double CA[3][3], NN[3][3];
      for (int l = 0; l < 3; ++l) {
        const double col[3] = {sym_at(Gaa, 0, l), sym_at(Gaa, 1, l), sym_at(Gaa, 2, l)};
        double r3[3];
        cross(Q, col, r3);
        for (int i = 0; i < 3; ++i) CA[i][l] = r3[i];
      }
      for (int i = 0; i < 3; ++i) cross(Q, CA[i], NN[i]);
      for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
        o[23 + 3 * a + b] = -P.g4 * (v12[a] * cv[b] * iDc + NN[a][b]);           // T4
      double n4[3];
      cross(Q, GAa, n4);
      for (int a = 0; a < 3; ++a) o[32 + a] = P.g4 * n4[a];                      // n4
    }
  } else {
    const int g = job - 4;            // 0: G (Q = k1' - k1), 1: G~ (Q = k2' - k1)
    double* o = rec + 4 * kRecX + kRecD * g;
    double Q[3];
    for (int a = 0; a < 3; ++a) Q[a] = (g == 0 ? c.kap[2][a] : c.kap[3][a]) - c.kap[0][a];
    const double Q2 = fma(Q[0], Q[0], fma(Q[1], Q[1], Q[2] * Q[2]));
    const double iDQ = 1.0 / (Q2 + P.m2);
    const double coef = 2.0 * R0 * (-P.G2 * (P.al - P.be * Q2) * iDQ * iDQ + 2.0 * P.gD * iDQ);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) o[3 * a + b] = coef * Q[a] * Q[b];
    o[9] = 2.0 * R0 * P.gE2;
  }
}

// ------------------------------------------------------------------------------------------
// Phase 2: lane = 16 g + 4 mu + nu  (g = 0: G, 1: G~;  mu, nu = Pauli index of nucleon 1, 2).
// Adds this pass's coefficient of sigma_1^mu sigma_2^nu in each of the six isospin blocks
//   blk 0 pp->pp, 1 pn->pn, 2 np->np, 3 nn->nn, 4 (row pn, col np), 5 (row np, col pn)
// Scalar and tensor coefficients are real; vector ones (exactly one of mu, nu zero) carry a factor i.
// Isospin operators O1 = 1, O2 = t1z, O3 = t2z, O4 = t1.t2, O5 = i (t1 x t2)_z.
// ------------------------------------------------------------------------------------------
NO_HD void phase2_lane(const double* rec, int lane, double nsp, double esum, double scale, double blk[6]) {
  const int g = lane >> 4, mu = (lane >> 2) & 3, nu = lane & 3;
  const double* r1 = rec + kRecX * (2 * g);        // exchange of nucleon 1
  const double* r2 = rec + kRecX * (2 * g + 1);    // exchange of nucleon 2
  const double* rd = rec + 4 * kRecX + kRecD * g;
  double C1 = 0, C2 = 0, C3 = 0, C4 = 0, C5 = 0;
  if (mu > 0 && nu > 0) {
    const int i = mu - 1, j = nu - 1;
    const double tA = r1[3 * i + j], tB = r1[9 + 3 * i + j];
    const double uA = r2[3 * j + i], uB = r2[9 + 3 * j + i];
    const double t4 = r1[23 + 3 * i + j], u4 = r2[23 + 3 * j + i];
    C2 = -0.5 * esum * (uA + uB) + esum * u4;
    C3 = -0.5 * esum * (tA + tB) + esum * t4;
    C4 = nsp * (rd[3 * i + j] - 0.5 * (tA + tB) - 0.5 * (uA + uB) - t4 - u4);
    C5 = -0.5 * esum * ((tB - tA) + (uA - uB));
  } else if (mu == 0 && nu == 0) {
    const double s1 = r1[18] + r1[22], s2 = r2[18] + r2[22], eE = r1[22], dE = rd[9];
    C1 = -1.5 * nsp * (s1 + s2);
    C2 = esum * (0.5 * s1 - eE + dE);
    C3 = esum * (0.5 * s2 - eE + dE);
    C4 = nsp * (dE - 2.0 * eE);
  } else if (nu == 0) {          // sigma_1^i: i wC of the nucleon-1 exchange; i n4 of the nucleon-2 exchange
    const int i = mu - 1;
    const double w = r1[19 + i], n4 = r2[32 + i];
    C1 = -1.5 * nsp * w;
    C2 = 0.5 * esum * w + esum * n4;
    C4 = -nsp * n4;
  } else {                       // sigma_2^j
    const int j = nu - 1;
    const double w = r2[19 + j], n4 = r1[32 + j];
    C1 = -1.5 * nsp * w;
    C3 = 0.5 * esum * w + esum * n4;
    C4 = -nsp * n4;
  }
  blk[0] += scale * (C1 + C2 + C3 + C4);
  blk[1] += scale * (C1 + C2 - C3 - C4);
  blk[2] += scale * (C1 - C2 + C3 - C4);
  blk[3] += scale * (C1 - C2 - C3 + C4);
  blk[4] += scale * (2.0 * C4 - 2.0 * C5);
  blk[5] += scale * (2.0 * C4 + 2.0 * C5);
}

// ------------------------------------------------------------------------------------------
// Phase 3: matrix element M[row][col] from the block coefficients coef[(16 g + 4 mu + nu) * 6 + blk].
//   M = G - P12 G~ : row (s1,s2,t1,t2) of G~ is read at (s2,s1,t2,t1).
// ------------------------------------------------------------------------------------------
NO_HD int iso_block(int to, int ti) {   // to, ti = 2 t1 + t2; -1 if charge is not conserved
  if (to == ti) return to;              // 0,1,2,3
  if (to == 1 && ti == 2) return 4;
  if (to == 2 && ti == 1) return 5;
  return -1;
}

// <a| sigma^mu |b> = (re + i im); returns false if zero
NO_HD bool pauli_elem(int mu, int a, int b, double& re, double& im) {
  re = 0; im = 0;
  if (mu == 0) { if (a != b) return false; re = 1; return true; }
  if (mu == 3) { if (a != b) return false; re = a == 0 ? 1.0 : -1.0; return true; }
  if (a == b) return false;
  if (mu == 1) { re = 1; return true; }
  im = a == 0 ? -1.0 : 1.0;             // sigma_y[0][1] = -i, [1][0] = +i
  return true;
}

NO_HD void spin_elem(const double* coef, int g, int blk, int s1o, int s2o, int s1i, int s2i, double& re, double& im) {
  re = 0; im = 0;
  for (int mu = 0; mu < 4; ++mu) {
    double ar, ai;
    if (!pauli_elem(mu, s1o, s1i, ar, ai)) continue;
    for (int nu = 0; nu < 4; ++nu) {
      double br, bi;
      if (!pauli_elem(nu, s2o, s2i, br, bi)) continue;
      const double cf = coef[(16 * g + 4 * mu + nu) * 6 + blk];
      double pr = ar * br - ai * bi, pi = ar * bi + ai * br;
      if ((mu == 0) != (nu == 0)) { const double t = pr; pr = -pi; pi = t; }   // vector coefficient: times i
      re = fma(cf, pr, re);
      im = fma(cf, pi, im);
    }
  }
}

NO_HD void phase3_elem(const double* coef, int row, int col, double& re, double& im) {
  re = 0; im = 0;
  const int s1o = (row >> 3) & 1, s2o = (row >> 2) & 1, t1o = (row >> 1) & 1, t2o = row & 1;
  const int s1i = (col >> 3) & 1, s2i = (col >> 2) & 1, ti = col & 3;
  const int b0 = iso_block(2 * t1o + t2o, ti);
  if (b0 < 0) return;
  const int b1 = iso_block(2 * t2o + t1o, ti);
  double gr, gi, hr, hi;
  spin_elem(coef, 0, b0, s1o, s2o, s1i, s2i, gr, gi);
  spin_elem(coef, 1, b1, s2o, s1o, s1i, s2i, hr, hi);
  re = gr - hr;
  im = gi - hi;
}

}  // namespace no3n
