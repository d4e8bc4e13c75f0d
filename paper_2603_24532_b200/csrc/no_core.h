// no_core.h -- arithmetic of the 3N normal-ordering kernel, written as plain inline functions so
// that the SAME source is compiled into the sm_100a kernel (no_kernel.cuh) and into the host-side
// lane-by-lane emulation that the CPU unit tests drive (tests/host_emu.cpp).  Nothing here is
// shared with oracle/.
//
// Formulation.  With A_123 = (1 - P12)(1 - P13 - P23) (reading R4)
//     M(p,p',P) = G(p,p',P) - P12 G(p,-p',P),      G = T_id - T_13 - T_23,
// and every traced term is expanded in Pauli operators of the two external nucleons.  All k3
// dependence sits in a few scalar "moments"; with k3 = r u (u = unit direction) and the four
// legs x_l = k3 - kappa_l (kappa = k1, k2, k1', k2'), D_l = x_l^2 + mpi^2 = r^2 + bet_l r + gam_l:
//     first level (one direction, sum over the radial nodes, 17 registers):
//        R0 = sum wF,   S_l^k = sum wF r^k / D_l   (k = 0,1; 4 legs),
//        G_t^k = sum wF r^k / (D_x D_y)             (k = 0,1; 4 exchange pairs t = (x,y))
//     per direction, from those:  S_l^2 = sum wF r^2/D_l = R0 - bet_l S_l^1 - gam_l S_l^0
//                                 (c4 only) G_t^2 = S_y^0 - bet_x G_t^1 - gam_x G_t^0
//     second level (sum over directions with the angular weight, lane-private shared memory):
//        A0 = sum S^0, A1 = sum S^1 u, A2 = sum S^2 u u^T   (per leg)
//        Gm0 = sum G^0, Gm1 = sum G^1 u  [, Gm2 = sum G^2 u u^T]   (per pair)
//     epilogue: with a.b = -x_x.x_y = c_xy - (D_x + D_y)/2 every moment of g (a.b)^j, g = wF/(D_x D_y),
//        follows from the ones above (phase1_job), e.g.
//        sum g a.b = c Gm0 - (A0_x + A0_y)/2,
//        sum g (a.b)^2 = c^2 Gm0 - c (A0_x + A0_y) + R0 + [(gam_x-gam_y)(A0_y-A0_x) - 2 (kappa_x-kappa_y).(A1_y-A1_x)]/4,
//        sum wF x/D = A1 - kappa A0,  sum wF x x^T/D = A2 - A1 kappa^T - kappa (A1 - kappa A0)^T, ...
// The regulator is evaluated as F = exp(-E0) exp(-dE(d^2)), E0 = (p^2/L^2)^n + (p'^2/L^2)^n the
// k3-independent part of the exponent, dE a degree-n polynomial in d^2 = |k3 - P/2|^2 without a
// constant term: identical to Eq. (13) applied to the in- and outgoing triples (R5), but the
// node-dependent rounding error scales with dE (O(1) where the integrand is large) instead of
// with the full exponent.  exp(-dE) is a branch-free 2^(s/N), s = -N log2(e) dE, N = kExpTab = 256:
// table of 2^(j/N), degree-4 polynomial on the remainder, exponent added as an integer.
#pragma once

#include <math.h>
#include <stdint.h>
#include <string.h>

#ifdef __CUDACC__
#define NO_HD __host__ __device__ __forceinline__
#else
#define NO_HD inline
#endif

namespace no3n {

constexpr int kLanes = 32;
constexpr int kMaxRegPoly = 12;   // largest regulator exponent of the generic path
constexpr int kMaxNr = 128;      // largest radial order (n_r_pad <= kMaxNr)
#ifndef NO_EXPTAB
#define NO_EXPTAB 256
#endif
constexpr int kExpTab = NO_EXPTAB;   // entries of the 2^(j/kExpTab) table at the start of the device tables (64 or 256)
static_assert(kExpTab == 64 || kExpTab == 256, "exp table size");
#ifndef NO_NPT
#define NO_NPT 4
#endif
constexpr int kNodesPerTrip = NO_NPT;
static_assert(128 % NO_NPT == 0, "n_r_pad must not exceed kMaxNr");  // radial nodes per trip of the hot loop (n_r is padded to a multiple)

// kernel-wide constants, all in fm units
struct DevParams {
  const double* tab;      // device tables, see table layout below
  int n_r, n_cos, n_phi;
  int n_list;             // > 0: caller-supplied angular rule of n_list directions replaces the cos x phi grid
  int n_r_pad;            // n_r rounded up to a multiple of kNodesPerTrip; padding nodes have weight 0
  int n_pass;             // number of Fermi spheres to integrate (1 or 2)
  int tab_doubles;        // doubles to stage into shared memory (exp table + all passes), multiple of 2
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
  double kf_max;          // largest Fermi momentum of the passes
  double radk[2][kMaxNr][2];  // per pass: (r_i, w_i r_i^2/(2 pi)^3), i < n_r_pad (weight 0 on the padding):
                              // read in the hot loop through the constant bank (uniform operands)
};

// table layout: tab[0..kExpTab) = 2^(j/kExpTab); then for each pass: radial nodes as [n_r_pad][2] =
// (r, w_r r^2/(2 pi)^3), then cos(theta)[n_cos], sin(theta)[n_cos], w_cos[n_cos], cos(phi)[n_phi],
// sin(phi)[n_phi], w_phi[n_phi] (padded to a multiple of 4 doubles: every radial block 32-byte aligned)
// (list mode: the six angular arrays are replaced by dirs[n_list][4] = (ux, uy, uz, w))
NO_HD int tab_pass_doubles(int n_r_pad, int n_cos, int n_phi, int n_list) {
  return n_list > 0 ? 2 * n_r_pad + 4 * n_list : (2 * n_r_pad + 3 * n_cos + 3 * n_phi + 3) & ~3;
}

// second-level accumulator rows
template <bool C4> struct Layout {
  static constexpr int kPairRows = C4 ? 10 : 4;     // Gm0, Gm1[3] (, Gm2[6])
  static constexpr int kRowLeg = 0;                 // leg l at 10 l: A0, A1[3], A2[6]
  static constexpr int kRowPair = 40;               // pair t at 40 + kPairRows t
  static constexpr int kRowR0 = 40 + 4 * kPairRows; // R0 is the last row
  static constexpr int kRows = kRowR0 + 1;          // 57 or 81
  // the accumulators are lane-major in shared memory, acc[lane * kStride + row], and are read and
  // written as 16-byte pairs; kStride / 2 is odd, so the eight lanes of a quarter warp hit eight
  // different 16-byte bank groups
  static constexpr int kStride = kRows + 1;         // 58 or 82
};

// legs of the four exchange terms.  pair t uses x-leg kPairX[t] (incoming) and y-leg kPairY[t] (outgoing)
//   t = 0: P13 of G   (a = k3-k1, b = k1'-k3)      t = 1: P23 of G   (a = k3-k2, b = k2'-k3)
//   t = 2: P13 of G~  (a = k3-k1, b = k2'-k3)      t = 3: P23 of G~  (a = k3-k2, b = k1'-k3)
#define NO_PAIR_X(t) ((t) & 1)
#define NO_PAIR_Y(t) (2 + (((t) & 1) ^ ((t) >> 1)))

// per-configuration constants; the kernel keeps one copy per warp in shared memory
struct CfgConst {
  double kap[4][3];   // k1, k2, k1', k2'
  double gam[4];      // |kappa_l|^2 + mpi^2
  double hP[3];       // P/2
  double gamd;        // |P/2|^2
  double cpair[4];    // |kappa_x - kappa_y|^2/2 + mpi^2
  double E0;          // k3-independent part of the regulator exponent
  double rs[kMaxRegPoly];  // s = -64 log2(e) dE = sum_k rs[k-1] (d^2)^k, k = 1..n
  double smin;        // lower bound of s over the Fermi spheres (s at d^2 = 2 (kF_max^2 + |P/2|^2)); NaN if cfg is not finite
  double pad_[2];     // 40 doubles: keeps what follows in shared memory 32-byte aligned
};
constexpr int kCfgDoubles = sizeof(CfgConst) / sizeof(double);
static_assert(kCfgDoubles == 40, "CfgConst layout");

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
  for (int k = 0; k < kMaxRegPoly; ++k) c.rs[k] = 0;
  for (int k = 0; k < 2; ++k) c.pad_[k] = 0;
  c.smin = 0;
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
    const double scale = -1.4426950408889634 * kExpTab;   // -kExpTab log2(e)
    double binom = 1.0;                       // C(n, k), exact in double
    for (int k = 1; k <= n; ++k) {
      binom = binom * (double)(n - k + 1) / (double)k;
      c.rs[k - 1] = scale * (binom * (px0[n - k] + px1[n - k]) * ps3[k]);
    }
    c.E0 = px0[n] + px1[n];
    // s = d2 h(d2) decreases with d2 (all rs <= 0); d2 = |k3 - P/2|^2 <= (kF_max + |P/2|)^2 <= 2 (kF_max^2 + |P/2|^2)
    // (the second bound needs no square root: 21 dependent FP64 instructions less in every prologue; it is only used
    //  to decide whether the hot loop needs its underflow guard)
    const double d2max = 2.0 * fma(P.kf_max, P.kf_max, c.gamd);
    double h = c.rs[n - 1];
    for (int k = n - 2; k >= 0; --k) h = fma(d2max, h, c.rs[k]);
    c.smin = d2max * h;
  }
}

// the hot loop may skip the underflow guard of exp2_table when s >= kFlushBelow at every node
constexpr double kFlushBelow = -1015.625 * kExpTab;   // -65000 for 64 entries: exp(-dE) < 1e-305
NO_HD bool needs_flush(const CfgConst& c) { return !(c.smin > kFlushBelow); }

// ---- bit access to doubles ----
NO_HD int hi32(double x) {
#ifdef __CUDA_ARCH__
  return __double2hiint(x);
#else
  uint64_t u; memcpy(&u, &x, 8); return (int)(uint32_t)(u >> 32);
#endif
}
NO_HD int lo32(double x) {
#ifdef __CUDA_ARCH__
  return __double2loint(x);
#else
  uint64_t u; memcpy(&u, &x, 8); return (int)(uint32_t)u;
#endif
}
NO_HD double hilo(int hi, int lo) {
#ifdef __CUDA_ARCH__
  return __hiloint2double(hi, lo);
#else
  const uint64_t u = ((uint64_t)(uint32_t)hi << 32) | (uint32_t)lo; double x; memcpy(&x, &u, 8); return x;
#endif
}

// exp(-dE(d2)) = 2^(s/64), s = d2 * h(d2) <= 0, h = rs0 + d2 (rs1 + ...).  Branch free:
//   tm = s + 1.5 2^52 holds round(s) in its low mantissa bits, f = s - round(s) in [-1/2, 1/2],
//   2^(s/N) = 2^floor(ky/N) * tab[ky mod N] * exp(f ln2/N)  (Taylor polynomial, |error| < 4e-17).
// Below s = -65000 (exp(-dE) < 1e-305) the result is replaced by a subnormal (< 3e-308), i.e. zero
// (FLUSH); configurations whose bound smin shows that no node gets there run without that guard.
// The stages are separate functions so that the W nodes of one trip can be interleaved.
template <int NREG>
NO_HD double reg_h(const double* rs, int n_reg, double d2) {
  if (NREG == 1) return rs[0];
  if (NREG == 2) return fma(d2, rs[1], rs[0]);
  if (NREG == 3) return fma(d2, fma(d2, rs[2], rs[1]), rs[0]);
  if (NREG == 4) return fma(d2, fma(d2, fma(d2, rs[3], rs[2]), rs[1]), rs[0]);
  double h = rs[n_reg - 1];
  for (int k = n_reg - 2; k >= 0; --k) h = fma(d2, h, rs[k]);
  return h;
}

constexpr double kMagic = 6755399441055744.0;             // 1.5 * 2^52

// scaled table value 2^(ky/64) from tm = s + kMagic and kf = round(s).  Index and exponent are taken
// with multiply-adds only (n = floor(ky/64) as the high word of ky 2^26): on B200 the logic/shift
// pipe shares issue bandwidth with the FP64 pipe, the integer multiply-add pipe does not.
NO_HD int mulhi32(int a, int b) {
#ifdef __CUDA_ARCH__
  return __mulhi(a, b);
#else
  return (int)(((long long)a * (long long)b) >> 32);
#endif
}

template <bool FLUSH>
NO_HD double exp2_table(double tm, double kf, const double* e2tab) {
  const int ky = lo32(tm);
  const int n = mulhi32(ky, (int)(4294967296LL / kExpTab));   // floor(ky / kExpTab)
  const double T = e2tab[ky - kExpTab * n];               // ky mod kExpTab in [0, kExpTab)
  int hiT = hi32(T) + n * 1048576;                        // exponent field += n
  if (FLUSH) hiT = !(kf >= kFlushBelow) ? 0 : hiT;        // kf below the bound (or not finite): flush
  return hilo(hiT, lo32(T));
}

// exp(f ln2/kExpTab), |f| <= 1/2: Taylor polynomial, degree 5 for 64 entries (|error| < 4e-17), degree 4
// for 256 entries (|x| <= 1.36e-3, x^5/120 < 4e-17); coefficients (ln2/kExpTab)^m / m!
NO_HD double exp2_poly(double f) {
  if (kExpTab == 64) {
    const double c1 = 0.010830424696249145, c2 = 5.864904955056169e-05, c3 = 2.1173137155464774e-07, c4 = 5.732851688640402e-10, c5 = 1.2417843701716923e-12;
    double p = fma(f, c5, c4);
    p = fma(f, p, c3);
    p = fma(f, p, c2);
    p = fma(f, p, c1);
    return fma(f, p, 1.0);
  } else {
    const double c1 = 0.0027076061740622863, c2 = 3.665565596910106e-06, c3 = 3.308302680541371e-09, c4 = 2.239395190875157e-12;
    double p = fma(f, c4, c3);
    p = fma(f, p, c2);
    p = fma(f, p, c1);
    return fma(f, p, 1.0);
  }
}

// hardware seed of 1/x (relative error <= 2^-20, measured), x normal and positive
NO_HD double rcp_seed(double d) {
#ifdef __CUDA_ARCH__
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(d));
  return x;
#else
  return hilo(hi32(1.0 / hilo(hi32(d), 0)), 0);           // emulation of the seed: high word only
#endif
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

// first-level sums of one direction
struct First {
  double R0;
  double S[4][2];
  double G[4][2];
};

NO_HD void first_zero(First& f) {
  f.R0 = 0;
  for (int l = 0; l < 4; ++l) f.S[l][0] = f.S[l][1] = 0;
  for (int t = 0; t < 4; ++t) f.G[t][0] = f.G[t][1] = 0;
}

// per-warp radial table entry (shared memory): r^2 + |P/2|^2, r^2 + gam_l (l = 0..3), pad
constexpr int kRadT = 6;

NO_HD void radial_entry(const CfgConst& c, double r, double* T) {
  T[0] = fma(r, r, c.gamd);
  for (int l = 0; l < 4; ++l) T[1 + l] = fma(r, r, c.gam[l]);
  T[5] = 0.0;
}

// W k3 nodes of one direction at once (the HOT loop body): r, wr = w_r r^2/(2 pi)^3
// (the same for every lane: the kernel passes them from the constant bank, i.e. as uniform-register
// operands), T = radial_entry.  Every step is written for all W nodes before the next one, so that the W
// independent dependency chains interleave in the instruction stream (FP64 latency is 8 cycles at
// one instruction per 2 cycles).
//
// An FP64 instruction with three distinct 64-bit REGISTER operands occupies the pipe for 3 cycles
// instead of 2 (profiles/r01b.md), so the body is arranged to need at most two: the weight wF is
// folded into the shared reciprocal, y = wF/(D0 D1 D2 D3), the pair and leg terms are products of y
// with the D's, the k = 0 sums are plain additions and the k = 1 sums are FMAs with the uniform r.
//
// FWD: forward configurations p' = p (the Hartree-Fock contractions): k1' = k1 and k2' = k2, so legs 2, 3 coincide
// with legs 0, 1 and pair 3 with pair 2.  The duplicates are not computed: D2 = D0, D3 = D1 (the common
// subexpressions collapse), S[2], S[3], G[3] are not accumulated (first_fwd_fill copies them per direction).
template <int NREG, int W, bool FLUSH, bool FWD = false>
NO_HD void nodes(const double* rs, int n_reg, const double* e2tab, const DirConst& d, const double* r,
                 const double* wr, const double (*T)[5], First& f) {
  double F[W], D0[W], D1[W], D2[W], D3[W], q02[W], q13[W], q03[W], q12[W], den[W], x[W];
#pragma unroll
  for (int k = 0; k < W; ++k) {
    D0[k] = fma(d.bet[0], r[k], T[k][1]);
    D1[k] = fma(d.bet[1], r[k], T[k][2]);
    D2[k] = FWD ? D0[k] : fma(d.bet[2], r[k], T[k][3]);
    D3[k] = FWD ? D1[k] : fma(d.bet[3], r[k], T[k][4]);
  }
#pragma unroll
  for (int k = 0; k < W; ++k) { q02[k] = D0[k] * D2[k]; q13[k] = D1[k] * D3[k]; }
#pragma unroll
  for (int k = 0; k < W; ++k) den[k] = q02[k] * q13[k];
#pragma unroll
  for (int k = 0; k < W; ++k) x[k] = rcp_seed(den[k]);
#pragma unroll
  for (int k = 0; k < W; ++k) { q03[k] = D0[k] * D3[k]; q12[k] = FWD ? q03[k] : D1[k] * D2[k]; }
  if (NREG >= 0) {
    double d2[W], h[W], tm[W], kf[W], fr[W], Ts[W];
#pragma unroll
    for (int k = 0; k < W; ++k) d2[k] = fma(d.betd, r[k], T[k][0]);
#pragma unroll
    for (int k = 0; k < W; ++k) h[k] = reg_h<NREG>(rs, n_reg, d2[k]);
#pragma unroll
    for (int k = 0; k < W; ++k) tm[k] = fma(d2[k], h[k], kMagic);
#pragma unroll
    for (int k = 0; k < W; ++k) kf[k] = tm[k] - kMagic;                 // round(s), exact
#pragma unroll
    for (int k = 0; k < W; ++k) fr[k] = fma(d2[k], h[k], -kf[k]);       // s - round(s), one rounding
#pragma unroll
    for (int k = 0; k < W; ++k) Ts[k] = exp2_table<FLUSH>(tm[k], kf[k], e2tab);
#pragma unroll
    for (int k = 0; k < W; ++k) F[k] = exp2_poly(fr[k]);
#pragma unroll
    for (int k = 0; k < W; ++k) F[k] *= Ts[k];
  } else {
#pragma unroll
    for (int k = 0; k < W; ++k) F[k] = 1.0;
  }
  // 1/den: seed and one cubic step, x (1 + e + e^2), e = 1 - den x (relative error 2^-60 + rounding)
  double e[W];
#pragma unroll
  for (int k = 0; k < W; ++k) e[k] = fma(-den[k], x[k], 1.0);
#pragma unroll
  for (int k = 0; k < W; ++k) e[k] = fma(e[k], e[k], e[k]);
#pragma unroll
  for (int k = 0; k < W; ++k) x[k] = fma(x[k], e[k], x[k]);
  double wf[W], y[W], g0[W], g1[W], g2[W], g3[W], i0[W], i1[W], i2[W], i3[W];
#pragma unroll
  for (int k = 0; k < W; ++k) wf[k] = F[k] * wr[k];
#pragma unroll
  for (int k = 0; k < W; ++k) y[k] = x[k] * wf[k];
#pragma unroll
  for (int k = 0; k < W; ++k) {
    g0[k] = y[k] * q13[k];   // wF/(D0 D2): pair 0 = legs (0, 2)
    g1[k] = y[k] * q02[k];   // wF/(D1 D3): pair 1 = legs (1, 3)
    g2[k] = y[k] * q12[k];   // wF/(D0 D3): pair 2 = legs (0, 3)
    g3[k] = FWD ? g2[k] : y[k] * q03[k];   // wF/(D1 D2): pair 3 = legs (1, 2)
  }
#pragma unroll
  for (int k = 0; k < W; ++k) {
    i0[k] = g0[k] * D2[k];   // wF/D0
    i2[k] = FWD ? i0[k] : g0[k] * D0[k];   // wF/D2
    i1[k] = g1[k] * D3[k];   // wF/D1
    i3[k] = FWD ? i1[k] : g1[k] * D1[k];   // wF/D3
  }
#pragma unroll
  for (int k = 0; k < W; ++k) {
    f.R0 += wf[k];
    f.S[0][0] += i0[k];
    f.S[1][0] += i1[k];
    if (!FWD) { f.S[2][0] += i2[k]; f.S[3][0] += i3[k]; }
    f.G[0][0] += g0[k];
    f.G[1][0] += g1[k];
    f.G[2][0] += g2[k];
    if (!FWD) f.G[3][0] += g3[k];
    f.S[0][1] = fma(i0[k], r[k], f.S[0][1]);
    f.S[1][1] = fma(i1[k], r[k], f.S[1][1]);
    if (!FWD) { f.S[2][1] = fma(i2[k], r[k], f.S[2][1]); f.S[3][1] = fma(i3[k], r[k], f.S[3][1]); }
    f.G[0][1] = fma(g0[k], r[k], f.G[0][1]);
    f.G[1][1] = fma(g1[k], r[k], f.G[1][1]);
    f.G[2][1] = fma(g2[k], r[k], f.G[2][1]);
    if (!FWD) f.G[3][1] = fma(g3[k], r[k], f.G[3][1]);
  }
}

// second level: acc[lane * kStride + row] += w_ang * (first-level sum) * (1 | u | u u^T)
// The rows are updated in groups (all loads of a group, then the FMAs, then the stores) so that the
// shared-memory latency is paid once per group; the compiler fences at both ends keep it from
// carrying the rows in registers across the direction loop.
#define NO_FENCE() asm volatile("" ::: "memory")

struct alignas(16) Pair { double x, y; };

// a: 10 consecutive rows of one lane (16-byte aligned): 1 | u | u u^T
// FIRST: the rows hold nothing yet (first direction of the lane in this pass): they are written, not updated, which
// saves the zero fill of the accumulators and one round of loads; fma(a, b, 0) and a * b round alike.
template <bool FIRST>
NO_HD void rmw_rank012(double* a, const double* wt, double s0, double s1, double s2) {
  Pair* p = reinterpret_cast<Pair*>(a);
  Pair v[5];
  for (int k = 0; k < 5; ++k) v[k] = FIRST ? Pair{0.0, 0.0} : p[k];
  v[0].x = fma(wt[0], s0, v[0].x); v[0].y = fma(wt[1], s1, v[0].y);
  v[1].x = fma(wt[2], s1, v[1].x); v[1].y = fma(wt[3], s1, v[1].y);
  v[2].x = fma(wt[4], s2, v[2].x); v[2].y = fma(wt[5], s2, v[2].y);
  v[3].x = fma(wt[6], s2, v[3].x); v[3].y = fma(wt[7], s2, v[3].y);
  v[4].x = fma(wt[8], s2, v[4].x); v[4].y = fma(wt[9], s2, v[4].y);
  for (int k = 0; k < 5; ++k) p[k] = v[k];
}

// FWD: the rows of legs 2, 3 and of pair 3 are left untouched (the kernel copies them from legs 0, 1 and pair 2
// after the lane reduction)
template <bool C4, bool FWD = false, bool FIRST = false>
NO_HD void second_level(const First& f, const DirConst& d, const double* gam, double w, double* acc /* this lane's rows */) {
  const double ux = d.u[0], uy = d.u[1], uz = d.u[2];
  double wt[10];      // w * (1, ux, uy, uz, ux ux, ux uy, ux uz, uy uy, uy uz, uz uz)
  wt[0] = w; wt[1] = w * ux; wt[2] = w * uy; wt[3] = w * uz;
  wt[4] = wt[1] * ux; wt[5] = wt[1] * uy; wt[6] = wt[1] * uz; wt[7] = wt[2] * uy; wt[8] = wt[2] * uz; wt[9] = wt[3] * uz;
  NO_FENCE();
  for (int l = 0; l < (FWD ? 2 : 4); ++l) {
    const double S2 = fma(-gam[l], f.S[l][0], fma(-d.bet[l], f.S[l][1], f.R0));   // sum wF r^2 / D_l
    rmw_rank012<FIRST>(acc + Layout<C4>::kRowLeg + 10 * l, wt, f.S[l][0], f.S[l][1], S2);
  }
  if (C4) {
    for (int t = 0; t < (FWD ? 3 : 4); ++t) {
      const int x = NO_PAIR_X(t), y = FWD ? (NO_PAIR_Y(t) - 2) : NO_PAIR_Y(t);          // FWD: leg y coincides with y - 2
      const double G2 = fma(-gam[x], f.G[t][0], fma(-d.bet[x], f.G[t][1], f.S[y][0]));   // sum wF r^2/(D_x D_y)
      rmw_rank012<FIRST>(acc + Layout<C4>::kRowPair + 10 * t, wt, f.G[t][0], f.G[t][1], G2);     // Gm0, Gm1, Gm2
    }
  } else {
    Pair* p = reinterpret_cast<Pair*>(acc + Layout<C4>::kRowPair);   // Gm0, Gm1[3] of the four pairs
    constexpr int np = FWD ? 3 : 4;
    Pair v[8];
    for (int k = 0; k < 2 * np; ++k) v[k] = FIRST ? Pair{0.0, 0.0} : p[k];
    for (int t = 0; t < np; ++t) {
      v[2 * t].x = fma(wt[0], f.G[t][0], v[2 * t].x);
      v[2 * t].y = fma(wt[1], f.G[t][1], v[2 * t].y);
      v[2 * t + 1].x = fma(wt[2], f.G[t][1], v[2 * t + 1].x);
      v[2 * t + 1].y = fma(wt[3], f.G[t][1], v[2 * t + 1].y);
    }
    for (int k = 0; k < 2 * np; ++k) p[k] = v[k];
  }
  acc[Layout<C4>::kRowR0] = FIRST ? w * f.R0 : fma(w, f.R0, acc[Layout<C4>::kRowR0]);
  NO_FENCE();
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
  const double R0 = mom[Layout<C4>::kRowR0];
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
    // moments of g (a.b)^j, g = wF/(D_x D_y), a.b = c_xy - (D_x + D_y)/2, from Gm0, Gm1 and the leg moments
    const int lx = Layout<C4>::kRowLeg + 10 * x, ly = Layout<C4>::kRowLeg + 10 * y;
    const double Gm0 = mom[pb], ct = c.cpair[t];
    const double sA0 = mom[lx] + mom[ly], dA0 = mom[ly] - mom[lx];
    const double GA0 = fma(ct, Gm0, -0.5 * sA0);                       // sum g a.b
    double GA1[3], dkA1 = 0;                                           // sum g a.b r u
    for (int a = 0; a < 3; ++a) {
      GA1[a] = fma(ct, mom[pb + 1 + a], -0.5 * (mom[lx + 1 + a] + mom[ly + 1 + a]));
      dkA1 = fma(kx[a] - ky[a], mom[ly + 1 + a] - mom[lx + 1 + a], dkA1);
    }
    const double gx = x == 0 ? c.gam[0] : c.gam[1], gy = y == 2 ? c.gam[2] : c.gam[3];
    const double GAA0 = fma(ct, GA0 - 0.5 * sA0, R0) + 0.25 * fma(gx - gy, dA0, -2.0 * dkA1);   // sum g (a.b)^2
    const double BS = fma(P.al, GA0, P.be * GAA0);                     // sum h a.b, h = g (al + be a.b)
    const double B0 = fma(P.al, Gm0, P.be * GA0);                      // sum h
    double B1[3];                                                      // sum h r u
    for (int a = 0; a < 3; ++a) B1[a] = fma(P.al, mom[pb + 1 + a], P.be * GA1[a]);
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
      double G0, Ga[3], Gaa[6], GAa[3];
      leg_moments(mom, pb, kx, G0, Ga, Gaa);
      for (int a = 0; a < 3; ++a) GAa[a] = fma(-kx[a], GA0, GA1[a]);
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

// sum_{mu,nu} coef[g][mu][nu][blk] <ao|sigma^mu|ai> <bo|sigma^nu|bi>, times i for the vector coefficients
// (exactly one of mu, nu zero).  For given spin projections only two mu contribute: (0, 3) on the
// diagonal, (1, 2) off it, with <a|1|a> = <a|sigma_x|b> = 1, <a|sigma_z|a> = +1/-1 and
// <0|sigma_y|1> = -i, <1|sigma_y|0> = +i; every term is coef * i^k, k = ka + kb + kv (mod 4).
NO_HD void spin_elem(const double* coef, int g, int blk, int ao, int bo, int ai, int bi, double& re, double& im) {
  const int da = ao ^ ai, db = bo ^ bi;
  const int mu[2] = {da, 3 - da}, nu[2] = {db, 3 - db};
  const int ka[2] = {0, da ? (ao ? 1 : 3) : (ao ? 2 : 0)};
  const int kb[2] = {0, db ? (bo ? 1 : 3) : (bo ? 2 : 0)};
  re = 0; im = 0;
#ifdef __CUDA_ARCH__
#pragma unroll
#endif
  for (int x = 0; x < 2; ++x) {
#ifdef __CUDA_ARCH__
#pragma unroll
#endif
    for (int y = 0; y < 2; ++y) {
      const double cf = coef[(16 * g + 4 * mu[x] + nu[y]) * 6 + blk];
      const int k = ka[x] + kb[y] + (((mu[x] == 0) != (nu[y] == 0)) ? 1 : 0);
      const double v = (k & 2) ? -cf : cf;
      if (k & 1) im += v; else re += v;
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

// ------------------------------------------------------------------------------------------
// Phase 3, lane-mapped (what the kernel runs for the full matrix): lane = 2 sc + h, sc = 8 s1o + 4 s2o +
// 2 s1i + s2i a fixed spin element; the six charge-conserving isospin blocks nb = 2 it + h are visited
// in three steps, the ten structurally zero blocks in five.  For a fixed spin element only four
// (mu, nu) terms of G and four of G~ contribute, each with a constant unit i^k: offsets and units are
// computed once per lane, a block costs 8 loads and 16 multiply-adds.  Same sum as phase3_elem.
// ------------------------------------------------------------------------------------------
struct P3Lane {
  int spin_off;             // element offset of the spin part: 16 (8 s1o + 4 s2o) + 8 s1i + 4 s2i
  int cof[2][4];            // coefficient offsets (16 g + 4 mu + nu) 6 of the four terms of G (0) and G~ (1)
  double pr[2][4], pi[2][4];   // their units i^k as (re, im)
};

NO_HD void phase3_terms(int g, int ao, int bo, int ai, int bi, int* cof, double* pr, double* pi) {
  const int da = ao ^ ai, db = bo ^ bi;
  const int mu[2] = {da, 3 - da}, nu[2] = {db, 3 - db};
  const int ka[2] = {0, da ? (ao ? 1 : 3) : (ao ? 2 : 0)};
  const int kb[2] = {0, db ? (bo ? 1 : 3) : (bo ? 2 : 0)};
  for (int x = 0; x < 2; ++x)
    for (int y = 0; y < 2; ++y) {
      const int k = (ka[x] + kb[y] + (((mu[x] == 0) != (nu[y] == 0)) ? 1 : 0)) & 3;
      cof[2 * x + y] = (16 * g + 4 * mu[x] + nu[y]) * 6;
      pr[2 * x + y] = k == 0 ? 1.0 : (k == 2 ? -1.0 : 0.0);
      pi[2 * x + y] = k == 1 ? 1.0 : (k == 3 ? -1.0 : 0.0);
    }
}

NO_HD void phase3_lane_setup(int lane, P3Lane& L) {
  const int sc = lane >> 1;
  const int s1o = (sc >> 3) & 1, s2o = (sc >> 2) & 1, s1i = (sc >> 1) & 1, s2i = sc & 1;
  L.spin_off = 16 * (8 * s1o + 4 * s2o) + 8 * s1i + 4 * s2i;
  phase3_terms(0, s1o, s2o, s1i, s2i, L.cof[0], L.pr[0], L.pi[0]);
  phase3_terms(1, s2o, s1o, s1i, s2i, L.cof[1], L.pr[1], L.pi[1]);      // row of G~ read at (s2, s1, t2, t1)
}

// charge-conserving block nb = 0..5: (to, ti) = (0,0) (1,1) (2,2) (3,3) (1,2) (2,1); returns the element offset
NO_HD int phase3_block(const double* coef, const P3Lane& L, int nb, double& re, double& im) {
  const int to = nb < 4 ? nb : nb - 3, ti = nb < 4 ? nb : 6 - nb;
  const int b0 = nb;                                  // iso_block(to, ti)
  const int b1 = nb == 0 ? 0 : (nb == 3 ? 3 : 6 - nb);   // iso_block(swap(to), ti): 0 5 4 3 2 1
  double gr = 0, gi = 0, hr = 0, hi = 0;
  for (int x = 0; x < 4; ++x) {
    const double cg = coef[L.cof[0][x] + b0], ch = coef[L.cof[1][x] + b1];
    gr = fma(cg, L.pr[0][x], gr); gi = fma(cg, L.pi[0][x], gi);
    hr = fma(ch, L.pr[1][x], hr); hi = fma(ch, L.pi[1][x], hi);
  }
  re = gr - hr;
  im = gi - hi;
  return L.spin_off + 16 * to + ti;
}

// structurally zero block nz = 0..9 (charge not conserved): element offset
NO_HD int phase3_zero_off(const P3Lane& L, int nz) {
  // (to, ti) in the order (0,1) (0,2) (0,3) (1,0) (1,3) (2,0) (2,3) (3,0) (3,1) (3,2)
  const int to = nz < 3 ? 0 : (nz < 5 ? 1 : (nz < 7 ? 2 : 3));
  const int ti = nz < 3 ? nz + 1 : (nz == 3 ? 0 : (nz == 4 ? 3 : (nz == 5 ? 0 : (nz == 6 ? 3 : nz - 7))));
  return L.spin_off + 16 * to + ti;
}

}  // namespace no3n
