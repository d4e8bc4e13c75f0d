// no_host.h -- host-side setup of the 3N normal-ordering library (step a0 of SURVEY.md 8(a)):
// parameter validation, unit conversion, Gauss-Legendre rules, k3 tables, kernel-variant choice.
// Plain C++ (no CUDA calls) so that the CPU unit tests can drive it through tests/host_emu.cpp.
#pragma once

#include <cmath>
#include <vector>

#include "../../include/no.h"
#include "no_core.h"

namespace no3n {

constexpr double kHbarc = 197.3269804;   // MeV fm (reading R9)
constexpr int kMaxOrder = 128;

// Gauss-Legendre rule of order n on [lo, hi].  Roots of P_n by Newton's method started from the
// Chebyshev-like guess, evaluated with the three-term recurrence in long double; the rule is
// built for the non-negative roots and mirrored so that nodes and weights are exactly symmetric.
inline void gl_rule(int n, double lo, double hi, std::vector<double>& x, std::vector<double>& w) {
  x.resize(n);
  w.resize(n);
  const long double pi = 3.141592653589793238462643383279502884L;
  const long double c = 0.5L * ((long double)hi + (long double)lo), h = 0.5L * ((long double)hi - (long double)lo);
  const int half = n / 2;
  for (int k = 0; k < half; ++k) {          // k-th largest root, t > 0
    long double t = cosl(pi * (4 * k + 3) / (4 * n + 2));
    long double dp = 1;
    for (int it = 0; it < 64; ++it) {
      long double pm = 1, pc = t;            // P_0, P_1
      for (int m = 2; m <= n; ++m) {
        const long double pn = ((2 * m - 1) * t * pc - (m - 1) * pm) / m;
        pm = pc;
        pc = pn;
      }
      dp = n * (pm - t * pc) / (1 - t * t);  // P_n'(t)
      const long double step = pc / dp;
      t -= step;
      if (fabsl(step) <= 4e-20L) {
        // derivative at the final root
        pm = 1; pc = t;
        for (int m = 2; m <= n; ++m) {
          const long double pn = ((2 * m - 1) * t * pc - (m - 1) * pm) / m;
          pm = pc;
          pc = pn;
        }
        dp = n * (pm - t * pc) / (1 - t * t);
        break;
      }
    }
    const long double wt = 2 / ((1 - t * t) * dp * dp);
    x[n - 1 - k] = (double)(c + h * t);
    x[k] = (double)(c - h * t);
    w[n - 1 - k] = w[k] = (double)(h * wt);
  }
  if (n & 1) {                               // middle root t = 0: P_n'(0) from the recurrence
    long double pm = 1, pc = 0;
    for (int m = 2; m <= n; ++m) {
      const long double pn = (-(long double)(m - 1) * pm) / m;   // t = 0
      pm = pc;
      pc = pn;
    }
    // after the loop pc = P_n(0) = 0 (n odd), pm = P_{n-1}(0);  P_n'(0) = n P_{n-1}(0)
    const long double dp = n * pm;
    x[half] = (double)c;
    w[half] = (double)(h * 2 / (dp * dp));
  }
}

struct HostPlan {
  DevParams dp;               // dp.tab is filled by the caller after the upload
  std::vector<double> tab;    // host copy of the device tables
  int nreg_variant;           // -1 unregulated, 0 generic, 1..4 unrolled
  bool has_c4;
  int n_sph;                  // distinct non-zero Fermi momenta
  double kf_n, kf_p;          // Fermi momenta as given (fm^-1)
  long long evals_per_cfg;
};

// product Gauss-Legendre grid of one Fermi sphere, [n_r n_cos n_phi][4] = (kx, ky, kz, W),
// W = r^2 w_r w_cos w_phi / (2 pi)^3 (hole sum Eq. (6), fixed lab frame: readings R7, R11, R13)
inline void sphere_nodes(int n_r, int n_cos, int n_phi, double kf, std::vector<double>& out) {
  const double pi = 3.14159265358979323846;
  const double norm = 1.0 / (8.0 * pi * pi * pi);
  std::vector<double> xr, wr, xc, wc, xp, wp;
  gl_rule(n_r, 0.0, kf, xr, wr);
  gl_rule(n_cos, -1.0, 1.0, xc, wc);
  gl_rule(n_phi, 0.0, 2.0 * pi, xp, wp);
  out.resize(4 * (size_t)n_r * n_cos * n_phi);
  size_t m = 0;
  for (int i = 0; i < n_r; ++i)
    for (int j = 0; j < n_cos; ++j)
      for (int l = 0; l < n_phi; ++l, ++m) {
        const double st = std::sqrt((1.0 - xc[j]) * (1.0 + xc[j]));
        out[4 * m + 0] = xr[i] * st * std::cos(xp[l]);
        out[4 * m + 1] = xr[i] * st * std::sin(xp[l]);
        out[4 * m + 2] = xr[i] * xc[j];
        out[4 * m + 3] = xr[i] * xr[i] * wr[i] * wc[j] * wp[l] * norm;
      }
}

inline bool finite_all(const no_params& p) {
  const double v[] = {p.kf_n, p.kf_p, p.c1, p.c3, p.c4, p.cD, p.cE, p.gA, p.fpi, p.mpi, p.lambda_chi, p.Lambda};
  for (double d : v) if (!std::isfinite(d)) return false;
  return true;
}

constexpr int kMaxList = 4096;   // directions of a caller-supplied angular rule

// dirs != nullptr: angular rule [n_dir][4] = (ux, uy, uz, w), sum w = 4 pi, instead of the cos x phi grid
inline int build_plan(const no_params* p, HostPlan& plan, const double* dirs = nullptr, int n_dir = 0) {
  if (!p || !finite_all(*p)) return NO_ERR_INVALID;
  if (p->kf_n < 0 || p->kf_p < 0 || !(p->fpi > 0) || !(p->mpi > 0)) return NO_ERR_INVALID;
  if (p->n_r < 1 || p->n_r > kMaxOrder || p->n_cos < 1 || p->n_cos > kMaxOrder || p->n_phi < 1 ||
      p->n_phi > kMaxOrder)
    return NO_ERR_INVALID;
  if (dirs) {
    if (n_dir < 1 || n_dir > kMaxList) return NO_ERR_INVALID;
    for (int i = 0; i < 4 * n_dir; ++i) if (!std::isfinite(dirs[i])) return NO_ERR_INVALID;
    // the kernel uses |u| = 1 (D_l = r^2 + bet_l r + gam_l, and the bound on |k3 - P/2| that elides the
    // underflow guard of the regulator): a direction that is not a unit vector is refused, not renormalised
    for (int i = 0; i < n_dir; ++i) {
      const double* u = dirs + 4 * i;
      if (std::fabs(u[0] * u[0] + u[1] * u[1] + u[2] * u[2] - 1.0) > 1e-12) return NO_ERR_INVALID;
    }
  }
  const bool regulated = p->Lambda > 0;
  if (regulated && (p->n_reg < 1 || p->n_reg > kMaxRegPoly)) return NO_ERR_INVALID;

  DevParams& d = plan.dp;
  d = DevParams();
  d.tab = nullptr;
  d.n_r = p->n_r; d.n_cos = p->n_cos; d.n_phi = p->n_phi;
  d.n_list = dirs ? n_dir : 0;
  const double mpi = p->mpi / kHbarc, fpi = p->fpi / kHbarc;
  const double Lchi = (p->lambda_chi > 0 ? p->lambda_chi : 700.0) / kHbarc;
  const double c1 = p->c1 * 1e-3 * kHbarc, c3 = p->c3 * 1e-3 * kHbarc, c4 = p->c4 * 1e-3 * kHbarc;
  const double f2 = fpi * fpi;
  d.m2 = mpi * mpi;
  d.inv_L2 = regulated ? (kHbarc / p->Lambda) * (kHbarc / p->Lambda) : 0.0;
  d.al = -4.0 * c1 * d.m2 / f2;
  d.be = 2.0 * c3 / f2;
  d.G2 = (p->gA / (2.0 * fpi)) * (p->gA / (2.0 * fpi));
  d.gD = -p->gA * p->cD / (8.0 * f2 * f2 * Lchi);
  d.gE2 = p->cE / (f2 * f2 * Lchi);
  d.g4 = d.G2 * c4 / f2;
  d.n_reg = regulated ? p->n_reg : 0;
  plan.nreg_variant = !regulated ? -1 : (p->n_reg <= 4 ? p->n_reg : 0);
  plan.has_c4 = (p->c4 != 0.0);

  // passes: equal non-zero Fermi momenta share one grid with the full isospin trace (R12)
  struct Pass { double kf, nsp, esum; };
  std::vector<Pass> passes;
  if (p->kf_n > 0 && p->kf_n == p->kf_p) {
    passes.push_back({p->kf_n, 2.0, 0.0});
  } else {
    if (p->kf_p > 0) passes.push_back({p->kf_p, 1.0, +1.0});
    if (p->kf_n > 0) passes.push_back({p->kf_n, 1.0, -1.0});
  }
  plan.kf_n = p->kf_n;
  plan.kf_p = p->kf_p;
  d.n_pass = (int)passes.size();
  d.kf_max = 0.0;
  for (const Pass& q : passes) d.kf_max = q.kf > d.kf_max ? q.kf : d.kf_max;
  plan.n_sph = d.n_pass;
  plan.evals_per_cfg = (long long)p->n_r * (dirs ? (long long)n_dir : (long long)p->n_cos * p->n_phi) * d.n_pass;

  d.n_r_pad = (p->n_r + kNodesPerTrip - 1) / kNodesPerTrip * kNodesPerTrip;
  const int per = tab_pass_doubles(d.n_r_pad, p->n_cos, p->n_phi, d.n_list);
  int total = kExpTab + per * d.n_pass;
  total = (total + 1) & ~1;               // 16-byte granularity of the bulk copy
  d.tab_doubles = total;
  plan.tab.assign(total, 0.0);
  for (int j = 0; j < kExpTab; ++j) plan.tab[j] = (double)exp2l((long double)j / kExpTab);   // 2^(j/kExpTab)
  const double pi = 3.14159265358979323846;
  const double norm = 1.0 / (8.0 * pi * pi * pi);
  std::vector<double> xr, wr, xc, wc, xp, wp;
  gl_rule(p->n_cos, -1.0, 1.0, xc, wc);
  gl_rule(p->n_phi, 0.0, 2.0 * pi, xp, wp);
  for (int s = 0; s < d.n_pass; ++s) {
    d.pass_off[s] = kExpTab + per * s;
    d.nsp[s] = passes[s].nsp;
    d.esum[s] = passes[s].esum;
    double* T = plan.tab.data() + d.pass_off[s];
    gl_rule(p->n_r, 0.0, passes[s].kf, xr, wr);
    for (int i = 0; i < d.n_r_pad; ++i) {
      const int k = i < p->n_r ? i : p->n_r - 1;        // padding node: a valid radius with weight 0
      T[2 * i + 0] = xr[k];
      T[2 * i + 1] = i < p->n_r ? wr[k] * xr[k] * xr[k] * norm : 0.0;
      d.radk[s][i][0] = T[2 * i + 0];
      d.radk[s][i][1] = T[2 * i + 1];
    }
    double* A = T + 2 * d.n_r_pad;
    if (dirs) {
      for (int i = 0; i < 4 * n_dir; ++i) A[i] = dirs[i];
      continue;
    }
    for (int j = 0; j < p->n_cos; ++j) {
      A[j] = xc[j];
      A[p->n_cos + j] = std::sqrt((1.0 - xc[j]) * (1.0 + xc[j]));
      A[2 * p->n_cos + j] = wc[j];
    }
    double* B = A + 3 * p->n_cos;
    for (int l = 0; l < p->n_phi; ++l) {
      B[l] = std::cos(xp[l]);
      B[p->n_phi + l] = std::sin(xp[l]);
      B[2 * p->n_phi + l] = wp[l];
    }
  }
  return NO_OK;
}

}  // namespace no3n
