// tests/host_emu.cpp -- lane-by-lane HOST emulation of the CUDA kernel's warp program, for the CPU
// unit tests only (tests/test_host_logic.py).  It compiles the kernel's own arithmetic
// (paper_2603_24532_b200/csrc/no_core.h, no_host.h) with g++ and walks the 32 lanes of one warp
// sequentially through the same phases, in the same order, as no3n_kernel in no_kernel.cuh.
// It is NOT part of the product library and is never loaded by the package: the product has no
// CPU path.  It lets the host logic (tables, kernel-variant choice, moment algebra, epilogue) be
// checked against the oracle on a machine without a GPU.
#include <cstring>
#include <cstdint>
#include <cmath>
#include <vector>

#include "../paper_2603_24532_b200/csrc/no_host.h"

using namespace no3n;

// one trip of the hot loop: the kernel's load pattern followed by no3n::nodes
template <int NREG>
static void trip(const double* rs, int n_reg, const double* e2tab, const DirConst& d, const double* rad,
                 const double* ttab, int i, First& f, bool flush) {
  double r[kNodesPerTrip], wr[kNodesPerTrip], T[kNodesPerTrip][5];
  for (int k = 0; k < kNodesPerTrip; ++k) {
    r[k] = rad[2 * (i + k)];
    wr[k] = rad[2 * (i + k) + 1];
    for (int q = 0; q < 5; ++q) T[k][q] = ttab[kRadT * (i + k) + q];
  }
  if (flush) nodes<NREG, kNodesPerTrip, true>(rs, n_reg, e2tab, d, r, wr, T, f);
  else nodes<NREG, kNodesPerTrip, false>(rs, n_reg, e2tab, d, r, wr, T, f);
}

static int n_dir_of(const DevParams& P) { return P.n_list > 0 ? P.n_list : P.n_cos * P.n_phi; }

template <int NREG, bool C4>
static void emu_cfg(const HostPlan& plan, const double* cfg, double* out /*[512]*/) {
  using L = Layout<C4>;
  const DevParams& P = plan.dp;
  CfgConst c;
  cfg_setup<NREG>(P, cfg, c);
  std::vector<double> acc(L::kStride * kLanes + 2), mom(L::kStride), rec(kRecDoubles), coef(32 * 6, 0.0);
  double* acc16 = acc.data() + ((reinterpret_cast<uintptr_t>(acc.data()) & 15) ? 1 : 0);   // 16-byte aligned rows
  std::vector<double> ttab(kRadT * P.n_r_pad);
  const double* e2tab = plan.tab.data();
  for (int pass = 0; pass < P.n_pass; ++pass) {
    const double* rad = plan.tab.data() + P.pass_off[pass];
    for (int i = 0; i < P.n_r_pad; ++i) radial_entry(c, rad[2 * i], &ttab[kRadT * i]);
    const double* ct = rad + 2 * P.n_r_pad;
    const double* st = ct + P.n_cos;
    const double* wc = st + P.n_cos;
    const double* cph = wc + P.n_cos;
    const double* sph = cph + P.n_phi;
    const double* wph = sph + P.n_phi;
    // as in the kernel: rows are written by a lane's first direction; only lanes without a direction clear theirs.
    // NaN everywhere else, so that a row the first direction failed to write cannot go unnoticed
    std::fill(acc.begin(), acc.end(), NAN);
    for (int lane = n_dir_of(P); lane < kLanes; ++lane)
      for (int row = 0; row < L::kStride; ++row) acc16[lane * L::kStride + row] = 0.0;
    const int n_dir = P.n_list > 0 ? P.n_list : P.n_cos * P.n_phi;
    for (int lane = 0; lane < kLanes; ++lane) {
      for (int m = lane; m < n_dir; m += kLanes) {
        DirConst d;
        double w;
        if (P.n_list > 0) {
          dir_setup(c, ct[4 * m], ct[4 * m + 1], ct[4 * m + 2], d);
          w = ct[4 * m + 3];
        } else {
          const int j = m / P.n_phi, l = m - j * P.n_phi;
          dir_setup(c, st[j] * cph[l], st[j] * sph[l], ct[j], d);
          w = wc[j] * wph[l];
        }
        First f;
        first_zero(f);
        for (int i = 0; i < P.n_r_pad; i += kNodesPerTrip) trip<NREG>(c.rs, P.n_reg, e2tab, d, rad, ttab.data(), i, f, NREG >= 0 && needs_flush(c));
        if (m == lane) second_level<C4, false, true>(f, d, c.gam, w, acc16 + lane * L::kStride);   // first direction writes
        else second_level<C4>(f, d, c.gam, w, acc16 + lane * L::kStride);
      }
    }
    for (int lane = 0; lane < kLanes; ++lane)
      for (int pr = lane; pr < L::kStride / 2; pr += kLanes)       // a lane adds one pair of adjacent rows (see the kernel)
        for (int h = 0; h < 2; ++h) {
          const int row = 2 * pr + h;
          double s4[4] = {0.0, 0.0, 0.0, 0.0};
          for (int t = 0; t < 8; ++t)
            for (int q = 0; q < 4; ++q) s4[q] += acc16[((2 * lane + t + 8 * q) & 31) * L::kStride + row];
          mom[row] = (s4[0] + s4[1]) + (s4[2] + s4[3]);
        }
    for (int lane = 0; lane < 6; ++lane) phase1_job<C4>(P, c, mom.data(), lane, rec.data());
    for (int lane = 0; lane < kLanes; ++lane)
      phase2_lane(rec.data(), lane, P.nsp[pass], P.esum[pass], NREG >= 0 ? exp(-c.E0) : 1.0, &coef[lane * 6]);
  }
  for (int e = 0; e < 512; ++e) out[e] = -777.0;      // every element must be written exactly once below
  for (int lane = 0; lane < kLanes; ++lane) {
    P3Lane pl;
    phase3_lane_setup(lane, pl);
    const int h = lane & 1;
    for (int it = 0; it < 3; ++it) {
      double re, im;
      const int off = phase3_block(coef.data(), pl, 2 * it + h, re, im);
      // the lane-mapped expansion is the same sum as the per-element definition
      double re0, im0;
      phase3_elem(coef.data(), off >> 4, off & 15, re0, im0);
      if (re != re0 || im != im0 || out[2 * off] != -777.0) { re = im = NAN; }
      out[2 * off] = re;
      out[2 * off + 1] = im;
    }
    for (int it = 0; it < 5; ++it) {
      const int off = phase3_zero_off(pl, 2 * it + h);
      double re0, im0;
      phase3_elem(coef.data(), off >> 4, off & 15, re0, im0);
      out[2 * off] = (re0 == 0.0 && im0 == 0.0 && out[2 * off] == -777.0) ? 0.0 : NAN;
      out[2 * off + 1] = out[2 * off];
    }
  }
}

template <bool C4>
static void emu_dispatch(const HostPlan& plan, const double* cfg, double* out) {
  switch (plan.nreg_variant) {
    case -1: emu_cfg<-1, C4>(plan, cfg, out); break;
    case 1: emu_cfg<1, C4>(plan, cfg, out); break;
    case 2: emu_cfg<2, C4>(plan, cfg, out); break;
    case 3: emu_cfg<3, C4>(plan, cfg, out); break;
    case 4: emu_cfg<4, C4>(plan, cfg, out); break;
    default: emu_cfg<0, C4>(plan, cfg, out); break;
  }
}

extern "C" {

int emu_eval_angular(const no_params* p, const double* dirs, int n_dir, const double* cfg, long long n_cfg,
                     double* out) {
  HostPlan plan;
  const int rc = build_plan(p, plan, dirs, n_dir);
  if (rc != NO_OK) return rc;
  for (long long i = 0; i < n_cfg; ++i) {
    if (plan.has_c4) emu_dispatch<true>(plan, cfg + 9 * i, out + 512 * i);
    else emu_dispatch<false>(plan, cfg + 9 * i, out + 512 * i);
  }
  return NO_OK;
}

int emu_eval(const no_params* p, const double* cfg, long long n_cfg, double* out) {
  HostPlan plan;
  const int rc = build_plan(p, plan);
  if (rc != NO_OK) return rc;
  for (long long i = 0; i < n_cfg; ++i) {
    if (plan.has_c4) emu_dispatch<true>(plan, cfg + 9 * i, out + 512 * i);
    else emu_dispatch<false>(plan, cfg + 9 * i, out + 512 * i);
  }
  return NO_OK;
}

// plan facts for the host-logic tests
int emu_plan(const no_params* p, int* n_pass, int* nreg_variant, int* has_c4, long long* evals_per_cfg,
             int* tab_doubles, double* tab_out, int tab_cap) {
  HostPlan plan;
  const int rc = build_plan(p, plan);
  if (rc != NO_OK) return rc;
  *n_pass = plan.dp.n_pass;
  *nreg_variant = plan.nreg_variant;
  *has_c4 = plan.has_c4 ? 1 : 0;
  *evals_per_cfg = plan.evals_per_cfg;
  *tab_doubles = plan.dp.tab_doubles;
  for (int i = 0; i < plan.dp.tab_doubles && i < tab_cap; ++i) tab_out[i] = plan.tab[i];
  return NO_OK;
}

void emu_gl_rule(int n, double lo, double hi, double* x, double* w) {
  std::vector<double> xs, ws;
  gl_rule(n, lo, hi, xs, ws);
  for (int i = 0; i < n; ++i) { x[i] = xs[i]; w[i] = ws[i]; }
}

}  // extern "C"

// debugging aid: reduced moments of one pass (c4 layout not supported)
extern "C" int emu_moments(const no_params* p, const double* cfg, int pass, double* mom_out) {
  HostPlan plan;
  const int rc = build_plan(p, plan);
  if (rc != NO_OK) return rc;
  using L = Layout<false>;
  const DevParams& P = plan.dp;
  CfgConst c;
  cfg_setup<-1>(P, cfg, c);
  std::vector<double> acc(L::kStride * kLanes + 2, 0.0);
  double* acc16 = acc.data() + ((reinterpret_cast<uintptr_t>(acc.data()) & 15) ? 1 : 0);
  const double* rad = plan.tab.data() + P.pass_off[pass];
  std::vector<double> ttab(kRadT * P.n_r_pad);
  for (int i = 0; i < P.n_r_pad; ++i) radial_entry(c, rad[2 * i], &ttab[kRadT * i]);
  const double* ct = rad + 2 * P.n_r_pad;
  const double* st = ct + P.n_cos;
  const double* wc = st + P.n_cos;
  const double* cph = wc + P.n_cos;
  const double* sph = cph + P.n_phi;
  const double* wph = sph + P.n_phi;
  for (int m = 0; m < P.n_cos * P.n_phi; ++m) {
    const int j = m / P.n_phi, l = m - j * P.n_phi;
    DirConst d;
    dir_setup(c, st[j] * cph[l], st[j] * sph[l], ct[j], d);
    First f;
    first_zero(f);
    for (int i = 0; i < P.n_r_pad; i += kNodesPerTrip) trip<-1>(c.rs, P.n_reg, plan.tab.data(), d, rad, ttab.data(), i, f, false);
    second_level<false>(f, d, c.gam, wc[j] * wph[l], acc16 + (m & 31) * L::kStride);
  }
  for (int row = 0; row < L::kRows; ++row) {
    double s = 0;
    for (int t = 0; t < kLanes; ++t) s += acc16[t * L::kStride + row];
    mom_out[row] = s;
  }
  return NO_OK;
}

extern "C" int emu_records(const no_params* p, const double* cfg, const double* mom, double* rec_out) {
  HostPlan plan;
  const int rc = build_plan(p, plan);
  if (rc != NO_OK) return rc;
  CfgConst c;
  cfg_setup<-1>(plan.dp, cfg, c);
  for (int lane = 0; lane < 6; ++lane) phase1_job<false>(plan.dp, c, mom, lane, rec_out);
  return NO_OK;
}
