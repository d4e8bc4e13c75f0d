// tests/host_emu_sanitize_main.cpp -- TEST ONLY.  The product's host logic and kernel arithmetic (no_host.h, no_core.h,
// compiled for the host by tests/host_emu.cpp, included verbatim) as a standalone program under
// -fsanitize=address,undefined: plans and lane-by-lane emulated evaluations for every kernel variant (regulator
// exponents 1-4, generic, unregulated; c4 on/off; one and two Fermi spheres; product grid and direction list; ragged
// orders incl. the maximum 128).  Exit 0 = no sanitizer report and every output finite.
#include <cstdio>

#include "host_emu.cpp"

static int run(no_params p, const double* dirs, int n_dir) {
  const double cfg[2 * 9] = {0.3, -0.2, 0.5, -0.1, 0.4, 0.2, 0.2, 0.1, -0.3,
                             1.1, 0.4, -0.7, 0.2, -0.9, 0.5, -0.6, 0.3, 0.8};
  static double out[2 * 512];
  const int rc = dirs ? emu_eval_angular(&p, dirs, n_dir, cfg, 2, out) : emu_eval(&p, cfg, 2, out);
  if (rc != 0) return 1;
  for (int i = 0; i < 2 * 512; ++i) if (!std::isfinite(out[i])) return 2;
  return 0;
}

int main() {
  no_params base;
  base.kf_n = 1.2; base.kf_p = 0.9; base.c1 = -0.81; base.c3 = -3.2; base.c4 = 0.0; base.cD = 1.0; base.cE = -0.5;
  base.gA = 1.27; base.fpi = 92.4; base.mpi = 138.04; base.lambda_chi = 700.0; base.Lambda = 500.0;
  base.n_reg = 4; base.n_r = 3; base.n_cos = 4; base.n_phi = 5; base.device = 0;
  int n_run = 0;
  for (int nreg = 0; nreg <= 6; ++nreg)
    for (int c4 = 0; c4 < 2; ++c4)
      for (int geo = 0; geo < 3; ++geo) {
        no_params p = base;
        if (nreg == 0) p.Lambda = -1.0; else p.n_reg = nreg;
        p.c4 = c4 ? 5.4 : 0.0;
        if (geo == 1) { p.kf_p = 0.0; }
        if (geo == 2) { p.kf_p = p.kf_n; }
        if (int rc = run(p, nullptr, 0)) { printf("grid nreg=%d c4=%d geo=%d rc=%d\n", nreg, c4, geo, rc); return 1; }
        ++n_run;
      }
  {
    no_params p = base; p.n_r = 128; p.n_cos = 1; p.n_phi = 2;
    if (run(p, nullptr, 0)) return 2;
    p.n_r = 1; p.n_cos = 128; p.n_phi = 1;
    if (run(p, nullptr, 0)) return 2;
    n_run += 2;
  }
  {
    // six-point octahedral rule as a direction list
    const double w = 4.0 * 3.14159265358979323846 / 6.0;
    const double dirs[6 * 4] = {1, 0, 0, w, -1, 0, 0, w, 0, 1, 0, w, 0, -1, 0, w, 0, 0, 1, w, 0, 0, -1, w};
    no_params p = base; p.n_cos = 1; p.n_phi = 1; p.c4 = 5.4;
    if (run(p, dirs, 6)) return 3;
    const double bad[4] = {1, 1, 0, w};                     // not a unit vector: refused
    static double out[512];
    const double cfg[9] = {0};
    if (emu_eval_angular(&p, bad, 1, cfg, 1, out) == 0) return 4;
    ++n_run;
  }
  printf("host emulation sanitized: %d runs ok\n", n_run);
  return 0;
}
