// tests/oracle_sanitize_main.cpp -- TEST ONLY.  Builds the CPU oracle (oracle/no_oracle.cpp, included
// verbatim) into a standalone program so that it can run under -fsanitize=address,undefined
// (SURVEY.md section 5): pin P11 (level 0 == level 1) on a 2 x 2 x 2 grid in asymmetric matter with all
// topologies incl. c4, the caller-supplied direction list, the double instantiation and the
// brute-force Hartree-Fock sum.  Exit code 0 = every comparison held and no sanitizer report was printed
// (a report aborts the program: -fno-sanitize-recover).
#include <cstdio>

#include "../oracle/no_oracle.cpp"

int main() {
  Params p;
  p.kf_n = 1.2; p.kf_p = 0.9;
  p.c1 = -0.81; p.c3 = -3.2; p.c4 = 5.4; p.cD = 1.0; p.cE = -0.5;
  p.gA = 1.27; p.fpi = 92.4; p.mpi = 138.04; p.lambda_chi = 700.0; p.Lambda = 500.0;
  p.n_reg = 4; p.n_r = 2; p.n_cos = 2; p.n_phi = 2;
  const double cfg[2 * 9] = {0.3, -0.2, 0.5, -0.1, 0.4, 0.2, 0.2, 0.1, -0.3,
                             1.1, 0.4, -0.7, 0.2, -0.9, 0.5, -0.6, 0.3, 0.8};
  static double a[2 * 512], b[2 * 512], c[2 * 512], d[2 * 512];
  oracle_no_level0_ld(&p, cfg, 2, a);
  oracle_no_level1_ld(&p, cfg, 2, b);
  oracle_no_level1_f64(&p, cfg, 2, c);
  double mx = 0, e01 = 0, e1d = 0;
  for (int i = 0; i < 2 * 512; ++i) {
    mx = std::fmax(mx, std::fabs(a[i]));
    e01 = std::fmax(e01, std::fabs(a[i] - b[i]));
    e1d = std::fmax(e1d, std::fabs(b[i] - c[i]));
  }
  // the product grid handed over as a direction list (built here with the oracle's own rule: only the code
  // path is exercised, the pin that uses numpy's rule lives in tests/test_oracle_pins.py)
  std::vector<long double> x, wx, ph, wph;
  gauss_legendre<long double>(2, -1.0L, 1.0L, x, wx);
  gauss_legendre<long double>(2, 0.0L, 2 * PI_LD, ph, wph);
  double dirs[4 * 4];
  for (int j = 0; j < 2; ++j) for (int l = 0; l < 2; ++l) {
    const long double st = sqrtl(1 - x[j] * x[j]);
    double* u = dirs + 4 * (2 * j + l);
    u[0] = (double)(st * cosl(ph[l])); u[1] = (double)(st * sinl(ph[l])); u[2] = (double)x[j];
    u[3] = (double)(wx[j] * wph[l]);
  }
  oracle_no_level1_dirs_ld(&p, cfg, 2, dirs, 4, d);
  double eld = 0;
  for (int i = 0; i < 2 * 512; ++i) eld = std::fmax(eld, std::fabs(b[i] - d[i]));
  p.n_r = 1;
  const double e = oracle_hf3n_bruteforce(&p);
  std::printf("max %.6e  level0-level1 %.3e  ld-f64 %.3e  grid-list %.3e  hf %.6e\n", mx, e01, e1d, eld, e);
  const bool ok = mx > 1e-3 && e01 < 1e-15 * mx && e1d < 1e-12 * mx && eld < 1e-14 * mx && std::isfinite(e) && e != 0.0;
  return ok ? 0 : 1;
}
