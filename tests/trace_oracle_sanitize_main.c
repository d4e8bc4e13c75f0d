/* tests/trace_oracle_sanitize_main.c -- TEST ONLY.  Builds the brute-force trace oracle (oracle/trace_oracle.c,
 * included verbatim) into a standalone program that runs under -fsanitize=address,undefined: a third-order ring and a
 * second-order ladder with a self-consistent check (ladder = trace of the matrix product, computed here with plain loops),
 * the isospin-assignment counter, and the out-of-range guards.  Exit code 0 = every check held and no sanitizer report
 * was printed (a report aborts: -fno-sanitize-recover). */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "../oracle/trace_oracle.c"

int main(void) {
  const int ladder2[8] = {0, 1, 2, 3, 2, 3, 0, 1};
  const int ring3[12] = {0, 1, 4, 3, 2, 3, 0, 5, 4, 5, 2, 1};
  double *V = malloc(sizeof(double) * 2 * 3 * 512);
  unsigned long long st = 88172645463325252ULL;
  for (int i = 0; i < 2 * 3 * 512; ++i) {
    st ^= st << 13; st ^= st >> 7; st ^= st << 17;
    V[i] = (double)(st >> 11) / 9007199254740992.0 - 0.5;
  }
  double out[4];
  if (oracle_trace_bruteforce(2, ladder2, V, 2, out) != 0) return 1;
  for (int s = 0; s < 2; ++s) {                     /* Tr[V_1 V_0] */
    const double *A = V + (size_t)s * 2 * 512 + 512, *B = V + (size_t)s * 2 * 512;
    double tr = 0, ti = 0;
    for (int i = 0; i < 16; ++i)
      for (int k = 0; k < 16; ++k) {
        const double ar = A[2 * (16 * i + k)], ai = A[2 * (16 * i + k) + 1];
        const double br = B[2 * (16 * k + i)], bi = B[2 * (16 * k + i) + 1];
        tr += ar * br - ai * bi; ti += ar * bi + ai * br;
      }
    if (fabs(tr - out[2 * s]) > 1e-12 * fabs(tr) + 1e-13 || fabs(ti - out[2 * s + 1]) > 1e-12 * fabs(ti) + 1e-13) return 2;
  }
  if (oracle_trace_bruteforce(3, ring3, V, 2, out) != 0) return 3;
  if (!(isfinite(out[0]) && isfinite(out[3]))) return 4;
  if (oracle_trace_isospin_configs(2, ladder2) != 6) return 5;
  if (oracle_trace_bruteforce(0, ladder2, V, 1, out) != 1 || oracle_trace_bruteforce(7, ladder2, V, 1, out) != 1) return 6;
  if (oracle_trace_isospin_configs(9, ladder2) != -1) return 7;
  free(V);
  printf("trace oracle sanitized: ok\n");
  return 0;
}
