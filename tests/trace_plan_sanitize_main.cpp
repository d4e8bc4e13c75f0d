// tests/trace_plan_sanitize_main.cpp -- TEST ONLY.  The product's host-side trace planner
// (paper_2603_24532_b200/csrc/no_trace_host.h) as a standalone program under -fsanitize=address,undefined: ladders and
// rings of order 1-6, the complete fifth-order graph, a few hundred pseudo-random closed topologies (self-loops,
// disconnected pieces, frontiers that need slicing), each planned with and without the charge-conservation flag;
// every table entry the kernel would use must stay inside the shared-memory buffers.  Exit 0 = no report, all in range.
#include <cstdio>
#include <cstdlib>

#include "../paper_2603_24532_b200/csrc/no_trace_host.h"

using namespace no3n;

static int check_plan(int n, const int* topo, bool charge, long long* planned) {
  TracePlan plan;
  if (build_trace_plan(n, topo, plan, charge) != 0) return 0;     // refused topologies are fine here
  ++*planned;
  if (plan.max_open > kTrMaxOpen || plan.n_sliced > kTrMaxSlice || plan.n_slice_iter > 64) return 1;
  for (int k = 0; k < n; ++k) {
    const TraceStep& s = plan.steps[k];
    if (s.vertex < 0 || s.vertex >= n || s.nA * s.nB > 256 || s.nC > 256) return 2;
    for (int a = 0; a < s.nA; ++a)
      for (int g = 0; g < s.nC; g += (s.nC > 16 ? 7 : 1)) {
        const int lim = s.r_vertex >= 0 ? kTrMatW : kTrMat;
        if (s.baseR[a] + s.offR[g] >= lim) return 3;
      }
    for (int b = 0; b < s.nB; ++b)
      for (int g = 0; g < s.nC; g += (s.nC > 16 ? 7 : 1))
        for (int it = 0; it < plan.n_slice_iter; ++it)
          if (s.baseW[b] + s.offW[g] + s.sliceW[it] >= kTrMatW) return 4;
    if (s.big) {
      for (int a = 0; a < 16; ++a)
        for (int b = 0; b < 16; ++b) {
          if (s.outA[a] + s.outB[b] >= kTrMat) return 5;
          if (s.fuse_last && s.lastW[a + 16 * b] >= kTrMatW) return 6;
        }
    }
  }
  return 0;
}

int main() {
  long long planned = 0;
  int topo[4 * kTrMaxVertex];
  for (int n = 1; n <= 6; ++n)
    for (int kind = 0; kind < 2; ++kind) {
      for (int v = 0; v < n; ++v) {
        topo[4 * v + 0] = 2 * v; topo[4 * v + 1] = 2 * v + 1;
        topo[4 * v + 2] = 2 * ((v + n - 1) % n);
        topo[4 * v + 3] = kind == 0 ? 2 * ((v + n - 1) % n) + 1 : 2 * ((v + 1) % n) + 1;
      }
      for (int c = 0; c < 2; ++c)
        if (int rc = check_plan(n, topo, c != 0, &planned)) { printf("chain n=%d kind=%d rc=%d\n", n, kind, rc); return 1; }
    }
  unsigned long long st = 0x9E3779B97F4A7C15ULL;
  auto rnd = [&](int m) { st ^= st << 13; st ^= st >> 7; st ^= st << 17; return (int)(st % (unsigned long long)m); };
  for (int trial = 0; trial < 300; ++trial) {
    const int n = 2 + trial % 4, L = 2 * n;
    int outs[kTrMaxLines], ins[kTrMaxLines];
    for (int l = 0; l < L; ++l) outs[l] = ins[l] = l;
    for (int l = L - 1; l > 0; --l) { int j = rnd(l + 1), t = outs[l]; outs[l] = outs[j]; outs[j] = t; j = rnd(l + 1); t = ins[l]; ins[l] = ins[j]; ins[j] = t; }
    for (int v = 0; v < n; ++v) { topo[4 * v] = outs[2 * v]; topo[4 * v + 1] = outs[2 * v + 1]; topo[4 * v + 2] = ins[2 * v]; topo[4 * v + 3] = ins[2 * v + 1]; }
    for (int c = 0; c < 2; ++c)
      if (int rc = check_plan(n, topo, c != 0, &planned)) { printf("random trial %d rc=%d\n", trial, rc); return 1; }
  }
  const int bad[4] = {0, 1, 0, 0};
  TracePlan p;
  if (build_trace_plan(1, bad, p) == 0 || build_trace_plan(7, topo, p) == 0) return 2;
  printf("trace planner sanitized: %lld plans ok\n", planned);
  return 0;
}
