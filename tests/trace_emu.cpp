// tests/trace_emu.cpp -- HOST emulation of the trace kernel's step program, for the CPU unit tests only
// (tests/test_trace_host_logic.py).  It compiles the product's planner (paper_2603_24532_b200/csrc/no_trace_host.h)
// with g++ and runs the planned program -- the same tables, the same step semantics as trace_kernel in no_trace.cu --
// with plain serial loops.  It is NOT part of the product library and is never loaded by the package.
#include <complex>
#include <vector>

#include "../paper_2603_24532_b200/csrc/no_trace_host.h"

using namespace no3n;
typedef std::complex<double> cplx;

extern "C" {

// info: [cmacs, max_open, n_sliced, n_isospin, n_slice_iter, order[6], (nA, nB, nC)[6], dmma_products]
int trace_emu_plan(int n, const int* topo, int charge, long long* info) {
  TracePlan plan;
  if (build_trace_plan(n, topo, plan, charge != 0) != 0) return 1;
  info[29] = plan.dmma_products;
  info[0] = plan.cmacs; info[1] = plan.max_open; info[2] = plan.n_sliced; info[3] = plan.n_isospin;
  info[4] = plan.n_slice_iter;
  for (int v = 0; v < 6; ++v) info[5 + v] = v < n ? plan.order[v] : -1;
  for (int k = 0; k < 6; ++k) {
    info[11 + 3 * k] = k < n ? plan.steps[k].nA : 0;
    info[12 + 3 * k] = k < n ? plan.steps[k].nB : 0;
    info[13 + 3 * k] = k < n ? plan.steps[k].nC : 0;
  }
  return 0;
}

// V: [n_sample][n][16][16][2]; out: [n_sample][2]
int trace_emu_eval(int n, const int* topo, int charge, const double* V, long long n_sample, double* out) {
  TracePlan plan;
  if (build_trace_plan(n, topo, plan, charge != 0) != 0) return 1;
  std::vector<cplx> R(kTrMat), Rn(kTrMat), W(n * kTrMatW);
  for (long long smp = 0; smp < n_sample; ++smp) {
    // the kernel's shared-memory image of the sample: every matrix row padded to kTrRow elements
    const cplx* Vs = reinterpret_cast<const cplx*>(V) + smp * n * 256;
    for (int v = 0; v < n; ++v)
      for (int e = 0; e < 256; ++e) W[v * kTrMatW + tr_padw(e)] = Vs[v * 256 + e];
    cplx total = 0;
    for (int it = 0; it < plan.n_slice_iter; ++it) {
      R.assign(kTrMat, cplx(0, 0));
      R[0] = 1.0;
      for (int k = 0; k < n; ++k) {
        const TraceStep& s = plan.steps[k];
        if (s.skip) continue;                         // folded into a neighbouring step
        const cplx* Wv = W.data() + s.vertex * kTrMatW + s.sliceW[it];
        const cplx* Rsrc = s.r_vertex >= 0 ? W.data() + s.r_vertex * kTrMatW + plan.steps[0].sliceW[it] : R.data();
        for (int b = 0; b < s.nB; ++b)
          for (int a = 0; a < s.nA; ++a) {
            cplx v = 0;
            for (int g = 0; g < s.nC; ++g) {
              // 16 x 16 x 16 steps: only the tile products the plan keeps (all of them unless it was made for
              // charge-conserving vertices); a, b tiles of 8, k-steps of 4 in the plan's enumeration
              if (s.big && !(s.tile_mask[g >> 2] >> (2 * (a >> 3) + (b >> 3)) & 1)) continue;
              v += Rsrc[s.baseR[a] + s.offR[g]] * Wv[s.baseW[b] + s.offW[g]];
            }
            Rn[s.big ? s.outA[a] + s.outB[b] : tr_pad(a + s.nA * b)] = v;
          }
        R.swap(Rn);
        if (s.fuse_last) {                            // the last vertex closes everything: one dot product
          const TraceStep& sl = plan.steps[n - 1];
          const cplx* Wl = W.data() + sl.vertex * kTrMatW + sl.sliceW[it];
          cplx t = 0;
          for (int b = 0; b < 16; ++b)
            for (int a = 0; a < 16; ++a) t += R[s.outA[a] + s.outB[b]] * Wl[s.lastW[a + 16 * b]];
          R[0] = t;
        }
      }
      total += R[0];
    }
    out[2 * smp] = total.real();
    out[2 * smp + 1] = total.imag();
  }
  return 0;
}

}  // extern "C"
