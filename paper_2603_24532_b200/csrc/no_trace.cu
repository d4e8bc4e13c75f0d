// no_trace.cu -- spin-isospin trace kernel and its C ABI (include/no_trace.h; PAPER.md:155-157,
// 639-653).  One warp contracts the tensor network of one Monte-Carlo sample: the n vertex matrices of the sample
// (n x 4 KiB, contiguous in HBM) arrive in shared memory through asynchronous 16-byte copies (cp.async, coalesced
// 512-byte warp reads) into rows padded by one element, the partial result (<= 256 complex numbers) ping-pongs
// between two padded shared-memory buffers, and every step of the host-planned program (no_trace_host.h) is a small
// complex matrix product whose index arithmetic is tabulated.  The dominant step shape (16 x 16 x 16: ladders and
// rings) runs on the FP64 tensor cores (mma.sync m8n8k4, SASS DMMA: 64 per step against 16 shared-memory fragment
// loads); a vector-FP64 register-tiled variant of it is kept for comparison.  sm_100a only; there is no CPU path.
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <new>

#include "../../include/no_trace.h"
#include "no_tma.cuh"
#include "no_trace_host.h"

using namespace no3n;

namespace {

struct DevTracePlan {
  int n_vertex, n_slice_iter, pad_[2];
  TraceStep steps[kTrMaxVertex];
};
static_assert(sizeof(TraceStep) % 16 == 0 && sizeof(DevTracePlan) % 16 == 0, "plan is staged with 16-byte copies");

__device__ __forceinline__ void cfma(double2& acc, const double2 a, const double2 b) {
  acc.x = fma(a.x, b.x, acc.x);
  acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y);
  acc.y = fma(a.y, b.x, acc.y);
}

constexpr int kTrStagesDefault = 1;
constexpr int kTrPathDefault = 1;

__device__ __forceinline__ double2 shfl_xor2(double2 v, int m) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}

// m8n8k4 FP64 tensor-core product D = A B + C (SASS DMMA): lane l holds A[l / 4][l % 4], B[l % 4][l / 4] and
// C[l / 4][2 (l % 4)], C[l / 4][2 (l % 4) + 1]
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// shared memory: plan (n_vertex steps) | per warp: the scalar 1 (16 B) | vertex buffers [stages][n][16][17] complex | R [1 or 2][16][17] complex
__host__ __device__ inline size_t trace_plan_bytes(int n) { return 16 + (size_t)n * sizeof(TraceStep); }
// Partial results ping-pong between a dedicated buffer and, when every vertex is read only once (no sliced lines), the
// slot of the first absorbed vertex, which is dead by the time the second buffer is first written (r_bufs = 1);
// with sliced lines the vertices are re-read in every outer iteration and both buffers are dedicated (r_bufs = 2).
__host__ __device__ inline size_t trace_warp_bytes(int n, int stages, int r_bufs) {
  return 16 + (size_t)(stages * n * kTrMatW + r_bufs * kTrMat) * 16;
}

// request vertex matrix v of a sample: 256 complex numbers, one 16-byte cp.async (LDGSTS) per lane and element --
// coalesced 512-byte warp reads from HBM, written into the padded rows of the vertex's slot, no registers held while in
// flight.  (One TMA bulk copy per sample cannot pad the rows, and one per row is bound by the TMA issue rate: 80
// descriptors per sample ran at 1.17e8 samples/s, profiles/r02b.md.)
__device__ __forceinline__ void request_vertex(double2* dst, const double2* src, int v, int lane) {
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const int rc = lane + 32 * j;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;"
                 ::"r"(smem_u32(dst + v * kTrMatW + (rc >> 4) * kTrRowW + (rc & 15))), "l"(src + v * 256 + rc) : "memory");
  }
}

// Packed input (NO_PACK_CHARGE of include/no.h: the 96 charge-conserving entries, [16 spin elements][6 isospin blocks]):
// padded offset of packed entry pk inside a vertex slot, and of the z-th of the 160 entries that form cannot hold
__device__ __forceinline__ int packed_pos(int pk) {
  const int sp = pk / 6, nb = pk - 6 * sp;
  const int to = nb < 4 ? nb : nb - 3, ti = nb < 4 ? nb : 6 - nb;
  return (4 * (sp >> 2) + to) * kTrRowW + 4 * (sp & 3) + ti;
}
__device__ __forceinline__ int forbidden_pos(int z) {
  const int sp = z / 10, nz = z - 10 * sp;
  // (to, ti) over (0,1) (0,2) (0,3) (1,0) (1,3) (2,0) (2,3) (3,0) (3,1) (3,2)
  const int to = (int)((0x3332211000ULL >> (4 * nz)) & 15), ti = (int)((0x2103030321ULL >> (4 * nz)) & 15);
  return (4 * (sp >> 2) + to) * kTrRowW + 4 * (sp & 3) + ti;
}
__device__ __forceinline__ void request_vertex_packed(double2* dst, const double2* src, int v, int lane) {
#pragma unroll
  for (int j = 0; j < 3; ++j) {
    const int pk = lane + 32 * j;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;"
                 ::"r"(smem_u32(dst + v * kTrMatW + packed_pos(pk))), "l"(src + v * 96 + pk) : "memory");
  }
}

// NO_PACK_ISOSPIN (isospin-symmetric matter): 32 entries per vertex, [16 spin elements][(pn,pn), (pn,np)].  Lane 2 sp + h
// copies its entry to the two places it stands for, (pn,pn) and (np,np) or (pn,np) and (np,pn); the pp and nn entries
// are their sum and are filled in after the copies have landed (isospin_fixup).
__device__ __forceinline__ int iso_pos(int sp, int to, int ti) { return (4 * (sp >> 2) + to) * kTrRowW + 4 * (sp & 3) + ti; }
__device__ __forceinline__ void request_vertex_iso(double2* dst, const double2* src, int v, int lane) {
  const int sp = lane >> 1, h = lane & 1;
  const double2* g = src + v * 32 + lane;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;"
               ::"r"(smem_u32(dst + v * kTrMatW + iso_pos(sp, 1, h ? 2 : 1))), "l"(g) : "memory");
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;"
               ::"r"(smem_u32(dst + v * kTrMatW + iso_pos(sp, 2, h ? 1 : 2))), "l"(g) : "memory");
}
__device__ __forceinline__ void isospin_fixup(double2* slots, int n, int lane) {
  const int sp = lane >> 1, h = lane & 1;
  for (int v = 0; v < n; ++v) {
    double2* m = slots + v * kTrMatW;
    const double2 d = m[iso_pos(sp, 1, 1)], x = m[iso_pos(sp, 1, 2)];
    m[h ? iso_pos(sp, 3, 3) : iso_pos(sp, 0, 0)] = make_double2(d.x + x.x, d.y + x.y);   // T = 1: pp = nn = (pn,pn) + (pn,np)
  }
}

// all n vertex matrices of the sample at src as ONE cp.async group (packed: 0 full matrices, 1 NO_PACK_CHARGE, 2 NO_PACK_ISOSPIN)
__device__ __forceinline__ void request_sample(double2* dst, const double2* src, int n, bool valid, int lane, int packed) {
  if (valid)
    for (int v = 0; v < n; ++v) {
      if (packed == 2) request_vertex_iso(dst, src, v, lane);
      else if (packed == 1) request_vertex_packed(dst, src, v, lane);
      else request_vertex(dst, src, v, lane);
    }
  asm volatile("cp.async.commit_group;" ::: "memory");
}

// path: 0 = vector FP64 (DFMA) register tiles, 1 = FP64 tensor cores (DMMA m8n8k4) for the 16 x 16 x 16 steps
__global__ void __launch_bounds__(384, 1)
trace_kernel(const DevTracePlan* __restrict__ plan_g, const double2* __restrict__ V, long long n_sample,
             double2* __restrict__ out, int stages, int path, int packed) {
  extern __shared__ __align__(128) unsigned char tsm[];
  const int n = plan_g->n_vertex, n_iter = plan_g->n_slice_iter;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, n_warps = blockDim.x >> 5;
  // ---- stage the plan (header + n steps) ----
  {
    const uint4* src = reinterpret_cast<const uint4*>(plan_g);
    uint4* dst = reinterpret_cast<uint4*>(tsm);
    const int n16 = (int)(trace_plan_bytes(n) / 16);
    for (int i = threadIdx.x; i < n16; i += blockDim.x) dst[i] = src[i];
  }
  const TraceStep* steps = reinterpret_cast<const TraceStep*>(tsm + 16);
  const int r_bufs = n_iter == 1 ? 1 : 2;
  unsigned char* wb = tsm + trace_plan_bytes(n) + (size_t)warp * trace_warp_bytes(n, stages, r_bufs);
  double2* one = reinterpret_cast<double2*>(wb);                         // the empty contraction: the scalar 1
  double2* vbuf = reinterpret_cast<double2*>(wb + 16);                   // [stages][n][16][17]
  double2* Rb = vbuf + (size_t)stages * n * kTrMatW;                      // [r_bufs][16][17]
  if (lane == 0) *one = make_double2(1.0, 0.0);
  const int vs = packed == 2 ? 32 : (packed ? 96 : 256);                  // complex numbers per vertex in HBM
  if (packed)                                                             // the entries the packed form leaves out stay zero
    for (int i = lane; i < stages * n * kTrMatW; i += 32) vbuf[i] = make_double2(0.0, 0.0);
  __syncthreads();

  const long long first = (long long)blockIdx.x * n_warps + warp, stride = (long long)gridDim.x * n_warps;
  // Loads.  Default (stages = 1): ONE set of vertex slots per warp; the whole next sample is requested when this sample
  // is done and awaited at the top of the loop: the other warps of the SM compute meanwhile (8 warps per SM at fifth
  // order).  Measured alternatives, both slower (profiles/r02b.md): requesting the next sample's vertices step by step
  // as their slots fall free (one cp.async group per executed step: -11 %, the copies compete with the fragment
  // loads of the running steps), and stages = 2, a second set of slots per warp (4 warps per SM instead of 7).
  request_sample(vbuf, V + first * n * vs, n, first < n_sample, lane, packed);
  int stage = 0;
  for (long long smp = first; smp < n_sample; smp += stride) {
    const long long nxt = smp + stride;
    if (stages == 2) {
      // the other buffer's last readers finished before the __syncwarp that ended the previous iteration
      request_sample(vbuf + (size_t)(stage ^ 1) * n * kTrMatW, V + nxt * n * vs, n, nxt < n_sample, lane, packed);
      asm volatile("cp.async.wait_group 1;" ::: "memory");      // this sample has landed; the next one is in flight
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncwarp();
    if (packed == 2) {
      isospin_fixup(vbuf + (size_t)stage * n * kTrMatW, n, lane);
      __syncwarp();
    }
    const double2* W = vbuf + (size_t)stage * n * kTrMatW;

    double2 total = make_double2(0.0, 0.0);
    for (int it = 0; it < n_iter; ++it) {
      double2* const RA = Rb;
      // second buffer: dedicated, or the slot of the first absorbed vertex (its matrix is consumed by the first
      // executed step, whose result goes to RA; the padded row strides of the two layouts are the same)
      double2* const RB = r_bufs == 2 ? Rb + kTrMat : vbuf + ((size_t)stage * n + steps[0].vertex) * kTrMatW;
      const double2* Rin = one;                         // nothing open, nothing contracted yet
      double2 last = make_double2(0.0, 0.0);
      for (int k = 0; k < n; ++k) {
        const TraceStep& s = steps[k];
        if (s.skip) continue;                           // folded into a neighbouring step (warp uniform)
        const double2* Wv = W + s.vertex * kTrMatW + s.sliceW[it];
        const int nA = s.nA, nB = s.nB, nC = s.nC, nOut = nA * nB;
        double2* const Rout = Rin == RA ? RB : RA;
        if (s.big) {
          // R of this step: the partial result, or (first vertex folded in) the first vertex's matrix itself
          const double2* Rs = s.r_vertex >= 0 ? W + s.r_vertex * kTrMatW + steps[0].sliceW[it] : Rin;
          // last vertex folded in: it closes all four lines, T = sum_{a,b} R'[a,b] W_last[lastW[a + 16 b]]
          const double2* Wl = s.fuse_last ? W + steps[n - 1].vertex * kTrMatW + steps[n - 1].sliceW[it] : nullptr;
          double2 dot = make_double2(0.0, 0.0);
          if (path == 1 && s.block_diag) {
            // charge-conserving vertices: the product is block diagonal in the isospin-pair enumeration, two 8 x 8 x 8
            // complex blocks (k-steps 2 p, 2 p + 1 -> output tile (p, p)); 16 tensor-core products instead of 64
            const int r = lane >> 2, c = lane & 3, valid = s.ks_valid;
            double cre[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, cim[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
#pragma unroll
            for (int p = 0; p < 2; ++p) {
              const int aR = s.baseR[8 * p + r], bW = s.baseW[8 * p + r];
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                const int ks = 2 * p + j;
                if (!(valid >> ks & 1)) continue;           // warp uniform
                const double2 A = Rs[aR + s.offR[4 * ks + c]], B = Wv[s.offW[4 * ks + c] + bW];
                dmma884(cre[p][0], cre[p][1], A.x, B.x);
                dmma884(cim[p][0], cim[p][1], A.x, B.y);
                dmma884(cre[p][0], cre[p][1], -A.y, B.y);
                dmma884(cim[p][0], cim[p][1], A.y, B.x);
              }
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
              for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int a = 8 * mt + r, b = 8 * nt + 2 * c + e;
                  if (Wl) {
                    if (mt == nt) cfma(dot, make_double2(cre[mt][e], cim[mt][e]), Wl[s.lastW[a + 16 * b]]);
                  } else {
                    // the off-diagonal tiles are stored as zeros: the next step reads whole tiles
                    Rout[s.outA[a] + s.outB[b]] = mt == nt ? make_double2(cre[mt][e], cim[mt][e]) : make_double2(0.0, 0.0);
                  }
                }
          } else if (path == 1) {
            // 16 x 16 x 16 complex product on the FP64 tensor cores: four real products per (8 x 8 tile, k-step of 4),
            // Re = Re Re - Im Im, Im = Re Im + Im Re; fragments come straight from the tabulated offsets
            const int r = lane >> 2, c = lane & 3;
            int aR[2], bW[2], gR[4], gW[4];
#pragma unroll
            for (int t = 0; t < 2; ++t) { aR[t] = s.baseR[8 * t + r]; bW[t] = s.baseW[8 * t + r]; }
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) { gR[ks] = s.offR[4 * ks + c]; gW[ks] = s.offW[4 * ks + c]; }
            double cre[2][2][2], cim[2][2][2];
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
              for (int nt = 0; nt < 2; ++nt) cre[mt][nt][0] = cre[mt][nt][1] = cim[mt][nt][0] = cim[mt][nt][1] = 0.0;
#pragma unroll
            for (int ks = 0; ks < 4; ++ks) {
              double2 A[2], B[2];
#pragma unroll
              for (int t = 0; t < 2; ++t) { A[t] = Rs[aR[t] + gR[ks]]; B[t] = Wv[gW[ks] + bW[t]]; }
              // one term over all four tiles before the next: dependent DMMAs are eight apart
#pragma unroll
              for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) dmma884(cre[mt][nt][0], cre[mt][nt][1], A[mt].x, B[nt].x);
#pragma unroll
              for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) dmma884(cim[mt][nt][0], cim[mt][nt][1], A[mt].x, B[nt].y);
#pragma unroll
              for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) dmma884(cre[mt][nt][0], cre[mt][nt][1], -A[mt].y, B[nt].y);
#pragma unroll
              for (int mt = 0; mt < 2; ++mt)
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) dmma884(cim[mt][nt][0], cim[mt][nt][1], A[mt].y, B[nt].x);
            }
#pragma unroll
            for (int mt = 0; mt < 2; ++mt)
#pragma unroll
              for (int nt = 0; nt < 2; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const int a = 8 * mt + r, b = 8 * nt + 2 * c + e;
                  const double2 v = make_double2(cre[mt][nt][e], cim[mt][nt][e]);
                  if (Wl) cfma(dot, v, Wl[s.lastW[a + 16 * b]]);
                  else Rout[s.outA[a] + s.outB[b]] = v;
                }
          } else {
            // vector FP64 variant: lane (la, lb) owns the 4 x 2 tile a = la + 4 i, b = lb + 8 j
            const int la = lane >> 3, lb = lane & 7;
            int rA[4], wB[2];
#pragma unroll
            for (int i = 0; i < 4; ++i) rA[i] = s.baseR[la + 4 * i];
#pragma unroll
            for (int j = 0; j < 2; ++j) wB[j] = s.baseW[lb + 8 * j];
            double2 acc[4][2];
#pragma unroll
            for (int i = 0; i < 4; ++i) acc[i][0] = acc[i][1] = make_double2(0.0, 0.0);
#pragma unroll 4
            for (int g = 0; g < 16; ++g) {
              const int oR = s.offR[g], oW = s.offW[g];
              double2 rr[4], w[2];
#pragma unroll
              for (int i = 0; i < 4; ++i) rr[i] = Rs[rA[i] + oR];
#pragma unroll
              for (int j = 0; j < 2; ++j) w[j] = Wv[wB[j] + oW];
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                cfma(acc[i][0], rr[i], w[0]);
                cfma(acc[i][1], rr[i], w[1]);
              }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
              for (int j = 0; j < 2; ++j) {
                const int a = la + 4 * i, b = lb + 8 * j;
                if (Wl) cfma(dot, acc[i][j], Wl[s.lastW[a + 16 * b]]);
                else Rout[s.outA[a] + s.outB[b]] = acc[i][j];
              }
          }
          if (Wl) {                                     // add the 32 partial dot products (fixed butterfly)
#pragma unroll
            for (int m = 16; m > 0; m >>= 1) {
              const double2 u = shfl_xor2(dot, m);
              dot.x += u.x; dot.y += u.y;
            }
            last = dot;
          }
        } else if (nOut >= 32) {
          const int mA = nA - 1, shA = 31 - __clz(nA);
          for (int o = lane; o < nOut; o += 32) {
            const int rA = s.baseR[o & mA], wB = s.baseW[o >> shA];
            double2 v = make_double2(0.0, 0.0);
            for (int g = 0; g < nC; ++g) cfma(v, Rin[rA + s.offR[g]], Wv[wB + s.offW[g]]);
            Rout[o + (o >> 4)] = v;
          }
        } else {
          // fewer outputs than lanes: P = 32 / nOut lanes share one output, each sums every P-th closed label,
          // partial sums added by a fixed butterfly
          const int P = 32 / nOut, o = lane / P, part = lane - o * P;
          const int mA = nA - 1, shA = 31 - __clz(nA);
          const int rA = s.baseR[o & mA], wB = s.baseW[o >> shA];
          double2 v = make_double2(0.0, 0.0);
          for (int g = part; g < nC; g += P) cfma(v, Rin[rA + s.offR[g]], Wv[wB + s.offW[g]]);
          for (int m = P >> 1; m > 0; m >>= 1) {
            const double2 u = shfl_xor2(v, m);
            v.x += u.x; v.y += u.y;
          }
          if (part == 0) Rout[o + (o >> 4)] = v;
          if (nOut == 1) last = v;
        }
        __syncwarp();
        Rin = Rout;
      }
      total.x += last.x; total.y += last.y;
    }
    if (lane == 0) out[smp] = total;
    __syncwarp();
    if (packed && r_bufs == 1) {
      // the slot of the first absorbed vertex served as the second partial-result buffer: the entries the packed
      // form does not carry must be zero again before the slot's next sample is used
      double2* slot = vbuf + ((size_t)stage * n + steps[0].vertex) * kTrMatW;
#pragma unroll
      for (int j = 0; j < 5; ++j) slot[forbidden_pos(lane + 32 * j)] = make_double2(0.0, 0.0);
    }
    if (stages == 2) stage ^= 1;
    else request_sample(vbuf, V + nxt * n * vs, n, nxt < n_sample, lane, packed);
  }
}

thread_local char g_trace_err[256] = "";

int trace_cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_trace_err, sizeof(g_trace_err), "%s: %s (%s)", where, cudaGetErrorName(e), cudaGetErrorString(e));
  return NO_ERR_CUDA;
}

struct TrDeviceGuard {
  int prev;
  bool ok;
  explicit TrDeviceGuard(int dev) : prev(-1), ok(false) {
    if (cudaGetDevice(&prev) != cudaSuccess) return;
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) return;
    ok = true;
  }
  ~TrDeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

struct no_trace_plan {
  TracePlan plan;
  int device;
  DevTracePlan* d_plan;
  int warps;        // warps per CTA
  int n_sm;
  int stages;       // vertex buffers per warp: 2 = the next sample's copy runs under this sample's arithmetic
  int path;         // 0 vector FP64 tiles, 1 FP64 tensor cores for the 16 x 16 x 16 steps
};

extern "C" {

const char* no_trace_last_cuda_error(void) { return g_trace_err; }

int no_trace_init(no_trace_plan** out, int n_vertex, const int* topo, int flags, int device) {
  if (!out || !topo || (flags & ~NO_TRACE_CHARGE_CONSERVING)) return NO_ERR_INVALID;
  no_trace_plan* p = new (std::nothrow) no_trace_plan();
  if (!p) return NO_ERR_ALLOC;
  p->d_plan = nullptr;
  if (build_trace_plan(n_vertex, topo, p->plan, (flags & NO_TRACE_CHARGE_CONSERVING) != 0) != 0) { delete p; return NO_ERR_INVALID; }
  int n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess) { delete p; return trace_cuda_fail(e, "cudaGetDeviceCount"); }
  if (device < 0 || device >= n_dev) { delete p; return NO_ERR_INVALID; }
  p->device = device;
  TrDeviceGuard guard(device);
  if (!guard.ok) { delete p; return trace_cuda_fail(cudaGetLastError(), "cudaSetDevice"); }
  int smem_optin = 0;
  e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, device);
  if (e != cudaSuccess) { delete p; return trace_cuda_fail(e, "cudaDeviceGetAttribute"); }
  // one CTA per SM, as many warps (samples in flight) as its shared memory holds
  p->stages = kTrStagesDefault;
  p->path = kTrPathDefault;
  const size_t avail = (size_t)smem_optin - trace_plan_bytes(n_vertex) - 128;
  const int r_bufs = p->plan.n_slice_iter == 1 ? 1 : 2;
  int warps = (int)(avail / trace_warp_bytes(n_vertex, p->stages, r_bufs));
  if (warps > 12) warps = 12;      // __launch_bounds__(384): up to 170 registers per thread, no spills
  if (warps < 1) { delete p; return NO_ERR_INVALID; }
  p->warps = warps;
  e = cudaFuncSetAttribute((const void*)trace_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
  if (e != cudaSuccess) { delete p; return trace_cuda_fail(e, "cudaFuncSetAttribute(smem)"); }
  DevTracePlan hp;
  hp.n_vertex = p->plan.n_vertex;
  hp.n_slice_iter = p->plan.n_slice_iter;
  hp.pad_[0] = hp.pad_[1] = 0;
  for (int k = 0; k < kTrMaxVertex; ++k) hp.steps[k] = p->plan.steps[k];
  e = cudaMalloc((void**)&p->d_plan, sizeof(DevTracePlan));
  if (e != cudaSuccess) { delete p; trace_cuda_fail(e, "cudaMalloc(trace plan)"); return NO_ERR_ALLOC; }
  e = cudaMemcpy(p->d_plan, &hp, sizeof(DevTracePlan), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaFree(p->d_plan); delete p; return trace_cuda_fail(e, "cudaMemcpy(trace plan)"); }
  *out = p;
  return NO_OK;
}

namespace {
int trace_launch(const no_trace_plan* p, const double* d_vertices, long long n_sample, double* d_out, void* cuda_stream, int packed);
}

int no_trace_eval(const no_trace_plan* p, const double* d_vertices, long long n_sample, double* d_out, void* cuda_stream) {
  return trace_launch(p, d_vertices, n_sample, d_out, cuda_stream, 0);
}

int no_trace_eval_packed(const no_trace_plan* p, int format, const double* d_packed, long long n_sample, double* d_out,
                         void* cuda_stream) {
  if (format != NO_PACK_CHARGE && format != NO_PACK_ISOSPIN) return NO_ERR_INVALID;
  return trace_launch(p, d_packed, n_sample, d_out, cuda_stream, format == NO_PACK_CHARGE ? 1 : 2);
}

namespace {
int trace_launch(const no_trace_plan* p, const double* d_vertices, long long n_sample, double* d_out, void* cuda_stream, int packed) {
  if (!p || n_sample < 0) return NO_ERR_INVALID;
  if (n_sample == 0) return NO_OK;
  if (!d_vertices || !d_out) return NO_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_vertices) & 15u) || (reinterpret_cast<uintptr_t>(d_out) & 15u)) return NO_ERR_INVALID;
  TrDeviceGuard guard(p->device);
  if (!guard.ok) return trace_cuda_fail(cudaGetLastError(), "cudaSetDevice");
  // persistent CTAs: warps stride over the samples; small batches are spread over the SMs first
  int warps = p->warps;
  long long blocks = (n_sample + warps - 1) / warps;
  if (blocks < p->n_sm) {
    warps = (int)((n_sample + p->n_sm - 1) / p->n_sm);
    blocks = (n_sample + warps - 1) / warps;
  } else {
    blocks = p->n_sm;
  }
  const size_t smem = trace_plan_bytes(p->plan.n_vertex) + (size_t)warps * trace_warp_bytes(p->plan.n_vertex, p->stages, p->plan.n_slice_iter == 1 ? 1 : 2);
  trace_kernel<<<(unsigned)blocks, warps * 32, smem, static_cast<cudaStream_t>(cuda_stream)>>>(
      p->d_plan, reinterpret_cast<const double2*>(d_vertices), n_sample, reinterpret_cast<double2*>(d_out), p->stages,
      p->path, packed);
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return trace_cuda_fail(e, "trace_kernel launch");
  return NO_OK;
}
}  // namespace

int no_trace_info(const no_trace_plan* p, long long* cmacs, int* max_open, int* n_sliced, long long* n_iso, int* order,
                  long long* tensor_products) {
  if (!p) return NO_ERR_INVALID;
  if (cmacs) *cmacs = p->plan.cmacs;
  if (tensor_products) *tensor_products = p->plan.dmma_products;
  if (max_open) *max_open = p->plan.max_open;
  if (n_sliced) *n_sliced = p->plan.n_sliced;
  if (n_iso) *n_iso = p->plan.n_isospin;
  if (order) for (int v = 0; v < p->plan.n_vertex; ++v) order[v] = p->plan.order[v];
  return NO_OK;
}

int no_trace_free(no_trace_plan* p) {
  if (!p) return NO_OK;
  TrDeviceGuard guard(p->device);
  if (p->d_plan) cudaFree(p->d_plan);
  delete p;
  return NO_OK;
}

}  // extern "C"
