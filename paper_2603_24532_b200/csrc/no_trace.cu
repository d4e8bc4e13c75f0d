// no_trace.cu -- spin-isospin trace kernel and its C ABI (include/no_trace.h; PAPER.md:155-157,
// 639-653).  One warp contracts the tensor network of one Monte-Carlo sample: the n vertex matrices of the sample
// (n x 4 KiB, contiguous in HBM) arrive in shared memory with ONE TMA bulk copy per sample (cp.async.bulk + mbarrier,
// double buffered: the next sample's copy runs under this sample's arithmetic), the partial result (<= 256 complex
// numbers) ping-pongs between two shared-memory buffers, and every step of the host-planned program
// (no_trace_host.h) is a small complex matrix product whose index arithmetic is tabulated.  The dominant step shape
// (16 x 16 x 16: ladders and rings) has a register-tiled path: a lane owns a 4 x 2 tile of the product, its operands
// are warp-broadcast 16-byte shared-memory loads, 32 DFMA per 6 loads.  sm_100a only; there is no CPU path.
#include <cuda_runtime.h>

#include <cstdio>
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

__device__ __forceinline__ double2 shfl_xor2(double2 v, int m) {
  return make_double2(__shfl_xor_sync(0xffffffffu, v.x, m), __shfl_xor_sync(0xffffffffu, v.y, m));
}

constexpr int kTrStages = 2;     // vertex buffers per warp (TMA double buffering)

// shared memory: plan (n_vertex steps) | per warp: mbarriers (16 B) | vertex buffers [kTrStages][n][256] complex | R [2][256] complex
__host__ __device__ inline size_t trace_plan_bytes(int n) { return 16 + (size_t)n * sizeof(TraceStep); }
__host__ __device__ inline size_t trace_warp_bytes(int n) { return 16 + (size_t)kTrStages * n * 4096 + 2 * 4096; }

__global__ void __launch_bounds__(512, 1)
trace_kernel(const DevTracePlan* __restrict__ plan_g, const double2* __restrict__ V, long long n_sample,
             double2* __restrict__ out) {
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
  unsigned char* wb = tsm + trace_plan_bytes(n) + (size_t)warp * trace_warp_bytes(n);
  uint64_t* bar = reinterpret_cast<uint64_t*>(wb);                       // [kTrStages]
  double2* vbuf = reinterpret_cast<double2*>(wb + 16);                   // [kTrStages][n][256]
  double2* Rb = vbuf + (size_t)kTrStages * n * 256;                      // [2][256]
  const uint32_t sample_bytes = (uint32_t)n * 4096u;
  if (lane == 0)
    for (int s = 0; s < kTrStages; ++s) mbar_init(bar + s, 1);
  __syncthreads();

  const long long first = (long long)blockIdx.x * n_warps + warp, stride = (long long)gridDim.x * n_warps;
  // prologue: request the first sample
  if (lane == 0 && first < n_sample) {
    mbar_expect_tx(bar, sample_bytes);
    tma_bulk_g2s(vbuf, V + first * n * 256, sample_bytes, bar);
  }
  uint32_t phase[kTrStages] = {0, 0};
  int stage = 0;
  for (long long smp = first; smp < n_sample; smp += stride) {
    // request the next sample into the other buffer (its last reader finished before the __syncwarp that ended
    // the previous iteration; the proxy fence orders those generic-proxy reads before the async-proxy write)
    const long long nxt = smp + stride;
    if (lane == 0 && nxt < n_sample) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(bar + (stage ^ 1), sample_bytes);
      tma_bulk_g2s(vbuf + (size_t)(stage ^ 1) * n * 256, V + nxt * n * 256, sample_bytes, bar + (stage ^ 1));
    }
    mbar_wait(bar + stage, phase[stage]);
    phase[stage] ^= 1;
    const double2* W = vbuf + (size_t)stage * n * 256;

    double2 total = make_double2(0.0, 0.0);
    for (int it = 0; it < n_iter; ++it) {
      double2* Rin = Rb;
      double2* Rout = Rb + 256;
      double2 last = make_double2(0.0, 0.0);
      for (int k = 0; k < n; ++k) {
        const TraceStep& s = steps[k];
        const double2* Wv = W + s.vertex * 256 + s.sliceW[it];
        const int nA = s.nA, nB = s.nB, nC = s.nC, nOut = nA * nB;
        if (nA == 1 && nC == 1) {
          // nothing is open on the input side (first vertex of a component): R' = the vertex's own entries,
          // times the scalar carried so far (1 at the start; the trace of the finished components otherwise)
          const double2 c = k == 0 ? make_double2(1.0, 0.0) : Rin[0];
          for (int o = lane; o < nB; o += 32) {
            double2 v = make_double2(0.0, 0.0);
            cfma(v, c, Wv[s.baseW[o]]);
            if (nB == 1) last = v;
            Rout[o] = v;
          }
        } else if (nA == 16 && nB == 16 && nC == 16) {
          // register-tiled 16 x 16 x 16 complex product: lane (la, lb) owns a = 4 la + i, b = 2 lb + j
          const int la = lane >> 3, lb = lane & 7;
          int rA[4], wB[2];
#pragma unroll
          for (int i = 0; i < 4; ++i) rA[i] = s.baseR[4 * la + i];
#pragma unroll
          for (int j = 0; j < 2; ++j) wB[j] = s.baseW[2 * lb + j];
          double2 acc[4][2];
#pragma unroll
          for (int i = 0; i < 4; ++i) acc[i][0] = acc[i][1] = make_double2(0.0, 0.0);
#pragma unroll 4
          for (int g = 0; g < 16; ++g) {
            const int oR = s.offR[g], oW = s.offW[g];
            double2 r[4], w[2];
#pragma unroll
            for (int i = 0; i < 4; ++i) r[i] = Rin[rA[i] + oR];
#pragma unroll
            for (int j = 0; j < 2; ++j) w[j] = Wv[wB[j] + oW];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
              cfma(acc[i][0], r[i], w[0]);
              cfma(acc[i][1], r[i], w[1]);
            }
          }
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            Rout[(4 * la + i) + 16 * (2 * lb)] = acc[i][0];
            Rout[(4 * la + i) + 16 * (2 * lb + 1)] = acc[i][1];
          }
        } else if (nOut >= 32) {
          const int mA = nA - 1, shA = 31 - __clz(nA);
          for (int o = lane; o < nOut; o += 32) {
            const int rA = s.baseR[o & mA], wB = s.baseW[o >> shA];
            double2 v = make_double2(0.0, 0.0);
            for (int g = 0; g < nC; ++g) cfma(v, Rin[rA + s.offR[g]], Wv[wB + s.offW[g]]);
            Rout[o] = v;
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
          if (part == 0) Rout[o] = v;
          if (nOut == 1) last = v;
        }
        __syncwarp();
        double2* t = Rin; Rin = Rout; Rout = t;
      }
      total.x += last.x; total.y += last.y;
    }
    if (lane == 0) out[smp] = total;
    __syncwarp();
    stage ^= 1;
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
  size_t smem;
};

extern "C" {

const char* no_trace_last_cuda_error(void) { return g_trace_err; }

int no_trace_init(no_trace_plan** out, int n_vertex, const int* topo, int device) {
  if (!out || !topo) return NO_ERR_INVALID;
  no_trace_plan* p = new (std::nothrow) no_trace_plan();
  if (!p) return NO_ERR_ALLOC;
  p->d_plan = nullptr;
  if (build_trace_plan(n_vertex, topo, p->plan) != 0) { delete p; return NO_ERR_INVALID; }
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
  const size_t avail = (size_t)smem_optin - trace_plan_bytes(n_vertex) - 128;
  int warps = (int)(avail / trace_warp_bytes(n_vertex));
  if (warps > 16) warps = 16;
  if (warps < 1) { delete p; return NO_ERR_INVALID; }
  p->warps = warps;
  p->smem = trace_plan_bytes(n_vertex) + (size_t)warps * trace_warp_bytes(n_vertex);
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

int no_trace_eval(const no_trace_plan* p, const double* d_vertices, long long n_sample, double* d_out, void* cuda_stream) {
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
  const size_t smem = trace_plan_bytes(p->plan.n_vertex) + (size_t)warps * trace_warp_bytes(p->plan.n_vertex);
  trace_kernel<<<(unsigned)blocks, warps * 32, smem, static_cast<cudaStream_t>(cuda_stream)>>>(
      p->d_plan, reinterpret_cast<const double2*>(d_vertices), n_sample, reinterpret_cast<double2*>(d_out));
  const cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return trace_cuda_fail(e, "trace_kernel launch");
  return NO_OK;
}

int no_trace_info(const no_trace_plan* p, long long* cmacs, int* max_open, int* n_sliced, long long* n_iso, int* order) {
  if (!p) return NO_ERR_INVALID;
  if (cmacs) *cmacs = p->plan.cmacs;
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
