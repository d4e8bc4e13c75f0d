// no_api.cu -- C ABI of libno3n.so (include/no.h): no_init / no_eval / no_eval_host / no_free and
// the small query and probe entry points.  Host setup lives in no_host.h, the kernel in
// no_kernel.cuh.  sm_100a only; there is no CPU path.
#include <cuda_runtime.h>

#include <atomic>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/no.h"
#include "no_host.h"
#include "no_kernel.cuh"

using namespace no3n;

namespace {

thread_local char g_cuda_err[256] = "";

int cuda_fail(cudaError_t e, const char* where) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s)", where, cudaGetErrorName(e), cudaGetErrorString(e));
  return NO_ERR_CUDA;
}

#define NO_CUDA(call)                                 \
  do {                                                \
    cudaError_t e_ = (call);                          \
    if (e_ != cudaSuccess) return cuda_fail(e_, #call); \
  } while (0)

#ifndef NO_WARPS
#define NO_WARPS 2
#endif
#ifndef NO_MINB
#define NO_MINB 6
#endif
constexpr int kWarps = NO_WARPS;       // configurations per CTA
constexpr int kMinBlocks = NO_MINB;   // resident CTAs per SM the register allocation must allow

typedef void (*KernelFn)(const DevParams, const double*, long long, double*, int);

constexpr long long kMaxGrid = 2147483647LL;   // gridDim.x limit; larger batches are cut into several launches
constexpr int kSplit = 4;       // warps per configuration of the small-batch layout (one configuration per CTA)

struct Variant {
  KernelFn fn;
  size_t smem;
  KernelFn fn_split;   // small-batch layout: the CTA's kSplit warps share one configuration
  size_t smem_split;
  KernelFn fn_fwd;     // throughput layout for launches whose configurations all have p' = p (Hartree-Fock)
};

template <int NREG, bool C4>
Variant make_variant(int tab_doubles, int n_r_pad) {
  Variant v;
  v.fn = no3n_kernel<NREG, C4, kWarps, kMinBlocks>;
  v.smem = smem_bytes<C4>(tab_doubles, n_r_pad, kWarps);
  v.fn_split = no3n_kernel<NREG, C4, kSplit, 3, kSplit>;
  v.fn_fwd = no3n_kernel<NREG, C4, kWarps, kMinBlocks, 1, true>;
  v.smem_split = smem_bytes<C4>(tab_doubles, n_r_pad, kSplit);
  return v;
}

template <bool C4>
Variant pick_nreg(int nreg, int tab_doubles, int n_r_pad) {
  switch (nreg) {
    case -1: return make_variant<-1, C4>(tab_doubles, n_r_pad);
    case 1: return make_variant<1, C4>(tab_doubles, n_r_pad);
    case 2: return make_variant<2, C4>(tab_doubles, n_r_pad);
    case 3: return make_variant<3, C4>(tab_doubles, n_r_pad);
    case 4: return make_variant<4, C4>(tab_doubles, n_r_pad);
    default: return make_variant<0, C4>(tab_doubles, n_r_pad);
  }
}

}  // namespace

struct no_handle {
  HostPlan plan;
  int device;
  double* d_tab;
  Variant var;
  // scratch of the host-buffer path
  double* d_cfg;
  double* d_out;
  long long scratch_cfg;      // configurations d_cfg holds
  long long scratch_out;      // doubles d_out holds
  double* hf_arena;           // grow-only device scratch of no_hf_energy / no_sp_energy
  long long hf_arena_doubles;
  std::atomic<int> layout;    // 0 automatic, 1 always one warp per configuration, 2 always one CTA per configuration;
                              // every entry point reads it ONCE per call (no_set_layout may run concurrently)
  std::atomic_flag busy;      // set while an entry point that uses the handle-owned scratch is running
  long long max_grid;         // CTAs per launch (kMaxGrid; the test hook no_set_max_grid lowers it)
  long long wave_cfg;         // configurations of one full wave of resident CTAs (chunk granularity of the host path)
  cudaStream_t copy_stream;   // device-to-host copies of finished chunks overlap the next chunk's kernel
  cudaEvent_t ev_chunk[2], ev_copied;
  bool host_path_ready;
};

namespace {

struct DeviceGuard {
  int prev;
  bool ok;
  explicit DeviceGuard(int dev) : prev(-1), ok(false) {
    if (cudaGetDevice(&prev) != cudaSuccess) return;
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) return;
    ok = true;
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

// kernel layout of one call: 1 = one warp per configuration, 2 = one CTA of kSplit warps per configuration.
// Decided ONCE per entry-point call from the handle's setting and the size of the whole batch, so that every
// chunk of a call (and hence every configuration of it) runs the same summation order.
int resolve_layout(const no_handle* h, long long n_cfg) {
  const int want = h->layout.load(std::memory_order_relaxed);
  if (want == 1 || want == 2) return want;
  // automatic: even with kSplit warps each the configurations do not fill the warp slots -> one CTA each
  return n_cfg * kSplit <= h->wave_cfg ? 2 : 1;
}


int launch(const no_handle* h, const double* d_cfg, long long n_cfg, double* d_out, cudaStream_t s, int layout,
           int mode = kModeFull, bool forward = false) {
  const long long out_doubles = no3n::out_doubles(mode);
  const bool split = layout == 2;
  const long long per_cta = split ? 1 : kWarps;
  const KernelFn fn = split ? h->var.fn_split : (forward ? h->var.fn_fwd : h->var.fn);
  const size_t smem = split ? h->var.smem_split : h->var.smem;
  const int threads = split ? kSplit * 32 : kWarps * 32;
  const long long max_cfg = h->max_grid * per_cta;
  for (long long c0 = 0; c0 < n_cfg; c0 += max_cfg) {
    const long long cnt = n_cfg - c0 < max_cfg ? n_cfg - c0 : max_cfg;
    const long long blocks = (cnt + per_cta - 1) / per_cta;
    fn<<<(unsigned)blocks, threads, smem, s>>>(h->plan.dp, d_cfg + 9 * c0, cnt, d_out + out_doubles * c0, mode);
    NO_CUDA(cudaGetLastError());
  }
  return NO_OK;
}

// entry points that use the handle-owned scratch (host path, Hartree-Fock contractions) are not re-entrant for
// one handle: a second concurrent call is refused instead of racing on the scratch
struct BusyGuard {
  no_handle* h;
  bool ok;
  explicit BusyGuard(no_handle* h_) : h(h_), ok(!h_->busy.test_and_set(std::memory_order_acquire)) {}
  ~BusyGuard() { if (ok) h->busy.clear(std::memory_order_release); }
};

// grow-only scratch of the Hartree-Fock entry points (allocation inside a timed call costs far more than the
// kernels when another process queries the driver, e.g. nvidia-smi)
int hf_scratch(no_handle* h, long long doubles, double** out) {
  if (doubles > h->hf_arena_doubles) {
    if (h->hf_arena) cudaFree(h->hf_arena);
    h->hf_arena = nullptr;
    h->hf_arena_doubles = 0;
    const cudaError_t e = cudaMalloc((void**)&h->hf_arena, sizeof(double) * (size_t)doubles);
    if (e != cudaSuccess) { cuda_fail(e, "cudaMalloc(HF scratch)"); return NO_ERR_ALLOC; }
    h->hf_arena_doubles = doubles;
  }
  *out = h->hf_arena;
  return NO_OK;
}

}  // namespace

extern "C" {

int no_init(no_handle** out, const no_params* p) { return no_init_angular(out, p, nullptr, 0); }

int no_init_angular(no_handle** out, const no_params* p, const double* h_dirs, int n_dir) {
  if (!out || !p) return NO_ERR_INVALID;
  if (!h_dirs && n_dir != 0) return NO_ERR_INVALID;
  no_handle* h = new (std::nothrow) no_handle();
  if (!h) return NO_ERR_ALLOC;
  h->d_tab = nullptr; h->d_cfg = nullptr; h->d_out = nullptr; h->scratch_cfg = 0; h->scratch_out = 0; h->host_path_ready = false;
  h->layout.store(0); h->busy.clear();
  h->max_grid = kMaxGrid;
  h->hf_arena = nullptr; h->hf_arena_doubles = 0;
  int rc = build_plan(p, h->plan, h_dirs, n_dir);
  if (rc != NO_OK) { delete h; return rc; }
  int n_dev = 0;
  cudaError_t e = cudaGetDeviceCount(&n_dev);
  if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaGetDeviceCount"); }
  if (p->device < 0 || p->device >= n_dev) { delete h; return NO_ERR_INVALID; }
  h->device = p->device;
  DeviceGuard guard(h->device);
  if (!guard.ok) { delete h; return cuda_fail(cudaGetLastError(), "cudaSetDevice"); }
  h->var = h->plan.has_c4 ? pick_nreg<true>(h->plan.nreg_variant, h->plan.dp.tab_doubles, h->plan.dp.n_r_pad)
                          : pick_nreg<false>(h->plan.nreg_variant, h->plan.dp.tab_doubles, h->plan.dp.n_r_pad);
  // the limit is a property of the kernel, shared by every handle that uses the same variant: raise it
  // to the device maximum once, so that handles with different table sizes never lower it for each other
  int smem_optin = 0;
  e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, h->device);
  if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaDeviceGetAttribute(smem optin)"); }
  if (h->var.smem > (size_t)smem_optin || h->var.smem_split > (size_t)smem_optin) { delete h; return NO_ERR_INVALID; }
  e = cudaFuncSetAttribute((const void*)h->var.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
  if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaFuncSetAttribute(smem)"); }
  e = cudaFuncSetAttribute((const void*)h->var.fn_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
  if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaFuncSetAttribute(smem, forward)"); }
  e = cudaFuncSetAttribute((const void*)h->var.fn_split, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
  if (e != cudaSuccess) { delete h; return cuda_fail(e, "cudaFuncSetAttribute(smem, split)"); }
  {
    int occ = 0, sms = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void*)h->var.fn, kWarps * 32, h->var.smem);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device);
    if (e != cudaSuccess || occ < 1 || sms < 1) { delete h; return cuda_fail(e, "occupancy query"); }
    h->wave_cfg = (long long)occ * sms * kWarps;
  }
  const size_t bytes = sizeof(double) * (size_t)(h->plan.dp.tab_doubles > 0 ? h->plan.dp.tab_doubles : 2);
  e = cudaMalloc((void**)&h->d_tab, bytes);
  if (e != cudaSuccess) { delete h; cuda_fail(e, "cudaMalloc(tables)"); return NO_ERR_ALLOC; }
  if (h->plan.dp.tab_doubles > 0) {
    e = cudaMemcpy(h->d_tab, h->plan.tab.data(), sizeof(double) * h->plan.dp.tab_doubles, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(h->d_tab); delete h; return cuda_fail(e, "cudaMemcpy(tables)"); }
  }
  h->plan.dp.tab = h->d_tab;
  *out = h;
  return NO_OK;
}

int no_eval(const no_handle* h, const double* d_cfg, long long n_cfg, double* d_out, void* cuda_stream) {
  if (!h || n_cfg < 0) return NO_ERR_INVALID;
  if (n_cfg == 0) return NO_OK;
  if (!d_cfg || !d_out) return NO_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_cfg) & 7u) || (reinterpret_cast<uintptr_t>(d_out) & 15u)) return NO_ERR_INVALID;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  return launch(h, d_cfg, n_cfg, d_out, static_cast<cudaStream_t>(cuda_stream), resolve_layout(h, n_cfg));
}

int no_set_layout(no_handle* h, int layout) {
  if (!h || layout < 0 || layout > 2) return NO_ERR_INVALID;
  h->layout.store(layout, std::memory_order_relaxed);
  return NO_OK;
}

int no_set_max_grid(no_handle* h, long long max_ctas) {
  if (!h || max_ctas < 0 || max_ctas > kMaxGrid) return NO_ERR_INVALID;
  h->max_grid = max_ctas == 0 ? kMaxGrid : max_ctas;
  return NO_OK;
}

int no_eval_diag(const no_handle* h, const double* d_cfg, long long n_cfg, double* d_out, void* cuda_stream) {
  if (!h || n_cfg < 0) return NO_ERR_INVALID;
  if (n_cfg == 0) return NO_OK;
  if (!d_cfg || !d_out) return NO_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_cfg) & 7u) || (reinterpret_cast<uintptr_t>(d_out) & 7u)) return NO_ERR_INVALID;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  return launch(h, d_cfg, n_cfg, d_out, static_cast<cudaStream_t>(cuda_stream), resolve_layout(h, n_cfg), kModeDiag);
}

int no_hf_energy(no_handle* h, int n_r, int n_cos, int n_phi, double* e_over_v, void* cuda_stream) {
  if (!h || !e_over_v) return NO_ERR_INVALID;
  if (n_r < 1 || n_r > kMaxOrder || n_cos < 1 || n_cos > kMaxOrder || n_phi < 1 || n_phi > kMaxOrder) return NO_ERR_INVALID;
  BusyGuard busy(h);
  if (!busy.ok) return NO_ERR_BUSY;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int layout = h->layout.load(std::memory_order_relaxed) == 2 ? 2 : 1;
  // single-particle grids of the two species (t = 0 proton, 1 neutron), [n][4] = (kx, ky, kz, W)
  const double kf[2] = {h->plan.kf_p, h->plan.kf_n};
  // equal Fermi momenta: the four (t1, t2) pair grids coincide, so the pair grid is integrated ONCE and the
  // four isospin columns of the traced diagonal are added in the reduction (same sum, a quarter of the work)
  const bool fused = kf[0] > 0 && kf[0] == kf[1];
  std::vector<double> nodes[2];
  for (int t = 0; t < 2; ++t)
    if (kf[t] > 0 && !(fused && t == 1)) sphere_nodes(n_r, n_cos, n_phi, kf[t], nodes[t]);
  const long long n1 = (long long)n_r * n_cos * n_phi;
  const long long chunk = n1 * n1 < (1LL << 20) ? n1 * n1 : (1LL << 20);
  double* base = nullptr;
  int rc = hf_scratch(h, 8 * n1 + 14 * chunk + 2, &base);
  if (rc != NO_OK) return rc;
  double* d_nodes[2] = {base, fused ? base : base + 4 * n1};
  double *d_cfg = base + 8 * n1, *d_w = d_cfg + 9 * chunk, *d_diag = d_w + chunk, *d_acc = d_diag + 4 * chunk;
  for (int t = 0; t < 2; ++t)
    if (!nodes[t].empty())
      NO_CUDA(cudaMemcpyAsync(d_nodes[t], nodes[t].data(), sizeof(double) * 4 * (size_t)n1, cudaMemcpyHostToDevice, s));
  NO_CUDA(cudaMemsetAsync(d_acc, 0, sizeof(double), s));
  for (int t1 = 0; t1 < 2; ++t1)
    for (int t2 = 0; t2 < 2; ++t2) {
      if (!(kf[t1] > 0) || !(kf[t2] > 0)) continue;
      if (fused && (t1 || t2)) continue;
      for (long long c0 = 0; c0 < n1 * n1; c0 += chunk) {
        const long long count = n1 * n1 - c0 < chunk ? n1 * n1 - c0 : chunk;
        hf_pairs_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(d_nodes[t1], d_nodes[t2], n1, c0, count, d_cfg, d_w);
        NO_CUDA(cudaGetLastError());
        rc = launch(h, d_cfg, count, d_diag, s, layout, kModeDiag, true);   // p' = p by construction
        if (rc != NO_OK) return rc;
        hf_reduce_kernel<<<1, 1024, 0, s>>>(d_diag, d_w, count, fused ? -1 : 2 * t1 + t2, d_acc);
        NO_CUDA(cudaGetLastError());
      }
    }
  double acc = 0.0;
  NO_CUDA(cudaMemcpyAsync(&acc, d_acc, sizeof(double), cudaMemcpyDeviceToHost, s));
  NO_CUDA(cudaStreamSynchronize(s));
  *e_over_v = acc / 6.0;
  return NO_OK;
}

int no_sp_energy(no_handle* h, const double* h_k1, int n_k, int n_r, int n_cos, int n_phi, double* h_sigma,
                 void* cuda_stream) {
  if (!h || n_k < 0) return NO_ERR_INVALID;
  if (n_k == 0) return NO_OK;
  if (!h_k1 || !h_sigma) return NO_ERR_INVALID;
  if (n_r < 1 || n_r > kMaxOrder || n_cos < 1 || n_cos > kMaxOrder || n_phi < 1 || n_phi > kMaxOrder) return NO_ERR_INVALID;
  BusyGuard busy(h);
  if (!busy.ok) return NO_ERR_BUSY;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int layout = h->layout.load(std::memory_order_relaxed) == 2 ? 2 : 1;
  const double kf[2] = {h->plan.kf_p, h->plan.kf_n};
  const bool fused = kf[0] > 0 && kf[0] == kf[1];   // one particle-2 grid serves both species (see no_hf_energy)
  const long long n2 = (long long)n_r * n_cos * n_phi;
  const long long rows_chunk = (1LL << 20) / n2 > 0 ? ((1LL << 20) / n2 < n_k ? (1LL << 20) / n2 : n_k) : 1;
  std::vector<double> k1w(4 * (size_t)n_k), nodes2[2];
  for (int i = 0; i < n_k; ++i) {
    for (int a = 0; a < 3; ++a) k1w[4 * i + a] = h_k1[3 * i + a];
    k1w[4 * i + 3] = 1.0;                              // particle 1 is not summed: unit weight
  }
  const long long pairs = rows_chunk * n2;
  double* base = nullptr;
  int rc = hf_scratch(h, 4LL * n_k + 8 * n2 + 14 * pairs + 2LL * n_k, &base);
  if (rc != NO_OK) return rc;
  double* d_k1 = base;
  double* d_nodes2[2] = {d_k1 + 4LL * n_k, d_k1 + 4LL * n_k + 4 * n2};
  double *d_cfg = d_nodes2[1] + 4 * n2, *d_w = d_cfg + 9 * pairs, *d_diag = d_w + pairs, *d_sigma = d_diag + 4 * pairs;
  NO_CUDA(cudaMemcpyAsync(d_k1, k1w.data(), sizeof(double) * 4 * (size_t)n_k, cudaMemcpyHostToDevice, s));
  NO_CUDA(cudaMemsetAsync(d_sigma, 0, sizeof(double) * 2 * (size_t)n_k, s));
  for (int t2 = 0; t2 < 2; ++t2) {
    if (!(kf[t2] > 0) || (fused && t2 == 1)) continue;
    sphere_nodes(n_r, n_cos, n_phi, kf[t2], nodes2[t2]);   // each species keeps its own host and device copy
    NO_CUDA(cudaMemcpyAsync(d_nodes2[t2], nodes2[t2].data(), sizeof(double) * 4 * (size_t)n2, cudaMemcpyHostToDevice, s));
    for (long long r0 = 0; r0 < n_k; r0 += rows_chunk) {
      const long long rows = n_k - r0 < rows_chunk ? n_k - r0 : rows_chunk, count = rows * n2;
      hf_pairs_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(d_k1, d_nodes2[t2], n2, r0 * n2, count, d_cfg, d_w);
      NO_CUDA(cudaGetLastError());
      rc = launch(h, d_cfg, count, d_diag, s, layout, kModeDiag, true);   // p' = p by construction
      if (rc != NO_OK) return rc;
      // (1/2) from xi = 1/2 of Eq. (10), (1/2) from averaging the spin of particle 1 out of the traced diagonal
      sp_reduce_kernel<<<(unsigned)rows, 256, 0, s>>>(d_diag, d_w, n2, fused ? -1 : t2, 0.25, r0, d_sigma);
      NO_CUDA(cudaGetLastError());
    }
  }
  NO_CUDA(cudaMemcpyAsync(h_sigma, d_sigma, sizeof(double) * 2 * (size_t)n_k, cudaMemcpyDeviceToHost, s));
  NO_CUDA(cudaStreamSynchronize(s));
  return NO_OK;
}

namespace {

// body of no_eval_host after the scratch is in place; any failure is reported after the copy stream has drained
int host_path(no_handle* h, const double* h_cfg, long long n_cfg, double* h_out, cudaStream_t s, int mode) {
  const long long od = no3n::out_doubles(mode);
  NO_CUDA(cudaMemcpyAsync(h->d_cfg, h_cfg, sizeof(double) * 9 * (size_t)n_cfg, cudaMemcpyHostToDevice, s));
  // chunks of whole waves of resident CTAs (about n/8, at most ~64 Ki configurations): the copy of chunk k
  // (copy stream) runs under the kernel of chunk k + 1 (caller's stream).  One layout for the whole call.
  const int layout = resolve_layout(h, n_cfg);
  long long waves = n_cfg / 8 / h->wave_cfg;
  if (waves < 1) waves = 1;
  if (waves * h->wave_cfg > 65536) waves = 65536 / h->wave_cfg > 0 ? 65536 / h->wave_cfg : 1;
  const long long chunk = waves * h->wave_cfg;
  int k = 0;
  for (long long c0 = 0; c0 < n_cfg; c0 += chunk, ++k) {
    const long long cnt = n_cfg - c0 < chunk ? n_cfg - c0 : chunk;
    const int rc = launch(h, h->d_cfg + 9 * c0, cnt, h->d_out + od * c0, s, layout, mode);
    if (rc != NO_OK) return rc;
    NO_CUDA(cudaEventRecord(h->ev_chunk[k & 1], s));
    NO_CUDA(cudaStreamWaitEvent(h->copy_stream, h->ev_chunk[k & 1], 0));
    NO_CUDA(cudaMemcpyAsync(h_out + od * c0, h->d_out + od * c0, sizeof(double) * (size_t)(od * cnt),
                            cudaMemcpyDeviceToHost, h->copy_stream));
  }
  NO_CUDA(cudaEventRecord(h->ev_copied, h->copy_stream));
  NO_CUDA(cudaStreamWaitEvent(s, h->ev_copied, 0));
  NO_CUDA(cudaStreamSynchronize(s));
  return NO_OK;
}

}  // namespace

namespace {

// kernel output mode of a packed format for this handle; -1 if the format does not apply
int packed_mode(const no_handle* h, int format) {
  if (format == NO_PACK_CHARGE) return kModePacked;
  // the isospin-reduced form exists only where the effective interaction is isospin invariant: one Fermi sphere
  // shared by both species (kF_n = kF_p), traced over the full isospin of the third nucleon
  if (format == NO_PACK_ISOSPIN && h->plan.dp.n_pass == 1 && h->plan.dp.esum[0] == 0.0 && h->plan.dp.nsp[0] == 2.0)
    return kModeIso;
  return -1;
}

int eval_host_mode(no_handle* h, const double* h_cfg, long long n_cfg, double* h_out, void* cuda_stream, int mode) {
  if (n_cfg == 0) return NO_OK;
  if (!h_cfg || !h_out) return NO_ERR_INVALID;
  BusyGuard busy(h);
  if (!busy.ok) return NO_ERR_BUSY;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const long long need_out = no3n::out_doubles(mode) * n_cfg;
  if (n_cfg > h->scratch_cfg) {
    if (h->d_cfg) cudaFree(h->d_cfg);
    h->d_cfg = nullptr;
    h->scratch_cfg = 0;
    const cudaError_t e = cudaMalloc((void**)&h->d_cfg, sizeof(double) * 9 * (size_t)n_cfg);
    if (e != cudaSuccess) { cuda_fail(e, "cudaMalloc(cfg scratch)"); return NO_ERR_ALLOC; }
    h->scratch_cfg = n_cfg;
  }
  if (need_out > h->scratch_out) {
    if (h->d_out) cudaFree(h->d_out);
    h->d_out = nullptr;
    h->scratch_out = 0;
    const cudaError_t e = cudaMalloc((void**)&h->d_out, sizeof(double) * (size_t)need_out);
    if (e != cudaSuccess) { cuda_fail(e, "cudaMalloc(out scratch)"); return NO_ERR_ALLOC; }
    h->scratch_out = need_out;
  }
  if (!h->host_path_ready) {
    NO_CUDA(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
    cudaError_t e = cudaEventCreateWithFlags(&h->ev_chunk[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_chunk[1], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_copied, cudaEventDisableTiming);
    if (e != cudaSuccess) {
      // cudaEventDestroy of a never-created (zero) event only returns an error code: nothing leaks
      cudaEventDestroy(h->ev_chunk[0]); cudaEventDestroy(h->ev_chunk[1]); cudaEventDestroy(h->ev_copied);
      cudaStreamDestroy(h->copy_stream);
      h->ev_chunk[0] = h->ev_chunk[1] = h->ev_copied = nullptr;
      return cuda_fail(e, "cudaEventCreateWithFlags");
    }
    h->host_path_ready = true;
  }
  const int rc = host_path(h, h_cfg, n_cfg, h_out, s, mode);
  if (rc != NO_OK) {
    // nothing of this call may still be writing into the caller's buffers or the scratch when it returns
    cudaStreamSynchronize(h->copy_stream);
    cudaStreamSynchronize(s);
  }
  return rc;
}

}  // namespace

int no_eval_host(no_handle* h, const double* h_cfg, long long n_cfg, double* h_out, void* cuda_stream) {
  if (!h || n_cfg < 0) return NO_ERR_INVALID;
  return eval_host_mode(h, h_cfg, n_cfg, h_out, cuda_stream, kModeFull);
}

int no_eval_host_packed(no_handle* h, int format, const double* h_cfg, long long n_cfg, double* h_packed,
                        void* cuda_stream) {
  if (!h || n_cfg < 0) return NO_ERR_INVALID;
  const int mode = packed_mode(h, format);
  if (mode < 0) return NO_ERR_INVALID;
  return eval_host_mode(h, h_cfg, n_cfg, h_packed, cuda_stream, mode);
}

int no_packed_doubles(const no_handle* h, int format) {
  if (!h) return 0;
  const int mode = packed_mode(h, format & ~NO_PACK_FORWARD);
  return mode < 0 ? 0 : no3n::out_doubles(mode);
}

int no_eval_packed(const no_handle* h, int format, const double* d_cfg, long long n_cfg, double* d_packed,
                   void* cuda_stream) {
  if (!h || n_cfg < 0) return NO_ERR_INVALID;
  // NO_PACK_FORWARD: the caller promises p' = p for every configuration -> the forward kernel (legs 2, 3 and pair 3
  // are copies of legs 0, 1 and pair 2: 39 instead of 51 FP64 instructions per node); same output form
  const bool forward = (format & NO_PACK_FORWARD) != 0;
  const int mode = packed_mode(h, format & ~NO_PACK_FORWARD);
  if (mode < 0) return NO_ERR_INVALID;
  if (n_cfg == 0) return NO_OK;
  if (!d_cfg || !d_packed) return NO_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_cfg) & 7u) || (reinterpret_cast<uintptr_t>(d_packed) & 15u)) return NO_ERR_INVALID;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  return launch(h, d_cfg, n_cfg, d_packed, static_cast<cudaStream_t>(cuda_stream), resolve_layout(h, n_cfg), mode, forward);
}

int no_unpack(int format, const double* d_packed, long long n_cfg, double* d_out, void* cuda_stream) {
  if (n_cfg < 0 || (format != NO_PACK_CHARGE && format != NO_PACK_ISOSPIN)) return NO_ERR_INVALID;
  if (n_cfg == 0) return NO_OK;
  if (!d_packed || !d_out) return NO_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_packed) & 15u) || (reinterpret_cast<uintptr_t>(d_out) & 15u)) return NO_ERR_INVALID;
  // runs on the device that owns the pointers (the caller's current device), like a memcpy
  const int mode = format == NO_PACK_CHARGE ? kModePacked : kModeIso;
  const long long pd = no3n::out_doubles(mode);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  for (long long c0 = 0; c0 < n_cfg; c0 += kMaxGrid) {
    const long long cnt = n_cfg - c0 < kMaxGrid ? n_cfg - c0 : kMaxGrid;
    unpack_kernel<<<(unsigned)cnt, 256, 0, s>>>(reinterpret_cast<const double2*>(d_packed + pd * c0), cnt,
                                                reinterpret_cast<double2*>(d_out + 512 * c0), mode);
    NO_CUDA(cudaGetLastError());
  }
  return NO_OK;
}

int no_free(no_handle* h) {
  if (!h) return NO_OK;
  DeviceGuard guard(h->device);
  if (h->d_tab) cudaFree(h->d_tab);
  if (h->d_cfg) cudaFree(h->d_cfg);
  if (h->d_out) cudaFree(h->d_out);
  if (h->hf_arena) cudaFree(h->hf_arena);
  if (h->host_path_ready) {
    cudaStreamDestroy(h->copy_stream);
    cudaEventDestroy(h->ev_chunk[0]);
    cudaEventDestroy(h->ev_chunk[1]);
    cudaEventDestroy(h->ev_copied);
  }
  delete h;
  return NO_OK;
}

const char* no_strerror(int code) {
  switch (code) {
    case NO_OK: return "success";
    case NO_ERR_INVALID: return "invalid argument (parameter out of range, null or misaligned pointer, n_cfg < 0, format not applicable)";
    case NO_ERR_CUDA: return "CUDA runtime or launch failure (see no_last_cuda_error)";
    case NO_ERR_ALLOC: return "allocation failed";
    case NO_ERR_BUSY: return "handle busy: another thread is inside a non-re-entrant entry point on it (retry later; not an argument error)";
    case NO_ERR_LIMIT: return "problem larger than the fixed, compiled-in capacity of an entry point that never allocates";
    default: return "unknown error code";
  }
}

const char* no_last_cuda_error(void) { return g_cuda_err; }

int no_kernel_info(const no_handle* h, int* regs, int* smem, int* threads, int* ctas_per_sm, int* n_sm,
                   int* cfg_per_cta) {
  if (!h) return NO_ERR_INVALID;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  cudaFuncAttributes a;
  NO_CUDA(cudaFuncGetAttributes(&a, (const void*)h->var.fn));
  int occ = 0;
  NO_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void*)h->var.fn, kWarps * 32, h->var.smem));
  int sms = 0;
  NO_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device));
  if (regs) *regs = a.numRegs;
  if (smem) *smem = (int)h->var.smem;
  if (threads) *threads = kWarps * 32;
  if (ctas_per_sm) *ctas_per_sm = occ;
  if (n_sm) *n_sm = sms;
  if (cfg_per_cta) *cfg_per_cta = kWarps;
  return NO_OK;
}

long long no_evals_per_cfg(const no_handle* h) { return h ? h->plan.evals_per_cfg : 0; }

int no_probe_fp64_peak(int device, int millis, double* tflops, int* n_sm, void* cuda_stream) {
  if (!tflops || millis < 1) return NO_ERR_INVALID;
  int n_dev = 0;
  NO_CUDA(cudaGetDeviceCount(&n_dev));
  if (device < 0 || device >= n_dev) return NO_ERR_INVALID;
  DeviceGuard guard(device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  int sms = 0;
  NO_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
  const int threads = 256, blocks = sms * 8;
  // everything the probe allocates is released on every exit
  struct Res {
    double* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ~Res() {
      if (e0) cudaEventDestroy(e0);
      if (e1) cudaEventDestroy(e1);
      if (sink) cudaFree(sink);
    }
  } r;
  NO_CUDA(cudaMalloc((void**)&r.sink, sizeof(double) * threads * blocks));
  NO_CUDA(cudaEventCreate(&r.e0));
  NO_CUDA(cudaEventCreate(&r.e1));
  int iters = 1 << 12;
  double best = 0.0;
  float ms = 0.f;
  // grow the launch until it lasts about `millis`, keep the best rate of the long launches
  for (int rep = 0; rep < 24; ++rep) {
    NO_CUDA(cudaEventRecord(r.e0, s));
    dfma_probe_kernel<<<blocks, threads, 0, s>>>(r.sink, iters, 1.0);
    NO_CUDA(cudaGetLastError());
    NO_CUDA(cudaEventRecord(r.e1, s));
    NO_CUDA(cudaEventSynchronize(r.e1));
    NO_CUDA(cudaEventElapsedTime(&ms, r.e0, r.e1));
    const double flops = 2.0 * 16.0 * (double)iters * threads * (double)blocks;
    const double rate = flops / (ms * 1e-3) * 1e-12;
    if (ms >= 0.5f * millis) {
      if (rate > best) best = rate;
      if (rep >= 3 && ms >= (float)millis) break;
    }
    if (ms < (float)millis && iters < (1 << 28)) iters *= 2;
  }
  *tflops = best;
  if (n_sm) *n_sm = sms;
  return NO_OK;
}

int no_probe_fp64_operands(int device, int millis, double* tflops_two, double* tflops_three, void* cuda_stream) {
  if (!tflops_two || !tflops_three || millis < 1) return NO_ERR_INVALID;
  int n_dev = 0;
  NO_CUDA(cudaGetDeviceCount(&n_dev));
  if (device < 0 || device >= n_dev) return NO_ERR_INVALID;
  DeviceGuard guard(device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  int sms = 0;
  NO_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device));
  const int threads = 256, blocks = sms * 4;
  struct Res {
    double* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ~Res() {
      if (e0) cudaEventDestroy(e0);
      if (e1) cudaEventDestroy(e1);
      if (sink) cudaFree(sink);
    }
  } r;
  NO_CUDA(cudaMalloc((void**)&r.sink, sizeof(double) * threads * blocks));
  NO_CUDA(cudaEventCreate(&r.e0));
  NO_CUDA(cudaEventCreate(&r.e1));
  double* res[2] = {tflops_two, tflops_three};
  for (int variant = 0; variant < 2; ++variant) {
    int iters = 1 << 12;
    double best = 0.0;
    float ms = 0.f;
    for (int rep = 0; rep < 24; ++rep) {
      NO_CUDA(cudaEventRecord(r.e0, s));
      if (variant) dfma_operand_probe_kernel<true><<<blocks, threads, 0, s>>>(r.sink, iters, 1.0);
      else dfma_operand_probe_kernel<false><<<blocks, threads, 0, s>>>(r.sink, iters, 1.0);
      NO_CUDA(cudaGetLastError());
      NO_CUDA(cudaEventRecord(r.e1, s));
      NO_CUDA(cudaEventSynchronize(r.e1));
      NO_CUDA(cudaEventElapsedTime(&ms, r.e0, r.e1));
      const double rate = 2.0 * 16.0 * (double)iters * threads * (double)blocks / (ms * 1e-3) * 1e-12;
      if (ms >= 0.5f * millis) {
        if (rate > best) best = rate;
        if (rep >= 3 && ms >= (float)millis) break;
      }
      if (ms < (float)millis && iters < (1 << 28)) iters *= 2;
    }
    *res[variant] = best;
  }
  return NO_OK;
}

}  // extern "C"


// ---- no_hf_energy_static: the Hartree-Fock energy for callers that must not allocate --------------------------------
// no_hf_energy keeps its intermediates (pair grids, generated configurations, weights, traced diagonals, the
// accumulator) in a handle-owned arena that it cudaMallocs and grows on demand.  The variant below runs the same
// kernels with the same arguments except that the arena is this fixed array, which is part of the library image:
// the CUDA runtime places it in the memory of every GPU whose context loads libno3n.so and keeps it until the
// process exits, whether or not the entry point is ever called.
namespace {

constexpr long long kStaticMaxNodes = NO_HF_STATIC_MAX_NODES;   // n_r n_cos n_phi of particles 1 and 2
constexpr long long kStaticChunk = 1LL << 16;                   // pair configurations per pass through the kernels
constexpr long long kStaticAccSlot = 32;                        // doubles reserved for the accumulator (256 bytes)
constexpr long long kStaticDoubles = kStaticAccSlot + 8 * kStaticMaxNodes + 14 * kStaticChunk;
static_assert(kStaticDoubles * 8 == NO_HF_STATIC_BYTES, "include/no.h states the size of the static scratch");

static __device__ __align__(256) double g_hf_static[kStaticDoubles];

// In host code `g_hf_static` names a host-side shadow of the array, NOT memory a kernel can use; the address the
// kernels need is a per-device fact that cudaGetSymbolAddress reports for the device that is current.  It is
// looked up once per device (first call on that device) and kept here.  The mutex of a slot also serialises the
// calls on that device: they all work in the one array, so two of them in flight together would corrupt each other.
constexpr int kStaticMaxDevices = 64;
struct StaticSlot {
  std::mutex mu;
  double* base = nullptr;
};
StaticSlot g_static_slot[kStaticMaxDevices];

}  // namespace

extern "C" int no_hf_energy_static(no_handle* h, int n_r, int n_cos, int n_phi, double* e_over_v, void* cuda_stream) {
  if (!h || !e_over_v) return NO_ERR_INVALID;
  if (n_r < 1 || n_r > kMaxOrder || n_cos < 1 || n_cos > kMaxOrder || n_phi < 1 || n_phi > kMaxOrder) return NO_ERR_INVALID;
  const long long n1 = (long long)n_r * n_cos * n_phi;
  if (n1 > kStaticMaxNodes) return NO_ERR_LIMIT;                 // the array cannot hold the two pair grids
  if (h->device < 0 || h->device >= kStaticMaxDevices) return NO_ERR_LIMIT;
  DeviceGuard guard(h->device);
  if (!guard.ok) return cuda_fail(cudaGetLastError(), "cudaSetDevice");
  StaticSlot& slot = g_static_slot[h->device];
  std::lock_guard<std::mutex> serial(slot.mu);                   // held until this call's stream has drained
  if (!slot.base) {
    // set-up, once per device, with that device current (DeviceGuard above)
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_hf_static);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(static HF scratch)");
    if (!p) return cuda_fail(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(static HF scratch) returned NULL");
    slot.base = p;
  }
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const int layout = h->layout.load(std::memory_order_relaxed) == 2 ? 2 : 1;
  const double kf[2] = {h->plan.kf_p, h->plan.kf_n};
  const bool fused = kf[0] > 0 && kf[0] == kf[1];                // as in no_hf_energy: one pair grid serves all four
  std::vector<double> nodes[2];                                  // host heap only (a few KB of quadrature nodes)
  for (int t = 0; t < 2; ++t)
    if (kf[t] > 0 && !(fused && t == 1)) sphere_nodes(n_r, n_cos, n_phi, kf[t], nodes[t]);
  const long long chunk = n1 * n1 < kStaticChunk ? n1 * n1 : kStaticChunk;
  double* d_acc = slot.base;
  double* d_nodes[2] = {slot.base + kStaticAccSlot, fused ? slot.base + kStaticAccSlot : slot.base + kStaticAccSlot + 4 * n1};
  double *d_cfg = slot.base + kStaticAccSlot + 8 * kStaticMaxNodes, *d_w = d_cfg + 9 * chunk, *d_diag = d_w + chunk;
  for (int t = 0; t < 2; ++t)
    if (!nodes[t].empty())
      NO_CUDA(cudaMemcpyAsync(d_nodes[t], nodes[t].data(), sizeof(double) * 4 * (size_t)n1, cudaMemcpyHostToDevice, s));
  // the array still holds whatever the previous call left: the accumulator is the one place that is added to
  // before it is written, so it is cleared here; every other element read below is written first in this call
  NO_CUDA(cudaMemsetAsync(d_acc, 0, sizeof(double), s));
  for (int t1 = 0; t1 < 2; ++t1)
    for (int t2 = 0; t2 < 2; ++t2) {
      if (!(kf[t1] > 0) || !(kf[t2] > 0)) continue;
      if (fused && (t1 || t2)) continue;
      for (long long c0 = 0; c0 < n1 * n1; c0 += chunk) {
        const long long count = n1 * n1 - c0 < chunk ? n1 * n1 - c0 : chunk;
        hf_pairs_kernel<<<(unsigned)((count + 255) / 256), 256, 0, s>>>(d_nodes[t1], d_nodes[t2], n1, c0, count, d_cfg, d_w);
        NO_CUDA(cudaGetLastError());
        const int rc = launch(h, d_cfg, count, d_diag, s, layout, kModeDiag, true);   // p' = p by construction
        if (rc != NO_OK) { cudaStreamSynchronize(s); return rc; }
        hf_reduce_kernel<<<1, 1024, 0, s>>>(d_diag, d_w, count, fused ? -1 : 2 * t1 + t2, d_acc);
        NO_CUDA(cudaGetLastError());
      }
    }
  double acc = 0.0;
  NO_CUDA(cudaMemcpyAsync(&acc, d_acc, sizeof(double), cudaMemcpyDeviceToHost, s));
  NO_CUDA(cudaStreamSynchronize(s));
  *e_over_v = acc / 6.0;
  return NO_OK;
}
