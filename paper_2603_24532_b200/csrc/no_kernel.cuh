// no_kernel.cuh -- the sm_100a kernel of the 3N normal ordering.
//
// One warp integrates one configuration (p, p', P): lanes stride over the angular directions
// of the k3 grid, every lane runs the radial loop of its direction, kNodesPerTrip nodes per trip, with
// the 17 first-level sums in registers (no3n::nodes, the hot loop, branch free; the radial nodes and
// weights are read from the kernel-parameter block, i.e. as uniform-register operands), folds them into
// lane-private shared-memory accumulators (no3n::second_level), then the warp reduces the 57
// (81 with c4) moments, turns them into Pauli-operator coefficients and writes the 16x16 complex
// matrix.  A CTA holds WARPS warps; the 2^(j/256) table and the quadrature tables of every Fermi
// sphere are staged once per CTA into shared memory with one TMA bulk copy (cp.async.bulk +
// mbarrier); r^2 + gam_l of the configuration is tabulated per warp.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "no_core.h"
#include "no_tma.cuh"

namespace no3n {

constexpr int kModeFull = 0;   // out[n_cfg][16][16][2]
constexpr int kModeDiag = 1;   // out[n_cfg][4]
constexpr int kModePacked = 2; // out[n_cfg][16 spin elements][6 charge-conserving isospin blocks][2]   (include/no.h NO_PACK_CHARGE)
constexpr int kModeIso = 3;    // out[n_cfg][16 spin elements][(pn,pn), (pn,np)][2], isospin-symmetric matter (NO_PACK_ISOSPIN)

__host__ __device__ constexpr int out_doubles(int mode) {
  return mode == kModeDiag ? 4 : (mode == kModePacked ? 192 : (mode == kModeIso ? 64 : 512));
}

// shared memory per CTA, in doubles:
//   tables | mbarrier (2) | per warp: CfgConst (40) | radial table [n_r_pad][6] aliased with mom[rows_pad] | acc[32][stride]
// (the reduced moments are written after the last read of the radial table of a pass, and the table is rebuilt
//  at the start of the next pass: the two share one region, sized for the larger)
template <bool C4> __host__ __device__ constexpr int rows_pad() { return (Layout<C4>::kRows + 3) & ~3; }

template <bool C4> __host__ __device__ inline int warp_doubles(int n_r_pad) {
  const int shared_region = kRadT * n_r_pad > rows_pad<C4>() ? kRadT * n_r_pad : rows_pad<C4>();
  return kCfgDoubles + shared_region + Layout<C4>::kStride * kLanes;
}

template <bool C4>
inline size_t smem_bytes(int tab_doubles, int n_r_pad, int warps) {
  return sizeof(double) * (size_t)(tab_doubles + 2 + warps * warp_doubles<C4>(n_r_pad));
}

// radial loop of one direction: kNodesPerTrip independent nodes per trip
template <int NREG, bool FLUSH, bool FWD>
__device__ __forceinline__ void radial_loop(const DevParams& P, int pass, const double* rsp, const double* e2tab,
                                            const DirConst& d, const double2* tt2, const double* ttab, First& f) {
#pragma unroll 1
  for (int i = 0; i < P.n_r_pad; i += kNodesPerTrip) {
    double r[kNodesPerTrip], wr[kNodesPerTrip], T[kNodesPerTrip][5];
#pragma unroll
    for (int k = 0; k < kNodesPerTrip; ++k) {
      const double2 t0 = tt2[3 * (i + k)], t1 = tt2[3 * (i + k) + 1];
      const double t2 = ttab[kRadT * (i + k) + 4];
      r[k] = P.radk[pass][i + k][0]; wr[k] = P.radk[pass][i + k][1];
      T[k][0] = t0.x; T[k][1] = t0.y; T[k][2] = t1.x; T[k][3] = t1.y; T[k][4] = t2;
    }
    nodes<NREG, kNodesPerTrip, FLUSH, FWD>(rsp, P.n_reg, e2tab, d, r, wr, T, f);
  }
}

// SPLIT = 1: one warp per configuration, WARPS configurations per CTA (the throughput layout).
// SPLIT = WARPS > 1: the whole CTA integrates ONE configuration, the directions dealt round-robin to its warps,
// the reduced moments of the warps added in a fixed order by warp 0, which then runs the epilogue alone: the
// small-batch layout (fewer configurations than warp slots), chosen by the launcher.
// FWD: every configuration of the launch has p' = p exactly (set by the Hartree-Fock entry points, which build
// the configurations themselves): duplicate legs and pairs are skipped, see no3n::nodes.
template <int NREG, bool C4, int WARPS, int MINB, int SPLIT = 1, bool FWD = false>
__global__ void __launch_bounds__(WARPS * 32, MINB)
no3n_kernel(const __grid_constant__ DevParams P, const double* __restrict__ cfg, long long n_cfg, double* __restrict__ out,
            int mode) {
  extern __shared__ __align__(128) double smem[];
  using L = Layout<C4>;
  double* s_tab = smem;
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + P.tab_doubles);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* wbase = smem + P.tab_doubles + 2 + warp * warp_doubles<C4>(P.n_r_pad);
  CfgConst* cc = reinterpret_cast<CfgConst*>(wbase);
  double* ttab = wbase + kCfgDoubles;
  double* mom = ttab;                                 // alias, see the layout comment
  double* acc = ttab + (kRadT * P.n_r_pad > rows_pad<C4>() ? kRadT * P.n_r_pad : rows_pad<C4>());

  // the configuration is requested first: its global-load latency overlaps the table staging
  static_assert(SPLIT == 1 || SPLIT == WARPS, "a split CTA holds one configuration");
  const long long ic = SPLIT == 1 ? (long long)blockIdx.x * WARPS + warp : (long long)blockIdx.x;
  const int part = SPLIT == 1 ? 0 : warp;             // which share of the directions this warp takes
  double q[9];
#pragma unroll
  for (int a = 0; a < 9; ++a) q[a] = ic < n_cfg ? __ldg(cfg + ic * 9 + a) : 0.0;

  // ---- a0: stage the exp table and the quadrature tables (TMA bulk copy, one per CTA) ----
  if (threadIdx.x == 0) {
    mbar_init(bar, 1);
    const uint32_t bytes = (uint32_t)P.tab_doubles * 8u;
    mbar_expect_tx(bar, bytes);
    tma_bulk_g2s(s_tab, P.tab, bytes, bar);
  }
  __syncthreads();

  if (ic >= n_cfg) return;

  // ---- a1: per-configuration constants, one copy per warp in shared memory ----
  {
    CfgConst c;
    cfg_setup<NREG>(P, q, c);
    if (lane == 0) *cc = c;
  }
  __syncwarp();
  double rs[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) rs[k] = cc->rs[k];
  // The coefficients are the same in every lane.  A warp reduction (SASS REDUX) returns its result in a UNIFORM
  // register, and ptxas then keeps the rebuilt double there: the Horner steps of the regulator polynomial read it as a
  // uniform operand and need two register-file operands instead of three (2 instead of 3 FP64 pipe cycles each,
  // DESIGN.md section 5.2; +1.1 % on the large grids, profiles/r02a.md).  The reduction is over identical values.
  if (NREG >= 1) {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const unsigned lo = __reduce_max_sync(0xffffffffu, (unsigned)__double2loint(rs[k]));
      const unsigned hi = __reduce_max_sync(0xffffffffu, (unsigned)__double2hiint(rs[k]));
      rs[k] = __hiloint2double((int)hi, (int)lo);
    }
  }
  const double* rsp = NREG >= 1 ? rs : cc->rs;     // unrolled exponents keep the coefficients in registers
  const bool flush = NREG >= 0 && needs_flush(*cc);   // warp uniform
  mbar_wait(bar, 0);
  const double* e2tab = s_tab;

  double blk[6] = {0, 0, 0, 0, 0, 0};
  for (int pass = 0; pass < P.n_pass; ++pass) {
    const double* rad = s_tab + P.pass_off[pass];
    const double* ct = rad + 2 * P.n_r_pad;
    const double* st = ct + P.n_cos;
    const double* wc = st + P.n_cos;
    const double* cph = wc + P.n_cos;
    const double* sph = cph + P.n_phi;
    const double* wph = sph + P.n_phi;
    for (int i = lane; i < P.n_r_pad; i += kLanes) radial_entry(*cc, rad[2 * i], ttab + kRadT * i);
    // ---- a2 + a3: hot loop over the k3 nodes of this sphere ----
    const int n_dir = P.n_list > 0 ? P.n_list : P.n_cos * P.n_phi;
    const int dstep = kLanes * SPLIT, m0 = lane + kLanes * part;
    // a lane's accumulator rows are WRITTEN by its first direction of the pass (second_level<.., FIRST>) and updated
    // by the others; only a lane without any direction clears its rows (in FWD launches the rows of the duplicate legs
    // are never written: the lane reduction adds whatever they hold and the copy after it overwrites the result)
    if (m0 >= n_dir) {
      Pair* z = reinterpret_cast<Pair*>(acc + lane * L::kStride);
#pragma unroll
      for (int k = 0; k < L::kStride / 2; ++k) z[k] = Pair{0.0, 0.0};
    }
    __syncwarp();
    const int dj = dstep / P.n_phi, dl = dstep - dj * P.n_phi;     // (j, l) advance by dstep directions per trip
    int j = m0 / P.n_phi, l = m0 - j * P.n_phi;
    const double4* dlist = reinterpret_cast<const double4*>(ct);   // list mode: (ux, uy, uz, w), 32-byte aligned
    const double2* tt2 = reinterpret_cast<const double2*>(ttab);
#pragma unroll 1
    for (int m = m0; m < n_dir; m += dstep) {
      DirConst d;
      double w;
      if (P.n_list > 0) {                                   // caller-supplied angular rule (e.g. Lebedev)
        const double4 q = dlist[m];
        dir_setup(*cc, q.x, q.y, q.z, d);
        w = q.w;
      } else {
        const double sj = st[j];
        dir_setup(*cc, sj * cph[l], sj * sph[l], ct[j], d);
        w = wc[j] * wph[l];
      }
      First f;
      first_zero(f);
      if (flush) radial_loop<NREG, true, FWD>(P, pass, rsp, e2tab, d, tt2, ttab, f);
      else radial_loop<NREG, false, FWD>(P, pass, rsp, e2tab, d, tt2, ttab, f);
      if (m == m0) second_level<C4, FWD, true>(f, d, cc->gam, w, acc + lane * L::kStride);
      else second_level<C4, FWD, false>(f, d, cc->gam, w, acc + lane * L::kStride);
      j += dj; l += dl;
      if (l >= P.n_phi) { l -= P.n_phi; ++j; }
    }
    __syncwarp();

    // ---- a3: reduce the moments over the 32 lanes (fixed order) ----
    // a lane adds one PAIR of adjacent rows over the 32 lanes: 16-byte loads, four independent chains of eight
    // (fixed order: bit reproducible), then a fixed tree.  Lane l starts at source lane 2 l: with an odd number of
    // 16-byte units per lane (29 or 41) the eight lanes of a quarter warp then hit eight different bank groups.
    {
      const Pair* acc2 = reinterpret_cast<const Pair*>(acc);
      Pair* mom2 = reinterpret_cast<Pair*>(mom);
      constexpr int kUnits = L::kStride / 2;
      for (int pr = lane; pr < kUnits; pr += kLanes) {
        Pair s0 = {0.0, 0.0}, s1 = {0.0, 0.0}, s2 = {0.0, 0.0}, s3 = {0.0, 0.0};
#pragma unroll
        for (int t = 0; t < 8; ++t) {
          const Pair a0 = acc2[((2 * lane + t) & 31) * kUnits + pr], a1 = acc2[((2 * lane + t + 8) & 31) * kUnits + pr];
          const Pair a2 = acc2[((2 * lane + t + 16) & 31) * kUnits + pr], a3 = acc2[((2 * lane + t + 24) & 31) * kUnits + pr];
          s0.x += a0.x; s0.y += a0.y; s1.x += a1.x; s1.y += a1.y;
          s2.x += a2.x; s2.y += a2.y; s3.x += a3.x; s3.y += a3.y;
        }
        mom2[pr] = Pair{(s0.x + s1.x) + (s2.x + s3.x), (s0.y + s1.y) + (s2.y + s3.y)};
      }
    }
    __syncwarp();

    if (FWD) {                                          // legs 2, 3 = legs 0, 1; pair 3 = pair 2
      __syncwarp();
      if (lane < 20) mom[L::kRowLeg + 20 + lane] = mom[L::kRowLeg + lane];
      if (lane < L::kPairRows) mom[L::kRowPair + 3 * L::kPairRows + lane] = mom[L::kRowPair + 2 * L::kPairRows + lane];
      __syncwarp();
    }
    if (SPLIT > 1) {                                    // add the warps' partial moments (fixed order)
      __syncthreads();
      if (warp == 0)
        for (int row = lane; row < L::kRows; row += kLanes) {
          double s = mom[row];
#pragma unroll
          for (int w = 1; w < SPLIT; ++w) s += mom[w * warp_doubles<C4>(P.n_r_pad) + row];
          mom[row] = s;
        }
      __syncthreads();                                  // the other warps may now reuse their regions
    }

    // ---- a4: epilogue, phases 1 and 2 (records live in the dead accumulator area) ----
    if (SPLIT == 1 || warp == 0) {
      double* rec = acc;
      __syncwarp();
      if (lane < 6) phase1_job<C4>(P, *cc, mom, lane, rec);
      __syncwarp();
      phase2_lane(rec, lane, P.nsp[pass], P.esum[pass], NREG >= 0 ? exp(-cc->E0) : 1.0, blk);
      __syncwarp();
    }
  }
  if (SPLIT > 1 && warp != 0) return;

  // ---- a4: phase 3, (1 - P12) and expansion to the 16x16 complex matrix ----
  double* coef = acc;
#pragma unroll
  for (int b = 0; b < 6; ++b) coef[lane * 6 + b] = blk[b];
  __syncwarp();
  if (mode == kModeDiag) {
    // spin-traced diagonal per isospin pair: out[ic][2 t1 + t2] = sum_{s1 s2} Re M[(s1 s2 t1 t2), (s1 s2 t1 t2)]
    // (the input of the Hartree-Fock contraction, Eq. (1)/(9): the 16x16 matrix never leaves the SM)
    double re = 0.0, im = 0.0;
    if (lane < 16) phase3_elem(coef, lane, lane, re, im);
    re += __shfl_xor_sync(0xffffffffu, re, 4);
    re += __shfl_xor_sync(0xffffffffu, re, 8);
    if (lane < 4) out[ic * 4 + lane] = re;
    return;
  }
  P3Lane pl;
  phase3_lane_setup(lane, pl);
  const int h = lane & 1;
  if (mode == kModePacked) {
    // only the 96 entries that charge conservation allows, [spin element][block]
    double2* o = reinterpret_cast<double2*>(out) + ic * 96 + (lane >> 1) * 6 + h;
#pragma unroll
    for (int it = 0; it < 3; ++it) {
      double re, im;
      phase3_block(coef, pl, 2 * it + h, re, im);
      o[2 * it] = make_double2(re, im);
    }
    return;
  }
  if (mode == kModeIso) {
    // isospin-symmetric matter: the (pn,pn) and (pn,np) blocks determine the other four (pin P9); one 512-byte warp store
    double re, im;
    phase3_block(coef, pl, h ? 4 : 1, re, im);
    reinterpret_cast<double2*>(out)[ic * 32 + lane] = make_double2(re, im);
    return;
  }
  double2* o = reinterpret_cast<double2*>(out) + ic * 256;
#pragma unroll
  for (int it = 0; it < 3; ++it) {
    double re, im;
    const int off = phase3_block(coef, pl, 2 * it + h, re, im);
    o[off] = make_double2(re, im);
  }
#pragma unroll
  for (int it = 0; it < 5; ++it) o[phase3_zero_off(pl, 2 * it + h)] = make_double2(0.0, 0.0);
}

// ---- reconstruction of the 16x16 matrix from a packed form ----
// one thread per element of the full matrix: charge-violating entries are 0; format kModeIso fills the four other
// charge-conserving blocks from isospin symmetry, (pp,pp) = (nn,nn) = (pn,pn) + (pn,np), (np,np) = (pn,pn), (np,pn) = (pn,np)
__global__ void __launch_bounds__(256) unpack_kernel(const double2* __restrict__ packed, long long n_cfg,
                                                     double2* __restrict__ out, int mode) {
  const long long c = blockIdx.x;
  const int e = threadIdx.x, row = e >> 4, col = e & 15;
  const int sp = 4 * (row >> 2) + (col >> 2), nb = iso_block(row & 3, col & 3);
  double2 v = make_double2(0.0, 0.0);
  if (nb >= 0) {
    if (mode == kModePacked) {
      v = packed[c * 96 + 6 * sp + nb];
    } else {
      const double2 d = packed[c * 32 + 2 * sp], x = packed[c * 32 + 2 * sp + 1];
      if (nb == 0 || nb == 3) v = make_double2(d.x + x.x, d.y + x.y);
      else v = nb < 3 ? d : x;
    }
  }
  if (c < n_cfg) out[c * 256 + e] = v;
}

// ---- Hartree-Fock contraction helpers ----
// configurations of the node pairs [c0, c0 + count) of two single-particle grids: pair c = i1 * n2 + i2,
// (p, p', P) = ((k1 - k2)/2, (k1 - k2)/2, k1 + k2), weight W1 W2.  nodes: [n][4] = (kx, ky, kz, W).
__global__ void hf_pairs_kernel(const double* __restrict__ nodes1, const double* __restrict__ nodes2, long long n2,
                                long long c0, long long count, double* __restrict__ cfg, double* __restrict__ w) {
  const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= count) return;
  const long long pair = c0 + c, i1 = pair / n2, i2 = pair - i1 * n2;
  const double* a = nodes1 + 4 * i1;
  const double* b = nodes2 + 4 * i2;
#pragma unroll
  for (int x = 0; x < 3; ++x) {
    const double p = 0.5 * (a[x] - b[x]);
    cfg[9 * c + x] = p;
    cfg[9 * c + 3 + x] = p;
    cfg[9 * c + 6 + x] = a[x] + b[x];
  }
  w[c] = a[3] * b[3];
}

// sigma[(row0 + i1) 2 + t1] += scale sum_{i2 < n2} w[i1 n2 + i2] diag[i1 n2 + i2][2 t1 + t2], t1 = 0, 1: one CTA per
// momentum k1 (row i1 of the chunk), fixed summation order.  t2 < 0: both species of particle 2 share this grid
// (equal Fermi momenta), their two columns are added
__global__ void __launch_bounds__(256) sp_reduce_kernel(const double* __restrict__ diag, const double* __restrict__ w,
                                                        long long n2, int t2, double scale, long long row0,
                                                        double* __restrict__ sigma) {
  __shared__ double sh[2][256];
  const long long base = (long long)blockIdx.x * n2;
  double s0 = 0.0, s1 = 0.0;
  for (long long i2 = threadIdx.x; i2 < n2; i2 += 256) {
    const double wv = w[base + i2];
    const double* d = diag + 4 * (base + i2);
    s0 = fma(wv, t2 < 0 ? d[0] + d[1] : d[t2], s0);
    s1 = fma(wv, t2 < 0 ? d[2] + d[3] : d[2 + t2], s1);
  }
  sh[0][threadIdx.x] = s0;
  sh[1][threadIdx.x] = s1;
  __syncthreads();
  for (int half = 128; half > 0; half >>= 1) {
    if ((int)threadIdx.x < half) {
      sh[0][threadIdx.x] += sh[0][threadIdx.x + half];
      sh[1][threadIdx.x] += sh[1][threadIdx.x + half];
    }
    __syncthreads();
  }
  if (threadIdx.x < 2) sigma[2 * (row0 + blockIdx.x) + threadIdx.x] += scale * sh[threadIdx.x][0];
}

// acc[0] += sum_c w[c] diag[c][blk], one CTA, fixed summation order (bit reproducible); blk < 0: the four isospin
// pairs share this pair grid (equal Fermi momenta) and their columns are added
__global__ void __launch_bounds__(1024) hf_reduce_kernel(const double* __restrict__ diag, const double* __restrict__ w,
                                                         long long count, int blk, double* __restrict__ acc) {
  __shared__ double sh[1024];
  double s = 0.0;
  for (long long c = threadIdx.x; c < count; c += 1024) {
    const double* d = diag + 4 * c;
    s = fma(w[c], blk < 0 ? (d[0] + d[1]) + (d[2] + d[3]) : d[blk], s);
  }
  sh[threadIdx.x] = s;
  __syncthreads();
  for (int half = 512; half > 0; half >>= 1) {
    if ((int)threadIdx.x < half) sh[threadIdx.x] += sh[threadIdx.x + half];
    __syncthreads();
  }
  if (threadIdx.x == 0) acc[0] += sh[0];
}

// ---- FP64 roofline probe: 16 independent DFMA chains per thread ----
__global__ void __launch_bounds__(256) dfma_probe_kernel(double* sink, int iters, double seed) {
  double a[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) a[k] = seed + k + threadIdx.x;
  const double x = 1.0 - 1e-9 * seed, y = 1e-9;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = fma(a[k], x, y);
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k];
  if (s == 123.456) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ---- FP64 operand-delivery probe: the same 16 DFMA chains with TWO or THREE fresh register operands ----
// two:   a[k] = fma(a[k], x, y)        x, y loop invariant (one register-file read per instruction after reuse)
// three: a[k] = fma(b[k], c[k'], a[k]) three distinct 64-bit registers per instruction (b, c rotate so that no
//        operand-reuse slot hits)
template <bool THREE>
__global__ void __launch_bounds__(256) dfma_operand_probe_kernel(double* sink, int iters, double seed) {
  double a[16], b[16], c[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    a[k] = seed + k + threadIdx.x;
    b[k] = 1.0 - 1e-9 * (seed + k + threadIdx.x);       // thread dependent: plain registers, not uniform ones
    c[k] = 1e-9 * (k + 1 + threadIdx.x);
  }
  const double x = 1.0 - 1e-9 * seed, y = 1e-9;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = THREE ? fma(b[k], c[(k + 5) & 15], a[k]) : fma(a[k], x, y);
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < 16; ++k) s += a[k] + (THREE ? b[k] + c[k] : 0.0);
  if (s == 123.456) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace no3n
