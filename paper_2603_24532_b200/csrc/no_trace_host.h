// no_trace_host.h -- host-side planning of the spin-isospin trace kernel (PAPER.md:155-157 and
// Appendix B): turns a diagram topology into a short program of tensor contractions.
// Plain C++ (no CUDA calls) so that the CPU tests can drive it through tests/trace_emu.cpp.  Nothing here is shared
// with oracle/.
//
// The trace of a closed two-body diagram,
//     T = sum over the labels x_j = 2 s_j + t_j of its 2 n lines of prod_v V_v[pair(o1, o2)][pair(i1, i2)],
// is the full contraction of a tensor network whose nodes are the vertex matrices.  The paper loops over the labels
// (restricted to charge-conserving isospin assignments) with the most connected vertex pair innermost
// (PAPER.md:643-651).  Here the network is contracted vertex by vertex instead: the partial result R carries the
// labels of the lines that are cut by the frontier ("open" lines, at most kMaxOpen = 4, i.e. 256 complex numbers that
// live in shared memory), and absorbing a vertex is one small complex matrix product
//     R'[a, b] = sum_g R[a, g] W_v[g, b]        a: labels of the open lines that stay open  (nA = 4^kept values)
//                                                g: labels of the lines the vertex closes     (nC = 4^closed)
//                                                b: labels of the lines the vertex opens      (nB = 4^new)
// which turns the exponential label sum (4^(2n) terms) into n products of at most 16 x 16 x 16.  Topologies whose
// frontier would exceed four lines are handled by "slicing": the labels of up to kMaxSlice lines are fixed in an outer
// loop; a line that starts and ends on the same vertex is summed inside that vertex's step.  The order of the vertices and the sliced
// lines are chosen here, on the host, by exhaustive search for the fewest complex multiply-adds.
//
// All index arithmetic of the kernel is tabulated here: with x the label of a line attached to slot q of a vertex
// (q = 0, 1: outgoing 1, 2; q = 2, 3: incoming 1, 2) the element offset inside the 16 x 16 matrix of include/no.h
// (row = outgoing pair, column = incoming pair, pair index 8 s1 + 4 s2 + 2 t1 + t2) is the sum over the four slots of
// slot_off(q, x); offsets into R are sums of label * 4^(position of the line in the open list); the new partial result
// is stored at index a + nA b (kept labels, then opened labels).
#pragma once

#include <stdint.h>

#include <algorithm>
#include <vector>

namespace no3n {

constexpr int kTrMaxVertex = 6;
constexpr int kTrMaxLines = 2 * kTrMaxVertex;
constexpr int kTrMaxOpen = 4;        // open lines of the partial result: 4^4 = 256 complex numbers
constexpr int kTrMaxSlice = 3;       // lines whose labels are fixed in the outer loop
constexpr int kTrTab = 256;

// Shared-memory layouts (complex elements).  Both the vertex matrices and the partial result are held as 16 rows of
// kTrRow = 17 elements (one element of padding per row): consecutive rows start one 16-byte bank group apart, so a
// warp access whose lanes differ in row AND column bits spreads over all banks.  Padding is additive on offsets
// that occupy disjoint digits, so every table below holds padded offsets and the kernel only adds them.
constexpr int kTrRow = 17;
constexpr int kTrMat = 16 * kTrRow;  // elements of one padded 16 x 16 matrix
inline int tr_pad(int idx) { return idx + (idx >> 4); }   // canonical index (16 row + col) -> padded offset
// row stride of the VERTEX matrices in shared memory: padded like R (written by 16-byte cp.async).  Unpadded rows
// filled by one TMA bulk copy per vertex were measured too: 2.12e8 against 2.43e8 samples/s (profiles/r02b.md)
constexpr int kTrRowW = kTrRow;
constexpr int kTrMatW = 16 * kTrRowW;
inline int tr_padw(int idx) { return (idx >> 4) * kTrRowW + (idx & 15); }

inline int slot_off(int slot, int x) {
  const int s = x >> 1, t = x & 1;
  switch (slot) {
    case 0: return kTrRowW * (8 * s + 2 * t);   // outgoing 1: row bits s1, t1
    case 1: return kTrRowW * (4 * s + t);       // outgoing 2: row bits s2, t2
    case 2: return 8 * s + 2 * t;               // incoming 1: column bits
    default: return 4 * s + t;                  // incoming 2
  }
}

// one absorption step, as the kernel runs it (offsets in complex elements)
struct TraceStep {
  int vertex;                 // which vertex matrix of the sample
  int nA, nB, nC;             // kept, opened, closed label combinations (powers of 4); nA * nB <= 256
  int skip;                   // 1: this step only copies its vertex into R and the next step reads the vertex directly
  int r_vertex;               // >= 0: R of this step IS that vertex matrix (baseR, offR hold offsets into it); -1: R
  int fuse_last;              // 1: the next (last) step closes all four lines: its sum is folded into this step,
                              //    lastW[o] = offset in the LAST vertex of the element that multiplies R'[o]
  int big;                    // 1: 16 x 16 x 16 step (two kept, two closed, two opened lines), tile tables below are valid
  uint16_t baseR[kTrTab];     // [a]  offset of the kept labels in R (all offsets padded, see kTrRow)
  uint16_t offR[kTrTab];      // [g]  offset of the closed labels in R
  uint16_t baseW[kTrTab];     // [b]  offset of the opened labels in the vertex matrix
  uint16_t offW[kTrTab];      // [g]  offset of the closed labels in the vertex matrix
  uint16_t sliceW[64];        // [outer iteration] offset of the sliced labels in the vertex matrix
  uint16_t lastW[kTrTab];     // [o = a + 16 b] see fuse_last
  // 16 x 16 x 16 steps only.  The 16 label combinations of a line pair are enumerated isospin-major,
  // e = 4 iso + spin, iso over (t1,t2) = (0,1) (1,0) (0,0) (1,1), spin = s1 + 2 s2: a tensor-core tile of 8 holds
  // two isospin combinations, a k-step of 4 holds one.  R'[a, b] is stored at outA[a] + outB[b] (padded offsets of
  // the canonical index); lastW is indexed by a + 16 b of this enumeration.
  uint16_t outA[16], outB[16];
  // tile_mask[ks] bit (2 mt + nt): the 8 x 8 x 4 product of m-tile mt, n-tile nt, k-step ks can be non-zero; all
  // ones unless the plan was made for charge-conserving vertices.  There the product is block diagonal: k-steps 0, 1
  // feed output tile (0, 0), k-steps 2, 3 feed tile (1, 1), the off-diagonal tiles are zero (block_diag = 1,
  // ks_valid bit ks: the k-step contributes).
  uint8_t tile_mask[4];
  uint8_t block_diag, ks_valid;
  uint8_t pad2_[10];
};

struct TracePlan {
  int n_vertex;
  int n_slice_iter;           // 4^(number of sliced lines)
  int n_sliced;
  int sliced[kTrMaxSlice];    // line ids
  int order[kTrMaxVertex];    // vertices in absorption order
  int max_open;               // widest frontier
  long long cmacs;            // complex multiply-adds per sample (all outer iterations)
  long long n_isospin;        // charge-conserving isospin assignments of the lines, for information
  long long dmma_products;    // 8 x 8 x 4 real tensor-core products per sample in the 16 x 16 x 16 steps (after skipping)
  int charge;                 // 1: planned for charge-conserving vertices (structurally zero tiles are skipped)
  TraceStep steps[kTrMaxVertex];
};

inline bool trace_topology_valid(int n, const int* topo) {
  if (n < 1 || n > kTrMaxVertex) return false;
  int outs[kTrMaxLines] = {0}, ins[kTrMaxLines] = {0};
  for (int v = 0; v < n; ++v)
    for (int q = 0; q < 4; ++q) {
      const int l = topo[4 * v + q];
      if (l < 0 || l >= 2 * n) return false;
      (q < 2 ? outs : ins)[l]++;
    }
  for (int l = 0; l < 2 * n; ++l) if (outs[l] != 1 || ins[l] != 1) return false;
  return true;
}

namespace trace_detail {

// frontier simulation of one (order, sliced set); returns the cost or -1 if the frontier exceeds kTrMaxOpen
inline long long simulate(int n, const int* topo, const int* order, unsigned sliced_mask, int* max_open) {
  int open[kTrMaxLines], n_open = 0;
  long long cost = 0;
  *max_open = 0;
  for (int k = 0; k < n; ++k) {
    const int v = order[k];
    int closed = 0, opened = 0, self = 0;
    for (int q = 0; q < 4; ++q) {
      const int l = topo[4 * v + q];
      if (sliced_mask >> l & 1) continue;
      bool twice = false;                      // a line that leaves and enters this vertex: summed inside the step
      for (int r = 0; r < 4; ++r) twice |= r != q && topo[4 * v + r] == l;
      if (twice) { self += q < 2; continue; }
      bool is_open = false;
      for (int j = 0; j < n_open; ++j) is_open |= open[j] == l;
      if (is_open) ++closed; else ++opened;
    }
    const int kept = n_open - closed;
    if (kept + opened > kTrMaxOpen) return -1;
    cost += (1LL << (2 * kept)) * (1LL << (2 * opened)) * (1LL << (2 * (closed + self)));
    // new frontier: kept lines in their old order, then the opened lines in slot order
    int next[kTrMaxLines], m = 0;
    for (int j = 0; j < n_open; ++j) {
      bool closes = false;
      for (int q = 0; q < 4; ++q) closes |= topo[4 * v + q] == open[j];
      if (!closes) next[m++] = open[j];
    }
    for (int q = 0; q < 4; ++q) {
      const int l = topo[4 * v + q];
      if (sliced_mask >> l & 1) continue;
      bool twice = false, was_open = false;
      for (int r = 0; r < 4; ++r) twice |= r != q && topo[4 * v + r] == l;
      for (int j = 0; j < n_open; ++j) was_open |= open[j] == l;
      if (!was_open && !twice) next[m++] = l;
    }
    n_open = m;
    for (int j = 0; j < m; ++j) open[j] = next[j];
    if (n_open > *max_open) *max_open = n_open;
  }
  return n_open == 0 ? cost : -1;
}

inline int popcount(unsigned m) { int c = 0; for (; m; m &= m - 1) ++c; return c; }

}  // namespace trace_detail

// 0 on success; 1 if the topology is malformed or cannot be contracted within the limits above
// charge: the caller promises that every vertex matrix is exactly zero outside the 96 charge-conserving entries
// (t_o1 + t_o2 = t_i1 + t_i2, what no_eval writes).  Then R[open labels] vanishes unless
// sum over the open lines of sigma_l t_l = 0 (sigma = +1: the line leaves the absorbed part, i.e. was opened at an
// outgoing slot; -1: it enters it) and the products of structurally zero tiles are skipped ("the
// subset of isospin configurations consistent with isospin conservation at each vertex").
inline int build_trace_plan(int n, const int* topo, TracePlan& plan, bool charge = false) {
  using namespace trace_detail;
  if (!trace_topology_valid(n, topo)) return 1;
  const int L = 2 * n;
  plan = TracePlan();
  plan.n_vertex = n;

  // charge-conserving isospin assignments (information only)
  plan.n_isospin = 0;
  for (unsigned m = 0; m < (1u << L); ++m) {
    bool ok = true;
    for (int v = 0; v < n && ok; ++v) {
      const int* t = topo + 4 * v;
      ok = (int)(m >> t[0] & 1) + (int)(m >> t[1] & 1) == (int)(m >> t[2] & 1) + (int)(m >> t[3] & 1);
    }
    plan.n_isospin += ok;
  }

  // exhaustive search: sliced sets of at most kTrMaxSlice lines x all vertex orders, fewest multiply-adds wins
  // (ties: fewer sliced lines, then the first order in lexicographic enumeration -- deterministic)
  long long best = -1;
  unsigned best_mask = 0;
  int best_order[kTrMaxVertex] = {0}, best_open = 0;
  for (int ns = 0; ns <= kTrMaxSlice; ++ns)
    for (unsigned mask = 0; mask < (1u << L); ++mask) {
      if (popcount(mask) != ns) continue;
      int order[kTrMaxVertex];
      for (int v = 0; v < n; ++v) order[v] = v;
      do {
        int mo = 0;
        const long long c = simulate(n, topo, order, mask, &mo);
        if (c < 0) continue;
        const long long total = c << (2 * ns);
        if (best < 0 || total < best) {
          best = total; best_mask = mask; best_open = mo;
          for (int v = 0; v < n; ++v) best_order[v] = order[v];
        }
      } while (std::next_permutation(order, order + n));
    }
  if (best < 0) return 1;
  plan.cmacs = best;
  plan.max_open = best_open;
  plan.n_sliced = 0;
  for (int l = 0; l < L; ++l) if (best_mask >> l & 1) plan.sliced[plan.n_sliced++] = l;
  plan.n_slice_iter = 1 << (2 * plan.n_sliced);
  for (int v = 0; v < n; ++v) plan.order[v] = best_order[v];

  plan.charge = charge ? 1 : 0;
  plan.dmma_products = 0;
  // isospin-major enumeration of a pair of line labels (16 x 16 x 16 steps): digit j of enumeration e
  static const int iso_t[4][2] = {{0, 1}, {1, 0}, {0, 0}, {1, 1}};
  auto big_digit = [](int e, int j) { return 2 * (((e & 3) >> j) & 1) + iso_t[(e >> 2) & 3][j]; };   // e < 16 is meaningful

  // tables of every step
  int open[kTrMaxLines], open_sigma[kTrMaxLines], n_open = 0;
  for (int k = 0; k < n; ++k) {
    const int v = plan.order[k];
    TraceStep& s = plan.steps[k];
    s.vertex = v;
    int kept_pos[kTrMaxOpen], n_kept = 0;            // positions (in the old open list) of the lines that stay open
    // closed lines: position in the old list (-1: a line that leaves and enters this vertex, it has no index in R),
    // slot of this vertex (and the second slot of such a self-loop, else -1)
    int closed_pos[4], closed_slot[4], closed_slot2[4], n_closed = 0;
    int opened_slot[4], opened_line[4], n_opened = 0;
    for (int j = 0; j < n_open; ++j) {
      int slot = -1;
      for (int q = 0; q < 4; ++q) if (topo[4 * v + q] == open[j]) slot = q;
      if (slot < 0) kept_pos[n_kept++] = j;
      else { closed_pos[n_closed] = j; closed_slot[n_closed] = slot; closed_slot2[n_closed++] = -1; }
    }
    for (int q = 0; q < 4; ++q) {
      const int l = topo[4 * v + q];
      if (best_mask >> l & 1) continue;
      int twin = -1;
      for (int r = 0; r < 4; ++r) if (r != q && topo[4 * v + r] == l) twin = r;
      if (twin >= 0) {
        if (q < twin) { closed_pos[n_closed] = -1; closed_slot[n_closed] = q; closed_slot2[n_closed++] = twin; }
        continue;
      }
      bool was_open = false;
      for (int j = 0; j < n_open; ++j) was_open |= open[j] == l;
      if (!was_open) { opened_slot[n_opened] = q; opened_line[n_opened++] = l; }
    }
    s.nA = 1 << (2 * n_kept);
    s.nB = 1 << (2 * n_opened);
    s.nC = 1 << (2 * n_closed);
    const bool big = n_kept == 2 && n_opened == 2 && n_closed == 2 && closed_slot2[0] < 0 && closed_slot2[1] < 0;
    s.big = big ? 1 : 0;
    auto digit = [&](int e, int j) { return big ? big_digit(e, j) : (e >> (2 * j)) & 3; };
    for (int a = 0; a < kTrTab; ++a) {
      int off = 0;
      for (int j = 0; j < n_kept; ++j) off += digit(a, j) << (2 * kept_pos[j]);
      s.baseR[a] = (uint16_t)(a < s.nA ? tr_pad(off) : 0);
    }
    for (int g = 0; g < kTrTab; ++g) {
      int offr = 0, offw = 0;
      for (int j = 0; j < n_closed; ++j) {
        const int x = digit(g, j);
        if (closed_pos[j] >= 0) offr += x << (2 * closed_pos[j]);
        offw += slot_off(closed_slot[j], x);
        if (closed_slot2[j] >= 0) offw += slot_off(closed_slot2[j], x);
      }
      s.offR[g] = (uint16_t)(g < s.nC ? tr_pad(offr) : 0);
      s.offW[g] = (uint16_t)(g < s.nC ? offw : 0);
    }
    for (int b = 0; b < kTrTab; ++b) {
      int off = 0;
      for (int j = 0; j < n_opened; ++j) off += slot_off(opened_slot[j], digit(b, j));
      s.baseW[b] = (uint16_t)(b < s.nB ? off : 0);
    }
    for (int e = 0; e < 16; ++e) {
      const int canon = big ? big_digit(e, 0) + 4 * big_digit(e, 1) : e;
      s.outA[e] = (uint16_t)tr_pad(canon);
      s.outB[e] = (uint16_t)tr_pad(16 * canon);
    }
    for (int ks = 0; ks < 4; ++ks) s.tile_mask[ks] = 0xF;
    s.block_diag = 0;
    s.ks_valid = 0xF;
    if (big && charge && plan.n_sliced == 0) {
      // signed charges: R side sigma (orientation of the open line), vertex side tau (+1 outgoing slot, -1 incoming)
      const int sk[2] = {open_sigma[kept_pos[0]], open_sigma[kept_pos[1]]};
      const int sc[2] = {open_sigma[closed_pos[0]], open_sigma[closed_pos[1]]};
      const int tc[2] = {closed_slot[0] < 2 ? 1 : -1, closed_slot[1] < 2 ? 1 : -1};
      const int to[2] = {opened_slot[0] < 2 ? 1 : -1, opened_slot[1] < 2 ? 1 : -1};
      uint8_t masks[4];
      bool diag = true;
      for (int ks = 0; ks < 4; ++ks) {
        const int qRg = sc[0] * iso_t[ks][0] + sc[1] * iso_t[ks][1], qWg = tc[0] * iso_t[ks][0] + tc[1] * iso_t[ks][1];
        int mset = 0, nset = 0;
        for (int i = 0; i < 4; ++i) {
          if (sk[0] * iso_t[i][0] + sk[1] * iso_t[i][1] + qRg == 0) mset |= 1 << (i >> 1);
          if (to[0] * iso_t[i][0] + to[1] * iso_t[i][1] + qWg == 0) nset |= 1 << (i >> 1);
        }
        int mask = 0;
        for (int mt = 0; mt < 2; ++mt)
          for (int nt = 0; nt < 2; ++nt)
            if ((mset >> mt & 1) && (nset >> nt & 1)) mask |= 1 << (2 * mt + nt);
        masks[ks] = (uint8_t)mask;
        // the isospin pairs {(0,1),(1,0)} and {(0,0),(1,1)} are mapped onto themselves by charge matching
        diag = diag && (mask == 0 || mask == (ks < 2 ? 1 : 8));
      }
      if (diag) {
        s.block_diag = 1;
        s.ks_valid = 0;
        for (int ks = 0; ks < 4; ++ks) { s.tile_mask[ks] = masks[ks]; if (masks[ks]) s.ks_valid |= (uint8_t)(1 << ks); }
      }
    }
    if (big)
      for (int ks = 0; ks < 4; ++ks) plan.dmma_products += 4LL * popcount(s.tile_mask[ks]) * plan.n_slice_iter;
    for (int it = 0; it < 64; ++it) {
      int off = 0;
      for (int i = 0; i < plan.n_sliced; ++i)
        for (int q = 0; q < 4; ++q)
          if (topo[4 * v + q] == plan.sliced[i]) off += slot_off(q, (it >> (2 * i)) & 3);
      s.sliceW[it] = (uint16_t)(it < plan.n_slice_iter ? off : 0);
    }
    // new frontier: kept lines in their old order, then the opened lines in slot order: R'[a + nA b]
    int next[kTrMaxLines], m = 0;
    int next_sigma[kTrMaxLines];
    for (int j = 0; j < n_kept; ++j) { next_sigma[m] = open_sigma[kept_pos[j]]; next[m++] = open[kept_pos[j]]; }
    for (int j = 0; j < n_opened; ++j) { next_sigma[m] = opened_slot[j] < 2 ? 1 : -1; next[m++] = opened_line[j]; }
    n_open = m;
    for (int j = 0; j < m; ++j) { open[j] = next[j]; open_sigma[j] = next_sigma[j]; }
  }
  if (n_open != 0) return 1;

  // fusions around the 16 x 16 x 16 steps (what ladders and rings consist of)
  for (int k = 0; k < n; ++k) { plan.steps[k].skip = 0; plan.steps[k].r_vertex = -1; plan.steps[k].fuse_last = 0; }
  auto is_big = [&](int k) { return plan.steps[k].big == 1; };
  // (1) first vertex: step 0 would copy its 256 entries into R (R[pad(b)] = W_0[baseW_0[b]], b = canonical index of
  //     the four opened lines).  Offsets are additive over disjoint digits, so step 1 can address the vertex itself.
  if (n >= 3 && plan.steps[0].nA == 1 && plan.steps[0].nC == 1 && plan.steps[0].nB == 256 && is_big(1)) {
    TraceStep& s0 = plan.steps[0];
    TraceStep& s1 = plan.steps[1];
    auto unpad = [](int p) { return p - p / kTrRow; };      // padded offset -> canonical index
    for (int a = 0; a < 16; ++a) s1.baseR[a] = s0.baseW[unpad(s1.baseR[a])];
    for (int g = 0; g < 16; ++g) s1.offR[g] = s0.baseW[unpad(s1.offR[g])];
    s1.r_vertex = s0.vertex;
    s0.skip = 1;
  }
  // (2) last vertex: it closes all four open lines, T = sum_o R'[o] W_last[offW_last[g(o)]] with g(o) the closed-label
  //     combination whose R offset is o: folded into the step that produces R'.
  if (n >= 3 && plan.steps[n - 1].nA == 1 && plan.steps[n - 1].nB == 1 && plan.steps[n - 1].nC == 256 && is_big(n - 2)) {
    TraceStep& sl = plan.steps[n - 1];
    TraceStep& sp = plan.steps[n - 2];
    uint16_t by_offset[kTrMat] = {0};                          // padded offset in R' -> offset in the last vertex
    for (int g = 0; g < 256; ++g) by_offset[sl.offR[g]] = sl.offW[g];
    for (int a = 0; a < 16; ++a)
      for (int b = 0; b < 16; ++b) sp.lastW[a + 16 * b] = by_offset[sp.outA[a] + sp.outB[b]];
    sp.fuse_last = 1;
    sl.skip = 1;
  }
  return 0;
}

}  // namespace no3n
