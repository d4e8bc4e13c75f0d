/* oracle/trace_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU oracle for the spin-isospin trace of a closed MBPT diagram at
 * the two-body level (arxiv/paper_2603_24532, Sec. III A, and Appendix B,
 * PAPER.md:639-653).  This is the "unoptimized trace" the paper cross-checks its optimised one
 * against: "the integrand function evaluated each vertex at the given momenta for
 * every spin and isospin configuration, yielding 2^4 x 2^4 = 256 matrix elements per vertex.  A
 * spin-isospin trace is then performed over the isospin and spin configurations for all propagators
 * in the diagram".  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.  It shares no code, header, table or constant with the CUDA path.
 *
 * Definition.  A diagram with n vertices has L = 2 n propagator lines; line j carries a spin label
 * s_j in {0 up, 1 down} and an isospin label t_j in {0 proton, 1 neutron}.  Vertex v is the complex
 * 16 x 16 matrix V_v[row][col] of include/no.h (row = outgoing pair, col = incoming pair, pair index
 * 8 s1 + 4 s2 + 2 t1 + t2) and is attached to four lines: topo[v] = (o1, o2, i1, i2), the ids of
 * the lines leaving the vertex in slots 1, 2 and of the lines entering it in slots 1, 2.  Every line
 * leaves exactly one vertex and enters exactly one vertex.  The trace is
 *
 *     T = sum_{s_0..s_{L-1}} sum_{t_0..t_{L-1}}  prod_v  V_v[ idx(o1, o2) ][ idx(i1, i2) ],
 *     idx(a, b) = 8 s_a + 4 s_b + 2 t_a + t_b,
 *
 * i.e. 4^L = 2^(4n) terms (2^20 at fifth order, 2^24 at sixth: PAPER.md:155).  Energy denominators,
 * momentum integrals, signs and symmetry factors of the diagram are not part of the trace.
 *
 * Nothing is hoisted, factorised or skipped: one odometer over all labels, n complex multiplications
 * per term, accumulation in long double.
 *
 * Pins (tests/test_trace_oracle_pins.py): n = 2 ladder = Tr[V_1 V_0] by a library matrix product;
 * n-vertex ladder = Tr[V_{n-1} ... V_0]; product vertices A (x) B factorise into one matrix-chain
 * trace per closed fermion loop; identity vertices give 4^(number of loops); multilinearity in every
 * vertex; invariance under relabelling of lines and of vertices; slot exchange = P12 on the rows or
 * columns; the count of charge-conserving isospin assignments (34 for the fifth-order ladder, at most
 * 36 "across all diagrams at fifth order").
 */
#include <stddef.h>

#define MAX_VERTEX 6

static int pair_index(int xa, int xb) {        /* x = 2 s + t */
  return 8 * (xa >> 1) + 4 * (xb >> 1) + 2 * (xa & 1) + (xb & 1);
}

/* V: [n_sample][n_vertex][16][16][2] (re, im);  out: [n_sample][2].  Returns 0, or 1 if n_vertex is out of range. */
int oracle_trace_bruteforce(int n_vertex, const int *topo, const double *V, long long n_sample, double *out) {
  if (n_vertex < 1 || n_vertex > MAX_VERTEX) return 1;
  const int L = 2 * n_vertex;
  long long n_terms = 1;
  for (int j = 0; j < L; ++j) n_terms *= 4;
  long long s;
#pragma omp parallel for schedule(dynamic, 1)
  for (s = 0; s < n_sample; ++s) {
    const double *Vs = V + (size_t)s * n_vertex * 512;
    long double tr = 0.0L, ti = 0.0L;
    int x[2 * MAX_VERTEX];
    for (long long term = 0; term < n_terms; ++term) {
      long long r = term;
      for (int j = 0; j < L; ++j) { x[j] = (int)(r & 3); r >>= 2; }      /* label of line j: x = 2 s + t */
      long double pr = 1.0L, pi = 0.0L;
      for (int v = 0; v < n_vertex; ++v) {
        const int *t = topo + 4 * v;
        const int row = pair_index(x[t[0]], x[t[1]]), col = pair_index(x[t[2]], x[t[3]]);
        const long double ar = Vs[(size_t)v * 512 + 2 * (16 * row + col)];
        const long double ai = Vs[(size_t)v * 512 + 2 * (16 * row + col) + 1];
        const long double nr = pr * ar - pi * ai, ni = pr * ai + pi * ar;
        pr = nr; pi = ni;
      }
      tr += pr; ti += pi;
    }
    out[2 * s] = (double)tr;
    out[2 * s + 1] = (double)ti;
  }
  return 0;
}

/* Number of isospin assignments t_0..t_{L-1} with t_o1 + t_o2 = t_i1 + t_i2 at every vertex ("the subset of
 * isospin configurations consistent with isospin conservation at each vertex"), by enumeration. */
long long oracle_trace_isospin_configs(int n_vertex, const int *topo) {
  if (n_vertex < 1 || n_vertex > MAX_VERTEX) return -1;
  const int L = 2 * n_vertex;
  long long count = 0;
  for (long long m = 0; m < (1LL << L); ++m) {
    int ok = 1;
    for (int v = 0; v < n_vertex && ok; ++v) {
      const int *t = topo + 4 * v;
      const int qo = (int)((m >> t[0]) & 1) + (int)((m >> t[1]) & 1);
      const int qi = (int)((m >> t[2]) & 1) + (int)((m >> t[3]) & 1);
      ok = qo == qi;
    }
    count += ok;
  }
  return count;
}
