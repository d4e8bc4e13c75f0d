/* no_trace.h -- C ABI of the spin-isospin trace kernel of libno3n.so (B200, sm_100a)   [SURVEY.md section 8(f) f4]
 *
 * Operation (arxiv/paper_2603_24532, /root/reference/PAPER.md:155-157 and Appendix B):
 *   "the evaluation of each diagram involves ... summing over isospin and spin degrees of freedom for propagators
 *   ... the integrand function evaluated each vertex at the given momenta for every spin and isospin
 *   configuration, yielding 2^4 x 2^4 = 256 matrix elements per vertex.  A spin-isospin trace is then performed over
 *   the isospin and spin configurations for all propagators in the diagram".  The paper accelerates this
 *   trace on the GPU because its cost grows by a factor 4 per MBPT order at the two-body level (2^20 label
 *   configurations at fifth order, 2^24 at sixth) and cross-checks the optimised trace "against an
 *   unoptimized trace".
 *
 * Definition.  A closed diagram with n vertices has 2 n propagator lines; line j carries a spin s_j (0 up, 1 down)
 * and an isospin t_j (0 proton, 1 neutron).  Vertex v is a complex 16 x 16 matrix V_v in the layout no_eval writes
 * (include/no.h: row = outgoing pair, column = incoming pair, pair index 8 s1 + 4 s2 + 2 t1 + t2) attached to the
 * lines topo[v] = (o1, o2, i1, i2): the lines leaving it in slots 1, 2 and entering it in slots 1, 2.  Then
 *
 *     T = sum_{s_0 .. s_{2n-1}} sum_{t_0 .. t_{2n-1}}  prod_v  V_v[ 8 s_o1 + 4 s_o2 + 2 t_o1 + t_o2 ][ 8 s_i1 + 4 s_i2 + 2 t_i1 + t_i2 ] .
 *
 * Energy denominators, momentum integration, signs and symmetry factors of the diagram are the caller's.
 * The library evaluates T for a batch of samples (one set of vertex matrices per Monte-Carlo sample) by contracting
 * the tensor network vertex by vertex in an order planned on the host; the result equals
 * the label sum up to floating-point summation order.
 *
 * All functions return 0 (NO_OK) or a positive NO_ERR_* code of include/no.h; they never throw and never exit.
 * There is no CPU fallback.
 */
#ifndef NO_TRACE_H_
#define NO_TRACE_H_

#include "no.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct no_trace_plan no_trace_plan;   /* opaque; owns its device tables */

#define NO_TRACE_MAX_VERTEX 6

/* flags of no_trace_init */
#define NO_TRACE_CHARGE_CONSERVING 1   /* the caller promises that every vertex matrix is EXACTLY zero outside the 96
                                          charge-conserving entries, t_o1 + t_o2 = t_i1 + t_i2 (what no_eval
                                          writes).  The plan then skips the blocks that isospin conservation at each vertex
                                          empties ("the subset of isospin configurations consistent with isospin conservation
                                          at each vertex"): a quarter of the tensor-core products of a ladder
                                          or ring remain.  With matrices that break the promise the result is unspecified. */

/* Plan the trace of one topology and upload its tables to device `device`.
 *   n_vertex : 1..NO_TRACE_MAX_VERTEX (the MBPT order at the two-body level)
 *   topo     : HOST, const, [n_vertex][4] ints = line ids (out 1, out 2, in 1, in 2) of every vertex; every id
 *              0 .. 2 n_vertex - 1 must appear exactly once among the outgoing and once among the incoming slots
 *   flags    : 0 (arbitrary complex vertex matrices) or NO_TRACE_CHARGE_CONSERVING
 * NO_ERR_INVALID: unknown flag, malformed topology, or one that cannot be contracted with at most four open lines after fixing
 * the labels of at most three lines in an outer loop (every ladder, ring and fifth-order diagram tested fits;
 * disconnected diagrams are accepted).  *plan is written only on success. */
int no_trace_init(no_trace_plan **plan, int n_vertex, const int *topo, int flags, int device);

/* Enqueue the trace of n_sample samples on `cuda_stream` (a cudaStream_t; NULL is the default stream).  No
 * synchronisation inside; one plan may be used from several streams and host threads at once.
 *   d_vertices : DEVICE, const, [n_sample][n_vertex][16][16][2] doubles (re, im), 16-byte aligned, dense, caller-owned
 *                (the matrices of one sample are contiguous: exactly what no_eval writes for n_vertex configurations)
 *   d_out      : DEVICE, [n_sample][2] doubles (re, im), 16-byte aligned, caller-owned
 * n_sample == 0 succeeds and does nothing.  Non-finite inputs give non-finite outputs.  Results are bit-reproducible. */
int no_trace_eval(const no_trace_plan *plan, const double *d_vertices, long long n_sample, double *d_out,
                  void *cuda_stream);

/* no_trace_eval reading the vertex matrices in a packed form of include/no.h (what no_eval_packed writes):
 *   NO_PACK_CHARGE  : the 96 charge-conserving entries, 1536 bytes per vertex instead of 4096; the kernel scatters
 *                     them into zeroed shared-memory matrices (7.7 instead of 20.5 KB per fifth-order sample cross HBM);
 *                     d_packed is [n_sample][n_vertex][96][2] doubles
 *   NO_PACK_ISOSPIN : isospin-symmetric matter, 32 entries = 512 bytes per vertex; the kernel rebuilds the other
 *                     charge-conserving entries as no_unpack does ((np,np) = (pn,pn), (np,pn) = (pn,np),
 *                     (pp,pp) = (nn,nn) = (pn,pn) + (pn,np)); d_packed is [n_sample][n_vertex][32][2] doubles
 * Any other format: NO_ERR_INVALID.  d_packed: DEVICE, const, 16-byte aligned, dense, caller-owned.
 * Otherwise as no_trace_eval; works with plans made with or without NO_TRACE_CHARGE_CONSERVING (a packed form cannot
 * express a charge-violating entry) and gives the same bits as no_trace_eval on the matrices no_unpack rebuilds. */
int no_trace_eval_packed(const no_trace_plan *plan, int format, const double *d_packed, long long n_sample, double *d_out,
                         void *cuda_stream);

/* Facts about a plan (each pointer may be NULL): complex multiply-adds per sample of the planned contraction,
 * widest frontier (open lines), number of sliced lines, number of charge-conserving isospin assignments of the lines
 * ("the subset of isospin configurations consistent with isospin conservation at each vertex"), the
 * vertex order (n_vertex ints), and the number of 8x8x4 FP64 tensor-core products per sample that the 16x16x16 steps
 * issue (64 per step for arbitrary vertices, 16 with NO_TRACE_CHARGE_CONSERVING). */
int no_trace_info(const no_trace_plan *plan, long long *cmacs_per_sample, int *max_open, int *n_sliced,
                  long long *n_isospin_configs, int *order, long long *tensor_products_per_sample);

/* Text of the last CUDA error seen by the calling thread in a no_trace_* call ("" if none). */
const char *no_trace_last_cuda_error(void);

/* Release the plan.  NULL is a no-op. */
int no_trace_free(no_trace_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* NO_TRACE_H_ */
