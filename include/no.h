/* no.h -- C ABI of the B200 (sm_100a) 3N normal-ordering library  (libno3n.so)
 *
 * Operation (arxiv/paper_2603_24532, /root/reference/PAPER.md):
 *   the second term of Eq. (10) with xi = 1,
 *
 *       M(p,p',P)[a',a] = sum_i < i a' | A_123 V_3N | i a > ,
 *
 *   i.e. the antisymmetrised chiral N2LO three-nucleon interaction with one nucleon summed
 *   over the occupied states of the reference state (hole sum of Eq. (6)-(7), PAPER.md:64-72:
 *   spin, isospin and int d^3k3/(2 pi)^3 theta(kF_tau - k3), separate neutron and proton
 *   Fermi spheres), evaluated "on the fly for given external momenta" by quadrature on the
 *   GPU, many vertices per asynchronous transaction.  The interaction is
 *   the operatorial definition as a 4^A x 4^A spin-isospin matrix with the
 *   permutation-invariant nonlocal regulator of Eq. (13).  The k3 rule
 *   is a Gauss-Legendre product grid radial x cos(theta) x phi in a fixed lab frame.
 *   The operator, the regulator exponent and every other reading of the paper are listed in
 *   DESIGN.md section 3 (R1-R20).
 *
 * Result: for every configuration c = (p, p', P) a complex 16x16 matrix in
 *   spin(1,2) x isospin(1,2) space, units fm^2 (hbar = c = 1; multiply by hbarc for MeV fm^3),
 *   index of a two-body state   idx = 8 s1 + 4 s2 + 2 t1 + t2,
 *   s = 0 spin up / 1 down, t = 0 proton / 1 neutron; row = outgoing (p'), column = incoming (p).
 *   k1 = P/2 + p, k2 = P/2 - p, k1' = P/2 + p', k2' = P/2 - p'.
 *   The caller multiplies by xi = 1/2 or 2/3 and adds the NN part.
 *
 * All functions return 0 (NO_OK) on success or a positive NO_ERR_* code; they never throw
 * and never exit.  There is no CPU fallback: without a CUDA device every call fails.
 */
#ifndef NO_H_
#define NO_H_

#ifdef __cplusplus
extern "C" {
#endif

#define NO_OK          0
#define NO_ERR_INVALID 1   /* bad parameter, null pointer, n_cfg < 0, misaligned pointer: a caller bug */
#define NO_ERR_CUDA    2   /* CUDA runtime or launch failure; text via no_last_cuda_error() */
#define NO_ERR_ALLOC   3   /* host or device allocation failed                              */
#define NO_ERR_BUSY    5   /* a second concurrent call of a non-re-entrant entry point (no_eval_host[_packed],
                              no_hf_energy, no_sp_energy) on ONE handle: returned at once, nothing was
                              launched, the call may simply be retried (or use one handle per thread)  */
#define NO_ERR_LIMIT   4   /* the problem does not fit the fixed capacity of an entry point that never
                              allocates (no_hf_energy_static); nothing was launched            */

typedef struct no_handle no_handle;   /* opaque; owns its device tables (and host-path scratch) */

typedef struct no_params {
  double kf_n, kf_p;        /* Fermi momenta, fm^-1; 0 allowed (empty sphere is skipped); <0 invalid */
  double c1, c3, c4;        /* GeV^-1; c4 = 0 in all BASELINE configs (reading R2)                   */
  double cD, cE;            /* dimensionless                                                         */
  double gA;                /* dimensionless                                                         */
  double fpi, mpi;          /* MeV, both > 0                                                         */
  double lambda_chi;        /* MeV; <= 0 means the default 700 (reading R3)                          */
  double Lambda;            /* MeV, 3N regulator cutoff; <= 0 means unregulated (f_R = 1)            */
  int    n_reg;             /* regulator exponent n >= 1: exp(-((p^2+3q^2/4)/Lambda^2)^n) (R5)       */
  int    n_r, n_cos, n_phi; /* Gauss-Legendre orders of the k3 grid, each 1..128                     */
  int    device;            /* CUDA device ordinal                                                   */
} no_params;

/* Build the handle: validates *p, converts units (hbarc = 197.3269804 MeV fm), computes the
 * Gauss-Legendre nodes and weights on [0,kF_tau], [-1,1], [0,2 pi] on the host (Newton on
 * P_N), uploads the k3 tables of every non-empty Fermi sphere (equal kF_n = kF_p share one
 * grid, full isospin trace of the third nucleon) to device `p->device`.
 * *h is written only on success.  HOST pointers. */
int no_init(no_handle **h, const no_params *p);

/* no_init with a caller-supplied ANGULAR rule instead of the cos(theta) x phi Gauss-Legendre grid:
 * the paper's own quadrature is "Gauss-Legendre radial x Lebedev angular" (16 radial points, order-15
 * Lebedev).  The k3 nodes of a sphere are r_i u_m, weights r_i^2 w_i w_m / (2 pi)^3.
 *   h_dirs : HOST, const, [n_dir][4] doubles = (ux, uy, uz, w): unit vectors in the fixed lab frame
 *            (| |u|^2 - 1 | <= 1e-12, NO_ERR_INVALID otherwise: the kernel relies on |u| = 1) and weights
 *            with sum w = 4 pi (not checked, used as given), all finite
 *   n_dir  : 1..4096 (NO_ERR_INVALID otherwise, or if the tables do not fit in shared memory)
 * p->n_cos and p->n_phi must still be valid orders but are otherwise unused; no_evals_per_cfg is
 * n_r * n_dir * (number of spheres).  h_dirs == NULL (with n_dir == 0) is no_init.  The array is
 * copied; the caller keeps ownership. */
int no_init_angular(no_handle **h, const no_params *p, const double *h_dirs, int n_dir);

/* Enqueue the normal ordering of n_cfg configurations on `cuda_stream` (a cudaStream_t; NULL is
 * the default stream).  No synchronisation inside: the call returns as soon as the work is
 * enqueued ("asynchronous GPU transaction"); one handle may be used from several
 * streams and host threads at once.  A batch that needs more CTAs than one grid holds is cut into several
 * launches on the same stream.
 *   d_cfg : DEVICE, const, [n_cfg][9] doubles = p(xyz), p'(xyz), P(xyz) in fm^-1, dense,
 *           8-byte aligned, caller-owned
 *   d_out : DEVICE, [n_cfg][16][16][2] doubles (re, im), row-major rows = outgoing state,
 *           16-byte aligned, dense, caller-owned; every element is written (structural zeros
 *           are written as 0)
 * n_cfg == 0 succeeds and does nothing.  Non-finite inputs propagate to non-finite outputs. */
int no_eval(const no_handle *h, const double *d_cfg, long long n_cfg, double *d_out, void *cuda_stream);

/* Work layout of the kernel: 0 (default) automatic, 1 one warp per configuration (throughput layout), 2 one CTA of
 * four warps per configuration (small-batch layout: the directions are dealt to the warps, their partial moments
 * added in a fixed order).  Automatic picks 2 when four warps per configuration still leave warp slots of the
 * device empty.  Both layouts compute the same sums in different (fixed) orders: results agree to rounding and
 * are bit-reproducible within a layout; with layout 0 the bits of a configuration therefore depend on the size of
 * the batch it is evaluated in (never on its position in the batch: every entry point decides ONCE per call, from
 * the whole batch).  The setting is atomic: it may be changed while other threads are inside no_eval (a call
 * in flight keeps the layout it read at entry).  Affects later no_eval / no_eval_diag / no_eval_host /
 * no_hf_energy / no_sp_energy calls. */
int no_set_layout(no_handle *h, int layout);

/* Test hook, not a tuning parameter: cap the number of CTAs per kernel launch for this handle (0 restores the
 * hardware limit of 2^31 - 1).  A batch that needs more is cut into several launches on the same stream, with the
 * same bits as a single launch; the hardware limit itself cannot be reached in a test, so the GPU tests lower it
 * to drive that path.  Not atomic: call it before the handle is used from other threads.  The library reads no
 * environment variables. */
int no_set_max_grid(no_handle *h, long long max_ctas);

/* Same operation with HOST buffers (pageable or pinned): copies h_cfg to a device scratch owned
 * by the handle, runs the kernels, copies the result back and SYNCHRONISES `cuda_stream` before
 * returning.  The batch is cut into chunks of a few waves: the device-to-host copy of a finished chunk
 * runs on an internal stream under the kernel of the next one (pinned h_out is needed for the copies to
 * be asynchronous; pageable memory is still correct).  Not re-entrant for one handle (the scratch is
 * shared): while one of no_eval_host / no_hf_energy / no_sp_energy runs on a handle, a second such call on
 * the same handle returns NO_ERR_BUSY (no_eval / no_eval_diag stay re-entrant).  On a CUDA failure both
 * streams are drained before the call returns.  Used for the end-to-end measurement. */
int no_eval_host(no_handle *h, const double *h_cfg, long long n_cfg, double *h_out, void *cuda_stream);

/* ---- Packed, symmetry-reduced output -------------------------------------------
 * "only up to 4^A C(2A,A) matrix elements can be non-zero ... only a subset of the remaining matrix
 * elements needs to be computed from which the entire matrix can be efficiently reconstructed."  For A = 2 that is
 * 96 of the 256 entries (charge conservation, t1' + t2' = t1 + t2); in isospin-symmetric matter the isospin
 * invariance of the effective interaction (it has the form A + B tau_1.tau_2) leaves 32.
 * A packed matrix is indexed [spin element sp][entry][2] (re, im), sp = 4 (2 s1' + s2') + (2 s1 + s2), i.e. the
 * full-matrix element is row = 8 s1' + 4 s2' + (row isospin pair), col = 8 s1 + 4 s2 + (column isospin pair),
 * isospin pair = 2 t1 + t2 (pp = 0, pn = 1, np = 2, nn = 3):
 *   NO_PACK_CHARGE  : 6 entries per spin element, (row pair, column pair) =
 *                     (pp,pp) (pn,pn) (np,np) (nn,nn) (pn,np) (np,pn): 96 complex = 192 doubles = 1536 bytes;
 *                     valid for every handle.
 *   NO_PACK_ISOSPIN : 2 entries per spin element, (pn,pn) and (pn,np): 32 complex = 64 doubles = 512 bytes;
 *                     only for handles with kF_n == kF_p > 0 (NO_ERR_INVALID otherwise).  Reconstruction:
 *                     (np,np) = (pn,pn), (np,pn) = (pn,np), (pp,pp) = (nn,nn) = (pn,pn) + (pn,np).
 * The packed kernels compute and store only the subset (the 160 structural zeros are neither computed nor written;
 * in isospin-symmetric matter 64 more entries are skipped). */
#define NO_PACK_CHARGE  1
#define NO_PACK_ISOSPIN 2
/* Flag for no_eval_packed / no_packed_doubles, ORed into `format`: FORWARD configurations.  The caller promises that
 * p' == p (bit for bit) in EVERY configuration of the call, as in the Hartree-Fock contractions and every diagonal
 * matrix element.  Then k1' = k1 and k2' = k2, half of the propagator legs coincide, and the kernel
 * runs its forward variant: 39 instead of 51 FP64 instructions per k3 node, same output form, results equal to the
 * general kernel's to rounding.  The promise cannot be checked on the device: a configuration with p' != p gets the
 * matrix of (p, p, P), silently.  In the one-CTA-per-configuration layout (small batches) the flag changes nothing. */
#define NO_PACK_FORWARD 0x100

/* Doubles per configuration of a packed format for this handle: 192 or 64; 0 if the format does not apply
 * to the handle (NO_PACK_ISOSPIN without kF_n == kF_p) or is unknown. */
int no_packed_doubles(const no_handle *h, int format);

/* no_eval writing the packed form.  Same arguments, ownership, alignment and asynchrony as no_eval, except
 *   d_packed : DEVICE, [n_cfg][no_packed_doubles(h, format)] doubles, 16-byte aligned, dense, caller-owned.
 * NO_ERR_INVALID if the format does not apply to the handle. */
int no_eval_packed(const no_handle *h, int format, const double *d_cfg, long long n_cfg, double *d_packed,
                   void *cuda_stream);

/* Rebuild the full matrices from a packed form on the device (one kernel, enqueued on `cuda_stream`, no
 * synchronisation; runs on the caller's current device, which must own both pointers):
 *   d_packed : DEVICE, const, [n_cfg][192 or 64] doubles as written by no_eval_packed, 16-byte aligned
 *   d_out    : DEVICE, [n_cfg][16][16][2] doubles as no_eval writes them, 16-byte aligned; every element is written.
 * With NO_PACK_CHARGE the result equals no_eval's bit for bit; with NO_PACK_ISOSPIN the pp and nn blocks are the
 * sum of the two stored entries (equal to no_eval's to rounding). */
int no_unpack(int format, const double *d_packed, long long n_cfg, double *d_out, void *cuda_stream);

/* no_eval_host shipping the packed form over PCIe: HOST buffers, h_packed [n_cfg][192 or 64] doubles; otherwise
 * as no_eval_host (chunked, copies overlapped, synchronises, not re-entrant for one handle).  The device-to-host
 * traffic per configuration drops from 4096 to 1536 or 512 bytes. */
int no_eval_host_packed(no_handle *h, int format, const double *h_cfg, long long n_cfg, double *h_packed,
                        void *cuda_stream);

/* Spin-traced diagonal of the normal-ordered matrix, reduced inside the kernel (the 16x16 matrix is
 * never written): the integrand of the Hartree-Fock contractions Eq. (1) and Eq. (9),
 * obtained "by repeatedly normal ordering".  Same arguments as no_eval except
 *   d_out : DEVICE, [n_cfg][4] doubles, d_out[c][2 t1 + t2] = sum_{s1,s2} Re M_c[a, a],
 *           a = (s1, s2, t1, t2), t = 0 proton / 1 neutron; 8-byte aligned, dense, caller-owned.
 * The configurations are arbitrary (for p' = p the diagonal is real by Hermiticity). */
int no_eval_diag(const no_handle *h, const double *d_cfg, long long n_cfg, double *d_out, void *cuda_stream);

/* 3N Hartree-Fock energy per volume (fm^-4; multiply by hbar c for MeV fm^-3),
 *   E/V = (1/6) sum_{123} n_1 n_2 n_3 <123| A_123 V_3N |123>        (xi-weights of Eq. (10))
 * by a second Fermi-sea quadrature over no_eval_diag: particles 1 and 2 run over Gauss-Legendre product
 * grids (n_r x n_cos x n_phi per Fermi sphere of the handle, fixed lab frame), particle 3 over the
 * handle's own k3 grid; configuration (p, p', P) = ((k1-k2)/2, (k1-k2)/2, k1+k2).  On the same grids this
 * equals the brute-force 9-dimensional sum exactly (pin P8).  Generates the pair configurations on the
 * device in chunks, enqueues on `cuda_stream`, SYNCHRONISES it, and writes the result to the HOST
 * double *e_over_v.  With kF_n = kF_p the four (t1, t2) pair grids coincide and are integrated once.
 * Uses a grow-only device scratch owned by the handle (not re-entrant for one handle, see no_eval_host). */
int no_hf_energy(no_handle *h, int n_r, int n_cos, int n_phi, double *e_over_v, void *cuda_stream);

/* no_hf_energy for callers that are not allowed to allocate GPU memory.
 *
 * Who that is.  The paper drives one GPU from many Monte-Carlo worker threads and MPI ranks at once
 * (PAPER.md:182-186).  cudaMalloc and cudaFree are device-wide operations: they take the driver's
 * allocation lock and wait for work in flight, so one worker that allocates stalls the transactions of all
 * the others, and it does so at a moment nobody chose (no_hf_energy grows its arena whenever a call needs
 * more than the last one did).  Other callers have no memory left to ask for: a host application that hands
 * all of HBM to its own pool at start-up (a framework's caching allocator, a fixed-budget service) makes
 * every later cudaMalloc fail with out-of-memory although the pool has room.  And some code simply runs
 * under a rule of "no allocation after initialisation" so that it cannot fail or fragment hours into a run.
 *
 * What it does.  Same arguments, same result (to rounding: the pair configurations go through the kernels
 * in passes of 65536 instead of 2^20, so the fixed summation order differs), same synchronisation of
 * `cuda_stream`, same HOST result pointer as no_hf_energy.  The only difference is where the intermediates
 * live: not in a handle-owned cudaMalloc arena but in ONE array of NO_HF_STATIC_BYTES (7.25 MiB) that is
 * compiled into libno3n.so as a `static __device__` variable.  Every GPU on which this process loads the
 * library carries that array from module load until the process exits, used or not; that is the price.
 * The call itself performs no cudaMalloc / cudaFree / cudaMallocAsync / cudaHostAlloc, creates no stream or
 * event and calls no library that could; the handle `h` (whose tables no_init did allocate) must exist already.
 * On the host it uses a little ordinary heap (the quadrature nodes, 32 bytes per node).
 *
 * Limit.  n_r * n_cos * n_phi <= NO_HF_STATIC_MAX_NODES (4096, e.g. 16 x 16 x 16); above that the call
 * returns NO_ERR_LIMIT before touching the GPU (use no_hf_energy).  The k3 grid of the handle is not limited.
 *
 * First call.  The first call on a device looks up where that device keeps the array
 * (cudaGetSymbolAddress with that device current) and remembers it; make this first call during
 * start-up, outside any stream capture.  Later calls only enqueue copies, a memset and kernels.
 *
 * Sharing.  There is one array per device, not per handle or per call, and it is not cleared between
 * calls: it holds the previous call's leftovers.  The function zeroes the one accumulator it adds into and
 * writes everything else before reading it, so a call never sees stale data.  Two calls working in the
 * array at the same time on one device would corrupt each other; the function therefore takes a per-device
 * lock for its whole duration (it returns only after its stream has drained), so threads of one process may
 * call it freely and are served one after the other, whatever handles and streams they use.  Do not defeat
 * this by other means.  Other processes have their own copy of the array. */
#define NO_HF_STATIC_MAX_NODES 4096
#define NO_HF_STATIC_BYTES     7602432
int no_hf_energy_static(no_handle *h, int n_r, int n_cos, int n_phi, double *e_over_v, void *cuda_stream);

/* 3N part of the Hartree-Fock single-particle energy (self-energy) of Eq. (9), isospin
 * dependent and spin averaged (unpolarised matter):
 *   Sigma_t1(k1) = sum_j <1j| Vbar_eff^(xi=1/2) |1j>|_3N = (1/4) sum_{t2} sum_{k2 in S(t2)} W2 D[2 t1 + t2],
 * D = no_eval_diag at (p, p', P) = ((k1-k2)/2, (k1-k2)/2, k1+k2); particle 2 on an n_r x n_cos x n_phi
 * Gauss-Legendre grid per Fermi sphere of the handle, particle 3 on the handle's own k3 grid.  Summed over
 * the Fermi sea of particle 1 it gives the energy: E/V = (1/3) sum_{t1} sum_{k1} 2 W1 Sigma_t1(k1).
 *   h_k1    : HOST, const, [n_k][3] momenta in fm^-1 (any momenta, inside or outside the Fermi sea)
 *   h_sigma : HOST, [n_k][2] doubles, (proton, neutron), fm^-1 (multiply by hbar c for MeV)
 * Enqueues on `cuda_stream`, SYNCHRONISES it; same handle-owned scratch as no_hf_energy (not re-entrant). */
int no_sp_energy(no_handle *h, const double *h_k1, int n_k, int n_r, int n_cos, int n_phi,
                 double *h_sigma, void *cuda_stream);

/* Release the handle and everything it owns.  NULL is a no-op. */
int no_free(no_handle *h);

/* Static description of a code. */
const char *no_strerror(int code);

/* Text of the last CUDA error seen by the calling thread ("" if none). */
const char *no_last_cuda_error(void);

/* Facts about the kernel no_eval launches for this handle (each pointer may be NULL):
 * registers per thread, dynamic shared memory per CTA in bytes, threads per CTA, resident CTAs
 * per SM (occupancy API), number of SMs, configurations per CTA. */
int no_kernel_info(const no_handle *h, int *regs, int *smem_bytes, int *threads, int *ctas_per_sm,
                   int *n_sm, int *cfg_per_cta);

/* Number of k3-point evaluations one configuration costs with this handle:
 * n_r * n_cos * n_phi * (number of distinct non-zero Fermi momenta). */
long long no_evals_per_cfg(const no_handle *h);

/* FP64 roofline probe: runs a register-resident chain of independent DFMAs on every SM of
 * `device` for about `millis` milliseconds on `cuda_stream`, synchronises, and writes the achieved
 * rate in TFLOP/s (2 flops per DFMA) and the SM count.  Used by bench.py to state the measured
 * FP64 peak next to the nominal one. */
int no_probe_fp64_peak(int device, int millis, double *tflops, int *n_sm, void *cuda_stream);

/* FP64 operand-delivery probe (the rule the hot loop is written around): the same 16
 * independent DFMA chains per thread, once with two fresh register operands per instruction (the other two loop
 * invariant) and once with three distinct 64-bit register operands per instruction; writes both rates in TFLOP/s.
 * On B200 the second runs at about two thirds of the first (3 instead of 2 pipe cycles per instruction). */
int no_probe_fp64_operands(int device, int millis, double *tflops_two_operands, double *tflops_three_operands,
                           void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* NO_H_ */
