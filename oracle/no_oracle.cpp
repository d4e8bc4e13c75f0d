// oracle/no_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU oracle for the normal ordering of the chiral N2LO
// three-nucleon force over the Fermi sea (arxiv/paper_2603_24532, Eq. (10) second term,
// PAPER.md:87-92).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call it.  It shares no code, header, table or constant with
// the CUDA path under paper_2603_24532_b200/csrc/.
//
// What it computes:
//
//   M[a',a] = sum_{tau3 in {p,n}, kF_tau3>0} sum_{i,j,l} W_ijl F(k3_ijl)
//             sum_{s3} < a' ; s3 tau3 | sum_{pi in S3} sgn(pi) Pi_pi V(q^pi) | a ; s3 tau3 >
//
//   hole sum        : Eq. (6)-(7), PAPER.md:64-72   -> int d^3k3/(2 pi)^3 theta(kF_tau - k3)
//   A_123           : Eq. (10) and text, PAPER.md:89-92 (unnormalised 6-term signed sum, R4)
//   operator        : "4^A x 4^A matrices in the spin-isospin space ... based on their
//                     operatorial definition", PAPER.md:161 (the N2LO 3N operator itself is
//                     not printed in the paper; reading R1 of DESIGN.md)
//   regulator       : Eq. (13), permutation invariant, reading R5
//   quadrature      : product rule, Gauss-Legendre radial x angular, reading R11
//
// Two levels.  Level 0 is the definition written out: the full 64x64 matrix of
// A_123 V at every k3 node, then the partial trace.  Level 1 uses only
// Pi_pi = Pi_pi^spin (x) Pi_pi^iso and Tr_3[S (x) T] = Tr_s3[S] (x) <tau3|T|tau3>, i.e. it traces
// the 8x8 spin factor and the 8x8 isospin factor separately (still explicit Pauli-Kronecker
// products).  Nothing is hoisted, blocked, or reordered beyond that.
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 cE closed form, P2 cE energy closed form,
// P3 PNM vanishing of cD/cE/c4, P4 Hermiticity, P5 antisymmetry, P6 sparsity, P7 kF->0 limit,
// P8 Hartree-Fock identity against a brute-force 9-D sum, P9 isospin symmetry, P10 linearity,
// P11 level 0 == level 1, P12 cross-implementation values, plus
// Gauss-Legendre exactness and operator permutation symmetry.  No function here is "parity unpinned".
//
// Arithmetic: every real is `long double` (x86 80-bit) in the `_ld` entry points, so that the
// oracle is more accurate than the FP64 CUDA path it judges (reading R19); the `_f64` entry
// points instantiate the same templates in double.

#include <cmath>
#include <complex>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const long double HBARC_LD = 197.3269804L;  // MeV fm (reading R9)
const long double PI_LD = 3.14159265358979323846264338327950288L;

struct Params {   // mirrors the argument list of north_star / include/no.h, plain doubles
  double kf_n, kf_p;
  double c1, c3, c4;      // GeV^-1
  double cD, cE;
  double gA, fpi, mpi;    // -, MeV, MeV
  double lambda_chi;      // MeV (<=0 -> 700, R3)
  double Lambda;          // MeV (<=0 -> unregulated)
  int n_reg;
  int n_r, n_cos, n_phi;
};

template <class T> using cx = std::complex<T>;

// ---------------------------------------------------------------------------------------
// Gauss-Legendre nodes and weights on [a,b]: Newton iteration on P_n (reading R11).
// ---------------------------------------------------------------------------------------
template <class T>
void gauss_legendre(int n, T a, T b, std::vector<T>& x, std::vector<T>& w) {
  x.assign(n, 0);
  w.assign(n, 0);
  for (int i = 0; i < (n + 1) / 2; ++i) {
    long double z = cosl(PI_LD * (i + 0.75L) / (n + 0.5L));
    long double pp = 0;
    for (int it = 0; it < 100; ++it) {
      long double p1 = 1, p2 = 0;
      for (int j = 1; j <= n; ++j) {
        long double p3 = p2;
        p2 = p1;
        p1 = ((2 * j - 1) * z * p2 - (j - 1) * p3) / j;
      }
      pp = n * (z * p1 - p2) / (z * z - 1);
      long double dz = p1 / pp;
      z -= dz;
      if (fabsl(dz) < 1e-19L) break;
    }
    // one more evaluation of the derivative at the converged root
    {
      long double p1 = 1, p2 = 0;
      for (int j = 1; j <= n; ++j) {
        long double p3 = p2;
        p2 = p1;
        p1 = ((2 * j - 1) * z * p2 - (j - 1) * p3) / j;
      }
      pp = n * (z * p1 - p2) / (z * z - 1);
    }
    if (2 * i + 1 == n) z = 0;   // middle node of an odd rule: exactly the midpoint
    long double wt = 2 / ((1 - z * z) * pp * pp);
    long double half = (long double)(b - a) / 2, mid = (long double)(b + a) / 2;
    x[i] = (T)(mid - half * z);
    x[n - 1 - i] = (T)(mid + half * z);
    w[i] = (T)(half * wt);
    w[n - 1 - i] = (T)(half * wt);
  }
}

// ---------------------------------------------------------------------------------------
// Pauli matrices and Kronecker products.  One-particle index: 0 = up / proton (eigenvalue +1),
// 1 = down / neutron (eigenvalue -1)  (reading R10).  Three-particle index = 4 i1 + 2 i2 + i3.
// ---------------------------------------------------------------------------------------
template <class T> struct M2 { cx<T> a[2][2]; };
template <class T> struct M8 { cx<T> a[8][8]; };

template <class T> M2<T> pauli(int k) {  // k = 0: identity, 1: x, 2: y, 3: z
  M2<T> m;
  for (auto& r : m.a) for (auto& e : r) e = 0;
  if (k == 0) { m.a[0][0] = 1; m.a[1][1] = 1; }
  if (k == 1) { m.a[0][1] = 1; m.a[1][0] = 1; }
  if (k == 2) { m.a[0][1] = cx<T>(0, -1); m.a[1][0] = cx<T>(0, 1); }
  if (k == 3) { m.a[0][0] = 1; m.a[1][1] = -1; }
  return m;
}

template <class T> M2<T> pauli_dot(const T v[3]) {  // sigma . v
  M2<T> m;
  m.a[0][0] = v[2];
  m.a[1][1] = -v[2];
  m.a[0][1] = cx<T>(v[0], -v[1]);
  m.a[1][0] = cx<T>(v[0], v[1]);
  return m;
}

template <class T> M8<T> kron3(const M2<T>& A, const M2<T>& B, const M2<T>& C) {
  M8<T> r;
  for (int i1 = 0; i1 < 2; ++i1) for (int i2 = 0; i2 < 2; ++i2) for (int i3 = 0; i3 < 2; ++i3)
    for (int j1 = 0; j1 < 2; ++j1) for (int j2 = 0; j2 < 2; ++j2) for (int j3 = 0; j3 < 2; ++j3)
      r.a[4 * i1 + 2 * i2 + i3][4 * j1 + 2 * j2 + j3] = A.a[i1][j1] * B.a[i2][j2] * C.a[i3][j3];
  return r;
}

// one-body operator `m` acting on particle `slot` (0,1,2), identity elsewhere
template <class T> M8<T> one_body(int slot, const M2<T>& m) {
  M2<T> id = pauli<T>(0);
  return kron3<T>(slot == 0 ? m : id, slot == 1 ? m : id, slot == 2 ? m : id);
}

template <class T> M8<T> mul(const M8<T>& A, const M8<T>& B) {
  M8<T> r;
  for (int i = 0; i < 8; ++i) for (int j = 0; j < 8; ++j) {
    cx<T> s = 0;
    for (int k = 0; k < 8; ++k) s += A.a[i][k] * B.a[k][j];
    r.a[i][j] = s;
  }
  return r;
}

template <class T> void axpy(M8<T>& Y, cx<T> c, const M8<T>& X) {
  for (int i = 0; i < 8; ++i) for (int j = 0; j < 8; ++j) Y.a[i][j] += c * X.a[i][j];
}

template <class T> M8<T> zero8() {
  M8<T> r;
  for (auto& row : r.a) for (auto& e : row) e = 0;
  return r;
}

template <class T> T dot3(const T a[3], const T b[3]) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }
template <class T> void cross3(const T a[3], const T b[3], T c[3]) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}

// ---------------------------------------------------------------------------------------
// Couplings in fm units (reading R9): MeV -> fm^-1 by /hbarc, GeV^-1 -> fm by *1e-3*hbarc.
// ---------------------------------------------------------------------------------------
template <class T> struct Coup {
  T mpi, fpi, gA, c1, c3, c4, cD, cE, Lchi, Lambda;
  int n_reg;
  bool regulated;
};

template <class T> Coup<T> couplings(const Params& p) {
  Coup<T> c;
  T hc = (T)HBARC_LD;
  c.mpi = (T)p.mpi / hc;
  c.fpi = (T)p.fpi / hc;
  c.gA = (T)p.gA;
  c.c1 = (T)p.c1 * (T)1e-3L * hc;
  c.c3 = (T)p.c3 * (T)1e-3L * hc;
  c.c4 = (T)p.c4 * (T)1e-3L * hc;
  c.cD = (T)p.cD;
  c.cE = (T)p.cE;
  c.Lchi = (T)(p.lambda_chi > 0 ? p.lambda_chi : 700.0) / hc;
  c.regulated = p.Lambda > 0;
  c.Lambda = c.regulated ? (T)p.Lambda / hc : (T)1;
  c.n_reg = p.n_reg;
  return c;
}

// ---------------------------------------------------------------------------------------
// The N2LO 3N operator (reading R1), written as a sum over isospin structures
//   V = sum_{ordered (i,j,k)} [ S^{2pi}_{ij} + S^{D}_{ij} ] (x) (t_i.t_j)
//     + sum_{ordered (i,j,k)} S^{4}_{ijk} (x) (t_i x t_j).t_k
//     + cE/(2 fpi^4 Lchi) sum_{ordered (j,k)} 1 (x) (t_j.t_k)
// with, for q = (q_1,q_2,q_3) the momentum transfers of the three particles,
//   S^{2pi}_{ij} = 1/2 (gA/2fpi)^2 (s_i.q_i)(s_j.q_j)/((q_i^2+mpi^2)(q_j^2+mpi^2))
//                  * ( -4 c1 mpi^2/fpi^2 + 2 c3/fpi^2 q_i.q_j )
//   S^{4}_{ijk}  = 1/2 (gA/2fpi)^2 c4/fpi^2 (s_i.q_i)(s_j.q_j)/((q_i^2+mpi^2)(q_j^2+mpi^2)) s_k.(q_i x q_j)
//   S^{D}_{ij}   = -gA/(8 fpi^2) cD/(fpi^2 Lchi) (s_j.q_j)(s_i.q_j)/(q_j^2+mpi^2)
// A "term" is (8x8 spin matrix, isospin kind, particles).  Both levels consume this list.
// ---------------------------------------------------------------------------------------
enum IsoKind { ISO_DOT = 0, ISO_TRIPLE = 1 };

template <class T> struct Term {
  M8<T> spin;
  int kind;   // ISO_DOT: t_i . t_j ; ISO_TRIPLE: (t_i x t_j) . t_k
  int i, j, k;
};

// Y += A(slot i) (x) B(slot j) (x) C(slot k): Kronecker product with the factors placed on the
// named particles (i, j, k a permutation of 0,1,2); zero entries of the 2x2 factors are skipped.
template <class T>
void add_kron_slots(M8<T>& Y, int i, const M2<T>& A, int j, const M2<T>& B, int k, const M2<T>& C) {
  const M2<T>* f[3];
  f[i] = &A; f[j] = &B; f[k] = &C;
  for (int r = 0; r < 8; ++r) for (int c = 0; c < 8; ++c) {
    cx<T> v = f[0]->a[(r >> 2) & 1][(c >> 2) & 1];
    if (v == cx<T>(0)) continue;
    cx<T> v1 = f[1]->a[(r >> 1) & 1][(c >> 1) & 1];
    if (v1 == cx<T>(0)) continue;
    cx<T> v2 = f[2]->a[r & 1][c & 1];
    if (v2 == cx<T>(0)) continue;
    Y.a[r][c] += v * v1 * v2;
  }
}

template <class T> M2<T> scaled(const M2<T>& m, T s) {
  M2<T> r;
  for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) r.a[a][b] = m.a[a][b] * s;
  return r;
}

template <class T>
void build_terms(const Coup<T>& c, const T q[3][3], std::vector<Term<T>>& terms) {
  terms.clear();
  terms.reserve(12);
  const T m2 = c.mpi * c.mpi, f2 = c.fpi * c.fpi;
  const T g2 = (c.gA / (2 * c.fpi)) * (c.gA / (2 * c.fpi));
  const T gD = -c.gA / (8 * f2) * c.cD / (f2 * c.Lchi);
  const T gE = c.cE / (2 * f2 * f2 * c.Lchi);
  T prop[3];
  for (int a = 0; a < 3; ++a) prop[a] = 1 / (dot3(q[a], q[a]) + m2);
  const M2<T> id = pauli<T>(0);
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    if (i == j) continue;
    int k = 3 - i - j;
    M2<T> s_qi = pauli_dot<T>(q[i]);   // sigma . q_i  (placed on particle i or k below)
    M2<T> s_qj = pauli_dot<T>(q[j]);   // sigma . q_j
    terms.emplace_back();
    Term<T>& t = terms.back();
    t.kind = ISO_DOT; t.i = i; t.j = j; t.k = k;
    t.spin = zero8<T>();
    // two-pion exchange c1, c3:  1/2 (gA/2fpi)^2 (s_i.q_i)(s_j.q_j) / (D_i D_j) * f_ij
    T f_ij = -4 * c.c1 * m2 / f2 + 2 * c.c3 / f2 * dot3(q[i], q[j]);
    add_kron_slots<T>(t.spin, i, scaled<T>(s_qi, T(0.5) * g2 * prop[i] * prop[j] * f_ij), j, s_qj, k, id);
    // one-pion-exchange-contact cD:  gD (s_j.q_j)(s_i.q_j) / D_j
    add_kron_slots<T>(t.spin, j, scaled<T>(s_qj, gD * prop[j]), i, s_qj, k, id);
    // contact cE: cE/(2 fpi^4 Lchi), one per ordered pair
    add_kron_slots<T>(t.spin, i, scaled<T>(id, gE), j, id, k, id);
    // two-pion exchange c4:  1/2 (gA/2fpi)^2 c4/fpi^2 (s_i.q_i)(s_j.q_j) s_k.(q_i x q_j) / (D_i D_j)
    if (c.c4 != 0) {
      T n[3];
      cross3(q[i], q[j], n);
      terms.emplace_back();
      Term<T>& u = terms.back();
      u.kind = ISO_TRIPLE; u.i = i; u.j = j; u.k = k;
      u.spin = zero8<T>();
      add_kron_slots<T>(u.spin, i, scaled<T>(s_qi, T(0.5) * g2 * c.c4 / f2 * prop[i] * prop[j]), j, s_qj,
                        k, pauli_dot<T>(n));
    }
  }
}

template <class T> M8<T> iso_matrix(int kind, int i, int j, int k) {
  M8<T> r = zero8<T>();
  if (kind == ISO_DOT) {
    for (int a = 1; a <= 3; ++a)
      axpy<T>(r, cx<T>(1), mul<T>(one_body<T>(i, pauli<T>(a)), one_body<T>(j, pauli<T>(a))));
  } else {
    for (int a = 1; a <= 3; ++a) for (int b = 1; b <= 3; ++b) for (int d = 1; d <= 3; ++d) {
      int eps = (a - b) * (b - d) * (d - a) / 2;  // Levi-Civita for indices 1..3
      if (eps == 0) continue;
      M8<T> m = mul<T>(mul<T>(one_body<T>(i, pauli<T>(a)), one_body<T>(j, pauli<T>(b))),
                       one_body<T>(k, pauli<T>(d)));
      axpy<T>(r, cx<T>((T)eps), m);
    }
  }
  return r;
}

// ---------------------------------------------------------------------------------------
// Permutations of S3.  perm[m] = pi(m): particle m goes to slot pi(m).
//   <b'|Pi_pi|b> = prod_m delta(b'_{pi(m)}, b_m),      q^pi_m = kout_{pi(m)} - kin_m  (R15)
// ---------------------------------------------------------------------------------------
const int PERMS[6][3] = {{0, 1, 2}, {1, 0, 2}, {2, 1, 0}, {0, 2, 1}, {1, 2, 0}, {2, 0, 1}};
const int SIGNS[6] = {+1, -1, -1, -1, +1, +1};

// row index b' (three one-particle labels packed 4 b1' + 2 b2' + b3') -> c with c_m = b'_{pi(m)}
inline int permute_row(int row, const int* pi) {
  int b[3] = {(row >> 2) & 1, (row >> 1) & 1, row & 1};
  return 4 * b[pi[0]] + 2 * b[pi[1]] + b[pi[2]];
}

// regulator exponent argument (R5): (1/6) [ (k1-k2)^2 + (k1-k3)^2 + (k2-k3)^2 ] = p_J^2 + 3 q_J^2 / 4
template <class T> T jacobi_x(const T k[3][3]) {
  T s = 0;
  for (int a = 0; a < 3; ++a) for (int b = a + 1; b < 3; ++b) {
    T d[3] = {k[a][0] - k[b][0], k[a][1] - k[b][1], k[a][2] - k[b][2]};
    s += dot3(d, d);
  }
  return s / 6;
}

template <class T> T ipow(T x, int n) {
  T r = 1;
  for (int i = 0; i < n; ++i) r *= x;
  return r;
}

// F = exp( -(X_in/Lambda^2)^n - (X_out/Lambda^2)^n ): ONE exponential of the summed exponent (R18)
template <class T> T regulator(const Coup<T>& c, const T kin[3][3], const T kout[3][3]) {
  if (!c.regulated) return 1;
  T L2 = c.Lambda * c.Lambda;
  T e = ipow<T>(jacobi_x<T>(kin) / L2, c.n_reg) + ipow<T>(jacobi_x<T>(kout) / L2, c.n_reg);
  return std::exp(-e);
}

// ---------------------------------------------------------------------------------------
// Level 0: the regulated, antisymmetrised 64x64 matrix  F * sum_pi sgn(pi) Pi_pi V(q^pi).
// 64-dim index = 8 * spin_index + iso_index, each 3-particle index = 4 b1 + 2 b2 + b3.
// ---------------------------------------------------------------------------------------
template <class T>
void av3n_level0(const Coup<T>& c, const T kin[3][3], const T kout[3][3], cx<T>* out /*[64*64]*/) {
  for (int e = 0; e < 64 * 64; ++e) out[e] = 0;
  std::vector<Term<T>> terms;
  std::vector<cx<T>> V(64 * 64);
  for (int ip = 0; ip < 6; ++ip) {
    const int* pi = PERMS[ip];
    T q[3][3];
    for (int m = 0; m < 3; ++m) for (int a = 0; a < 3; ++a) q[m][a] = kout[pi[m]][a] - kin[m][a];
    build_terms<T>(c, q, terms);
    for (auto& v : V) v = 0;
    for (const auto& t : terms) {
      M8<T> iso = iso_matrix<T>(t.kind, t.i, t.j, t.k);
      for (int s1 = 0; s1 < 8; ++s1) for (int s0 = 0; s0 < 8; ++s0) {
        cx<T> sv = t.spin.a[s1][s0];
        if (sv == cx<T>(0)) continue;
        for (int t1 = 0; t1 < 8; ++t1) for (int t0 = 0; t0 < 8; ++t0)
          V[(8 * s1 + t1) * 64 + 8 * s0 + t0] += sv * iso.a[t1][t0];
      }
    }
    for (int row = 0; row < 64; ++row) {
      int src = 8 * permute_row(row >> 3, pi) + permute_row(row & 7, pi);
      for (int col = 0; col < 64; ++col) out[row * 64 + col] += cx<T>((T)SIGNS[ip]) * V[src * 64 + col];
    }
  }
  T F = regulator<T>(c, kin, kout);
  for (int e = 0; e < 64 * 64; ++e) out[e] *= F;
}

// momenta of the normal-ordering kinematics (R6, R7): k1 = P/2 + p, k2 = P/2 - p, k3' = k3
template <class T>
void kinematics(const double* cfg, const T k3[3], T kin[3][3], T kout[3][3]) {
  for (int a = 0; a < 3; ++a) {
    T p = (T)cfg[a], pp = (T)cfg[3 + a], P = (T)cfg[6 + a];
    kin[0][a] = P / 2 + p;
    kin[1][a] = P / 2 - p;
    kin[2][a] = k3[a];
    kout[0][a] = P / 2 + pp;
    kout[1][a] = P / 2 - pp;
    kout[2][a] = k3[a];
  }
}

// output index of a two-body state: idx = 8 s1 + 4 s2 + 2 t1 + t2 (R10)
inline int out_index(int s1, int s2, int t1, int t2) { return 8 * s1 + 4 * s2 + 2 * t1 + t2; }

template <class T> struct Grid {
  std::vector<T> r, wr, x, wx, phi, wphi;
};

template <class T> Grid<T> make_grid(const Params& p, T kf) {
  Grid<T> g;
  gauss_legendre<T>(p.n_r, (T)0, kf, g.r, g.wr);
  gauss_legendre<T>(p.n_cos, (T)-1, (T)1, g.x, g.wx);
  gauss_legendre<T>(p.n_phi, (T)0, (T)(2 * PI_LD), g.phi, g.wphi);
  return g;
}

// species loop: tau3 = 0 proton (kf_p), tau3 = 1 neutron (kf_n); an empty sphere is skipped (R12)
inline double species_kf(const Params& p, int tau3) { return tau3 == 0 ? p.kf_p : p.kf_n; }

template <class T>
void normal_order_level0(const Params& p, const double* cfg, long long n_cfg, double* out) {
  Coup<T> c = couplings<T>(p);
  const T norm = 1 / (8 * (T)PI_LD * (T)PI_LD * (T)PI_LD);
#pragma omp parallel for schedule(dynamic, 1)
  for (long long ic = 0; ic < n_cfg; ++ic) {
    std::vector<cx<T>> acc(256, cx<T>(0)), AV(64 * 64);
    for (int tau3 = 0; tau3 < 2; ++tau3) {
      T kf = (T)species_kf(p, tau3);
      if (!(kf > 0)) continue;
      Grid<T> g = make_grid<T>(p, kf);
      for (int i = 0; i < p.n_r; ++i) for (int j = 0; j < p.n_cos; ++j) for (int l = 0; l < p.n_phi; ++l) {
        T st = std::sqrt(1 - g.x[j] * g.x[j]);
        T k3[3] = {g.r[i] * st * std::cos(g.phi[l]), g.r[i] * st * std::sin(g.phi[l]), g.r[i] * g.x[j]};
        T W = g.r[i] * g.r[i] * g.wr[i] * g.wx[j] * g.wphi[l] * norm;
        T kin[3][3], kout[3][3];
        kinematics<T>(cfg + 9 * ic, k3, kin, kout);
        av3n_level0<T>(c, kin, kout, AV.data());
        for (int s1o = 0; s1o < 2; ++s1o) for (int s2o = 0; s2o < 2; ++s2o)
        for (int t1o = 0; t1o < 2; ++t1o) for (int t2o = 0; t2o < 2; ++t2o)
        for (int s1 = 0; s1 < 2; ++s1) for (int s2 = 0; s2 < 2; ++s2)
        for (int t1 = 0; t1 < 2; ++t1) for (int t2 = 0; t2 < 2; ++t2)
        for (int s3 = 0; s3 < 2; ++s3) {
          int row = 8 * (4 * s1o + 2 * s2o + s3) + (4 * t1o + 2 * t2o + tau3);
          int col = 8 * (4 * s1 + 2 * s2 + s3) + (4 * t1 + 2 * t2 + tau3);
          acc[out_index(s1o, s2o, t1o, t2o) * 16 + out_index(s1, s2, t1, t2)] += W * AV[row * 64 + col];
        }
      }
    }
    for (int e = 0; e < 256; ++e) {
      out[(ic * 256 + e) * 2 + 0] = (double)acc[e].real();
      out[(ic * 256 + e) * 2 + 1] = (double)acc[e].imag();
    }
  }
}

// ---------------------------------------------------------------------------------------
// Level 1: same sum, the spin factor and the isospin factor of every term traced separately,
//   Tr_3[ Pi_pi (S (x) T) ] = sum_{s3} <s1' s2' s3| Pi^spin_pi S |s1 s2 s3>          (4x4, depends on k3)
//                         (x) <t1' t2' tau3| Pi^iso_pi T |t1 t2 tau3>                (4x4, constant)
// and, the isospin factor being the same at every node, the node sum is taken on the 4x4 spin
// factor of each (permutation, term) first (linearity of the sum; nothing else is regrouped).
// ---------------------------------------------------------------------------------------
// One k3 node: momentum and full weight r^2 w_r w_ang / (2 pi)^3.
template <class T> struct Node { T k3[3]; T W; };

// Nodes of one Fermi sphere in summation order.  Default: the Gauss-Legendre product grid in
// (r, cos theta, phi) of Params (BASELINE.json).  With a caller-supplied angular rule
// dirs[n_dir][4] = (ux, uy, uz, w), sum w = 4 pi (e.g. a Lebedev rule, the paper's choice:
// "Gauss-Legendre radial x Lebedev angular"), the angular part is that list.
template <class T>
std::vector<Node<T>> sphere_nodes(const Params& p, T kf, const double* dirs, int n_dir) {
  const T norm = 1 / (8 * (T)PI_LD * (T)PI_LD * (T)PI_LD);
  Grid<T> g = make_grid<T>(p, kf);
  std::vector<Node<T>> nodes;
  if (dirs) {
    for (int i = 0; i < p.n_r; ++i) for (int m = 0; m < n_dir; ++m) {
      Node<T> nd;
      for (int a = 0; a < 3; ++a) nd.k3[a] = g.r[i] * (T)dirs[4 * m + a];
      nd.W = g.r[i] * g.r[i] * g.wr[i] * (T)dirs[4 * m + 3] * norm;
      nodes.push_back(nd);
    }
  } else {
    for (int i = 0; i < p.n_r; ++i) for (int j = 0; j < p.n_cos; ++j) for (int l = 0; l < p.n_phi; ++l) {
      T st = std::sqrt(1 - g.x[j] * g.x[j]);
      Node<T> nd;
      nd.k3[0] = g.r[i] * st * std::cos(g.phi[l]);
      nd.k3[1] = g.r[i] * st * std::sin(g.phi[l]);
      nd.k3[2] = g.r[i] * g.x[j];
      nd.W = g.r[i] * g.r[i] * g.wr[i] * g.wx[j] * g.wphi[l] * norm;
      nodes.push_back(nd);
    }
  }
  return nodes;
}

template <class T>
void normal_order_level1(const Params& p, const double* cfg, long long n_cfg, double* out,
                         const double* dirs = nullptr, int n_dir = 0) {
  Coup<T> c = couplings<T>(p);
  // constant isospin matrices of the two kinds for every ordered pair (i,j)
  M8<T> iso_tab[2][3][3];
  for (int kind = 0; kind < 2; ++kind) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j)
    if (i != j) iso_tab[kind][i][j] = iso_matrix<T>(kind, i, j, 3 - i - j);
#pragma omp parallel for schedule(dynamic, 1)
  for (long long ic = 0; ic < n_cfg; ++ic) {
    std::vector<cx<T>> acc(256, cx<T>(0));
    std::vector<Term<T>> terms;
    for (int tau3 = 0; tau3 < 2; ++tau3) {
      T kf = (T)species_kf(p, tau3);
      if (!(kf > 0)) continue;
      const std::vector<Node<T>> nodes = sphere_nodes<T>(p, kf, dirs, n_dir);
      // node sums of the traced spin factors: [permutation][kind][i][j][4][4]
      cx<T> S4[6][2][3][3][4][4];
      for (auto& a : S4) for (auto& b : a) for (auto& d : b) for (auto& e : d) for (auto& f : e) for (auto& v : f) v = 0;
      for (const Node<T>& nd : nodes) {
        const T* k3 = nd.k3;
        const T W = nd.W;
        T kin[3][3], kout[3][3];
        kinematics<T>(cfg + 9 * ic, k3, kin, kout);
        T WF = W * regulator<T>(c, kin, kout);
        for (int ip = 0; ip < 6; ++ip) {
          const int* pi = PERMS[ip];
          T q[3][3];
          for (int m = 0; m < 3; ++m) for (int a = 0; a < 3; ++a) q[m][a] = kout[pi[m]][a] - kin[m][a];
          build_terms<T>(c, q, terms);
          for (const auto& t : terms)
            for (int ro = 0; ro < 4; ++ro) for (int co = 0; co < 4; ++co) {
              cx<T> s = 0;
              for (int s3 = 0; s3 < 2; ++s3) s += t.spin.a[permute_row(2 * ro + s3, pi)][2 * co + s3];
              S4[ip][t.kind][t.i][t.j][ro][co] += WF * s;
            }
        }
      }
      for (int ip = 0; ip < 6; ++ip) for (int kind = 0; kind < 2; ++kind)
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
        if (i == j) continue;
        const int* pi = PERMS[ip];
        const M8<T>& iso = iso_tab[kind][i][j];
        for (int so = 0; so < 4; ++so) for (int to = 0; to < 4; ++to)
        for (int si = 0; si < 4; ++si) for (int ti = 0; ti < 4; ++ti) {
          cx<T> I = iso.a[permute_row(2 * to + tau3, pi)][2 * ti + tau3];
          acc[(4 * so + to) * 16 + 4 * si + ti] += cx<T>((T)SIGNS[ip]) * S4[ip][kind][i][j][so][si] * I;
        }
      }
    }
    for (int e = 0; e < 256; ++e) {
      out[(ic * 256 + e) * 2 + 0] = (double)acc[e].real();
      out[(ic * 256 + e) * 2 + 1] = (double)acc[e].imag();
    }
  }
}

// ---------------------------------------------------------------------------------------
// Brute-force three-body Hartree-Fock energy density (pin P8), an independent loop nest:
//   E/V = (1/6) sum_{123} <123| A_123 V |123>,  sum_i as in Eq. (6), on a product grid per particle.
// ---------------------------------------------------------------------------------------
template <class T> double hf3n_bruteforce(const Params& p) {
  Coup<T> c = couplings<T>(p);
  const T norm = 1 / (8 * (T)PI_LD * (T)PI_LD * (T)PI_LD);
  struct Node { T k[3]; T w; int tau; };
  std::vector<Node> nodes;
  for (int tau = 0; tau < 2; ++tau) {
    T kf = (T)species_kf(p, tau);
    if (!(kf > 0)) continue;
    Grid<T> g = make_grid<T>(p, kf);
    for (int i = 0; i < p.n_r; ++i) for (int j = 0; j < p.n_cos; ++j) for (int l = 0; l < p.n_phi; ++l) {
      T st = std::sqrt(1 - g.x[j] * g.x[j]);
      Node n;
      n.k[0] = g.r[i] * st * std::cos(g.phi[l]);
      n.k[1] = g.r[i] * st * std::sin(g.phi[l]);
      n.k[2] = g.r[i] * g.x[j];
      n.w = g.r[i] * g.r[i] * g.wr[i] * g.wx[j] * g.wphi[l] * norm;
      n.tau = tau;
      nodes.push_back(n);
    }
  }
  const long long N = (long long)nodes.size();
  long double total = 0;
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : total)
  for (long long a = 0; a < N; ++a) {
    std::vector<cx<T>> AV(64 * 64);
    for (long long b = 0; b < N; ++b) for (long long d = 0; d < N; ++d) {
      T k[3][3];
      for (int x = 0; x < 3; ++x) { k[0][x] = nodes[a].k[x]; k[1][x] = nodes[b].k[x]; k[2][x] = nodes[d].k[x]; }
      av3n_level0<T>(c, k, k, AV.data());
      int iso = 4 * nodes[a].tau + 2 * nodes[b].tau + nodes[d].tau;
      cx<T> tr = 0;
      for (int s = 0; s < 8; ++s) tr += AV[(8 * s + iso) * 64 + 8 * s + iso];
      total += (long double)(nodes[a].w * nodes[b].w * nodes[d].w * tr.real());
    }
  }
  return (double)(total / 6);
}

}  // namespace

// ---------------------------------------------------------------------------------------
// C entry points (ctypes).  `params` is the struct above, laid out as 12 doubles + 4 ints.
// ---------------------------------------------------------------------------------------
extern "C" {

void oracle_gauss_legendre(int n, double a, double b, double* x, double* w) {
  std::vector<long double> xs, ws;
  gauss_legendre<long double>(n, (long double)a, (long double)b, xs, ws);
  for (int i = 0; i < n; ++i) { x[i] = (double)xs[i]; w[i] = (double)ws[i]; }
}

// bare operator V(q1,q2,q3) as a 64x64 complex matrix (identity permutation, no regulator)
void oracle_v3n(const Params* p, const double* q /*[3][3]*/, double* out /*[64][64][2]*/) {
  typedef long double T;
  Coup<T> c = couplings<T>(*p);
  T qq[3][3];
  for (int m = 0; m < 3; ++m) for (int a = 0; a < 3; ++a) qq[m][a] = q[3 * m + a];
  std::vector<Term<T>> terms;
  build_terms<T>(c, qq, terms);
  std::vector<cx<T>> V(64 * 64, cx<T>(0));
  for (const auto& t : terms) {
    M8<T> iso = iso_matrix<T>(t.kind, t.i, t.j, t.k);
    for (int s1 = 0; s1 < 8; ++s1) for (int s0 = 0; s0 < 8; ++s0)
      for (int t1 = 0; t1 < 8; ++t1) for (int t0 = 0; t0 < 8; ++t0)
        V[(8 * s1 + t1) * 64 + 8 * s0 + t0] += t.spin.a[s1][s0] * iso.a[t1][t0];
  }
  for (int e = 0; e < 64 * 64; ++e) { out[2 * e] = (double)V[e].real(); out[2 * e + 1] = (double)V[e].imag(); }
}

// regulated antisymmetrised matrix F * A_123 V for explicit momenta kin[3][3], kout[3][3]
void oracle_av3n(const Params* p, const double* kin, const double* kout, double* out /*[64][64][2]*/) {
  typedef long double T;
  Coup<T> c = couplings<T>(*p);
  T ki[3][3], ko[3][3];
  for (int m = 0; m < 3; ++m) for (int a = 0; a < 3; ++a) { ki[m][a] = kin[3 * m + a]; ko[m][a] = kout[3 * m + a]; }
  std::vector<cx<T>> AV(64 * 64);
  av3n_level0<T>(c, ki, ko, AV.data());
  for (int e = 0; e < 64 * 64; ++e) { out[2 * e] = (double)AV[e].real(); out[2 * e + 1] = (double)AV[e].imag(); }
}

void oracle_no_level0_ld(const Params* p, const double* cfg, long long n, double* out) {
  normal_order_level0<long double>(*p, cfg, n, out);
}
void oracle_no_level1_ld(const Params* p, const double* cfg, long long n, double* out) {
  normal_order_level1<long double>(*p, cfg, n, out);
}
void oracle_no_level1_f64(const Params* p, const double* cfg, long long n, double* out) {
  normal_order_level1<double>(*p, cfg, n, out);
}
// level 1 with a caller-supplied angular rule dirs[n_dir][4] = (ux, uy, uz, w) instead of the cos x phi grid
void oracle_no_level1_dirs_ld(const Params* p, const double* cfg, long long n, const double* dirs, int n_dir,
                              double* out) {
  normal_order_level1<long double>(*p, cfg, n, out, dirs, n_dir);
}
// the same template in double (timed as the CPU baseline by bench.py; the parity reference is the _ld one)
void oracle_no_level1_dirs_f64(const Params* p, const double* cfg, long long n, const double* dirs, int n_dir,
                               double* out) {
  normal_order_level1<double>(*p, cfg, n, out, dirs, n_dir);
}
double oracle_hf3n_bruteforce(const Params* p) { return hf3n_bruteforce<long double>(*p); }

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
