"""Pins of the CPU oracle (oracle/no_oracle.cpp) against what the paper and the mathematics fix.

None of these tests touches the CUDA path.  Each pin names the passage or the DESIGN.md /
SURVEY.md section 8(c) item it comes from.  A plausible mistake in the oracle (a dropped term, a
wrong sign, a transposed index, a wrong permutation convention, a wrong Jacobian or 1/(2 pi)^3)
fails at least one of them.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as O

HBARC = 197.3269804
PHYS = dict(c1=-0.81, c3=-3.2, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0,
            Lambda=500.0, n_reg=4)
RNG = np.random.default_rng(20260324)


def idx(s1, s2, t1, t2):
    return 8 * s1 + 4 * s2 + 2 * t1 + t2


def p12_matrix():
    """Exchange of (s1,t1) <-> (s2,t2) on the 16-dim two-body index."""
    P = np.zeros((16, 16))
    for s1 in range(2):
        for s2 in range(2):
            for t1 in range(2):
                for t2 in range(2):
                    P[idx(s2, s1, t2, t1), idx(s1, s2, t1, t2)] = 1.0
    return P


def rand_cfg(n, scale=1.0):
    return RNG.uniform(-1.0, 1.0, size=(n, 9)) * scale


def only(**kw):
    """Parameter set with every LEC zero except the named ones."""
    d = dict(PHYS)
    for k in ("c1", "c3", "cD", "cE"):
        d[k] = 0.0
    d["c4"] = 0.0
    d.update(kw)
    return d


# ----------------------------------------------------------------------------------------------
# Gauss-Legendre (reading R11): against numpy's library routine, and exactness on monomials.
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [1, 2, 3, 7, 16, 32, 40, 48, 64, 128])
def test_gauss_legendre_matches_library_and_is_exact(n):
    x, w = O.gauss_legendre(n, -1.0, 1.0)
    xr, wr = np.polynomial.legendre.leggauss(n)
    assert np.allclose(x, xr, rtol=0, atol=3e-15)
    assert np.allclose(w, wr, rtol=1e-10, atol=1e-16)      # numpy's own weights are only ~1e-12 accurate
    for k in {2 * n - 2, 2 * n - 1, n, min(2, 2 * n - 1)}:   # exact up to degree 2n-1 (numpy reaches ~1e-14)
        exact = 2.0 / (k + 1) if k % 2 == 0 else 0.0
        assert abs(np.dot(w, x ** k) - exact) <= 4e-16
    assert np.all(np.diff(x) > 0)
    assert np.array_equal(x, -x[::-1]) and np.array_equal(w, w[::-1])   # symmetric pairs enforced
    a, b = 0.0, 1.7
    x, w = O.gauss_legendre(n, a, b)
    for k in range(0, min(2 * n, 12)):
        exact = (b ** (k + 1) - a ** (k + 1)) / (k + 1)
        assert abs(np.dot(w, x ** k) - exact) <= 1e-14 * exact


# ----------------------------------------------------------------------------------------------
# Bare operator (reading R1): hand-evaluated matrix elements, Hermiticity, relabelling symmetry.
# ----------------------------------------------------------------------------------------------
def test_operator_hand_evaluated_elements():
    """All spins up, three protons, all transfers along z: every Pauli dot product is a number.
    t_i.t_j = 1 between protons, (sigma_i.q)(sigma_j.q') = q_z q'_z on |up up up>."""
    a, b = 0.7, -0.4
    q = np.array([[0, 0, a], [0, 0, b], [0, 0, -a - b]])
    m = PHYS["mpi"] / HBARC
    f = PHYS["fpi"] / HBARC
    L = PHYS["lambda_chi"] / HBARC
    qz = q[:, 2]
    D = qz ** 2 + m ** 2
    row = 8 * 0 + 0          # spin index 0 = up up up, isospin index 0 = p p p
    # cE: cE/(2 f^4 L) * sum_{j != k} 1
    V = O.v3n(q, **only(cE=-0.5))
    assert V[row, row] == pytest.approx(-0.5 / (2 * f ** 4 * L) * 6, rel=1e-14)
    # cD: -gA/(8 f^2) cD/(f^2 L) sum_{i != j} q_j^2 / D_j
    V = O.v3n(q, **only(cD=1.0))
    want = -PHYS["gA"] / (8 * f ** 2) * 1.0 / (f ** 2 * L) * 2 * np.sum(qz ** 2 / D)
    assert V[row, row] == pytest.approx(want, rel=1e-14)
    # c1, c3: 1/2 (gA/2f)^2 sum_{i != j} q_i q_j /(D_i D_j) (-4 c1 m^2/f^2 + 2 c3/f^2 q_i q_j)
    c1 = -0.81e-3 * HBARC
    c3 = -3.2e-3 * HBARC
    V = O.v3n(q, **only(c1=-0.81, c3=-3.2))
    want = 0.0
    for i in range(3):
        for j in range(3):
            if i != j:
                want += 0.5 * (PHYS["gA"] / (2 * f)) ** 2 * qz[i] * qz[j] / (D[i] * D[j]) * (
                    -4 * c1 * m ** 2 / f ** 2 + 2 * c3 / f ** 2 * qz[i] * qz[j])
    assert V[row, row] == pytest.approx(want, rel=1e-14)
    # c4: (t_i x t_j).t_k has no diagonal element between isospin product states with all t_z equal
    V = O.v3n(RNG.normal(size=(3, 3)), **only(c4=5.4))
    assert abs(V[row, row]) < 1e-18
    assert np.abs(V).max() > 1e-3


def test_c4_term_sign_and_size_by_hand():
    """The c4 part of the two-pion exchange (reading R1),
        1/2 (gA/2f)^2 c4/f^2 sum_{ijk} (s_i.q_i)(s_j.q_j)/(D_i D_j) (t_i x t_j).t_k s_k.(q_i x q_j),
    at q1 = (a,0,0), q2 = (0,b,0), q3 = 0: only (i,j,k) = (1,2,3) and (2,1,3) survive and are equal, so
        V = (gA/2f)^2 c4/f^2 a b/(D1 D2) [s_1x s_2y (a b s_3z)] [(t_1 x t_2).t_3].
    Every factor is a number between product states:
        <dn dn s3| s_1x s_2y s_3z |up up s3> = (1)(i)(+1 for s3 = up, -1 for s3 = down),
        <n p p| (t_1 x t_2).t_3 |p n p> = <n p|t_1x t_2y - t_1y t_2x|p n> <p|t_3z|p> = (1)(-i) - (i)(1) = -2i
        (and +2i with a spectator neutron, <n|t_3z|n> = -1),
    so the element is + 2 (gA/2f)^2 (c4/f^2) a^2 b^2 / (D1 D2) for (s3 up, t3 proton): fixes the sign, the
    factor 1/2 (gA/2f)^2 c4/f^2 and the Levi-Civita isospin factor of the term, none of which P3/P5/P10 see."""
    a, b = 0.9, -0.6
    q = np.array([[a, 0, 0], [0, b, 0], [0, 0, 0]])
    m, f = PHYS["mpi"] / HBARC, PHYS["fpi"] / HBARC
    c4 = 5.4e-3 * HBARC
    D1, D2 = a * a + m * m, b * b + m * m
    want = 2 * (PHYS["gA"] / (2 * f)) ** 2 * c4 / f ** 2 * a * a * b * b / (D1 * D2)
    V = O.v3n(q, **only(c4=5.4))

    def idx(s, t):                                         # s, t = (b1, b2, b3); 64-dim index = 8 spin + isospin
        return 8 * (4 * s[0] + 2 * s[1] + s[2]) + 4 * t[0] + 2 * t[1] + t[2]

    assert want > 0.01
    for s3, t3, sign in ((0, 0, +1), (1, 0, -1), (0, 1, -1), (1, 1, +1)):
        got = V[idx((1, 1, s3), (1, 0, t3)), idx((0, 0, s3), (0, 1, t3))]
        assert got.real == pytest.approx(sign * want, rel=1e-14) and abs(got.imag) < 1e-16 * want
    # the reverse isospin exchange |n p> -> |p n> has the opposite sign ((t_1 x t_2)_z is antisymmetric)
    got = V[idx((1, 1, 0), (0, 1, 0)), idx((0, 0, 0), (1, 0, 0))]
    assert got.real == pytest.approx(-want, rel=1e-14)
    # spectator spin or isospin changed, or the pair's isospin unchanged: no contribution from this topology
    assert abs(V[idx((1, 1, 1), (1, 0, 0)), idx((0, 0, 0), (0, 1, 0))]) < 1e-16 * want
    assert abs(V[idx((1, 1, 0), (0, 1, 0)), idx((0, 0, 0), (0, 1, 0))]) < 1e-16 * want
    # linear in c4, and nothing else of the operator is switched on by it
    V2 = O.v3n(q, **only(c4=-2.7))
    assert np.abs(V2 + 0.5 * V).max() < 1e-15 * np.abs(V).max()


def _perm_matrix64(pi):
    """<b'|Pi_pi|b> = prod_m delta(b'_{pi(m)}, b_m) on spin (x) isospin of three particles."""
    P8 = np.zeros((8, 8))
    for b in range(8):
        bits = [(b >> 2) & 1, (b >> 1) & 1, b & 1]
        out = [0, 0, 0]
        for m in range(3):
            out[pi[m]] = bits[m]
        P8[4 * out[0] + 2 * out[1] + out[2], b] = 1.0
    return np.kron(P8, P8)


def test_operator_is_hermitian_even_and_symmetric_under_relabelling():
    kw = dict(PHYS, c4=5.4)
    q = RNG.normal(size=(3, 3))
    q[2] = -q[0] - q[1]
    V = O.v3n(q, **kw)
    scale = np.abs(V).max()
    assert np.abs(V - V.conj().T).max() < 1e-15 * scale
    assert np.abs(V - O.v3n(-q, **kw)).max() < 1e-15 * scale
    for pi in ([1, 0, 2], [2, 1, 0], [0, 2, 1], [1, 2, 0], [2, 0, 1]):
        Pm = _perm_matrix64(pi)
        qp = np.empty_like(q)
        for m in range(3):
            qp[pi[m]] = q[m]          # particle m, relabelled pi(m), keeps its momentum transfer
        assert np.abs(Pm @ V @ Pm.T - O.v3n(qp, **kw)).max() < 2e-15 * scale


def test_antisymmetrised_matrix_is_antisymmetric_in_both_indices():
    """A_123 V A-symmetry at the untraced level, with the regulator on."""
    kw = dict(PHYS, c4=5.4)
    kin = RNG.normal(size=(3, 3)) * 0.6
    kout = RNG.normal(size=(3, 3)) * 0.6
    kout[2] = kin.sum(axis=0) - kout[0] - kout[1]
    AV = O.av3n(kin, kout, **kw)
    scale = np.abs(AV).max()
    assert scale > 1e-3
    for pi, sgn in (([1, 0, 2], -1), ([2, 1, 0], -1), ([1, 2, 0], +1)):
        Pm = _perm_matrix64(pi)
        ko = np.empty_like(kout)
        ki = np.empty_like(kin)
        for m in range(3):
            ko[pi[m]] = kout[m]
            ki[pi[m]] = kin[m]
        # permuting the outgoing labels (momenta with spin-isospin) gives the sign of pi
        assert np.abs(Pm @ AV - sgn * O.av3n(kin, ko, **kw)).max() < 4e-15 * scale
        assert np.abs(AV @ Pm.T - sgn * O.av3n(ki, kout, **kw)).max() < 4e-15 * scale


# ----------------------------------------------------------------------------------------------
# P1 / P2: closed forms of the contact term (north_star (c)).
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kf", [0.8, 1.33, 1.7])
@pytest.mark.parametrize("level", [0, 1])
def test_P1_cE_closed_form_snm_unregulated(kf, level):
    kw = only(cE=-0.5, Lambda=-1.0, kf_n=kf, kf_p=kf, n_r=3, n_cos=2, n_phi=2)
    cfg = rand_cfg(3, 2.0)
    M = O.normal_order(cfg, level=level, **kw)
    f = PHYS["fpi"] / HBARC
    L = PHYS["lambda_chi"] / HBARC
    pref = -(-0.5) * kf ** 3 / (math.pi ** 2 * f ** 4 * L)
    want = pref * (np.eye(16) - p12_matrix())
    for m in M:
        assert np.abs(m - want).max() < 2e-15 * abs(pref)
    # scales as kF^3, and the number quoted in SURVEY.md Appendix A for kF = 1.33
    if kf == 1.33:
        assert pref == pytest.approx(0.6988301080442392, rel=1e-12)


def test_P2_cE_energy_closed_form():
    kf = 1.33
    kw = only(cE=-0.5, Lambda=-1.0, kf_n=kf, kf_p=kf, n_r=2, n_cos=2, n_phi=2)
    M = O.normal_order(rand_cfg(1), **kw)[0]
    dens = kf ** 3 / (6 * math.pi ** 2)           # per spin-isospin state
    e_from_m = np.trace(M).real * dens ** 2 / 6
    rho = 2 * kf ** 3 / (3 * math.pi ** 2)
    f = PHYS["fpi"] / HBARC
    L = PHYS["lambda_chi"] / HBARC
    assert e_from_m == pytest.approx(-(3.0 / 16.0) * (-0.5) * rho ** 3 / (f ** 4 * L), rel=1e-14)


# ----------------------------------------------------------------------------------------------
# P3: cD, cE (and c4) vanish in pure neutron matter (Sec. VI A; reading R17).
# ----------------------------------------------------------------------------------------------
NN_BLOCK = [idx(s1, s2, 1, 1) for s1 in range(2) for s2 in range(2)]


@pytest.mark.parametrize("which", ["cD", "cE", "c4"])
def test_P3_pnm_vanishing(which):
    lec = {"cD": 1.0, "cE": -0.5, "c4": 5.4}[which]
    kw = only(**{which: lec}, kf_n=1.3, kf_p=0.0, n_r=3, n_cos=3, n_phi=3)
    cfg = rand_cfg(4, 1.5)
    M = O.normal_order(cfg, **kw)
    ref = O.normal_order(cfg, **only(c1=-0.81, c3=-3.2, kf_n=1.3, kf_p=0.0, n_r=3, n_cos=3, n_phi=3))
    scale = np.abs(ref[:, NN_BLOCK][:, :, NN_BLOCK]).max()
    assert scale > 1e-3                                       # c1/c3 do NOT vanish
    assert np.abs(M[:, NN_BLOCK][:, :, NN_BLOCK]).max() < 1e-16 * max(1.0, scale / 1e-2)
    assert np.abs(M).max() > 1e-3                             # blocks with an external proton do not (R17)
    # node by node, before the trace: the nnn isospin block of A_123 V vanishes identically
    kin = RNG.normal(size=(3, 3)) * 0.6
    kout = RNG.normal(size=(3, 3)) * 0.6
    kout[2] = kin.sum(axis=0) - kout[0] - kout[1]
    AV = O.av3n(kin, kout, **only(**{which: lec}))
    nnn = [8 * s + 7 for s in range(8)]
    assert np.abs(AV[np.ix_(nnn, nnn)]).max() < 1e-15 * np.abs(AV).max()


# ----------------------------------------------------------------------------------------------
# P4 Hermiticity, P5 antisymmetry, P6 sparsity, P9 isospin symmetry, P10 linearity, P11 levels.
# ----------------------------------------------------------------------------------------------
ASYM = dict(PHYS, c4=5.4, kf_n=1.2, kf_p=0.9, n_r=3, n_cos=4, n_phi=3)


def _swap(cfg, what):
    c = cfg.copy()
    if what == "p<->p'":
        c[:, 0:3], c[:, 3:6] = cfg[:, 3:6], cfg[:, 0:3]
    elif what == "-p'":
        c[:, 3:6] *= -1
    elif what == "-p":
        c[:, 0:3] *= -1
    return c


def test_P4_hermiticity():
    cfg = rand_cfg(4, 1.5)
    M = O.normal_order(cfg, **ASYM)
    Mt = O.normal_order(_swap(cfg, "p<->p'"), **ASYM)
    scale = np.abs(M).max()
    assert np.abs(M - np.conj(np.swapaxes(Mt, 1, 2))).max() < 4e-16 * scale


def test_P5_antisymmetry():
    cfg = rand_cfg(4, 1.5)
    P = p12_matrix()
    M = O.normal_order(cfg, **ASYM)
    scale = np.abs(M).max()
    assert np.abs(P @ O.normal_order(_swap(cfg, "-p'"), **ASYM) + M).max() < 4e-16 * scale
    assert np.abs(O.normal_order(_swap(cfg, "-p"), **ASYM) @ P + M).max() < 4e-16 * scale


@pytest.mark.parametrize("level", [0, 1])
def test_P6_sparsity(level):
    """Charge conservation: 4^A * C(2A,A) = 96 possible non-zeros for A = 2."""
    kw = dict(ASYM, n_r=2, n_cos=3, n_phi=2)
    M = O.normal_order(rand_cfg(2, 1.5), level=level, **kw)
    allowed = np.zeros((16, 16), bool)
    for r in range(16):
        for c in range(16):
            allowed[r, c] = ((r >> 1) & 1) + (r & 1) == ((c >> 1) & 1) + (c & 1)
    assert allowed.sum() == 96 == 4 ** 2 * math.comb(4, 2)
    for m in M:
        assert np.abs(m[~allowed]).max() < 1e-16 * np.abs(m).max()
        assert (np.abs(m[allowed]) > 1e-9 * np.abs(m).max()).all()


def test_P9_isospin_symmetry_snm_and_its_breaking_in_asymmetric_matter():
    def blocks(m):
        B = {}
        for a, (t1o, t2o) in enumerate(((0, 0), (0, 1), (1, 0), (1, 1))):
            for b, (t1, t2) in enumerate(((0, 0), (0, 1), (1, 0), (1, 1))):
                rows = [idx(s1, s2, t1o, t2o) for s1 in range(2) for s2 in range(2)]
                cols = [idx(s1, s2, t1, t2) for s1 in range(2) for s2 in range(2)]
                B[a, b] = m[np.ix_(rows, cols)]
        return B
    cfg = rand_cfg(2, 1.5)
    snm = dict(ASYM, kf_n=1.1, kf_p=1.1)
    for m in O.normal_order(cfg, **snm):
        B = blocks(m)
        scale = np.abs(m).max()
        t1 = (B[1, 1] + B[1, 2] + B[2, 1] + B[2, 2]) / 2
        assert np.abs(B[0, 0] - B[3, 3]).max() < 4e-16 * scale
        assert np.abs(B[0, 0] - t1).max() < 4e-16 * scale
        assert np.abs(B[1, 1] - B[1, 2] + B[2, 1] - B[2, 2]).max() < 4e-16 * scale
    m = O.normal_order(cfg, **ASYM)[0]
    B = blocks(m)
    assert np.abs(B[0, 0] - B[3, 3]).max() > 1e-3 * np.abs(m).max()


def test_P10_linearity_in_the_lecs():
    cfg = rand_cfg(2, 1.5)
    geo = dict(kf_n=1.2, kf_p=0.9, n_r=3, n_cos=2, n_phi=3)
    full = O.normal_order(cfg, **dict(PHYS, c4=5.4, **geo))
    each = [O.normal_order(cfg, **only(**{k: v}, **geo))
            for k, v in (("c1", -0.81), ("c3", -3.2), ("c4", 5.4), ("cD", 1.0), ("cE", -0.5))]
    assert min(np.abs(e).max() for e in each) > 1e-3          # every topology contributes
    # each part is rounded to double on output: tolerance = a few ulp of the largest part
    assert np.abs(full - sum(each)).max() < 4e-16 * sum(np.abs(e).max() for e in each)


@pytest.mark.parametrize("geo", [dict(kf_n=1.2, kf_p=0.9, n_r=2, n_cos=3, n_phi=4),
                                 dict(kf_n=1.0, kf_p=0.0, n_r=3, n_cos=2, n_phi=2),
                                 dict(kf_n=1.3, kf_p=1.3, n_r=2, n_cos=2, n_phi=5, Lambda=450.0, n_reg=3)])
def test_P11_level0_equals_level1(geo):
    cfg = rand_cfg(3, 2.0)
    kw = dict(PHYS, c4=5.4)
    kw.update(geo)
    M0 = O.normal_order(cfg, level=0, **kw)
    M1 = O.normal_order(cfg, level=1, **kw)
    assert np.abs(M0 - M1).max() < 1e-16 * np.abs(M0).max()
    M1d = O.normal_order(cfg, level=1, precision="f64", **kw)
    assert np.abs(M1d - M1).max() < 1e-14 * np.abs(M0).max()


# ----------------------------------------------------------------------------------------------
# P7: kF -> 0 (pins 1/(2 pi)^3, the weights and the r^2 Jacobian).
# ----------------------------------------------------------------------------------------------
def test_P7_low_density_limit():
    cfg = rand_cfg(1, 1.0)
    p, pp, P = cfg[0, 0:3], cfg[0, 3:6], cfg[0, 6:9]
    kin = np.array([P / 2 + p, P / 2 - p, np.zeros(3)])
    kout = np.array([P / 2 + pp, P / 2 - pp, np.zeros(3)])
    kw = dict(PHYS, c4=5.4)
    AV = O.av3n(kin, kout, **kw)
    # trace over the third particle's spin, third isospin fixed to neutron (t3 = 1)
    lim = np.zeros((16, 16), complex)
    for r in range(16):
        for c in range(16):
            s1o, s2o, t1o, t2o = (r >> 3) & 1, (r >> 2) & 1, (r >> 1) & 1, r & 1
            s1, s2, t1, t2 = (c >> 3) & 1, (c >> 2) & 1, (c >> 1) & 1, c & 1
            for s3 in range(2):
                lim[r, c] += AV[8 * (4 * s1o + 2 * s2o + s3) + 4 * t1o + 2 * t2o + 1,
                                8 * (4 * s1 + 2 * s2 + s3) + 4 * t1 + 2 * t2 + 1]
    errs = []
    for kf in (0.1, 0.01, 0.001):
        M = O.normal_order(cfg, kf_n=kf, kf_p=0.0, n_r=4, n_cos=4, n_phi=4, **kw)[0]
        assert np.abs(M).max() < 10 * kf ** 3          # M -> 0
        ratio = M / (kf ** 3 / (6 * math.pi ** 2))
        errs.append(np.abs(ratio - lim).max() / np.abs(lim).max())
    assert errs[0] < 2e-2 and errs[1] < 2e-4 and errs[2] < 2e-6      # O(kF^2)
    assert errs[0] / errs[1] == pytest.approx(100, rel=0.2)


# ----------------------------------------------------------------------------------------------
# P8: contracting once more over the Fermi sea gives the 3N Hartree-Fock energy of a brute-force
#     9-D quadrature on the same tiny grids (north_star (c)).
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("geo", [dict(kf_n=1.2, kf_p=0.9), dict(kf_n=1.1, kf_p=0.0)])
def test_P8_hartree_fock_identity(geo):
    n = 2
    kw = dict(PHYS, c4=5.4, n_r=n, n_cos=n, n_phi=n, **geo)
    e_brute = O.hf3n_bruteforce(**kw)
    # particles 1 and 2 on the same product grids, third particle integrated by normal ordering
    nodes = []
    for tau, kf in ((0, kw["kf_p"]), (1, kw["kf_n"])):
        if kf <= 0:
            continue
        r, wr = O.gauss_legendre(n, 0.0, kf)
        x, wx = O.gauss_legendre(n, -1.0, 1.0)
        ph, wp = O.gauss_legendre(n, 0.0, 2 * math.pi)
        for i in range(n):
            for j in range(n):
                for l in range(n):
                    st = math.sqrt(1 - x[j] ** 2)
                    k = r[i] * np.array([st * math.cos(ph[l]), st * math.sin(ph[l]), x[j]])
                    nodes.append((k, r[i] ** 2 * wr[i] * wx[j] * wp[l] / (2 * math.pi) ** 3, tau))
    cfgs, wts, isos = [], [], []
    for k1, w1, t1 in nodes:
        for k2, w2, t2 in nodes:
            p = (k1 - k2) / 2
            cfgs.append(np.concatenate([p, p, k1 + k2]))
            wts.append(w1 * w2)
            isos.append((t1, t2))
    M = O.normal_order(np.array(cfgs), **kw)
    e_no = 0.0
    for m, w, (t1, t2) in zip(M, wts, isos):
        for s1 in range(2):
            for s2 in range(2):
                e_no += w * m[idx(s1, s2, t1, t2), idx(s1, s2, t1, t2)].real
    e_no /= 6
    assert abs(e_brute) > 1e-6
    assert e_no == pytest.approx(e_brute, rel=1e-13)


# ----------------------------------------------------------------------------------------------
# P12: values of an independent transcription -- a third opinion.  The stored values are the
# survey's originals (never regenerated); tests/golden/make_survey_appendix_a.py is checked against them.
# ----------------------------------------------------------------------------------------------
def test_P12_cross_implementation_values():
    path = os.path.join(os.path.dirname(__file__), "golden", "survey_appendix_a.txt")
    rows = [l.split() for l in open(path) if l.strip() and not l.startswith("#")]
    cfg = np.array([[0.3, -0.2, 0.5, -0.1, 0.4, 0.2, 0.2, 0.1, -0.3]])
    for c4 in (0.0, 5.4):
        M = O.normal_order(cfg, level=0, kf_p=0.9, kf_n=1.2, n_r=4, n_cos=4, n_phi=4, c4=c4, **PHYS)[0]
        assert (np.abs(M) > 1e-14).sum() == 96
        for row in rows:
            if float(row[0]) != c4:
                continue
            r, c, re, im = int(row[1]), int(row[2]), float(row[3]), float(row[4])
            if r == -1:
                assert np.linalg.norm(M) == pytest.approx(re, rel=1e-13)
            elif r == -2:
                assert np.abs(M).max() == pytest.approx(re, rel=1e-13)
            else:
                assert abs(M[r, c] - complex(re, im)) < 1e-14


def test_P12_golden_file_is_regenerable_by_the_committed_numpy_transcription():
    """tests/golden/make_survey_appendix_a.py (numpy only; imports neither oracle/ nor the product package)
    reproduces every stored value (the survey's original digits) to 1e-13; the script never writes the file."""
    import subprocess
    import sys
    here = os.path.dirname(__file__)
    script = os.path.join(here, "golden", "make_survey_appendix_a.py")
    import ast
    mods = set()
    for node in ast.walk(ast.parse(open(script).read())):
        if isinstance(node, ast.Import):
            mods.update(a.name.split(".")[0] for a in node.names)
        elif isinstance(node, ast.ImportFrom):
            mods.add((node.module or "").split(".")[0])
    assert mods <= {"itertools", "os", "sys", "numpy"}, mods
    assert "--write" not in open(script).read() and 'open(' not in open(script).read()
    out = subprocess.run([sys.executable, script], check=True, capture_output=True, text=True).stdout

    def rows(text):
        return np.array([[float(x) for x in l.split()] for l in text.splitlines() if l.strip() and not l.startswith("#")])

    got, want = rows(out), rows(open(os.path.join(here, "golden", "survey_appendix_a.txt")).read())
    assert got.shape == want.shape == (22, 5)
    assert np.array_equal(got[:, :3], want[:, :3])
    assert np.abs(got[:, 3:] - want[:, 3:]).max() < 1e-13


def test_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the oracle, built with -fsanitize=address,undefined (tests/oracle_sanitize_main.cpp
    includes oracle/no_oracle.cpp verbatim), runs P11 on a 2^3 grid, the direction-list path, the double
    instantiation and the brute-force Hartree-Fock sum without a report."""
    import subprocess
    here = os.path.dirname(__file__)
    exe = str(tmp_path / "oracle_sanitized")
    subprocess.run(["g++", "-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                    "-fno-omit-frame-pointer", "-o", exe, os.path.join(here, "oracle_sanitize_main.cpp")], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr and "LeakSanitizer" not in r.stderr
    assert "level0-level1" in r.stdout


# ----------------------------------------------------------------------------------------------
# Regulator (reading R5): Jacobi form equals p^2 + |k3 - P/2|^2 / 3 and is ONE exponential.
# ----------------------------------------------------------------------------------------------
def test_regulator_reduces_to_the_normal_ordering_form():
    cfg = rand_cfg(1, 1.0)
    p, pp, P = cfg[0, 0:3], cfg[0, 3:6], cfg[0, 6:9]
    k3 = RNG.normal(size=3) * 0.5
    kin = np.array([P / 2 + p, P / 2 - p, k3])
    kout = np.array([P / 2 + pp, P / 2 - pp, k3])
    for Lam, n in ((500.0, 4), (450.0, 3), (400.0, 2)):
        reg = O.av3n(kin, kout, **only(cE=1.0, Lambda=Lam, n_reg=n))
        bare = O.av3n(kin, kout, **only(cE=1.0, Lambda=-1.0))
        L2 = (Lam / HBARC) ** 2
        d2 = np.dot(k3 - P / 2, k3 - P / 2)
        want = math.exp(-((p @ p + d2 / 3) / L2) ** n - ((pp @ pp + d2 / 3) / L2) ** n)
        i = np.unravel_index(np.abs(bare).argmax(), bare.shape)
        assert (reg[i] / bare[i]).real == pytest.approx(want, rel=1e-14)


# ----------------------------------------------------------------------------------------------
# the Hartree-Fock contraction functions of the oracle against what fixes them
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("geo", [dict(kf_n=1.2, kf_p=0.9), dict(kf_n=0.0, kf_p=1.0), dict(kf_n=1.1, kf_p=1.1)])
def test_hf_energy_function_equals_brute_force_on_equal_grids(geo):
    """pin P8 for O.hf_energy: exact reordering of the 9-D sum when all three particles share the grid."""
    kw = dict(PHYS, c4=5.4, n_r=2, n_cos=3, n_phi=2, **geo)
    e_brute = O.hf3n_bruteforce(**kw)
    e_no = O.hf_energy(2, 3, 2, **kw)
    assert abs(e_brute) > 1e-8
    assert e_no == pytest.approx(e_brute, rel=1e-12)


def test_hf_energy_function_cE_closed_form():
    """pin P2 for O.hf_energy: unregulated contact term in SNM, E/V = -(3/16) cE rho^3/(fpi^4 Lchi), any grids >= 2."""
    kF = 1.33
    kw = dict(kf_n=kF, kf_p=kF, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0, Lambda=-1.0,
              n_r=3, n_cos=2, n_phi=2)
    hbarc = 197.3269804
    rho = 2 * kF ** 3 / (3 * math.pi ** 2)
    want = -(3.0 / 16.0) * (-0.5) * rho ** 3 / ((92.4 / hbarc) ** 4 * (700.0 / hbarc))
    assert O.hf_energy(2, 2, 3, **kw) == pytest.approx(want, rel=1e-12)


def test_diag_trace_is_the_spin_trace_of_the_diagonal():
    kw = dict(PHYS, kf_n=1.2, kf_p=0.9, n_r=2, n_cos=2, n_phi=2)
    cfg = RNG.uniform(-1, 1, (3, 9))
    M = O.normal_order(cfg, **kw)
    D = O.diag_trace(cfg, **kw)
    for t1 in range(2):
        for t2 in range(2):
            want = sum(M[:, idx(s1, s2, t1, t2), idx(s1, s2, t1, t2)].real for s1 in range(2) for s2 in range(2))
            assert np.allclose(D[:, 2 * t1 + t2], want, rtol=0, atol=1e-15)
    assert np.abs(np.trace(M, axis1=1, axis2=2).real - D.sum(axis=1)).max() < 1e-14


def test_oracle_direction_list_equals_the_product_grid():
    """pin of the caller-supplied angular rule path of the oracle: the cos x phi Gauss-Legendre grid passed
    as a list (built here with numpy's leggauss, not with the oracle's rule) gives the default result."""
    kw = dict(PHYS, c4=5.4, kf_n=1.2, kf_p=0.9, n_r=3)
    x, wx = np.polynomial.legendre.leggauss(4)
    t, wt = np.polynomial.legendre.leggauss(5)
    ph, wp = math.pi * (t + 1), math.pi * wt
    dirs = np.array([[math.sqrt(1 - x[j] ** 2) * math.cos(ph[l]), math.sqrt(1 - x[j] ** 2) * math.sin(ph[l]), x[j],
                      wx[j] * wp[l]] for j in range(4) for l in range(5)])
    cfg = RNG.uniform(-1, 1, (2, 9))
    a = O.normal_order(cfg, n_cos=4, n_phi=5, **kw)
    b = O.normal_order(cfg, dirs=dirs, n_cos=1, n_phi=1, **kw)
    assert np.abs(a - b).max() < 1e-14 * np.abs(a).max()


def test_oracle_direction_list_cE_closed_form():
    """P1 with an angular rule of 6 directions: the constant integrand only needs sum w = 4 pi."""
    kF = 1.33
    dirs = np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=float)
    dirs = np.column_stack([dirs, np.full(6, 4 * math.pi / 6)])
    kw = dict(kf_n=kF, kf_p=kF, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0, Lambda=-1.0, n_r=2,
              n_cos=1, n_phi=1)
    M = O.normal_order(np.zeros((1, 9)), dirs=dirs, **kw)[0]
    hbarc = 197.3269804
    pref = -(-0.5) * kF ** 3 / (math.pi ** 2 * (92.4 / hbarc) ** 4 * (700.0 / hbarc))
    assert M[1, 1].real == pytest.approx(pref, rel=1e-13) and M[1, 2].real == pytest.approx(-pref, rel=1e-13)
    assert abs(M[0, 0]) < 1e-15


# ----------------------------------------------------------------------------------------------
# Hartree-Fock self-energy of Eq. (9), oracle function sp_energy
# ----------------------------------------------------------------------------------------------
def test_sp_energy_sum_rule_gives_the_hf_energy():
    """E/V = (1/3) sum_{t1} sum_{k1 in S(t1)} 2 W1 Sigma_t1(k1) (three equivalent ways to pick particle 1 out
    of the 1/6 of Eq. (1)): ties sp_energy to hf_energy, which pin P8 ties to the brute-force 9-D sum."""
    kw = dict(PHYS, c4=5.4, kf_n=1.2, kf_p=0.9, n_r=2, n_cos=3, n_phi=2)
    e = 0.0
    for t1, kf in ((0, kw["kf_p"]), (1, kw["kf_n"])):
        k1, w1 = O.sphere_nodes(2, 3, 2, kf)
        e += np.sum(2 * w1 * O.sp_energy(k1, 2, 3, 2, **kw)[:, t1]) / 3
    assert e == pytest.approx(O.hf3n_bruteforce(**kw), rel=1e-12)


def test_sp_energy_cE_closed_form():
    """unregulated contact term in SNM: from P1, D[t1 t2] = pref (4 - 2 delta_t1t2), so
    Sigma = (1/4) (kF^3/6 pi^2) 6 pref = pref kF^3/(4 pi^2), independent of k1 and of the isospin."""
    kF, hbarc = 1.33, 197.3269804
    kw = dict(kf_n=kF, kf_p=kF, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0, Lambda=-1.0,
              n_r=2, n_cos=2, n_phi=2)
    pref = -(-0.5) * kF ** 3 / (math.pi ** 2 * (92.4 / hbarc) ** 4 * (700.0 / hbarc))
    sig = O.sp_energy(np.array([[0.3, -0.2, 0.5], [2.0, 1.0, -3.0]]), 3, 2, 2, **kw)
    assert np.allclose(sig, pref * kF ** 3 / (4 * math.pi ** 2), rtol=1e-12, atol=0)


# ----------------------------------------------------------------------------------------------
# Packed, symmetry-reduced matrix, oracle functions pack / unpack
# ----------------------------------------------------------------------------------------------
def test_pack_format1_is_exactly_the_96_charge_conserving_entries():
    """"only up to 4^A C(2A,A) matrix elements can be non-zero": the index map of format 1 hits each of
    the 96 allowed (row, column) pairs once and nothing else (checked on a matrix of distinct labels, independent of the physics)."""
    label = (np.arange(256).reshape(1, 16, 16) + 1).astype(complex)
    P = O.pack(label, O.PACK_CHARGE)[0].real.astype(int) - 1
    assert len(set(P.tolist())) == 96 == 4 ** 2 * math.comb(4, 2)
    for e in P:
        r, c = divmod(int(e), 16)
        assert ((r >> 1) & 1) + (r & 1) == ((c >> 1) & 1) + (c & 1)
    # the element order: spin element major, then (pp,pp) (pn,pn) (np,np) (nn,nn) (pn,np) (np,pn)
    assert P[0] == 16 * idx(0, 0, 0, 0) + idx(0, 0, 0, 0) and P[4] == 16 * idx(0, 0, 0, 1) + idx(0, 0, 1, 0)
    assert P[6 * 7 + 5] == 16 * idx(0, 1, 1, 0) + idx(1, 1, 0, 1)
    U = O.unpack(O.pack(label, O.PACK_CHARGE), O.PACK_CHARGE)[0]
    allowed = U != 0
    assert allowed.sum() == 96 and (U[allowed] == label[0][allowed]).all()


@pytest.mark.parametrize("matter", ["snm", "pnm", "asym"])
def test_unpack_of_pack_reproduces_the_oracle_matrix(matter):
    """Format 1 loses nothing in any matter (P6); format 2 reconstructs the matrix only in isospin-symmetric matter
    (P9: pp = nn = T=1 combination, pn/np blocks equal) and must NOT be used elsewhere (pp != nn there)."""
    kf = {"snm": (1.1, 1.1), "pnm": (1.3, 0.0), "asym": (1.2, 0.9)}[matter]
    kw = dict(PHYS, c4=5.4, kf_n=kf[0], kf_p=kf[1], n_r=3, n_cos=3, n_phi=4)
    M = O.normal_order(rand_cfg(3, 1.5), **kw)
    scale = np.abs(M).max(axis=(1, 2), keepdims=True)
    U1 = O.unpack(O.pack(M, O.PACK_CHARGE), O.PACK_CHARGE)
    assert np.abs(U1 - M).max() <= 1e-16 * scale.max()        # only the O(1e-17) structural zeros of the oracle differ
    U2 = O.unpack(O.pack(M, O.PACK_ISOSPIN), O.PACK_ISOSPIN)
    err = (np.abs(U2 - M) / scale).max()
    if matter == "snm":
        assert err < 4e-16
    else:
        assert err > 1e-3
