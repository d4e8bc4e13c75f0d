#!/usr/bin/env python
"""Recomputes the table of tests/golden/survey_appendix_a.txt (pin P12): a plain numpy transcription of the
level-0 definition of SURVEY.md section 8(c) / DESIGN.md section 1-3.

    python tests/golden/make_survey_appendix_a.py            # prints the table

It never writes the golden file: the stored values are the survey session's originals and stay byte for byte as
first committed; this script is checked AGAINST them (tests/test_oracle_pins.py, 1e-13), not the other way round.

It imports nothing from oracle/ or paper_2603_24532_b200/ (numpy only: np.kron for the Pauli-Kronecker
products, numpy's leggauss for the quadrature rule) and is a THIRD implementation next to the C++ oracle
and the CUDA path -- not an authority: the paper prints no matrix element.  The
values in the committed file were first produced by the survey session's scratch;
this transcription reproduces them, and tests/test_oracle_pins.py checks both the file against the
oracle and this script against the file.

Definition transcribed (readings R1, R4-R10, R15):
  M[a',a] = sum_{tau3} sum_{ijl} W_ijl F(k3) sum_{s3} <a'; s3 tau3| sum_pi sgn(pi) Pi_pi V(q^pi) |a; s3 tau3>
  V = 1/2 (gA/2f)^2 sum_{ijk} (s_i.q_i)(s_j.q_j)/(D_i D_j) [ (t_i.t_j)(-4 c1 m^2/f^2 + 2 c3/f^2 q_i.q_j)
                                                          + c4/f^2 (t_i x t_j).t_k s_k.(q_i x q_j) ]
      - gA cD/(8 f^4 Lchi) sum_{ijk} (s_j.q_j)(s_i.q_j)/D_j (t_i.t_j) + cE/(2 f^4 Lchi) sum_{jk} t_j.t_k
"""
import itertools
import os
import sys

import numpy as np

HBARC = 197.3269804
INPUT = dict(p=(0.3, -0.2, 0.5), pp=(-0.1, 0.4, 0.2), P=(0.2, 0.1, -0.3), kf_p=0.9, kf_n=1.2,
             c1=-0.81, c3=-3.2, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, Lchi=700.0, Lambda=500.0, n_reg=4,
             grid=(4, 4, 4))
ENTRIES = [(0, 0), (3, 3), (15, 15), (1, 2), (3, 15), (5, 10), (6, 9), (7, 13), (1, 4)]

PAULI = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]], complex),
         np.array([[1, 0], [0, -1]], complex)]
ID2 = np.eye(2, dtype=complex)


def on(slot, m):
    """one-body operator m on particle `slot` of three: kron(particle 1, particle 2, particle 3)."""
    f = [ID2, ID2, ID2]
    f[slot] = m
    return np.kron(np.kron(f[0], f[1]), f[2])


def sdot(slot, v):
    return sum(v[a] * on(slot, PAULI[a]) for a in range(3))


TDOT = {(i, j): sum(on(i, PAULI[a]) @ on(j, PAULI[a]) for a in range(3))
        for i in range(3) for j in range(3) if i != j}


def levi(a, b, c):
    return (a - b) * (b - c) * (c - a) / 2


TTRIPLE = {(i, j): sum(levi(a, b, c) * on(i, PAULI[a]) @ on(j, PAULI[b]) @ on(3 - i - j, PAULI[c])
                       for a in range(3) for b in range(3) for c in range(3) if levi(a, b, c))
           for i in range(3) for j in range(3) if i != j}


def v3n(q, c):
    """64x64 = kron(spin 8x8, isospin 8x8) for momentum transfers q[3][3] (fm^-1)."""
    m2, f2 = c["mpi"] ** 2, c["fpi"] ** 2
    G2 = (c["gA"] / (2 * c["fpi"])) ** 2
    D = [q[i] @ q[i] + m2 for i in range(3)]
    V = np.zeros((64, 64), complex)
    for i, j in itertools.permutations(range(3), 2):
        k = 3 - i - j
        sisj = sdot(i, q[i]) @ sdot(j, q[j]) / (D[i] * D[j])
        V += 0.5 * G2 * (-4 * c["c1"] * m2 / f2 + 2 * c["c3"] / f2 * (q[i] @ q[j])) * np.kron(sisj, TDOT[i, j])
        V += 0.5 * G2 * c["c4"] / f2 * np.kron(sisj @ sdot(k, np.cross(q[i], q[j])), TTRIPLE[i, j])
        V += -c["gA"] * c["cD"] / (8 * f2 * f2 * c["Lchi"]) * np.kron(sdot(j, q[j]) @ sdot(i, q[j]) / D[j], TDOT[i, j])
        V += c["cE"] / (2 * f2 * f2 * c["Lchi"]) * np.kron(np.eye(8), TDOT[i, j])
    return V


def perm8(pi):
    """<b'|Pi_pi|b> = prod_m delta(b'_{pi(m)}, b_m) on three two-level systems."""
    P = np.zeros((8, 8))
    for b in range(8):
        bits = [(b >> 2) & 1, (b >> 1) & 1, b & 1]
        out = [0, 0, 0]
        for m in range(3):
            out[pi[m]] = bits[m]
        P[4 * out[0] + 2 * out[1] + out[2], b] = 1
    return P


PERMS = [((0, 1, 2), 1), ((1, 0, 2), -1), ((2, 1, 0), -1), ((0, 2, 1), -1), ((1, 2, 0), 1), ((2, 0, 1), 1)]


def gauss_legendre(n, a, b):
    x, w = np.polynomial.legendre.leggauss(n)
    return 0.5 * (b + a) + 0.5 * (b - a) * x, 0.5 * (b - a) * w


def normal_order(c4_gev):
    I = INPUT
    c = dict(mpi=I["mpi"] / HBARC, fpi=I["fpi"] / HBARC, gA=I["gA"], Lchi=I["Lchi"] / HBARC,
             c1=I["c1"] * 1e-3 * HBARC, c3=I["c3"] * 1e-3 * HBARC, c4=c4_gev * 1e-3 * HBARC, cD=I["cD"], cE=I["cE"])
    L2 = (I["Lambda"] / HBARC) ** 2
    p, pp, P = (np.array(I[k], float) for k in ("p", "pp", "P"))
    n_r, n_c, n_p = I["grid"]
    M = np.zeros((16, 16), complex)
    for tau3, kf in ((0, I["kf_p"]), (1, I["kf_n"])):
        r, wr = gauss_legendre(n_r, 0.0, kf)
        x, wx = gauss_legendre(n_c, -1.0, 1.0)
        ph, wp = gauss_legendre(n_p, 0.0, 2 * np.pi)
        for i, j, l in itertools.product(range(n_r), range(n_c), range(n_p)):
            st = np.sqrt(1 - x[j] ** 2)
            k3 = r[i] * np.array([st * np.cos(ph[l]), st * np.sin(ph[l]), x[j]])
            W = r[i] ** 2 * wr[i] * wx[j] * wp[l] / (2 * np.pi) ** 3
            kin = [P / 2 + p, P / 2 - p, k3]
            kout = [P / 2 + pp, P / 2 - pp, k3]

            def jac(k):
                return sum((k[a] - k[b]) @ (k[a] - k[b]) for a, b in ((0, 1), (0, 2), (1, 2))) / 6
            F = np.exp(-((jac(kin) / L2) ** I["n_reg"] + (jac(kout) / L2) ** I["n_reg"]))
            AV = np.zeros((64, 64), complex)
            for pi, sgn in PERMS:
                q = np.array([kout[pi[m]] - kin[m] for m in range(3)])
                P8 = perm8(pi)
                AV += sgn * np.kron(P8, P8) @ v3n(q, c)
            AV *= W * F
            for so, to, si, ti, s3 in itertools.product(range(4), range(4), range(4), range(4), range(2)):
                row = 8 * (2 * so + s3) + 2 * to + tau3          # spin (s1 s2 s3), isospin (t1 t2 tau3)
                col = 8 * (2 * si + s3) + 2 * ti + tau3
                M[4 * so + to, 4 * si + ti] += AV[row, col]      # idx = 8 s1 + 4 s2 + 2 t1 + t2
    return M


def table():
    lines = []
    for c4 in (0.0, 5.4):
        M = normal_order(c4)
        lines.append((c4, -1, -1, float(np.linalg.norm(M)), 0.0))
        lines.append((c4, -2, -2, float(np.abs(M).max()), 0.0))
        for r, cidx in ENTRIES:
            v = M[r, cidx]
            charge = lambda a: ((a >> 1) & 1) + (a & 1)
            if charge(r) != charge(cidx):
                assert abs(v) < 1e-15, (r, cidx, v)
                v = 0.0
            lines.append((c4, r, cidx, float(np.real(v)), float(np.imag(v))))
    return lines


HEADER = """# Cross-implementation values for pin P12.
# Source: /root/repo/SURVEY.md, Appendix A ("cross-implementation values from this session's scratch"):
# a numpy transcription of the level-0 definition written by the survey's author, independent of
# oracle/no_oracle.cpp.  NOT from the paper (the paper prints no matrix element, SURVEY.md section 4).
# (recomputed by tests/golden/make_survey_appendix_a.py; the committed file keeps the survey's original digits)
# Inputs: p=(0.3,-0.2,0.5) p'=(-0.1,0.4,0.2) P=(0.2,0.1,-0.3) fm^-1; kf_p=0.9 kf_n=1.2;
# c1=-0.81 c3=-3.2 GeV^-1 cD=1.0 cE=-0.5 gA=1.27 fpi=92.4 mpi=138.04 Lchi=700 Lambda=500 MeV n_reg=4;
# grid 4x4x4; output fm^2; idx = 8 s1 + 4 s2 + 2 t1 + t2, t=0 proton.
# columns: c4[GeV^-1]  row  col  real  imag      (row = -1: Frobenius norm in `real`; row = -2: max abs)
"""


def main():
    rows = table()
    text = HEADER + "".join(f"{c4:.1f}  {r:2d} {c:2d}  {re:.15e}  {im:.15e}\n" for c4, r, c, re, im in rows)
    sys.stdout.write(text)


if __name__ == "__main__":
    main()
