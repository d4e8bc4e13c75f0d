"""Angular quadrature rules on the unit sphere, as INPUT arrays for no_init_angular and for the oracle.

The paper integrates the Fermi sea with "Gauss-Legendre radial x Lebedev angular" quadrature
(16 radial points, order-15 Lebedev rule); BASELINE.json's configs use a
cos(theta) x phi Gauss-Legendre product grid.  Both are just lists of unit vectors and weights
(sum w = 4 pi), dirs[n,4] = (ux, uy, uz, w); the library and the oracle take such a list as an input.
This module holds no arithmetic of the normal-ordering method.

Lebedev-type rules are NOT copied from a table (none is available here): `octahedral_rule` solves
the moment equations of an octahedrally symmetric point set (orbits a1, a2, a3, b_k, c_k) so that
all monomials up to the requested degree are integrated exactly, starting from seeded random
guesses.  `check_rule` verifies the result against the closed-form monomial integrals.
"""
from __future__ import annotations

import functools
import itertools
import math

import numpy as np

# orbit structure (a1, a2, a3, n_b, n_c) of the octahedral rules by algebraic degree
STRUCTURES = {3: (1, 0, 0, 0, 0), 5: (1, 0, 1, 0, 0), 7: (1, 1, 1, 0, 0), 9: (1, 0, 1, 0, 1),
              11: (1, 1, 1, 1, 0), 15: (1, 0, 1, 2, 1), 17: (1, 0, 1, 3, 1)}


def product_rule(n_cos: int, n_phi: int) -> np.ndarray:
    """The cos(theta) x phi Gauss-Legendre product grid as a direction list (phi fastest)."""
    x, wx = np.polynomial.legendre.leggauss(n_cos)
    t, wt = np.polynomial.legendre.leggauss(n_phi)
    phi, wphi = math.pi * (t + 1.0), math.pi * wt
    st = np.sqrt((1.0 - x) * (1.0 + x))
    out = np.empty((n_cos, n_phi, 4))
    out[..., 0] = st[:, None] * np.cos(phi)[None, :]
    out[..., 1] = st[:, None] * np.sin(phi)[None, :]
    out[..., 2] = x[:, None]
    out[..., 3] = wx[:, None] * wphi[None, :]
    return out.reshape(-1, 4)


def monomial_integral(a: int, b: int, c: int) -> float:
    """int x^a y^b z^c dOmega over the unit sphere (closed form)."""
    if a % 2 or b % 2 or c % 2:
        return 0.0
    lg = math.lgamma
    return 2.0 * math.exp(lg((a + 1) / 2) + lg((b + 1) / 2) + lg((c + 1) / 2) - lg((a + b + c + 3) / 2))


_SIGNS = np.array(list(itertools.product((1.0, -1.0), repeat=3)))


def _orbit_a1() -> np.ndarray:
    e = np.eye(3)
    return np.vstack([e, -e])


def _orbit_a2() -> np.ndarray:
    r = math.sqrt(0.5)
    pts = []
    for zero in range(3):
        i, j = [k for k in range(3) if k != zero]
        for si in (r, -r):
            for sj in (r, -r):
                v = [0.0, 0.0, 0.0]
                v[i], v[j] = si, sj
                pts.append(v)
    return np.array(pts)


def _orbit_a3() -> np.ndarray:
    return _SIGNS * math.sqrt(1.0 / 3.0)


def _orbit_b(l: float) -> np.ndarray:
    m = math.sqrt(max(1.0 - 2.0 * l * l, 0.0))
    base = np.array([[l, l, m], [l, m, l], [m, l, l]])
    return (base[:, None, :] * _SIGNS[None, :, :]).reshape(-1, 3)          # 24 points


def _orbit_c(p: float) -> np.ndarray:
    q = math.sqrt(max(1.0 - p * p, 0.0))
    pts = []
    for zero in range(3):
        i, j = [k for k in range(3) if k != zero]
        for a, b in ((p, q), (q, p)):
            for sa in (1.0, -1.0):
                for sb in (1.0, -1.0):
                    v = [0.0, 0.0, 0.0]
                    v[i], v[j] = sa * a, sb * b
                    pts.append(v)
    return np.array(pts)                                                      # 24 points


def _orbits(struct, params):
    """list of points[n,3] per orbit; params = [l_1..l_nb, p_1..p_nc]."""
    a1, a2, a3, nb, nc = struct
    orbs = []
    if a1:
        orbs.append(_orbit_a1())
    if a2:
        orbs.append(_orbit_a2())
    if a3:
        orbs.append(_orbit_a3())
    for k in range(nb):
        orbs.append(_orbit_b(params[k]))
    for k in range(nc):
        orbs.append(_orbit_c(params[nb + k]))
    return orbs


def _exponents(degree: int):
    """even monomials x^a y^b z^c, a >= b >= c, a + b + c <= degree (the others follow by symmetry)."""
    return [(a, b, c) for a in range(0, degree + 1, 2) for b in range(0, a + 1, 2) for c in range(0, b + 1, 2)
            if a + b + c <= degree]


def octahedral_rule(degree: int, seed: int = 0, tries: int = 400) -> np.ndarray:
    """dirs[n,4] of the octahedrally symmetric rule exact to `degree` (3, 5, 7, 9, 11, 15, 17);
    6, 14, 26, 38, 50, 86, 110 points, positive weights.  Deterministic for a given seed; cached."""
    return _octahedral_rule(degree, seed, tries).copy()


@functools.lru_cache(maxsize=None)
def _octahedral_rule(degree: int, seed: int, tries: int) -> np.ndarray:
    from scipy.optimize import least_squares

    struct = STRUCTURES[degree]
    a1, a2, a3, nb, nc = struct
    n_orb = a1 + a2 + a3 + nb + nc
    expo = _exponents(degree)
    exact = np.array([monomial_integral(*e) for e in expo])

    ex = np.array(expo, dtype=float)

    def residual(z):
        w, par = z[:n_orb], z[n_orb:]
        r = -exact.copy()
        for wk, pts in zip(w, _orbits(struct, par)):
            mono = np.prod(np.abs(pts)[:, None, :] ** ex[None, :, :], axis=2)     # even exponents
            r += wk * mono.sum(axis=0)
        return r

    rng = np.random.default_rng(seed)
    lo = np.concatenate([np.full(n_orb, 1e-4), np.full(nb, 1e-3), np.full(nc, 1e-3)])
    hi = np.concatenate([np.full(n_orb, 4 * math.pi), np.full(nb, math.sqrt(0.5) - 1e-3), np.full(nc, 1.0 - 1e-3)])
    n_pts = 6 * a1 + 12 * a2 + 8 * a3 + 24 * (nb + nc)
    for _ in range(tries):
        z0 = np.concatenate([np.full(n_orb, 4 * math.pi / n_pts) * rng.uniform(0.5, 1.5, n_orb),
                             rng.uniform(0.02, 0.70, nb), rng.uniform(0.02, 0.98, nc)])
        sol = least_squares(residual, z0, bounds=(lo, hi), xtol=1e-15, ftol=1e-15, gtol=1e-15)
        if np.abs(sol.fun).max() < 1e-13:
            par = sol.x[n_orb:]
            lpar, ppar = np.sort(par[:nb]), par[nb:]
            if nb > 1 and np.min(np.diff(lpar)) < 1e-3:
                continue                                   # two b-orbits collapsed onto each other
            if any(abs(p * p - 0.5) < 1e-3 for p in ppar):
                continue                                   # c-orbit degenerated into a2
            order = np.argsort(par[:nb])
            w = sol.x[:n_orb].copy()
            base = a1 + a2 + a3
            w[base:base + nb] = w[base:base + nb][order]
            par = np.concatenate([lpar, ppar])
            rows = [np.column_stack([pts, np.full(len(pts), wk)]) for wk, pts in zip(w, _orbits(struct, par))]
            dirs = np.ascontiguousarray(np.vstack(rows))
            dirs[:, :3] /= np.linalg.norm(dirs[:, :3], axis=1, keepdims=True)
            return dirs
    raise RuntimeError(f"no octahedral rule of degree {degree} found in {tries} tries")


def check_rule(dirs: np.ndarray, degree: int) -> float:
    """largest absolute error over ALL monomials x^a y^b z^c with a + b + c <= degree."""
    worst = 0.0
    for a in range(degree + 1):
        for b in range(degree + 1 - a):
            for c in range(degree + 1 - a - b):
                got = float(np.sum(dirs[:, 3] * dirs[:, 0] ** a * dirs[:, 1] ** b * dirs[:, 2] ** c))
                worst = max(worst, abs(got - monomial_integral(a, b, c)))
    return worst
