"""ctypes face of the CPU oracle (oracle/no_oracle.cpp) -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  The product package (paper_2603_24532_b200) never does.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "no_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (OpenMP over configurations).  Returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC", "-Wall", "-Wextra",
               "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    from . import trace
    trace.build(force)          # the second oracle (spin-isospin trace, oracle/trace_oracle.c)
    return _LIB


class _Params(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in
                ("kf_n", "kf_p", "c1", "c3", "c4", "cD", "cE", "gA", "fpi", "mpi", "lambda_chi", "Lambda")] + \
               [(n, ctypes.c_int) for n in ("n_reg", "n_r", "n_cos", "n_phi")]


_DEFAULTS = dict(kf_n=0.0, kf_p=0.0, c1=0.0, c3=0.0, c4=0.0, cD=0.0, cE=0.0, gA=1.27, fpi=92.4,
                 mpi=138.04, lambda_chi=700.0, Lambda=500.0, n_reg=4, n_r=4, n_cos=4, n_phi=4)

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        pp = ctypes.POINTER(_Params)
        lib.oracle_gauss_legendre.argtypes = [ctypes.c_int, ctypes.c_double, ctypes.c_double, dp, dp]
        lib.oracle_v3n.argtypes = [pp, dp, dp]
        lib.oracle_av3n.argtypes = [pp, dp, dp, dp]
        for name in ("oracle_no_level0_ld", "oracle_no_level1_ld", "oracle_no_level1_f64"):
            getattr(lib, name).argtypes = [pp, dp, ctypes.c_longlong, dp]
            getattr(lib, name).restype = None
        for name in ("oracle_no_level1_dirs_ld", "oracle_no_level1_dirs_f64"):
            getattr(lib, name).argtypes = [pp, dp, ctypes.c_longlong, dp, ctypes.c_int, dp]
            getattr(lib, name).restype = None
        lib.oracle_hf3n_bruteforce.argtypes = [pp]
        lib.oracle_hf3n_bruteforce.restype = ctypes.c_double
        lib.oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _params(kw: dict) -> _Params:
    d = dict(_DEFAULTS)
    for k, v in kw.items():
        if k not in d:
            raise TypeError(f"unknown oracle parameter {k!r}")
        d[k] = v
    return _Params(**d)


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def gauss_legendre(n: int, a: float, b: float):
    x = np.empty(n)
    w = np.empty(n)
    _load().oracle_gauss_legendre(n, a, b, _dptr(x), _dptr(w))
    return x, w


def v3n(q, **params) -> np.ndarray:
    """Bare operator V(q1,q2,q3): complex [64,64]; index = 8*(4 s1+2 s2+s3) + (4 t1+2 t2+t3)."""
    q = np.ascontiguousarray(q, dtype=np.float64).reshape(3, 3)
    out = np.empty((64, 64, 2))
    _load().oracle_v3n(ctypes.byref(_params(params)), _dptr(q), _dptr(out))
    return out[..., 0] + 1j * out[..., 1]


def av3n(kin, kout, **params) -> np.ndarray:
    """Regulated antisymmetrised F * A_123 V for explicit momenta: complex [64,64]."""
    kin = np.ascontiguousarray(kin, dtype=np.float64).reshape(3, 3)
    kout = np.ascontiguousarray(kout, dtype=np.float64).reshape(3, 3)
    out = np.empty((64, 64, 2))
    _load().oracle_av3n(ctypes.byref(_params(params)), _dptr(kin), _dptr(kout), _dptr(out))
    return out[..., 0] + 1j * out[..., 1]


def normal_order(cfg, level: int = 1, precision: str = "ld", dirs=None, **params) -> np.ndarray:
    """M[n_cfg,16,16] complex for configurations cfg[n_cfg,9] = (p, p', P) in fm^-1; output fm^2.

    level 0 = definition (64x64 per node); level 1 = spin and isospin traced separately.
    precision "ld" = long double arithmetic (parity reference), "f64" = double (level 1 only).
    dirs: optional caller-supplied angular rule [n_dir,4] = (ux, uy, uz, w), sum w = 4 pi, used instead
    of the cos(theta) x phi Gauss-Legendre grid (level 1): radial GL x Lebedev.
    """
    cfg = np.ascontiguousarray(cfg, dtype=np.float64).reshape(-1, 9)
    n = cfg.shape[0]
    out = np.empty((n, 16, 16, 2))
    if dirs is not None:
        assert level == 1 and precision in ("ld", "f64")
        dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 4)
        if n:
            getattr(_load(), "oracle_no_level1_dirs_" + precision)(ctypes.byref(_params(params)), _dptr(cfg), n,
                                                                   _dptr(dirs), dirs.shape[0], _dptr(out))
        return out[..., 0] + 1j * out[..., 1]
    name = {(0, "ld"): "oracle_no_level0_ld", (1, "ld"): "oracle_no_level1_ld",
            (1, "f64"): "oracle_no_level1_f64"}[(level, precision)]
    if n:
        getattr(_load(), name)(ctypes.byref(_params(params)), _dptr(cfg), n, _dptr(out))
    return out[..., 0] + 1j * out[..., 1]


def hf3n_bruteforce(**params) -> float:
    """(1/6) sum_{123} <123|F A_123 V|123> on the product grid of every particle (pin P8); fm^-4."""
    return float(_load().oracle_hf3n_bruteforce(ctypes.byref(_params(params))))


def diag_trace(cfg, **params) -> np.ndarray:
    """D[n_cfg,4]: D[c, 2 t1 + t2] = sum_{s1,s2} Re M_c[a,a], a = 8 s1 + 4 s2 + 2 t1 + t2 (the integrand
    of the Hartree-Fock contractions Eq. (1), (9)): the definition, from normal_order."""
    M = normal_order(cfg, **params)
    D = np.zeros((M.shape[0], 4))
    for s1 in range(2):
        for s2 in range(2):
            for t in range(4):
                a = 8 * s1 + 4 * s2 + t
                D[:, t] += M[:, a, a].real
    return D


def sphere_nodes(n_r: int, n_cos: int, n_phi: int, kf: float):
    """Product Gauss-Legendre grid of one Fermi sphere (fixed lab frame): k[n,3], W[n] = r^2 w_r w_c w_phi/(2 pi)^3."""
    r, wr = gauss_legendre(n_r, 0.0, kf)
    x, wx = gauss_legendre(n_cos, -1.0, 1.0)
    ph, wp = gauss_legendre(n_phi, 0.0, 2.0 * np.pi)
    k, w = [], []
    for i in range(n_r):
        for j in range(n_cos):
            for l in range(n_phi):
                st = np.sqrt(1.0 - x[j] ** 2)
                k.append(r[i] * np.array([st * np.cos(ph[l]), st * np.sin(ph[l]), x[j]]))
                w.append(r[i] ** 2 * wr[i] * wx[j] * wp[l] / (2.0 * np.pi) ** 3)
    return np.array(k), np.array(w)


def hf_energy(n_r12: int, n_cos12: int, n_phi12: int, **params) -> float:
    """3N Hartree-Fock energy per volume (fm^-4) by repeated normal ordering:
    E/V = (1/6) sum_{t1 t2} sum_{k1 in S(t1)} sum_{k2 in S(t2)} W1 W2 sum_{s1 s2} M(p=(k1-k2)/2, p'=p, P=k1+k2)[a,a],
    particles 1, 2 on n_r12 x n_cos12 x n_phi12 grids, particle 3 inside M on the grid of `params`."""
    kf = {0: params.get("kf_p", 0.0), 1: params.get("kf_n", 0.0)}
    e = 0.0
    for t1 in (0, 1):
        for t2 in (0, 1):
            if kf[t1] <= 0 or kf[t2] <= 0:
                continue
            k1, w1 = sphere_nodes(n_r12, n_cos12, n_phi12, kf[t1])
            k2, w2 = sphere_nodes(n_r12, n_cos12, n_phi12, kf[t2])
            cfg = np.empty((len(k1), len(k2), 9))
            cfg[:, :, 0:3] = (k1[:, None, :] - k2[None, :, :]) / 2
            cfg[:, :, 3:6] = cfg[:, :, 0:3]
            cfg[:, :, 6:9] = k1[:, None, :] + k2[None, :, :]
            D = diag_trace(cfg.reshape(-1, 9), **params)[:, 2 * t1 + t2]
            e += float(np.sum((w1[:, None] * w2[None, :]).reshape(-1) * D))
    return e / 6.0


def sp_energy(k1, n_r12: int, n_cos12: int, n_phi12: int, **params) -> np.ndarray:
    """3N Hartree-Fock self-energy of Eq. (9), spin averaged: Sigma[n,2] (proton, neutron), fm^-1:
    Sigma_t1(k1) = (1/2) sum_{s2 t2} sum_{k2 in S(t2)} W2 (1/2) sum_{s1} M(p=(k1-k2)/2, p'=p, P=k1+k2)[a,a]."""
    k1 = np.ascontiguousarray(k1, dtype=np.float64).reshape(-1, 3)
    kf = {0: params.get("kf_p", 0.0), 1: params.get("kf_n", 0.0)}
    sig = np.zeros((k1.shape[0], 2))
    for t2 in (0, 1):
        if kf[t2] <= 0:
            continue
        k2, w2 = sphere_nodes(n_r12, n_cos12, n_phi12, kf[t2])
        cfg = np.empty((len(k1), len(k2), 9))
        cfg[:, :, 0:3] = (k1[:, None, :] - k2[None, :, :]) / 2
        cfg[:, :, 3:6] = cfg[:, :, 0:3]
        cfg[:, :, 6:9] = k1[:, None, :] + k2[None, :, :]
        D = diag_trace(cfg.reshape(-1, 9), **params).reshape(len(k1), len(k2), 4)
        for t1 in (0, 1):
            sig[:, t1] += 0.25 * np.sum(w2[None, :] * D[:, :, 2 * t1 + t2], axis=1)
    return sig


# ---- packed, symmetry-reduced form of the 16x16 matrix ----
# "only up to 4^A C(2A,A) matrix elements can be non-zero ... only a subset of the remaining matrix elements
# needs to be computed from which the entire matrix can be efficiently reconstructed."  The plain definitions
# of the two subsets the library writes, element by element.
#   format 1 ("charge"): the 96 = 4^2 C(4,2) entries with t1' + t2' = t1 + t2, as [16 spin elements][6 isospin blocks],
#       spin element sp = 4 (2 s1' + s2') + (2 s1 + s2), isospin block nb -> (row pair, column pair), pair = 2 t1 + t2:
#       (pp,pp) (pn,pn) (np,np) (nn,nn) (pn,np) (np,pn)
#   format 2 ("isospin"): isospin-symmetric matter only (kF_n = kF_p, pin P9): per spin element the two entries
#       (pn,pn) and (pn,np); the others follow from isospin invariance of the effective interaction,
#       (pp,pp) = (nn,nn) = (pn,pn) + (pn,np)   [T = 1],   (np,np) = (pn,pn),   (np,pn) = (pn,np).
PACK_CHARGE, PACK_ISOSPIN = 1, 2
PACK_BLOCKS = ((0, 0), (1, 1), (2, 2), (3, 3), (1, 2), (2, 1))     # (row isospin pair, column isospin pair)
PACKED_COMPLEX = {PACK_CHARGE: 96, PACK_ISOSPIN: 32}


def _spin_rc(sp: int):
    """row and column offsets 8 s1 + 4 s2 of spin element sp = 4 (2 s1' + s2') + (2 s1 + s2)."""
    return 4 * (sp >> 2), 4 * (sp & 3)


def pack(M, fmt: int) -> np.ndarray:
    """M[n,16,16] complex -> packed[n, 96 or 32] complex: copies the entries of the subset, nothing else."""
    M = np.asarray(M)
    out = np.zeros((M.shape[0], PACKED_COMPLEX[fmt]), dtype=complex)
    for sp in range(16):
        r0, c0 = _spin_rc(sp)
        if fmt == PACK_CHARGE:
            for nb, (to, ti) in enumerate(PACK_BLOCKS):
                out[:, 6 * sp + nb] = M[:, r0 + to, c0 + ti]
        else:
            out[:, 2 * sp + 0] = M[:, r0 + 1, c0 + 1]
            out[:, 2 * sp + 1] = M[:, r0 + 1, c0 + 2]
    return out


def unpack(P, fmt: int) -> np.ndarray:
    """packed[n, 96 or 32] complex -> M[n,16,16]: the 160 charge-violating entries are 0 (P6); format 2 fills the
    other four blocks from isospin symmetry (P9)."""
    P = np.asarray(P)
    M = np.zeros((P.shape[0], 16, 16), dtype=complex)
    for sp in range(16):
        r0, c0 = _spin_rc(sp)
        if fmt == PACK_CHARGE:
            for nb, (to, ti) in enumerate(PACK_BLOCKS):
                M[:, r0 + to, c0 + ti] = P[:, 6 * sp + nb]
        else:
            d, x = P[:, 2 * sp + 0], P[:, 2 * sp + 1]
            M[:, r0 + 1, c0 + 1] = d
            M[:, r0 + 2, c0 + 2] = d
            M[:, r0 + 1, c0 + 2] = x
            M[:, r0 + 2, c0 + 1] = x
            M[:, r0 + 0, c0 + 0] = d + x
            M[:, r0 + 3, c0 + 3] = d + x
    return M


def num_threads() -> int:
    return int(_load().oracle_num_threads())


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
