"""ctypes face of oracle/trace_oracle.c (brute-force spin-isospin trace) --
TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module; the product package never does."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "trace_oracle.c")
_LIB = os.path.join(_HERE, "libtrace_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.run(["gcc", "-O2", "-std=c99", "-fopenmp", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", _LIB, _SRC],
                       check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_trace_bruteforce.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                                ctypes.c_void_p]
        lib.oracle_trace_bruteforce.restype = ctypes.c_int
        lib.oracle_trace_isospin_configs.argtypes = [ctypes.c_int, ctypes.c_void_p]
        lib.oracle_trace_isospin_configs.restype = ctypes.c_longlong
        _lib = lib
    return _lib


def _topo(topo) -> np.ndarray:
    t = np.ascontiguousarray(topo, dtype=np.int32).reshape(-1, 4)
    n = t.shape[0]
    # every line id 0..2n-1 leaves exactly one vertex and enters exactly one vertex
    assert sorted(t[:, :2].reshape(-1).tolist()) == list(range(2 * n)), "outgoing slots must use every line once"
    assert sorted(t[:, 2:].reshape(-1).tolist()) == list(range(2 * n)), "incoming slots must use every line once"
    return t


def trace_bruteforce(topo, V) -> np.ndarray:
    """T[n_sample] complex: sum over the spin and isospin labels of all 2 n lines of prod_v V_v[out pair][in pair].
    topo [n,4] = line ids (out1, out2, in1, in2) per vertex; V [n_sample, n, 16, 16] complex."""
    t = _topo(topo)
    V = np.asarray(V, dtype=complex)
    assert V.ndim == 4 and V.shape[1:] == (t.shape[0], 16, 16)
    Vd = np.ascontiguousarray(np.stack([V.real, V.imag], axis=-1))
    out = np.zeros((V.shape[0], 2))
    rc = _load().oracle_trace_bruteforce(t.shape[0], t.ctypes.data, Vd.ctypes.data, V.shape[0], out.ctypes.data)
    assert rc == 0
    return out[:, 0] + 1j * out[:, 1]


def isospin_configs(topo) -> int:
    """number of isospin assignments of the lines that conserve charge at every vertex."""
    t = _topo(topo)
    return int(_load().oracle_trace_isospin_configs(t.shape[0], t.ctypes.data))
