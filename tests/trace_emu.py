"""ctypes face of tests/trace_emu.cpp (host emulation of the trace kernel's planned step program)."""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "trace_emu.cpp")
_LIB = os.path.join(_HERE, "libtrace_emu.so")
_DEPS = [_SRC, os.path.join(_HERE, "..", "paper_2603_24532_b200", "csrc", "no_trace_host.h")]
_lib = None


def load():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB) or any(os.path.getmtime(d) > os.path.getmtime(_LIB) for d in _DEPS):
            subprocess.run(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-Wall", "-Wextra", "-o", _LIB, _SRC], check=True)
        _lib = ctypes.CDLL(_LIB)
    return _lib


def plan(topo, charge=False):
    t = np.ascontiguousarray(topo, dtype=np.int32).reshape(-1, 4)
    info = np.zeros(30, dtype=np.int64)
    rc = load().trace_emu_plan(t.shape[0], ctypes.c_void_p(t.ctypes.data), int(charge), ctypes.c_void_p(info.ctypes.data))
    if rc != 0:
        return None
    n = t.shape[0]
    return dict(cmacs=int(info[0]), max_open=int(info[1]), n_sliced=int(info[2]), n_isospin=int(info[3]),
                n_slice_iter=int(info[4]), order=info[5:5 + n].tolist(), dmma_products=int(info[29]),
                steps=[tuple(int(x) for x in info[11 + 3 * k:14 + 3 * k]) for k in range(n)])


def evaluate(topo, V, charge=False):
    t = np.ascontiguousarray(topo, dtype=np.int32).reshape(-1, 4)
    V = np.asarray(V, dtype=complex)
    Vd = np.ascontiguousarray(np.stack([V.real, V.imag], axis=-1))
    out = np.zeros((V.shape[0], 2))
    rc = load().trace_emu_eval(t.shape[0], ctypes.c_void_p(t.ctypes.data), int(charge), ctypes.c_void_p(Vd.ctypes.data),
                               ctypes.c_longlong(V.shape[0]), ctypes.c_void_p(out.ctypes.data))
    if rc != 0:
        raise ValueError("topology rejected")
    return out[:, 0] + 1j * out[:, 1]
