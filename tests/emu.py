"""ctypes face of tests/host_emu.cpp (lane-by-lane host emulation of the kernel's warp program)."""
import ctypes
import os
import subprocess

import numpy as np

from paper_2603_24532_b200.binding import no_params

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "host_emu.cpp")
_LIB = os.path.join(_HERE, "libhost_emu.so")
_DEPS = [_SRC] + [os.path.join(_HERE, "..", "paper_2603_24532_b200", "csrc", f) for f in ("no_core.h", "no_host.h")]
_lib = None


def load():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB) or any(os.path.getmtime(d) > os.path.getmtime(_LIB) for d in _DEPS):
            subprocess.run(["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-Wall", "-Wextra",
                            "-o", _LIB, _SRC], check=True)
        _lib = ctypes.CDLL(_LIB)
    return _lib


def emu_eval(cfg, **params):
    cfg = np.ascontiguousarray(cfg, dtype=np.float64).reshape(-1, 9)
    out = np.empty((cfg.shape[0], 16, 16, 2))
    p = no_params(device=0, **params)
    rc = load().emu_eval(ctypes.byref(p), cfg.ctypes.data_as(ctypes.c_void_p), ctypes.c_longlong(cfg.shape[0]),
                         out.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError(rc)
    return out[..., 0] + 1j * out[..., 1]


def emu_eval_angular(cfg, dirs, **params):
    cfg = np.ascontiguousarray(cfg, dtype=np.float64).reshape(-1, 9)
    dirs = np.ascontiguousarray(dirs, dtype=np.float64).reshape(-1, 4)
    out = np.empty((cfg.shape[0], 16, 16, 2))
    params = dict(params)
    params.setdefault("n_cos", 1)
    params.setdefault("n_phi", 1)
    p = no_params(device=0, **params)
    rc = load().emu_eval_angular(ctypes.byref(p), dirs.ctypes.data_as(ctypes.c_void_p), ctypes.c_int(dirs.shape[0]),
                                 cfg.ctypes.data_as(ctypes.c_void_p), ctypes.c_longlong(cfg.shape[0]),
                                 out.ctypes.data_as(ctypes.c_void_p))
    if rc != 0:
        raise ValueError(rc)
    return out[..., 0] + 1j * out[..., 1]


def emu_plan(**params):
    p = no_params(device=0, **params)
    n_pass, nreg, c4, tabn = ctypes.c_int(), ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    evals = ctypes.c_longlong()
    tab = np.zeros(4096)
    rc = load().emu_plan(ctypes.byref(p), ctypes.byref(n_pass), ctypes.byref(nreg), ctypes.byref(c4),
                         ctypes.byref(evals), ctypes.byref(tabn), tab.ctypes.data_as(ctypes.c_void_p), 4096)
    if rc != 0:
        raise ValueError(rc)
    return dict(n_pass=n_pass.value, nreg_variant=nreg.value, has_c4=c4.value, evals_per_cfg=evals.value,
                tab_doubles=tabn.value, tab=tab[:tabn.value])


def emu_gl_rule(n, lo, hi):
    x, w = np.empty(n), np.empty(n)
    load().emu_gl_rule(n, ctypes.c_double(lo), ctypes.c_double(hi), x.ctypes.data_as(ctypes.c_void_p),
                       w.ctypes.data_as(ctypes.c_void_p))
    return x, w
