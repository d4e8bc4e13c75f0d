"""Thin ctypes binding of libno3n.so: the same names as include/no.h, argument marshalling only.

PyTorch is used by callers for device memory and streams; every step of the hot path runs in the
CUDA kernels behind no_eval.  There is no CPU fallback: if the library is missing or no CUDA
device is present the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libno3n.so")

NO_OK, NO_ERR_INVALID, NO_ERR_CUDA, NO_ERR_ALLOC, NO_ERR_LIMIT, NO_ERR_BUSY = 0, 1, 2, 3, 4, 5

EXPORTS = ("no_init", "no_init_angular", "no_eval", "no_eval_host", "no_eval_diag", "no_hf_energy", "no_sp_energy", "no_set_layout", "no_free", "no_strerror", "no_last_cuda_error",
           "no_kernel_info", "no_evals_per_cfg", "no_probe_fp64_peak",
           "no_packed_doubles", "no_eval_packed", "no_unpack", "no_eval_host_packed", "no_probe_fp64_operands",
           "no_hf_energy_static", "no_set_max_grid")

NO_PACK_CHARGE, NO_PACK_ISOSPIN = 1, 2
NO_PACK_FORWARD = 0x100      # flag ORed into the format of no_eval_packed: every configuration has p' == p (include/no.h)

TRACE_EXPORTS = ("no_trace_init", "no_trace_eval", "no_trace_eval_packed", "no_trace_info", "no_trace_free",
                 "no_trace_last_cuda_error")


class no_params(ctypes.Structure):
    """struct no_params of include/no.h."""
    _fields_ = [(n, ctypes.c_double) for n in
                ("kf_n", "kf_p", "c1", "c3", "c4", "cD", "cE", "gA", "fpi", "mpi", "lambda_chi", "Lambda")] + \
               [(n, ctypes.c_int) for n in ("n_reg", "n_r", "n_cos", "n_phi", "device")]


class NoError(RuntimeError):
    def __init__(self, code: int, where: str):
        lib = load()
        msg = lib.no_strerror(code).decode()
        cuda = lib.no_last_cuda_error().decode()
        super().__init__(f"{where}: {msg}" + (f" [{cuda}]" if code == NO_ERR_CUDA and cuda else ""))
        self.code = code


_lib = None


def load() -> ctypes.CDLL:
    """dlopen libno3n.so (built by `python -m paper_2603_24532_b200.build`); fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2603_24532_b200.build` "
                               "(the package has no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        H = ctypes.c_void_p
        lib.no_init.argtypes = [ctypes.POINTER(H), ctypes.POINTER(no_params)]
        lib.no_init_angular.argtypes = [ctypes.POINTER(H), ctypes.POINTER(no_params), ctypes.c_void_p, ctypes.c_int]
        lib.no_eval.argtypes = [H, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.no_eval_host.argtypes = [H, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.no_eval_diag.argtypes = [H, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.no_hf_energy.argtypes = [H, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                     ctypes.c_void_p]
        lib.no_hf_energy_static.argtypes = lib.no_hf_energy.argtypes
        lib.no_hf_energy_static.restype = ctypes.c_int
        lib.no_sp_energy.argtypes = [H, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_void_p, ctypes.c_void_p]
        lib.no_set_layout.argtypes = [H, ctypes.c_int]
        lib.no_set_max_grid.argtypes = [H, ctypes.c_longlong]
        lib.no_set_max_grid.restype = ctypes.c_int
        lib.no_packed_doubles.argtypes = [H, ctypes.c_int]
        lib.no_eval_packed.argtypes = [H, ctypes.c_int, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.no_unpack.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.no_eval_host_packed.argtypes = [H, ctypes.c_int, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p,
                                            ctypes.c_void_p]
        lib.no_free.argtypes = [H]
        lib.no_strerror.argtypes = [ctypes.c_int]
        lib.no_strerror.restype = ctypes.c_char_p
        lib.no_last_cuda_error.restype = ctypes.c_char_p
        ip = ctypes.POINTER(ctypes.c_int)
        lib.no_kernel_info.argtypes = [H, ip, ip, ip, ip, ip, ip]
        lib.no_evals_per_cfg.argtypes = [H]
        lib.no_evals_per_cfg.restype = ctypes.c_longlong
        lib.no_probe_fp64_peak.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double), ip,
                                           ctypes.c_void_p]
        for name in ("no_init", "no_init_angular", "no_eval", "no_eval_host", "no_eval_diag", "no_hf_energy", "no_sp_energy", "no_set_layout", "no_free", "no_kernel_info",
                     "no_probe_fp64_peak", "no_packed_doubles", "no_eval_packed", "no_unpack", "no_eval_host_packed"):
            getattr(lib, name).restype = ctypes.c_int
        lib.no_probe_fp64_operands.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double),
                                               ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]
        lib.no_probe_fp64_operands.restype = ctypes.c_int
        lib.no_trace_init.argtypes = [ctypes.POINTER(H), ctypes.c_int, ctypes.c_void_p, ctypes.c_int, ctypes.c_int]
        lib.no_trace_eval.argtypes = [H, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]
        lib.no_trace_eval_packed.argtypes = [H, ctypes.c_int, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p,
                                             ctypes.c_void_p]
        lib.no_trace_eval_packed.restype = ctypes.c_int
        lib.no_trace_info.argtypes = [H, ctypes.POINTER(ctypes.c_longlong), ip, ip, ctypes.POINTER(ctypes.c_longlong), ip,
                                      ctypes.POINTER(ctypes.c_longlong)]
        lib.no_trace_free.argtypes = [H]
        lib.no_trace_last_cuda_error.restype = ctypes.c_char_p
        for name in ("no_trace_init", "no_trace_eval", "no_trace_info", "no_trace_free"):
            getattr(lib, name).restype = ctypes.c_int
        _lib = lib
    return _lib


def no_init(device: int = 0, angular=None, **params) -> ctypes.c_void_p:
    """no_init: keyword arguments are the fields of struct no_params; returns the opaque handle.
    angular: optional host array [n_dir, 4] = (ux, uy, uz, w) -> no_init_angular (n_cos, n_phi default to 1)."""
    if angular is None:
        p = no_params(device=device, **params)
        h = ctypes.c_void_p()
        rc = load().no_init(ctypes.byref(h), ctypes.byref(p))
        if rc != NO_OK:
            raise NoError(rc, "no_init")
        return h
    import numpy as np
    dirs = np.ascontiguousarray(angular, dtype=np.float64).reshape(-1, 4)
    params = dict(params)
    params.setdefault("n_cos", 1)
    params.setdefault("n_phi", 1)
    p = no_params(device=device, **params)
    h = ctypes.c_void_p()
    rc = load().no_init_angular(ctypes.byref(h), ctypes.byref(p), ctypes.c_void_p(dirs.ctypes.data), dirs.shape[0])
    if rc != NO_OK:
        raise NoError(rc, "no_init_angular")
    return h


def no_eval(h, d_cfg_ptr: int, n_cfg: int, d_out_ptr: int, stream_ptr: Optional[int] = None) -> None:
    """no_eval with raw DEVICE pointers (e.g. tensor.data_ptr()) and a cudaStream_t value."""
    rc = load().no_eval(h, ctypes.c_void_p(d_cfg_ptr), n_cfg, ctypes.c_void_p(d_out_ptr),
                        ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_eval")


def no_eval_host(h, h_cfg_ptr: int, n_cfg: int, h_out_ptr: int, stream_ptr: Optional[int] = None) -> None:
    """no_eval_host with raw HOST pointers; synchronises the stream before returning."""
    rc = load().no_eval_host(h, ctypes.c_void_p(h_cfg_ptr), n_cfg, ctypes.c_void_p(h_out_ptr),
                             ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_eval_host")


def no_eval_diag(h, d_cfg_ptr: int, n_cfg: int, d_out_ptr: int, stream_ptr: Optional[int] = None) -> None:
    """no_eval_diag with raw DEVICE pointers: d_out is [n_cfg][4] doubles."""
    rc = load().no_eval_diag(h, ctypes.c_void_p(d_cfg_ptr), n_cfg, ctypes.c_void_p(d_out_ptr),
                             ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_eval_diag")


def no_packed_doubles(h, fmt: int) -> int:
    """doubles per configuration of packed format fmt for this handle (0: the format does not apply)."""
    return int(load().no_packed_doubles(h, fmt))


def no_eval_packed(h, fmt: int, d_cfg_ptr: int, n_cfg: int, d_packed_ptr: int, stream_ptr: Optional[int] = None) -> None:
    """no_eval_packed with raw DEVICE pointers: d_packed is [n_cfg][no_packed_doubles(h, fmt)] doubles."""
    rc = load().no_eval_packed(h, fmt, ctypes.c_void_p(d_cfg_ptr), n_cfg, ctypes.c_void_p(d_packed_ptr),
                               ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_eval_packed")


def no_unpack(fmt: int, d_packed_ptr: int, n_cfg: int, d_out_ptr: int, stream_ptr: Optional[int] = None) -> None:
    """no_unpack with raw DEVICE pointers: packed -> [n_cfg][16][16][2]."""
    rc = load().no_unpack(fmt, ctypes.c_void_p(d_packed_ptr), n_cfg, ctypes.c_void_p(d_out_ptr),
                          ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_unpack")


def no_eval_host_packed(h, fmt: int, h_cfg_ptr: int, n_cfg: int, h_packed_ptr: int,
                        stream_ptr: Optional[int] = None) -> None:
    """no_eval_host_packed with raw HOST pointers; synchronises the stream before returning."""
    rc = load().no_eval_host_packed(h, fmt, ctypes.c_void_p(h_cfg_ptr), n_cfg, ctypes.c_void_p(h_packed_ptr),
                                    ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_eval_host_packed")


def no_hf_energy(h, n_r: int, n_cos: int, n_phi: int, stream_ptr: Optional[int] = None) -> float:
    """no_hf_energy: 3N Hartree-Fock energy per volume in fm^-4 (synchronises the stream)."""
    e = ctypes.c_double(0.0)
    rc = load().no_hf_energy(h, n_r, n_cos, n_phi, ctypes.byref(e), ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_hf_energy")
    return float(e.value)


def no_hf_energy_static(h, n_r: int, n_cos: int, n_phi: int, stream_ptr: Optional[int] = None) -> float:
    """no_hf_energy_static: no_hf_energy without any GPU allocation (intermediates in the library's fixed 7.25 MiB
    device array; n_r * n_cos * n_phi <= 4096, NO_ERR_LIMIT beyond).  Synchronises the stream."""
    e = ctypes.c_double(0.0)
    rc = load().no_hf_energy_static(h, n_r, n_cos, n_phi, ctypes.byref(e), ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_hf_energy_static")
    return float(e.value)


def no_sp_energy(h, k1, n_r: int, n_cos: int, n_phi: int, stream_ptr: Optional[int] = None):
    """no_sp_energy: k1 host array [n,3] -> Sigma[n,2] (proton, neutron) in fm^-1 (synchronises the stream)."""
    import numpy as np
    k1 = np.ascontiguousarray(k1, dtype=np.float64).reshape(-1, 3)
    out = np.zeros((k1.shape[0], 2))
    rc = load().no_sp_energy(h, ctypes.c_void_p(k1.ctypes.data), k1.shape[0], n_r, n_cos, n_phi,
                             ctypes.c_void_p(out.ctypes.data), ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_sp_energy")
    return out


def no_set_max_grid(h, max_ctas: int) -> None:
    """test hook: cap the CTAs per launch of this handle (0 = hardware limit), include/no.h."""
    rc = load().no_set_max_grid(h, max_ctas)
    if rc != NO_OK:
        raise NoError(rc, "no_set_max_grid")


def no_set_layout(h, layout: int) -> None:
    """0 automatic, 1 one warp per configuration, 2 one CTA per configuration (include/no.h)."""
    rc = load().no_set_layout(h, layout)
    if rc != NO_OK:
        raise NoError(rc, "no_set_layout")


def no_free(h) -> None:
    rc = load().no_free(h)
    if rc != NO_OK:
        raise NoError(rc, "no_free")


def no_kernel_info(h) -> dict:
    v = [ctypes.c_int() for _ in range(6)]
    rc = load().no_kernel_info(h, *[ctypes.byref(x) for x in v])
    if rc != NO_OK:
        raise NoError(rc, "no_kernel_info")
    keys = ("regs", "smem_bytes", "threads", "ctas_per_sm", "n_sm", "cfg_per_cta")
    return {k: x.value for k, x in zip(keys, v)}


def no_evals_per_cfg(h) -> int:
    return int(load().no_evals_per_cfg(h))


def no_probe_fp64_peak(device: int = 0, millis: int = 200, stream_ptr: Optional[int] = None) -> dict:
    t = ctypes.c_double()
    n = ctypes.c_int()
    rc = load().no_probe_fp64_peak(device, millis, ctypes.byref(t), ctypes.byref(n), ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_probe_fp64_peak")
    return {"tflops": t.value, "n_sm": n.value}


def no_probe_fp64_operands(device: int = 0, millis: int = 100, stream_ptr: Optional[int] = None) -> dict:
    """DFMA rate (TFLOP/s) with two and with three fresh register operands per instruction (include/no.h)."""
    a, b = ctypes.c_double(), ctypes.c_double()
    rc = load().no_probe_fp64_operands(device, millis, ctypes.byref(a), ctypes.byref(b), ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_probe_fp64_operands")
    return {"two_operands_tflops": a.value, "three_operands_tflops": b.value}


# ---- include/no_trace.h: spin-isospin trace of a closed diagram ----
NO_TRACE_CHARGE_CONSERVING = 1


def no_trace_init(topo, device: int = 0, flags: int = 0) -> ctypes.c_void_p:
    """no_trace_init: topo host int array [n_vertex, 4] = line ids (out 1, out 2, in 1, in 2); returns the plan.
    flags: 0 or NO_TRACE_CHARGE_CONSERVING (vertex matrices exactly zero outside the 96 charge-conserving entries)."""
    import numpy as np
    t = np.ascontiguousarray(topo, dtype=np.int32).reshape(-1, 4)
    h = ctypes.c_void_p()
    rc = load().no_trace_init(ctypes.byref(h), t.shape[0], ctypes.c_void_p(t.ctypes.data), flags, device)
    if rc != NO_OK:
        raise NoError(rc, "no_trace_init")
    return h


def no_trace_eval(plan, d_vertices_ptr: int, n_sample: int, d_out_ptr: int, stream_ptr: Optional[int] = None) -> None:
    """no_trace_eval with raw DEVICE pointers: vertices [n_sample][n_vertex][16][16][2], out [n_sample][2]."""
    rc = load().no_trace_eval(plan, ctypes.c_void_p(d_vertices_ptr), n_sample, ctypes.c_void_p(d_out_ptr),
                              ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_trace_eval")


def no_trace_eval_packed(plan, fmt: int, d_packed_ptr: int, n_sample: int, d_out_ptr: int,
                         stream_ptr: Optional[int] = None) -> None:
    """no_trace_eval_packed with raw DEVICE pointers: packed vertices [n_sample][n_vertex][96][2] (NO_PACK_CHARGE)."""
    rc = load().no_trace_eval_packed(plan, fmt, ctypes.c_void_p(d_packed_ptr), n_sample, ctypes.c_void_p(d_out_ptr),
                                     ctypes.c_void_p(stream_ptr or 0))
    if rc != NO_OK:
        raise NoError(rc, "no_trace_eval_packed")


def no_trace_info(plan, n_vertex: int) -> dict:
    cm, iso, tp = ctypes.c_longlong(), ctypes.c_longlong(), ctypes.c_longlong()
    mo, ns = ctypes.c_int(), ctypes.c_int()
    order = (ctypes.c_int * 8)()
    rc = load().no_trace_info(plan, ctypes.byref(cm), ctypes.byref(mo), ctypes.byref(ns), ctypes.byref(iso), order,
                              ctypes.byref(tp))
    if rc != NO_OK:
        raise NoError(rc, "no_trace_info")
    return {"cmacs_per_sample": cm.value, "max_open": mo.value, "n_sliced": ns.value, "n_isospin_configs": iso.value,
            "order": [order[i] for i in range(n_vertex)], "tensor_products_per_sample": tp.value}


def no_trace_free(plan) -> None:
    rc = load().no_trace_free(plan)
    if rc != NO_OK:
        raise NoError(rc, "no_trace_free")
