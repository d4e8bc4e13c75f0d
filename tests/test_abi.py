"""The C-ABI library loads and exports every symbol include/no.h declares; argument validation
that needs no GPU.  No compute call is made here."""
import ctypes
import os
import re

import pytest

from paper_2603_24532_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def declared_symbols(header="no.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(no_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_boundary():
    syms = declared_symbols()
    for required in ("no_init", "no_eval", "no_free"):          # north_star (a)
        assert required in syms
    assert set(syms) == set(binding.EXPORTS)
    assert set(declared_symbols("no_trace.h")) == set(binding.TRACE_EXPORTS)


def test_every_declared_symbol_is_exported(lib):
    for name in declared_symbols() + declared_symbols("no_trace.h"):
        assert hasattr(lib, name), name


def test_params_struct_layout_matches_header():
    text = open(os.path.join(ROOT, "include", "no.h")).read()
    body = re.search(r"typedef struct no_params \{(.*?)\} no_params;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        typ, names = decl.split(None, 1)
        fields += [(n.strip(), typ) for n in names.split(",")]
    want = [(n, "double" if t is ctypes.c_double else "int") for n, t in binding.no_params._fields_]
    assert fields == want
    assert ctypes.sizeof(binding.no_params) == 12 * 8 + 5 * 4 + 4     # padded to 8


def test_error_strings_and_null_handling(lib):
    assert lib.no_strerror(0) == b"success"
    for code in (1, 2, 3, 4, 5, 99):
        assert len(lib.no_strerror(code)) > 0
    assert b"busy" in lib.no_strerror(binding.NO_ERR_BUSY) and b"busy" not in lib.no_strerror(binding.NO_ERR_INVALID)
    assert lib.no_free(None) == binding.NO_OK                      # NULL is a no-op
    assert lib.no_init(None, None) == binding.NO_ERR_INVALID
    assert lib.no_eval(None, None, 0, None, None) == binding.NO_ERR_INVALID
    assert lib.no_evals_per_cfg(None) == 0
    assert lib.no_trace_free(None) == binding.NO_OK
    assert lib.no_trace_init(None, 2, None, 0, 0) == binding.NO_ERR_INVALID
    assert lib.no_trace_eval(None, None, 0, None, None) == binding.NO_ERR_INVALID
    assert lib.no_trace_info(None, None, None, None, None, None, None) == binding.NO_ERR_INVALID


def test_malformed_trace_topologies_are_rejected_before_any_cuda_call(lib):
    import numpy as np
    for topo in ([[0, 1, 0, 0]],                        # a line entering twice
                 [[0, 1, 2, 3], [2, 3, 0, 4]],          # id out of range
                 [[0, 1, 2, 3], [2, 2, 0, 1]]):         # a line leaving twice
        t = np.array(topo, dtype=np.int32)
        h = ctypes.c_void_p()
        assert lib.no_trace_init(ctypes.byref(h), t.shape[0], ctypes.c_void_p(t.ctypes.data), 0, 0) == binding.NO_ERR_INVALID
        assert not h.value
    t = np.zeros((7, 4), dtype=np.int32)
    h = ctypes.c_void_p()
    assert lib.no_trace_init(ctypes.byref(h), 7, ctypes.c_void_p(t.ctypes.data), 0, 0) == binding.NO_ERR_INVALID
    t2 = np.array([[0, 1, 2, 3], [2, 3, 0, 1]], dtype=np.int32)
    assert lib.no_trace_init(ctypes.byref(h), 2, ctypes.c_void_p(t2.ctypes.data), 8, 0) == binding.NO_ERR_INVALID   # unknown flag


GOOD = dict(kf_n=1.0, kf_p=0.0, c1=-0.81, c3=-3.2, c4=0.0, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04,
            lambda_chi=700.0, Lambda=500.0, n_reg=4, n_r=16, n_cos=16, n_phi=16)


@pytest.mark.parametrize("bad", [dict(kf_n=-1.0), dict(kf_p=-0.1), dict(n_r=0), dict(n_cos=129), dict(n_phi=-3),
                                 dict(n_reg=0), dict(n_reg=13), dict(fpi=0.0), dict(mpi=-1.0),
                                 dict(c1=float("nan")), dict(Lambda=float("inf"))])
def test_invalid_parameters_are_rejected_before_any_cuda_call(lib, bad):
    p = binding.no_params(device=0, **dict(GOOD, **bad))
    h = ctypes.c_void_p()
    assert lib.no_init(ctypes.byref(h), ctypes.byref(p)) == binding.NO_ERR_INVALID
    assert not h.value


def test_product_fails_loudly_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    p = binding.no_params(device=0, **GOOD)
    h = ctypes.c_void_p()
    assert lib.no_init(ctypes.byref(h), ctypes.byref(p)) == binding.NO_ERR_CUDA
    assert len(lib.no_last_cuda_error()) > 0
    from paper_2603_24532_b200 import NormalOrdering
    with pytest.raises(RuntimeError):
        NormalOrdering(device=0, **GOOD)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2603_24532_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".h", ".cuh", ".cu", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", src, flags=re.M), f
                assert "no_oracle" not in src and "liboracle" not in src and "trace_oracle" not in src, f
