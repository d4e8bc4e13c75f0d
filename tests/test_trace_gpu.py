"""Parity of the CUDA spin-isospin trace (no_trace_* of libno3n.so, through the C ABI) with the brute-force oracle
(oracle/trace_oracle.c: the "unoptimized trace" of PAPER.md:653) on the same seeded inputs.  All tests need a B200.

Tolerance: both sides sum the same <= 4^(2n) products in different orders; with entries of magnitude <= sqrt(2) the
result of a sample carries an absolute error of a few eps times the sum of the term magnitudes, which for random
phases is ~ sqrt(number of terms) times larger than |T| at worst.  Written below: |got - want| <= 1e-11 max(|want|,
1e-3 rms of the batch)."""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O                                   # noqa: E402
from oracle import trace as T                                    # noqa: E402
from paper_2603_24532_b200 import NormalOrdering, SpinIsospinTrace, binding, build, trace_workloads as TW, workloads as W   # noqa: E402

pytestmark = pytest.mark.gpu
TOL = 1e-11


@pytest.fixture(scope="module", autouse=True)
def _built():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    build.build()
    binding.load()


def check(got, want, label=""):
    floor = 1e-3 * np.sqrt(np.mean(np.abs(want) ** 2)) if len(want) else 0.0
    err = np.abs(got - want) / np.maximum(np.abs(want), floor)
    worst = err.max() if len(err) else 0.0
    assert worst < TOL, f"{label}: max rel err {worst:.3e}"
    return worst


def gpu_trace(topo, V, charge=False):
    tr = SpinIsospinTrace(topo, charge_conserving=charge)
    out = tr(torch.from_numpy(V).cuda())
    torch.cuda.synchronize()
    info = tr.info()
    tr.close()
    return out.cpu().numpy(), info


def complete5():
    n = 5
    outs = {v: [] for v in range(n)}
    ins = {v: [] for v in range(n)}
    line = 0
    for a in range(n):
        for b in range(a + 1, n):
            src, dst = (a, b) if (a + b) % 2 else (b, a)
            outs[src].append(line); ins[dst].append(line); line += 1
    return np.array([outs[v] + ins[v] for v in range(n)], dtype=np.int32)


TOPOS = ([(f"ladder{n}", TW.ladder(n)) for n in (1, 2, 3, 4, 5, 6)] + [(f"ring{n}", TW.ring(n)) for n in (2, 3, 4, 5, 6)] +
         [("ladder5x", TW.exchange_slots(TW.ladder(5), out_mask=0b01010, in_mask=0b00110)),
          ("ring5x", TW.relabel(TW.exchange_slots(TW.ring(5), out_mask=0b10001), 3)),
          ("complete5", complete5())] +
         [(f"random{n}_{s}", TW.random_closed(n, s)) for n in (2, 3, 4, 5) for s in range(4)] +
         [(f"random6_{s}", TW.random_closed(6, s)) for s in range(2)])


@pytest.mark.parametrize("name,topo", TOPOS)
def test_trace_matches_the_unoptimized_trace(name, topo):
    n = len(topo)
    n_sample = 37 if n <= 5 else 5
    for dense in (False, True):
        V = TW.vertex_matrices(n_sample, n, seed=4, stream=n + 100 * dense, dense=dense)
        got, info = gpu_trace(topo, V)
        want = T.trace_bruteforce(topo, V)
        worst = check(got, want, f"{name} dense={dense}")
        if not dense:
            # plan for charge-conserving vertices (NO_TRACE_CHARGE_CONSERVING): structurally zero blocks skipped
            got_c, info_c = gpu_trace(topo, V, charge=True)
            worst = max(worst, check(got_c, want, f"{name} charge-conserving plan"))
            assert info_c["tensor_products_per_sample"] <= info["tensor_products_per_sample"]
    assert info["n_isospin_configs"] == T.isospin_configs(topo)
    print(f"{name}: {info}, max rel err {worst:.2e}")


@pytest.mark.parametrize("n_sample", [0, 1, 2, 31, 149, 2500])
def test_ragged_batches_persistent_warps_and_reproducibility(n_sample):
    topo = TW.ring(4)
    V = TW.vertex_matrices(max(n_sample, 1), 4, seed=5)[:n_sample]
    tr = SpinIsospinTrace(topo)
    d_V = torch.from_numpy(V).cuda()
    out = tr(d_V)
    torch.cuda.synchronize()
    want = T.trace_bruteforce(topo, V) if n_sample else np.zeros(0, complex)
    check(out.cpu().numpy(), want, f"n={n_sample}")
    if n_sample:
        # bit reproducible: same bits on another stream, and for the same sample at another position of the batch
        s2 = torch.cuda.Stream()
        out2 = torch.empty_like(out)
        s2.wait_stream(torch.cuda.current_stream())
        tr.eval_into(d_V, out2, stream=s2)
        s2.synchronize()
        assert torch.equal(out, out2)
        rev = tr(torch.flip(d_V, dims=[0]).contiguous())
        assert torch.equal(torch.flip(rev, dims=[0]), out)
    tr.close()


@pytest.mark.parametrize("name,topo", [("ring5", TW.ring(5)), ("ladder4", TW.ladder(4)), ("ladder2", TW.ladder(2)),
                                       ("complete5", complete5()), ("random4_1", TW.random_closed(4, 1))])
@pytest.mark.parametrize("charge_plan", [False, True])
def test_packed_vertex_input_gives_the_same_trace(name, topo, charge_plan):
    """no_trace_eval_packed reads the 96-entry form no_eval_packed writes; several samples per warp so
    that the re-zeroing of the aliased slot between samples is exercised; the packing itself is checked against the
    oracle's definition of the format"""
    n = len(topo)
    n_sample = 3000
    V = TW.vertex_matrices(n_sample, n, seed=8, stream=n)
    P = TW.pack_charge(V)
    assert np.array_equal(P.reshape(-1, 96), O.pack(V.reshape(-1, 16, 16), O.PACK_CHARGE))
    tr = SpinIsospinTrace(topo, charge_conserving=charge_plan)
    full = tr(torch.from_numpy(V).cuda())
    packed = tr.from_packed(torch.from_numpy(P).cuda())
    torch.cuda.synchronize()
    assert torch.equal(full, packed)
    idx = np.arange(0, n_sample, 97)
    check(packed.cpu().numpy()[idx], T.trace_bruteforce(topo, V[idx]), f"{name} packed input")
    # isospin form: vertices of the form A + B tau_1.tau_2 (what SNM normal ordering gives); the kernel rebuilds the
    # matrix as the oracle's unpack does
    Pi = np.ascontiguousarray(P.reshape(n_sample, n, 16, 6)[..., [1, 4]].reshape(n_sample, n, 32))
    Vi = O.unpack(Pi.reshape(-1, 32), O.PACK_ISOSPIN).reshape(n_sample, n, 16, 16)
    from_iso = tr.from_packed(torch.from_numpy(Pi).cuda(), binding.NO_PACK_ISOSPIN)
    ref_iso = tr(torch.from_numpy(np.ascontiguousarray(Vi)).cuda())
    torch.cuda.synchronize()
    assert torch.equal(from_iso, ref_iso)
    check(from_iso.cpu().numpy()[idx], T.trace_bruteforce(topo, Vi[idx]), f"{name} isospin-packed input")
    lib = binding.load()
    assert lib.no_trace_eval_packed(tr._p, 3, None, 0, None, None) == binding.NO_ERR_INVALID
    tr.close()


def test_trace_abi_argument_checks():
    lib = binding.load()
    topo = TW.ladder(3)
    p = binding.no_trace_init(topo)
    V = torch.zeros((4, 3, 16, 16), dtype=torch.complex128, device="cuda")
    out = torch.zeros((4,), dtype=torch.complex128, device="cuda")
    vp = ctypes.c_void_p
    assert lib.no_trace_eval(p, vp(V.data_ptr()), -1, vp(out.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_trace_eval(p, None, 4, vp(out.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_trace_eval(p, vp(V.data_ptr() + 8), 4, vp(out.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_trace_eval(p, vp(V.data_ptr()), 4, vp(out.data_ptr() + 8), None) == binding.NO_ERR_INVALID
    assert lib.no_trace_eval(p, None, 0, None, None) == binding.NO_OK
    assert lib.no_trace_eval(p, vp(V.data_ptr()), 4, vp(out.data_ptr()), None) == binding.NO_OK
    torch.cuda.synchronize()
    assert float(out.abs().sum()) == 0.0
    h = ctypes.c_void_p()
    t = np.ascontiguousarray(topo)
    assert lib.no_trace_init(ctypes.byref(h), 3, vp(t.ctypes.data), 0, 99) == binding.NO_ERR_INVALID
    binding.no_trace_free(p)
    # NaN in one sample stays in that sample (both kinds of plan)
    Vn = TW.vertex_matrices(6, 3, seed=6)
    Vn[2, 1, 0, 0] = np.nan
    for charge in (False, True):
        got, _ = gpu_trace(topo, Vn, charge=charge)
        assert np.isnan(got[2]) and np.isfinite(np.delete(got, 2)).all()


def test_normal_ordering_feeds_the_trace_on_the_device():
    """the data structure is shared: no_eval output of n x n_sample configurations IS the vertex array of n_sample
    samples.  Both pipelines run independently (CUDA: no_eval -> no_trace_eval; oracle: normal_order -> brute force)."""
    n, n_sample = 3, 6
    run = W.workload("cfg3").runs[0].shrunk(n * n_sample, 6)
    cfg = W.momentum_configurations(21, 0, n * n_sample, 1.5, 2.0 * run.kf_n)
    no = NormalOrdering(device=0, **run.params())
    M = no(torch.from_numpy(cfg).cuda())                      # [n n_sample, 16, 16] complex
    topo = TW.ring(n)
    tr = SpinIsospinTrace(topo, charge_conserving=True)       # no_eval writes exact zeros outside the 96 entries
    got = tr(M.reshape(n_sample, n, 16, 16)).cpu().numpy()
    torch.cuda.synchronize()
    want = T.trace_bruteforce(topo, O.normal_order(cfg, **run.params()).reshape(n_sample, n, 16, 16))
    err = np.abs(got - want) / np.maximum(np.abs(want), 1e-3 * np.sqrt(np.mean(np.abs(want) ** 2)))
    assert err.max() < 1e-9, err.max()       # n factors, each within 1e-10 of the oracle's matrix
    # the packed hand-over: no_eval_packed -> no_trace_eval_packed, same bits
    Pk = no.packed(torch.from_numpy(cfg).cuda(), binding.NO_PACK_CHARGE)
    got_p = tr.from_packed(Pk.reshape(n_sample, n, 96)).cpu().numpy()
    assert np.array_equal(got_p, got)
    # cfg3 is symmetric matter: the 512-byte isospin form carries the same information (pp = nn = pn,pn + pn,np to rounding)
    Pi = no.packed(torch.from_numpy(cfg).cuda(), binding.NO_PACK_ISOSPIN)
    got_i = tr.from_packed(Pi.reshape(n_sample, n, 32), binding.NO_PACK_ISOSPIN).cpu().numpy()
    err_i = np.abs(got_i - want) / np.maximum(np.abs(want), 1e-3 * np.sqrt(np.mean(np.abs(want) ** 2)))
    assert err_i.max() < 1e-9, err_i.max()
    no.close(); tr.close()


def test_bench_size_launch_sampled_against_the_oracle():
    """the launch bench.py --workload trace5 times (fifth-order ring, 2^18 samples), sampled outputs vs the oracle"""
    from bench import TRACE_BENCH
    topo = TW.ring(TRACE_BENCH["n_vertex"])
    n_sample = TRACE_BENCH["n_sample"]
    V = TW.vertex_matrices(n_sample, 5, seed=TRACE_BENCH["seed"])
    tr = SpinIsospinTrace(topo, charge_conserving=True)       # as bench.py runs it
    d_V = torch.from_numpy(V).cuda()
    out = tr(d_V).cpu().numpy()
    torch.cuda.synchronize()
    assert np.isfinite(out.view(np.float64)).all()
    dense_plan = SpinIsospinTrace(topo)
    out_d = dense_plan(d_V).cpu().numpy()
    assert np.abs(out - out_d).max() <= 1e-12 * np.abs(out_d).max()      # both plans, every sample
    dense_plan.close()
    idx = sorted(set(list(range(32)) + [int(i) for i in np.linspace(0, n_sample - 1, 33)]))
    worst = check(out[idx], T.trace_bruteforce(topo, V[idx]), "trace5 bench launch")
    print(f"trace5: {n_sample} samples, {len(idx)} compared, max rel err {worst:.2e}, plan {tr.info()}")
    tr.close()
