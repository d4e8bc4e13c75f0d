"""Parity of the CUDA path (libno3n.so through the C ABI) with the CPU oracle, element by element on
the same seeded inputs.  Tolerance (north_star, BASELINE.json): maximum relative error 1e-10 on every
element whose magnitude exceeds 1e-12 of its matrix maximum; structural zeros must be below that floor.
All tests here need a B200 (`-m gpu`)."""
import ctypes
import os

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import oracle as O                                   # noqa: E402
from paper_2603_24532_b200 import NormalOrdering, binding, build, workloads as W   # noqa: E402

pytestmark = pytest.mark.gpu

REL_TOL = 1e-10
MAG_FLOOR = 1e-12
PHYS = dict(c1=-0.81, c3=-3.2, c4=0.0, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0,
            Lambda=500.0, n_reg=4)


@pytest.fixture(scope="module", autouse=True)
def _built():
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    build.build()
    binding.load()


_last = {}


def gpu_eval(cfg, **params):
    """Result of the throughput layout (one warp per configuration).  The small-batch layout (one CTA per
    configuration) and the automatic choice are run too and kept for check_parity, so every parity case
    below covers both kernels element by element."""
    d_cfg = torch.from_numpy(np.ascontiguousarray(cfg)).cuda()
    res = []
    for layout in (0, 1, 2):
        no = NormalOrdering(device=0, layout=layout, **params)
        out = no(d_cfg)
        torch.cuda.synchronize()
        res.append(out.cpu().numpy())
        no.close()
    assert np.array_equal(res[0], res[1], equal_nan=True) or np.array_equal(res[0], res[2], equal_nan=True)
    _last.update(main=res[1], split=res[2])
    return res[1]


def _check(got, want, label):
    mx = np.abs(want).max(axis=(1, 2), keepdims=True)
    mask = np.abs(want) > MAG_FLOOR * mx
    rel = np.abs(got - want)[mask] / np.abs(want)[mask]
    worst = rel.max() if rel.size else 0.0
    assert worst < REL_TOL, f"{label}: max rel err {worst:.3e}"
    floor = np.broadcast_to(MAG_FLOOR * mx, got.shape)
    assert (np.abs(got)[~mask] <= floor[~mask]).all(), f"{label}: structural zero above the floor"
    return worst


def check_parity(got, want, label=""):
    worst = _check(got, want, label)
    if got is _last.get("main"):
        worst = max(worst, _check(_last["split"], want, label + " [one CTA per configuration]"))
    return worst


def sample_indices(n, k):
    """first k/2 and k/2 evenly strided configurations."""
    head = list(range(min(k // 2, n)))
    m = k - len(head)
    stride = [int(i) for i in np.linspace(0, n - 1, m + 1)[1:]] if n > len(head) and m > 0 else []   # ends at n - 1
    return sorted(set(head + stride))


# ----------------------------------------------------------------------------------------------
# config 1 in full; configs 2-5 at full size with sampled outputs; extra c4 case (R2)
# ----------------------------------------------------------------------------------------------
def test_cfg1_all_configurations():
    run = W.workload("cfg1").runs[0]
    cfg = run.configurations()
    got = gpu_eval(cfg, **run.params())
    want = O.normal_order(cfg, **run.params())
    worst = check_parity(got, want, "cfg1")
    nn = [3, 7, 11, 15]
    assert np.abs(got[:, nn][:, :, nn]).max() > 0            # c1/c3 survive in the nn block of PNM
    print(f"cfg1: 256 configurations, max rel err {worst:.2e}")


FULL_SIZE = [("cfg2", 16), ("cfg3", 32), ("cfg4", 32), ("cfg5", 16), ("paper", 64)]


def device_invariants(no, d_cfg, out, label, chunk=1 << 16):
    """Any-size properties of a whole launch, checked on ALL its matrices with torch reductions on the device (two
    more launches of the same size): every value finite; the 160 charge-violating entries exactly zero (P6);
    Hermiticity M(p, p', P) = M(p', p, P)^dagger (P4); antisymmetry P12 M(p, -p', P) = -M(p, p', P) (P5), the last
    two to 1e-12 of each matrix maximum.  `out` is the [n, 16, 16, 2] result of `no` on `d_cfg`."""
    n = out.shape[0]
    assert bool(torch.isfinite(out).all()), label
    idx = torch.arange(16, device=out.device)
    charge = ((idx >> 1) & 1) + (idx & 1)
    forbidden = charge[:, None] != charge[None, :]
    assert int(forbidden.sum()) == 160
    swap = 8 * ((idx >> 2) & 1) + 4 * ((idx >> 3) & 1) + 2 * (idx & 1) + ((idx >> 1) & 1)      # (P12 M)[r] = M[swap(r)]
    swapped = d_cfg.clone()
    swapped[:, 0:3], swapped[:, 3:6] = d_cfg[:, 3:6], d_cfg[:, 0:3]
    out_t = torch.empty_like(out)
    no.eval_into(swapped, out_t)
    flipped = d_cfg.clone()
    flipped[:, 3:6] *= -1
    out_f = torch.empty_like(out)
    no.eval_into(flipped, out_f)
    torch.cuda.synchronize()
    worst_h = worst_a = 0.0
    for c0 in range(0, n, chunk):
        M = torch.view_as_complex(out[c0:c0 + chunk])
        assert int(torch.count_nonzero(M[:, forbidden])) == 0, f"{label}: structural zero written as non-zero"
        mx = M.abs().amax(dim=(1, 2), keepdim=True).clamp_min(1e-300)      # an all-zero matrix must match exactly
        Mt = torch.view_as_complex(out_t[c0:c0 + chunk])
        dh = ((M - Mt.transpose(1, 2).conj()).abs() / mx).amax()
        Mf = torch.view_as_complex(out_f[c0:c0 + chunk])
        da = ((Mf[:, swap, :] + M).abs() / mx).amax()
        worst_h, worst_a = max(worst_h, float(dh)), max(worst_a, float(da))
    assert worst_h <= 1e-12, f"{label}: Hermiticity violated by {worst_h:.2e} of the matrix maximum"
    assert worst_a <= 1e-12, f"{label}: antisymmetry violated by {worst_a:.2e} of the matrix maximum"
    print(f"{label}: all {n} matrices finite, 160 structural zeros exact, Hermiticity {worst_h:.1e}, antisymmetry {worst_a:.1e}")


@pytest.mark.parametrize("name,n_sample", FULL_SIZE)
def test_full_size_launch_sampled_outputs(name, n_sample):
    """The launch bench.py times (all configurations of every run, full k3 grid); the oracle computes
    the sampled matrices one by one."""
    for run in W.workload(name).runs:
        cfg = run.configurations()
        no = NormalOrdering(device=0, angular=run.angular(), **run.params())
        d_cfg = torch.from_numpy(cfg).cuda()
        out = torch.empty((run.n_cfg, 16, 16, 2), dtype=torch.float64, device="cuda")
        no.eval_into(d_cfg, out)
        torch.cuda.synchronize()
        assert no.evals_per_cfg == run.nodes_per_cfg
        idx = sample_indices(run.n_cfg, n_sample)
        got = torch.view_as_complex(out[idx]).cpu().numpy()
        want = O.normal_order(cfg[idx], dirs=run.angular(), **run.params())
        worst = check_parity(got, want, run.name)
        # properties that hold at any size, on EVERY output of the launch, reduced on the device (P4, P5, P6)
        device_invariants(no, d_cfg, out, run.name)
        no.close()
        del out, d_cfg
        torch.cuda.empty_cache()
        print(f"{run.name}: {run.n_cfg} configurations x {run.nodes_per_cfg} nodes, "
              f"{len(idx)} sampled, max rel err {worst:.2e}")


def test_random_parameter_sweep():
    """24 seeded random parameter sets (matter composition, LECs incl. c4, cutoff, regulator exponent, ragged
    quadrature orders, product grid or Lebedev-type rule), a few configurations each, every element compared."""
    from paper_2603_24532_b200 import angular_rules as A
    rng = np.random.default_rng(20260324)
    worst = 0.0
    for case in range(24):
        kf = rng.uniform(0.6, 2.1, 2)
        comp = case % 4
        kf_n, kf_p = (kf[0], 0.0) if comp == 0 else ((0.0, kf[1]) if comp == 1 else ((kf[0], kf[0]) if comp == 2 else kf))
        kw = dict(kf_n=float(kf_n), kf_p=float(kf_p), c1=rng.uniform(-1.5, 0.5), c3=rng.uniform(-5, -1),
                  c4=0.0 if case % 3 else rng.uniform(2, 6), cD=rng.uniform(-2, 2), cE=rng.uniform(-1, 1),
                  gA=rng.uniform(1.2, 1.3), fpi=rng.uniform(88, 95), mpi=rng.uniform(134, 140),
                  lambda_chi=rng.uniform(600, 1000), Lambda=-1.0 if case % 7 == 6 else rng.uniform(380, 700),
                  n_reg=int(rng.integers(1, 7)), n_r=int(rng.integers(1, 13)))
        kw = {k: (float(v) if isinstance(v, np.floating) else v) for k, v in kw.items()}
        cfg = W.momentum_configurations(100 + case, 0, 3, float(rng.uniform(0.5, 3.0)), 2.0 * max(kf_n, kf_p))
        if case % 5 == 4:
            dirs = A.octahedral_rule([5, 9, 11, 15][case % 4])
            no = NormalOrdering(device=0, angular=dirs, layout=1 + case % 2, **kw)
            want = O.normal_order(cfg, dirs=dirs, n_cos=1, n_phi=1, **kw)
        else:
            grid = dict(n_cos=int(rng.integers(1, 12)), n_phi=int(rng.integers(1, 12)))
            no = NormalOrdering(device=0, layout=1 + case % 2, **kw, **grid)
            want = O.normal_order(cfg, **kw, **grid)
        got = no(torch.from_numpy(cfg).cuda()).cpu().numpy()
        no.close()
        if np.abs(want).max() < 1e-280:
            continue                                             # regulator underflow: nothing to compare (R18)
        worst = max(worst, check_parity(got, want, f"random case {case}: {kw}"))
    print(f"random sweep: worst rel err {worst:.2e}")


def test_c4_topology_extra_case():
    run = W.workload("c4").runs[0]
    cfg = run.configurations()
    got = gpu_eval(cfg, **run.params())
    idx = sample_indices(run.n_cfg, 32)
    want = O.normal_order(cfg[idx], **run.params())
    check_parity(got[idx], want, "c4")
    without = O.normal_order(cfg[idx[:2]], **dict(run.params(), c4=0.0))
    assert np.abs(without - want[:2]).max() > 1e-3 * np.abs(want[:2]).max()     # the term is exercised


# ----------------------------------------------------------------------------------------------
# edge cases
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n_cfg", [0, 1, 3, 4, 5, 7, 130])
def test_ragged_batch_sizes(n_cfg):
    """4 configurations per CTA: every remainder, plus the empty batch."""
    run = W.workload("cfg4").runs[0].shrunk(n_cfg, 6)
    cfg = run.configurations()
    got = gpu_eval(cfg, **run.params())
    assert got.shape == (n_cfg, 16, 16)
    if n_cfg:
        check_parity(got, O.normal_order(cfg, **run.params()), f"n_cfg={n_cfg}")


@pytest.mark.parametrize("orders", [(5, 7, 3), (1, 1, 1), (2, 33, 1), (3, 5, 13), (128, 3, 2), (2, 128, 2), (2, 2, 128)])
def test_ragged_and_maximum_quadrature_orders(orders):
    """direction counts that do not fill the 32 lanes, single-node rules, the maximum order per axis."""
    n_r, n_cos, n_phi = orders
    kw = dict(PHYS, kf_n=1.3, kf_p=0.9, n_r=n_r, n_cos=n_cos, n_phi=n_phi)
    cfg = W.momentum_configurations(3, 1, 6, 1.5, 2.0)
    check_parity(gpu_eval(cfg, **kw), O.normal_order(cfg, **kw), str(orders))


@pytest.mark.parametrize("geo", [dict(kf_n=1.0, kf_p=0.0), dict(kf_n=0.0, kf_p=0.8), dict(kf_n=1.33, kf_p=1.33),
                                 dict(kf_n=1.4, kf_p=0.8, Lambda=-1.0), dict(kf_n=1.4, kf_p=0.8, Lambda=400.0, n_reg=1),
                                 dict(kf_n=1.4, kf_p=0.8, Lambda=400.0, n_reg=2), dict(kf_n=1.4, kf_p=0.8, Lambda=450.0, n_reg=3),
                                 dict(kf_n=1.4, kf_p=0.8, Lambda=600.0, n_reg=6), dict(kf_n=1.4, kf_p=0.8, Lambda=700.0, n_reg=12)])
@pytest.mark.parametrize("c4", [0.0, 5.4])
def test_every_kernel_variant(geo, c4):
    """all regulator variants (unregulated, n = 1..4 unrolled, generic) x (c4 = 0, c4 != 0), each matter type."""
    kw = dict(PHYS, c4=c4, n_r=6, n_cos=7, n_phi=8)
    kw.update(geo)
    cfg = W.momentum_configurations(5, 2, 9, 1.5, 2.0)
    check_parity(gpu_eval(cfg, **kw), O.normal_order(cfg, **kw), f"{geo} c4={c4}")


def test_underflow_guard_path_strong_regulator():
    """Lambda = 100 MeV: far nodes have exp(-dE) below the double range (guarded hot loop, chosen per
    configuration from a bound on the exponent), near nodes are O(1); mixed with mild configurations."""
    kw = dict(PHYS, kf_n=1.4, kf_p=0.8, n_r=6, n_cos=7, n_phi=8)
    kw.update(Lambda=100.0, n_reg=4)
    cfg = np.array([[0.05, -0.02, 0.03, -0.04, 0.06, 0.01, 0.6, 0.8, 1.0],
                    [0.02, 0.01, 0.03, 0.01, -0.02, 0.02, 0.05, 0.02, -0.03],
                    [0.10, 0.05, -0.05, 0.02, -0.08, 0.04, -0.9, 0.5, 0.7],
                    [0.02, 0.01, 0.03, 0.01, -0.02, 0.02, 0.05, 0.02, -0.03],
                    [0.01, 0.00, 0.02, 0.00, 0.03, -0.01, 1.2, -1.1, 0.9]])
    want = O.normal_order(cfg, **kw)
    assert np.abs(want).max(axis=(1, 2)).min() > 1e-30
    check_parity(gpu_eval(cfg, **kw), want, "guarded hot loop")
    # generic exponent, extreme: everything underflows to exactly zero instead of garbage
    out = gpu_eval(np.full((2, 9), 3.0), **dict(kw, Lambda=50.0, n_reg=12))
    assert np.count_nonzero(out) == 0


def test_degenerate_inputs():
    kw = dict(PHYS, kf_n=1.2, kf_p=0.9, n_r=4, n_cos=4, n_phi=4)
    # empty Fermi sea: exactly zero
    assert np.count_nonzero(gpu_eval(np.ones((5, 9)), **dict(kw, kf_n=0.0, kf_p=0.0))) == 0
    # p = p' (forward), P = 0, p = 0: finite and equal to the oracle
    cfg = np.zeros((4, 9))
    cfg[0, 0:3] = cfg[0, 3:6] = (0.3, -0.2, 0.5)
    cfg[1, 0:3] = (0.4, 0.1, -0.2)
    cfg[1, 3:6] = (-0.4, -0.1, 0.2)                     # p' = -p
    cfg[2, 6:9] = (0.2, 0.1, -0.3)                      # p = p' = 0
    check_parity(gpu_eval(cfg[:3], **kw), O.normal_order(cfg[:3], **kw), "degenerate")
    # everything zero: the pion-exchange terms vanish, the contact term survives
    got = gpu_eval(cfg[3:], **kw)
    check_parity(got, O.normal_order(cfg[3:], **kw), "all-zero momenta")
    # non-finite inputs propagate (no checking on the hot path), neighbours are untouched
    bad = W.momentum_configurations(1, 1, 3, 1.0, 1.0)
    good = gpu_eval(bad, **kw)
    bad2 = bad.copy()
    bad2[1, 4] = np.nan
    out = gpu_eval(bad2, **kw)
    assert not np.isfinite(out[1].view(np.float64)).all()
    assert np.array_equal(out[0], good[0]) and np.array_equal(out[2], good[2])


def test_abi_pointer_checks_streams_and_host_path():
    run = W.workload("cfg3").runs[0].shrunk(37, 8)
    cfg = run.configurations()
    h = binding.no_init(device=0, **run.params())
    lib = binding.load()
    d_cfg = torch.from_numpy(cfg).cuda()
    out = torch.zeros((37, 16, 16, 2), dtype=torch.float64, device="cuda")
    s = torch.cuda.current_stream().cuda_stream
    vp = ctypes.c_void_p
    assert lib.no_eval(h, vp(d_cfg.data_ptr() + 4), 37, vp(out.data_ptr()), vp(s)) == binding.NO_ERR_INVALID
    assert lib.no_eval(h, vp(d_cfg.data_ptr()), 37, vp(out.data_ptr() + 8), vp(s)) == binding.NO_ERR_INVALID
    assert lib.no_eval(h, vp(d_cfg.data_ptr()), -1, vp(out.data_ptr()), vp(s)) == binding.NO_ERR_INVALID
    assert lib.no_eval(h, None, 5, vp(out.data_ptr()), vp(s)) == binding.NO_ERR_INVALID
    assert lib.no_eval(h, None, 0, None, vp(s)) == binding.NO_OK
    assert int(out.abs().sum().item()) == 0                      # nothing was written by the failed calls
    # default stream
    binding.no_eval(h, d_cfg.data_ptr(), 37, out.data_ptr(), None)
    torch.cuda.synchronize()
    ref = out.clone()
    # two user streams at once on one handle (threads time-share the GPU via streams)
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    o1, o2 = torch.empty_like(out), torch.empty_like(out)
    binding.no_eval(h, d_cfg.data_ptr(), 37, o1.data_ptr(), s1.cuda_stream)
    binding.no_eval(h, d_cfg.data_ptr(), 37, o2.data_ptr(), s2.cuda_stream)
    torch.cuda.synchronize()
    assert torch.equal(o1, ref) and torch.equal(o2, ref)         # bit-identical: fixed summation order
    # host-buffer path
    h_out = np.empty((37, 16, 16, 2))
    binding.no_eval_host(h, cfg.ctypes.data, 37, h_out.ctypes.data, None)
    assert np.array_equal(h_out, ref.cpu().numpy())
    binding.no_eval_host(h, cfg.ctypes.data, 5, h_out.ctypes.data, s1.cuda_stream)   # smaller batch reuses scratch
    assert np.array_equal(h_out[:5], ref[:5].cpu().numpy())
    info = binding.no_kernel_info(h)
    assert info["threads"] == 32 * info["cfg_per_cta"] and info["cfg_per_cta"] in (1, 2, 4) and info["ctas_per_sm"] >= 1 and info["n_sm"] > 0
    assert binding.no_evals_per_cfg(h) == 8 ** 3
    binding.no_free(h)
    check_parity(torch.view_as_complex(ref).cpu().numpy(), O.normal_order(cfg, **run.params()), "streams")
    with pytest.raises(binding.NoError):
        binding.no_init(device=99, **run.params())


def test_batches_larger_than_one_grid_are_cut_into_several_launches():
    """A batch that needs more CTAs than gridDim.x allows is chunked, not refused.  The limit (2^31 - 1 CTAs)
    cannot be reached in a test, so the test hook no_set_max_grid lowers it: same bits as one launch."""
    run = W.workload("cfg4").runs[0].shrunk(37, 6)
    cfg = torch.from_numpy(run.configurations()).cuda()
    ref = {}
    for layout in (1, 2):
        no = NormalOrdering(device=0, layout=layout, **run.params())
        ref[layout] = no(cfg).cpu().numpy()
        ref[layout, "diag"] = no.diag(cfg).cpu().numpy()
        no.close()
    for layout in (1, 2):
        no = NormalOrdering(device=0, layout=layout, **run.params())          # 37 configurations: 7 or 13 launches
        binding.no_set_max_grid(no._h, 3)
        assert np.array_equal(no(cfg).cpu().numpy(), ref[layout])
        assert np.array_equal(no.diag(cfg).cpu().numpy(), ref[layout, "diag"])
        h_out = np.empty((37, 16, 16, 2))
        h_cfg = run.configurations()                     # kept alive across the call (a raw pointer is passed)
        binding.no_eval_host(no._h, h_cfg.ctypes.data, 37, h_out.ctypes.data, None)
        assert np.array_equal(h_out[..., 0] + 1j * h_out[..., 1], ref[layout])
        no.close()


def test_host_path_uses_one_layout_per_call_and_refuses_concurrent_use():
    """no_eval_host decides the kernel layout once per call from the whole batch (a small tail chunk does not
    switch to the small-batch layout), and a second concurrent call on the same handle is refused."""
    import threading
    run = W.workload("cfg1").runs[0].shrunk(4000, 6)             # chunked: waves of 1776 configurations + a tail
    cfg = run.configurations()
    h = binding.no_init(device=0, **run.params())
    d_out = torch.empty((4000, 16, 16, 2), dtype=torch.float64, device="cuda")
    binding.no_set_layout(h, 1)
    binding.no_eval(h, torch.from_numpy(cfg).cuda().data_ptr(), 4000, d_out.data_ptr(), None)
    torch.cuda.synchronize()
    binding.no_set_layout(h, 0)
    h_out = torch.empty((4000, 16, 16, 2), dtype=torch.float64, pin_memory=True)
    binding.no_eval_host(h, cfg.ctypes.data, 4000, h_out.data_ptr(), None)
    assert torch.equal(h_out, d_out.cpu())                       # tail included: bit-identical to the one-warp layout
    # two threads on one handle: every call either succeeds with the right bits or is refused with NO_ERR_BUSY
    lib, results = binding.load(), []
    outs = [torch.empty((4000, 16, 16, 2), dtype=torch.float64, pin_memory=True) for _ in range(2)]
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]

    def work(i):
        for _ in range(20):
            rc = lib.no_eval_host(h, ctypes.c_void_p(cfg.ctypes.data), 4000, ctypes.c_void_p(outs[i].data_ptr()),
                                  ctypes.c_void_p(streams[i].cuda_stream))
            results.append((rc, rc != 0 or bool(torch.equal(outs[i], h_out))))

    th = [threading.Thread(target=work, args=(i,)) for i in range(2)]
    [t.start() for t in th]
    [t.join() for t in th]
    assert all(rc in (binding.NO_OK, binding.NO_ERR_BUSY) and good for rc, good in results)
    assert any(rc == binding.NO_OK for rc, _ in results)
    binding.no_free(h)


def test_handles_with_different_shared_memory_sizes_coexist():
    """Two handles on the same kernel variant, the larger table set created first: the dynamic shared
    memory limit is a property of the kernel, not of the handle that set it last."""
    kw2 = dict(PHYS, kf_n=1.4, kf_p=0.8, n_r=24, n_cos=20, n_phi=20)     # two spheres: larger tables
    kw1 = dict(PHYS, kf_n=1.4, kf_p=0.0, n_r=4, n_cos=4, n_phi=4)
    big, small = NormalOrdering(device=0, **kw2), NormalOrdering(device=0, **kw1)
    cfg = W.momentum_configurations(6, 1, 3, 1.5, 2.0)
    got = big(torch.from_numpy(cfg).cuda()).cpu().numpy()
    torch.cuda.synchronize()
    check_parity(got, O.normal_order(cfg, **kw2), "big handle after small init")
    big.close(); small.close()


# ----------------------------------------------------------------------------------------------
# Hartree-Fock contraction on the device
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("geo", [dict(kf_n=1.3, kf_p=0.9), dict(kf_n=1.33, kf_p=1.33), dict(kf_n=1.2, kf_p=0.0)])
def test_diag_trace_matches_oracle(geo):
    kw = dict(PHYS, c4=5.4, n_r=6, n_cos=5, n_phi=7, **geo)
    cfg = W.momentum_configurations(11, 2, 37, 1.5, 2.0)
    cfg[:20, 3:6] = cfg[:20, 0:3]                               # forward configurations p' = p, and generic ones
    no = NormalOrdering(device=0, **kw)
    got = no.diag(torch.from_numpy(cfg).cuda()).cpu().numpy()
    full = no(torch.from_numpy(cfg).cuda()).cpu().numpy()
    no.close()
    want = O.diag_trace(cfg, **kw)
    scale = np.abs(O.normal_order(cfg, **kw)).max(axis=(1, 2))[:, None]
    assert np.abs(got - want).max() / scale.max() < 1e-13
    assert (np.abs(got - want) <= 1e-12 * scale).all()          # relative to each matrix maximum
    mask = np.abs(want) > 1e-6 * scale
    assert (np.abs(got - want)[mask] / np.abs(want)[mask]).max() < 1e-10
    idx4 = [[8 * s1 + 4 * s2 + t for s1 in range(2) for s2 in range(2)] for t in range(4)]
    from_full = np.stack([sum(full[:, a, a].real for a in idx4[t]) for t in range(4)], axis=1)
    assert (np.abs(got - from_full) <= 1e-14 * scale).all()     # same kernel, same coefficients


@pytest.mark.parametrize("geo", [dict(kf_n=1.2, kf_p=0.9), dict(kf_n=1.1, kf_p=1.1), dict(kf_n=0.0, kf_p=1.0)])
def test_hf_energy_equals_brute_force_9d_sum(geo):
    """pin P8 on the device: all three particles on the same tiny grids."""
    kw = dict(PHYS, c4=5.4, n_r=2, n_cos=3, n_phi=2, **geo)
    no = NormalOrdering(device=0, **kw)
    got = no.hf_energy(2, 3, 2)
    no.close()
    want = O.hf3n_bruteforce(**kw)
    assert abs(want) > 1e-8
    assert got == pytest.approx(want, rel=1e-11)


def test_hf_energy_matches_oracle_contraction_and_closed_form():
    kw = dict(PHYS, kf_n=1.4, kf_p=1.0, n_r=5, n_cos=4, n_phi=6)
    no = NormalOrdering(device=0, **kw)
    got = no.hf_energy(3, 4, 3)                                 # grids of particles 1, 2 differ from the k3 grid
    assert got == no.hf_energy(3, 4, 3)                         # fixed summation order: bit reproducible
    no.close()
    assert got == pytest.approx(O.hf_energy(3, 4, 3, **kw), rel=1e-11)
    # P2: unregulated contact term in symmetric matter, E/V = -(3/16) cE rho^3 / (fpi^4 Lchi); chunked pair loop
    kF, hbarc = 1.33, 197.3269804
    kc = dict(kf_n=kF, kf_p=kF, c1=0.0, c3=0.0, c4=0.0, cD=0.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04,
              lambda_chi=700.0, Lambda=-1.0, n_r=2, n_cos=2, n_phi=2)
    rho = 2 * kF ** 3 / (3 * np.pi ** 2)
    want = -(3.0 / 16.0) * (-0.5) * rho ** 3 / ((92.4 / hbarc) ** 4 * (700.0 / hbarc))
    no = NormalOrdering(device=0, **kc)
    assert no.hf_energy(12, 10, 10) == pytest.approx(want, rel=1e-11)      # 1200^2 pairs: two chunks of 2^20
    no.close()


# ----------------------------------------------------------------------------------------------
# caller-supplied angular rule: Gauss-Legendre radial x Lebedev-type angular
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("degree,geo", [(15, dict(kf_n=1.33, kf_p=1.33)), (15, dict(kf_n=1.4, kf_p=0.8, c4=5.4)),
                                        (5, dict(kf_n=1.0, kf_p=0.0)), (17, dict(kf_n=1.4, kf_p=0.8))])
def test_lebedev_type_rule_matches_oracle(degree, geo):
    """the paper's production quadrature: 16 radial Gauss-Legendre points x the 86-point degree-15 rule
    (and 14 / 110 directions: ragged over the 32 lanes)."""
    from paper_2603_24532_b200 import angular_rules as A
    dirs = A.octahedral_rule(degree)
    kw = dict(PHYS, n_r=16)
    kw.update(geo)
    cfg = W.momentum_configurations(21, 3, 11, 1.5, 2.0)
    want = O.normal_order(cfg, dirs=dirs, n_cos=1, n_phi=1, **kw)
    for layout in (1, 2):                                        # one warp / one CTA per configuration
        no = NormalOrdering(device=0, angular=dirs, layout=layout, **kw)
        assert no.evals_per_cfg == 16 * len(dirs) * (1 if kw["kf_p"] in (0.0, kw["kf_n"]) else 2)
        got = no(torch.from_numpy(cfg).cuda()).cpu().numpy()
        torch.cuda.synchronize()
        no.close()
        check_parity(got, want, f"degree {degree}, layout {layout}")


def test_product_rule_as_list_equals_grid_path_and_bad_rules_are_refused():
    from paper_2603_24532_b200 import angular_rules as A
    kw = dict(PHYS, kf_n=1.3, kf_p=0.9, n_r=6)
    cfg = W.momentum_configurations(2, 1, 5, 1.5, 2.0)
    grid = gpu_eval(cfg, n_cos=7, n_phi=9, **kw)
    no = NormalOrdering(device=0, angular=A.product_rule(7, 9), **kw)
    lst = no(torch.from_numpy(cfg).cuda()).cpu().numpy()
    no.close()
    assert np.abs(grid - lst).max() <= 1e-13 * np.abs(grid).max()
    bad = A.product_rule(2, 2)
    bad[1, 2] = np.nan
    with pytest.raises(binding.NoError):
        binding.no_init(device=0, angular=bad, **kw)
    with pytest.raises(binding.NoError):
        binding.no_init(device=0, angular=np.zeros((5000, 4)), **kw)          # more than 4096 directions


def test_sp_energy_matches_oracle_and_sums_to_the_hf_energy():
    """Eq. (9): isospin-dependent 3N Hartree-Fock self-energy; chunked over k1 rows; sum rule with no_hf_energy."""
    kw = dict(PHYS, c4=5.4, kf_n=1.3, kf_p=0.9, n_r=4, n_cos=3, n_phi=5)
    k1 = np.array([[0.0, 0.0, 0.0], [0.3, -0.2, 0.5], [1.0, 0.4, -0.7], [0.0, 0.0, 2.5], [-1.9, 1.2, 0.3]])
    no = NormalOrdering(device=0, **kw)
    got = no.sp_energy(k1, 3, 4, 3)
    assert np.array_equal(got, no.sp_energy(k1, 3, 4, 3))                     # bit reproducible
    want = O.sp_energy(k1, 3, 4, 3, **kw)
    assert np.abs(got - want).max() < 1e-11 * np.abs(want).max()
    assert np.abs(want[:, 0] - want[:, 1]).max() > 1e-3 * np.abs(want).max()   # isospin dependence is there
    # sum rule on equal grids: E/V = (1/3) sum_t1 sum_k1 2 W1 Sigma_t1(k1)
    e = 0.0
    for t1, kf in ((0, kw["kf_p"]), (1, kw["kf_n"])):
        kk, ww = O.sphere_nodes(3, 4, 3, kf)
        e += np.sum(2 * ww * no.sp_energy(kk, 3, 4, 3)[:, t1]) / 3
    assert e == pytest.approx(no.hf_energy(3, 4, 3), rel=1e-11)
    no.close()
    # many momenta against a large particle-2 grid: several row chunks (2^20 pairs each)
    kc = dict(kf_n=1.33, kf_p=1.33, c1=0.0, c3=0.0, c4=0.0, cD=0.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04,
              lambda_chi=700.0, Lambda=-1.0, n_r=2, n_cos=2, n_phi=2)
    hbarc = 197.3269804
    pref = 0.5 * 1.33 ** 3 / (np.pi ** 2 * (92.4 / hbarc) ** 4 * (700.0 / hbarc))
    no = NormalOrdering(device=0, **kc)
    sig = no.sp_energy(W.momentum_configurations(4, 0, 100, 2.0, 2.0)[:, :3].copy(), 30, 30, 30)   # 100 x 27000 pairs
    no.close()
    assert np.allclose(sig, pref * 1.33 ** 3 / (4 * np.pi ** 2), rtol=1e-11, atol=0)


def test_no_eval_is_cuda_graph_capturable():
    """no_eval only enqueues (no synchronisation, no allocation): a batch of launches can be captured once in a
    CUDA graph and replayed (launch-bound inner loops of small batches)."""
    run = W.workload("cfg1").runs[0].shrunk(64, 8)
    h = binding.no_init(device=0, **run.params())
    cfg = torch.from_numpy(run.configurations()).cuda()
    ref = torch.empty((64, 16, 16, 2), dtype=torch.float64, device="cuda")
    binding.no_eval(h, cfg.data_ptr(), 64, ref.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    outs = [torch.zeros_like(ref) for _ in range(4)]
    g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream()
    with torch.cuda.stream(s):
        with torch.cuda.graph(g, stream=s):
            for o in outs:
                binding.no_eval(h, cfg.data_ptr(), 64, o.data_ptr(), torch.cuda.current_stream().cuda_stream)
    for o in outs:
        o.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert all(torch.equal(ref, o) for o in outs)
    del g
    binding.no_free(h)


def test_fp64_probe_reports_a_sane_peak():
    r = binding.no_probe_fp64_peak(0, 100)
    assert r["n_sm"] > 0 and 1.0 < r["tflops"] < 100.0
    print("FP64 DFMA probe:", r)


def test_fp64_operand_probe_shows_the_three_register_operand_penalty():
    """the rule the hot loop is arranged around: a DFMA with three distinct 64-bit register
    operands holds the FP64 pipe for 3 cycles instead of 2, i.e. runs at about two thirds of the rate"""
    r = binding.no_probe_fp64_operands(0, 100)
    ratio = r["three_operands_tflops"] / r["two_operands_tflops"]
    print("FP64 operand probe:", r, f"ratio {ratio:.3f}")
    assert 1.0 < r["two_operands_tflops"] < 100.0
    assert 0.55 < ratio < 0.8


def test_native_library_is_the_one_loaded():
    maps = open(f"/proc/{os.getpid()}/maps").read()
    assert "libno3n.so" in maps


# ----------------------------------------------------------------------------------------------
# packed, symmetry-reduced output and its reconstruction
# ----------------------------------------------------------------------------------------------
def _check_packed(got, want, label):
    """same criterion as _check, on packed rows: relative 1e-10 above 1e-12 of the row maximum"""
    mx = np.abs(want).max(axis=1, keepdims=True)
    mask = np.abs(want) > MAG_FLOOR * mx
    rel = np.abs(got - want)[mask] / np.abs(want)[mask]
    worst = rel.max() if rel.size else 0.0
    assert worst < REL_TOL, f"{label}: max rel err {worst:.3e}"
    return worst


@pytest.mark.parametrize("layout", [1, 2])
@pytest.mark.parametrize("matter", ["snm", "pnm", "asym", "snm_c4_lebedev"])
def test_packed_output_and_unpack_match_the_oracle(matter, layout):
    from paper_2603_24532_b200 import angular_rules
    kf = {"snm": (1.33, 1.33), "pnm": (1.2, 0.0), "asym": (1.3, 0.9), "snm_c4_lebedev": (1.1, 1.1)}[matter]
    kw = dict(PHYS, kf_n=kf[0], kf_p=kf[1], n_r=6, n_cos=7, n_phi=5)
    dirs = None
    if matter == "snm_c4_lebedev":
        kw.update(c4=5.4, n_cos=1, n_phi=1)
        dirs = angular_rules.octahedral_rule(7)
    cfg = W.momentum_configurations(11, 0, 37, 2.5, 2.0 * max(kf))
    want = O.normal_order(cfg, dirs=dirs, **kw)
    no = NormalOrdering(device=0, layout=layout, angular=dirs, **kw)
    d_cfg = torch.from_numpy(cfg).cuda()
    full = no(d_cfg)
    formats = [binding.NO_PACK_CHARGE] + ([binding.NO_PACK_ISOSPIN] if kf[0] == kf[1] else [])
    for fmt in formats:
        packed = no.packed(d_cfg, fmt)
        torch.cuda.synchronize()
        assert packed.shape == (37, O.PACKED_COMPLEX[fmt]) and binding.no_packed_doubles(no._h, fmt) == 2 * O.PACKED_COMPLEX[fmt]
        worst = _check_packed(packed.cpu().numpy(), O.pack(want, fmt), f"{matter} packed fmt {fmt}")
        rebuilt = NormalOrdering.unpack(packed, fmt)
        torch.cuda.synchronize()
        worst = max(worst, _check(rebuilt.cpu().numpy(), want, f"{matter} unpack fmt {fmt}"))
        # the oracle's own reconstruction of the oracle's packed form is the same matrix
        _check(rebuilt.cpu().numpy(), O.unpack(O.pack(want, fmt), fmt), f"{matter} unpack vs oracle unpack fmt {fmt}")
        if fmt == binding.NO_PACK_CHARGE:
            assert torch.equal(rebuilt, full)                    # format 1 loses nothing: bit for bit no_eval
        # the host path ships the same packed bits
        host = no.packed(torch.from_numpy(cfg), fmt)
        assert torch.equal(host, packed.cpu())
        print(f"{matter} layout {layout} fmt {fmt}: max rel err {worst:.2e}")
    if kf[0] != kf[1]:
        assert binding.no_packed_doubles(no._h, binding.NO_PACK_ISOSPIN) == 0
        with pytest.raises(binding.NoError):
            out = torch.empty((37, 32, 2), dtype=torch.float64, device="cuda")
            binding.no_eval_packed(no._h, binding.NO_PACK_ISOSPIN, d_cfg.data_ptr(), 37, out.data_ptr(), 0)
    no.close()


@pytest.mark.parametrize("matter", ["snm", "asym", "pnm"])
def test_forward_flag_of_the_packed_entry_point_matches_the_oracle(matter):
    """NO_PACK_FORWARD: configurations with p' = p through the forward kernel in packed mode, against
    the oracle's packed matrices and against the general kernel on the same configurations; at p' = p the matrix is
    Hermitian (pin P4), checked on the reconstruction."""
    kf = {"snm": (1.33, 1.33), "pnm": (1.2, 0.0), "asym": (1.3, 0.9)}[matter]
    kw = dict(PHYS, c4=5.4 if matter == "asym" else 0.0, kf_n=kf[0], kf_p=kf[1], n_r=6, n_cos=7, n_phi=5)
    cfg = W.momentum_configurations(13, 0, 41, 2.5, 2.0 * max(kf))
    cfg[:, 3:6] = cfg[:, 0:3]                                      # forward: p' = p
    want = O.normal_order(cfg, **kw)
    d_cfg = torch.from_numpy(cfg).cuda()
    for layout in (1, 2):
        no = NormalOrdering(device=0, layout=layout, **kw)
        for fmt in [binding.NO_PACK_CHARGE] + ([binding.NO_PACK_ISOSPIN] if kf[0] == kf[1] else []):
            assert binding.no_packed_doubles(no._h, fmt | binding.NO_PACK_FORWARD) == 2 * O.PACKED_COMPLEX[fmt]
            fwd = no.packed(d_cfg, fmt | binding.NO_PACK_FORWARD)
            gen = no.packed(d_cfg, fmt)
            torch.cuda.synchronize()
            worst = _check_packed(fwd.cpu().numpy(), O.pack(want, fmt), f"{matter} forward packed fmt {fmt} layout {layout}")
            _check_packed(fwd.cpu().numpy(), gen.cpu().numpy(), f"{matter} forward vs general kernel fmt {fmt}")
            if layout == 2:
                assert torch.equal(fwd, gen)                       # small-batch layout: the flag changes nothing
            M = NormalOrdering.unpack(fwd, fmt).cpu().numpy()
            mx = np.abs(M).max(axis=(1, 2), keepdims=True)
            assert (np.abs(M - np.conj(np.swapaxes(M, 1, 2))) <= 1e-12 * mx).all()
            print(f"{matter} forward fmt {fmt} layout {layout}: max rel err {worst:.2e}")
        no.close()


def test_packed_abi_argument_checks_and_full_size_launch():
    """raw C-ABI calls: bad formats, null / misaligned pointers, n = 0; then the bench-size paper-quadrature launch in
    packed form against the full no_eval launch (every configuration, bit for bit) and sampled against the oracle."""
    lib = binding.load()
    run = W.workload("paper").runs[0]
    no = NormalOrdering(device=0, angular=run.angular(), **run.params())
    h = no._h
    n = run.n_cfg
    cfg = run.configurations()
    d_cfg = torch.from_numpy(cfg).cuda()
    pk = torch.empty((n, 32, 2), dtype=torch.float64, device="cuda")
    vp = ctypes.c_void_p
    assert lib.no_eval_packed(h, 3, vp(d_cfg.data_ptr()), n, vp(pk.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_eval_packed(h, 0, vp(d_cfg.data_ptr()), n, vp(pk.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_eval_packed(h, 2, vp(d_cfg.data_ptr()), -1, vp(pk.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_eval_packed(h, 2, None, n, vp(pk.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_eval_packed(h, 2, vp(d_cfg.data_ptr()), n, vp(pk.data_ptr() + 8), None) == binding.NO_ERR_INVALID
    assert lib.no_eval_packed(h, 2, None, 0, None, None) == binding.NO_OK
    assert lib.no_unpack(5, vp(pk.data_ptr()), n, vp(pk.data_ptr()), None) == binding.NO_ERR_INVALID
    assert lib.no_unpack(2, None, 0, None, None) == binding.NO_OK
    assert lib.no_packed_doubles(h, 1) == 192 and lib.no_packed_doubles(h, 2) == 64 and lib.no_packed_doubles(h, 7) == 0
    assert lib.no_packed_doubles(None, 1) == 0
    # full size, isospin-reduced form (the paper workload is SNM)
    assert lib.no_eval_packed(h, 2, vp(d_cfg.data_ptr()), n, vp(pk.data_ptr()), None) == binding.NO_OK
    full = torch.empty((n, 16, 16, 2), dtype=torch.float64, device="cuda")
    no.eval_into(d_cfg, full)
    torch.cuda.synchronize()
    F = torch.view_as_complex(full)
    P = torch.view_as_complex(pk)
    sp = torch.arange(16, device="cuda")
    rows, cols = 4 * (sp >> 2), 4 * (sp & 3)
    assert torch.equal(P[:, 0::2], F[:, rows + 1, cols + 1]) and torch.equal(P[:, 1::2], F[:, rows + 1, cols + 2])
    idx = sample_indices(n, 16)
    want = O.normal_order(cfg[idx], dirs=run.angular(), **run.params())
    rebuilt = NormalOrdering.unpack(P[idx].contiguous(), 2).cpu().numpy()
    worst = _check(rebuilt, want, "paper packed")
    print(f"paper packed (isospin form, {n} configurations): max rel err {worst:.2e} on {len(idx)} sampled")
    no.close()
