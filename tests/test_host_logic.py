"""Host logic of the product, checked on the CPU: quadrature tables, kernel-variant choice, the seeded
workloads, and -- through tests/host_emu.cpp, which compiles the kernel's own arithmetic
(csrc/no_core.h) with g++ and walks one warp lane by lane -- the factored moment formulation and the
epilogue against the oracle.  The emulation is test-only; the product has no CPU path."""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2603_24532_b200 import workloads as W
from tests import emu

PHYS = dict(c1=-0.81, c3=-3.2, c4=0.0, cD=1.0, cE=-0.5, gA=1.27, fpi=92.4, mpi=138.04, lambda_chi=700.0,
            Lambda=500.0, n_reg=4)
REL_TOL = 1e-10      # north_star: max relative error on every element ...
MAG_FLOOR = 1e-12    # ... whose magnitude exceeds 1e-12 of the matrix maximum


def check_parity(got, want):
    mx = np.abs(want).max(axis=(1, 2), keepdims=True)
    mask = np.abs(want) > MAG_FLOOR * mx
    rel = np.abs(got - want)[mask] / np.abs(want)[mask]
    assert rel.max() < REL_TOL, rel.max()
    assert (np.abs(got)[~mask] <= MAG_FLOOR * np.broadcast_to(mx, got.shape)[~mask]).all()
    return rel.max()


@pytest.mark.parametrize("n", [1, 2, 3, 5, 16, 31, 32, 40, 48, 64, 127, 128])
def test_product_gauss_legendre_rule(n):
    x, w = emu.emu_gl_rule(n, -1.0, 1.0)
    xo, wo = O.gauss_legendre(n, -1.0, 1.0)             # independent implementation (oracle)
    assert np.abs(x - xo).max() <= 2.3e-16
    assert np.abs(w - wo).max() <= 1e-16 + 4e-16 * wo.max()
    assert np.array_equal(x, -x[::-1]) and np.array_equal(w, w[::-1])
    assert abs(math.fsum(w) - 2.0) < 4e-16
    k = 2 * n - 2
    assert abs(math.fsum(w * x ** k) - 2.0 / (k + 1)) < 4e-16
    x, w = emu.emu_gl_rule(n, 0.0, 2 * math.pi)
    assert abs(w.sum() - 2 * math.pi) < 4e-15 and x.min() > 0 and x.max() < 2 * math.pi


def test_plan_passes_variants_and_tables():
    base = dict(PHYS, n_r=3, n_cos=4, n_phi=5)
    p = emu.emu_plan(kf_n=1.2, kf_p=0.9, **base)
    assert (p["n_pass"], p["nreg_variant"], p["has_c4"], p["evals_per_cfg"]) == (2, 4, 0, 2 * 60)
    n_pad = 4                                           # n_r = 3 padded to a multiple of 4 with zero-weight nodes
    per = (2 * n_pad + 3 * 4 + 3 * 5 + 3) // 4 * 4      # each pass padded to 32 bytes
    assert p["tab_doubles"] == 256 + 2 * per
    t = p["tab"]
    assert t[0] == 1.0 and np.abs(t[:256] - 2.0 ** (np.arange(256) / 256.0)).max() < 2.3e-16   # 2^(j/256)
    t = t[256:]
    r, wr = O.gauss_legendre(3, 0.0, 0.9)               # pass 0 = protons
    assert np.allclose(t[0:6:2], r, rtol=0, atol=3e-16)
    assert np.allclose(t[1:6:2], wr * r * r / (2 * math.pi) ** 3, rtol=1e-14)
    assert t[6] == t[4] and t[7] == 0.0                 # padding node: valid radius, weight 0
    x, wx = O.gauss_legendre(4, -1.0, 1.0)
    assert np.allclose(t[8:12], x, atol=3e-16) and np.allclose(t[12:16], np.sqrt(1 - x * x), atol=3e-16)
    assert np.allclose(t[16:20], wx, rtol=1e-14)
    ph, wp = O.gauss_legendre(5, 0.0, 2 * math.pi)
    assert np.allclose(t[20:25], np.cos(ph), atol=1e-15) and np.allclose(t[25:30], np.sin(ph), atol=1e-15)
    assert np.allclose(t[30:35], wp, rtol=1e-14)
    rn, _ = O.gauss_legendre(3, 0.0, 1.2)               # pass 1 = neutrons
    assert np.allclose(t[per:per + 6:2], rn, atol=3e-16)
    # equal Fermi momenta share one grid; empty spheres are skipped; regulator variants
    assert emu.emu_plan(kf_n=1.3, kf_p=1.3, **base)["n_pass"] == 1
    assert emu.emu_plan(kf_n=1.3, kf_p=1.3, **base)["evals_per_cfg"] == 60
    assert emu.emu_plan(kf_n=1.3, kf_p=0.0, **base)["n_pass"] == 1
    assert emu.emu_plan(kf_n=0.0, kf_p=0.0, **base)["n_pass"] == 0
    assert emu.emu_plan(kf_n=1.0, kf_p=0.0, **dict(base, Lambda=-1.0))["nreg_variant"] == -1
    assert emu.emu_plan(kf_n=1.0, kf_p=0.0, **dict(base, n_reg=3))["nreg_variant"] == 3
    assert emu.emu_plan(kf_n=1.0, kf_p=0.0, **dict(base, n_reg=7))["nreg_variant"] == 0
    assert emu.emu_plan(kf_n=1.0, kf_p=0.0, **dict(base, c4=5.4))["has_c4"] == 1
    with pytest.raises(ValueError):
        emu.emu_plan(kf_n=-1.0, kf_p=0.0, **base)


GEOS = [dict(kf_n=1.2, kf_p=0.9), dict(kf_n=1.0, kf_p=0.0), dict(kf_n=1.33, kf_p=1.33), dict(kf_n=0.0, kf_p=0.8),
        dict(kf_n=1.4, kf_p=0.8, Lambda=450.0, n_reg=3), dict(kf_n=1.4, kf_p=0.8, Lambda=-1.0),
        dict(kf_n=1.4, kf_p=0.8, Lambda=600.0, n_reg=6), dict(kf_n=1.4, kf_p=0.8, Lambda=400.0, n_reg=2),
        dict(kf_n=1.4, kf_p=0.8, Lambda=400.0, n_reg=1)]


@pytest.mark.parametrize("c4", [0.0, 5.4])
@pytest.mark.parametrize("geo", GEOS)
def test_kernel_arithmetic_matches_oracle(geo, c4):
    rng = np.random.default_rng(5)
    kw = dict(PHYS, c4=c4, n_r=6, n_cos=7, n_phi=8)      # 56 directions: ragged over 32 lanes
    kw.update(geo)
    cfg = rng.uniform(-1, 1, (3, 9)) * 1.5
    check_parity(emu.emu_eval(cfg, **kw), O.normal_order(cfg, **kw))


def test_kernel_arithmetic_on_the_cfg1_distribution():
    """p, p' up to 4 fm^-1: regulators down to 1e-100; parity is per matrix (reading R18)."""
    run = W.workload("cfg1").runs[0].shrunk(24, 8)
    cfg = run.configurations()
    want = O.normal_order(cfg, **run.params())
    assert np.abs(want).max(axis=(1, 2)).min() < 1e-12      # some matrices are tiny in absolute terms
    check_parity(emu.emu_eval(cfg, **run.params()), want)


def test_underflow_guard_path_strong_regulator():
    """Lambda = 100 MeV: at the far nodes the regulator exponent exceeds 704 (exp(-dE) below the double
    range) while the near nodes are O(1): the configurations take the guarded (FLUSH) hot loop; a
    configuration with a mild exponent in the same batch takes the unguarded one."""
    kw = dict(PHYS, c4=0.0, kf_n=1.4, kf_p=0.8, n_r=6, n_cos=7, n_phi=8)
    kw.update(Lambda=100.0, n_reg=4)
    cfg = np.array([[0.05, -0.02, 0.03, -0.04, 0.06, 0.01, 0.6, 0.8, 1.0],
                    [0.10, 0.05, -0.05, 0.02, -0.08, 0.04, -0.9, 0.5, 0.7],
                    [0.02, 0.01, 0.03, 0.01, -0.02, 0.02, 0.05, 0.02, -0.03]])
    want = O.normal_order(cfg, **kw)
    assert np.abs(want).max(axis=(1, 2)).min() > 1e-30            # the matrices themselves are representable
    check_parity(emu.emu_eval(cfg, **kw), want)


# ----------------------------------------------------------------------------------------------
# caller-supplied angular rules (Gauss-Legendre radial x Lebedev angular)
# ----------------------------------------------------------------------------------------------
def test_octahedral_rules_integrate_monomials_exactly():
    from paper_2603_24532_b200 import angular_rules as A
    for deg, n_pts in ((3, 6), (5, 14), (7, 26), (9, 38), (11, 50), (15, 86)):
        d = A.octahedral_rule(deg)
        assert d.shape == (n_pts, 4) and (d[:, 3] > 0).all()
        assert np.abs(np.linalg.norm(d[:, :3], axis=1) - 1).max() < 1e-15
        assert A.check_rule(d, deg) < 5e-14                      # every monomial up to the degree
        assert A.check_rule(d, deg + 1) > 1e-6                   # and not beyond
    # octahedral symmetry of the point set: invariant under x -> -x and x <-> y
    d = A.octahedral_rule(15)
    key = lambda a: sorted(map(tuple, np.round(a, 12)))
    assert key(d * [-1, 1, 1, 1]) == key(d) and key(d[:, [1, 0, 2, 3]]) == key(d)
    p = A.product_rule(4, 5)
    assert p.shape == (20, 4) and abs(p[:, 3].sum() - 4 * np.pi) < 1e-14
    for k in (2, 4, 6):                                        # Gauss-Legendre in cos(theta): z^k exact
        assert abs(np.sum(p[:, 3] * p[:, 2] ** k) - 4 * np.pi / (k + 1)) < 1e-14


def test_product_rule_as_a_list_reproduces_the_grid_path():
    """the same nodes through the list path of the kernel arithmetic and through the cos x phi path."""
    from paper_2603_24532_b200 import angular_rules as A
    kw = dict(PHYS, c4=5.4, kf_n=1.3, kf_p=0.9, n_r=5)
    cfg = np.random.default_rng(9).uniform(-1, 1, (3, 9)) * 1.5
    grid = emu.emu_eval(cfg, n_cos=6, n_phi=7, **kw)
    lst = emu.emu_eval_angular(cfg, A.product_rule(6, 7), **kw)
    assert np.abs(grid - lst).max() < 1e-14 * np.abs(grid).max()
    check_parity(lst, O.normal_order(cfg, n_cos=6, n_phi=7, **kw))


@pytest.mark.parametrize("degree", [5, 15])
def test_kernel_arithmetic_with_a_lebedev_type_rule_matches_oracle(degree):
    from paper_2603_24532_b200 import angular_rules as A
    dirs = A.octahedral_rule(degree)                             # 14 and 86 directions: ragged over 32 lanes
    kw = dict(PHYS, c4=0.0, kf_n=1.3, kf_p=0.9, n_r=4)
    cfg = np.random.default_rng(11).uniform(-1, 1, (2, 9)) * 1.5
    want = O.normal_order(cfg, dirs=dirs, n_cos=1, n_phi=1, **kw)
    check_parity(emu.emu_eval_angular(cfg, dirs, **kw), want)
    assert emu.emu_eval_angular(cfg, dirs, **kw).shape == (2, 16, 16)


def test_lebedev_rule_converges_to_the_product_grid_result():
    """quadrature sanity (loose): 86 Lebedev-type directions and a 24 x 24 product grid agree to ~1e-4,
    far better than the 10 x 9 product grid with about the same number of directions."""
    from paper_2603_24532_b200 import angular_rules as A
    kw = dict(PHYS, c4=0.0, kf_n=1.2, kf_p=0.0, n_r=8, Lambda=500.0)
    cfg = np.array([[0.3, -0.2, 0.5, -0.1, 0.4, 0.2, 0.2, 0.1, -0.3]])
    fine = emu.emu_eval(cfg, n_cos=24, n_phi=24, **kw)
    leb = emu.emu_eval_angular(cfg, A.octahedral_rule(15), **kw)
    coarse = emu.emu_eval(cfg, n_cos=10, n_phi=9, **kw)
    e_leb = np.abs(leb - fine).max() / np.abs(fine).max()
    e_coarse = np.abs(coarse - fine).max() / np.abs(fine).max()
    assert e_leb < 1e-3 and e_leb < e_coarse


def test_empty_fermi_sea_gives_zero():
    out = emu.emu_eval(np.ones((2, 9)), kf_n=0.0, kf_p=0.0, n_r=2, n_cos=2, n_phi=2, **PHYS)
    assert np.count_nonzero(out) == 0


# ----------------------------------------------------------------------------------------------
# seeded synthetic workloads
# ----------------------------------------------------------------------------------------------
def test_workload_tables_match_baseline():
    evals = {n: W.workload(n).evals for n in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5")}
    assert evals["cfg1"] == 256 * 16 ** 3
    assert evals["cfg2"] == 12 * 8192 * 32 ** 3
    assert evals["cfg3"] == 65536 * 40 ** 3
    assert evals["cfg4"] == 131072 * 48 ** 3 * 2
    assert evals["cfg5"] == (1 << 20) * 64 ** 3 + (1 << 18) * 64 ** 3 * (1 + 2 + 2 + 2 + 1)
    r = W.workload("cfg4").runs[0]
    assert r.kf_n == pytest.approx(1.621540614038, abs=1e-11) and r.kf_p == pytest.approx(0.779555417944, abs=1e-11)
    assert (r.Lambda, r.n_reg, r.n_sph) == (450.0, 3, 2)
    kfs = [(q.kf_n, q.kf_p) for q in W.workload("cfg5").runs[1:]]
    want = [(2.116038959580, 0.0), (2.080166962512, 0.779555417944), (2.043013152886, 0.982178280627),
            (1.964356561255, 1.237467090512), (1.679501235221, 1.679501235221)]
    assert np.allclose(kfs, want, atol=1e-11)
    assert [q.n_sph for q in W.workload("cfg5").runs] == [1, 1, 2, 2, 2, 1]
    assert all(q.c4 == 0.0 for n in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5") for q in W.workload(n).runs)


def test_seeded_configurations_are_reproducible_and_in_range():
    r = W.workload("cfg2").runs[5]
    a = r.configurations(1000)
    assert np.array_equal(a, r.configurations(1000))
    assert np.array_equal(a[:100], r.configurations(100))              # a prefix of the same stream
    assert not np.array_equal(a[:100], W.workload("cfg2").runs[4].configurations(100))
    pn = np.linalg.norm(a[:, 0:3], axis=1)
    ppn = np.linalg.norm(a[:, 3:6], axis=1)
    Pn = np.linalg.norm(a[:, 6:9], axis=1)
    assert pn.max() < 4.0 and ppn.max() < 4.0 and Pn.max() < 2 * r.kf_n
    # uniform in the ball: <r^2>/R^2 = 3/5
    assert np.mean(pn ** 2) / 16.0 == pytest.approx(0.6, abs=0.03)
    assert np.mean(Pn ** 2) / (2 * r.kf_n) ** 2 == pytest.approx(0.6, abs=0.03)
    d = W.splitmix64_doubles(0, 0, 0, 5)
    assert np.array_equal(d, W.splitmix64_doubles(0, 0, 0, 8)[:5]) and (0 <= d).all() and (d < 1).all()
    assert np.array_equal(W.splitmix64_doubles(0, 0, 3, 2), W.splitmix64_doubles(0, 0, 0, 8)[3:5])


def test_angular_rule_with_non_unit_directions_is_refused():
    """The kernel relies on |u| = 1 (propagator polynomial in r, bound that elides the underflow guard):
    build_plan refuses a rule whose directions are not unit vectors instead of silently renormalising."""
    from paper_2603_24532_b200 import angular_rules as A
    kw = dict(PHYS, kf_n=1.2, kf_p=0.9, n_r=3)
    cfg = W.momentum_configurations(1, 0, 2, 1.5, 2.0)
    dirs = A.octahedral_rule(5)
    emu.emu_eval_angular(cfg, dirs, **kw)                       # accepted as generated
    bad = dirs.copy()
    bad[3, :3] *= 1.0 + 1e-9
    with pytest.raises(ValueError):
        emu.emu_eval_angular(cfg, bad, **kw)
    bad = dirs.copy()
    bad[0, :3] = 0.0
    with pytest.raises(ValueError):
        emu.emu_eval_angular(cfg, bad, **kw)


def test_host_logic_and_kernel_arithmetic_run_clean_under_sanitizers(tmp_path):
    """no_host.h + no_core.h (the product's planner and the kernel's arithmetic, compiled for the host) under
    -fsanitize=address,undefined: every kernel variant, both matter geometries, grid and direction list, maximum orders"""
    import os
    import subprocess
    here = os.path.dirname(__file__)
    exe = str(tmp_path / "host_emu_sanitized")
    subprocess.run(["g++", "-O1", "-g", "-std=c++17", "-ffp-contract=off", "-fsanitize=address,undefined",
                    "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-o", exe,
                    os.path.join(here, "host_emu_sanitize_main.cpp")], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
    assert "runs ok" in r.stdout
