"""Host logic of the spin-isospin trace (paper_2603_24532_b200/csrc/no_trace_host.h): the planner and its tables, run by
a serial host emulation of the kernel's step program (tests/trace_emu.cpp) and compared with the brute-force oracle.
No GPU needed; the product itself has no CPU path (this emulation is test code)."""
import numpy as np
import pytest

from oracle import trace as T
from paper_2603_24532_b200 import trace_workloads as TW
from tests import trace_emu as E


def rel_err(got, want):
    return np.abs(got - want).max() / np.abs(want).max()


@pytest.mark.parametrize("name,topo", [(f"ladder{n}", TW.ladder(n)) for n in (1, 2, 3, 4, 5)] +
                         [(f"ring{n}", TW.ring(n)) for n in (2, 3, 4, 5)] +
                         [("ladder5x", TW.exchange_slots(TW.ladder(5), out_mask=0b01010, in_mask=0b00110)),
                          ("ring5x", TW.relabel(TW.exchange_slots(TW.ring(5), out_mask=0b10001), 3))])
def test_planned_program_equals_the_brute_force_trace_on_chains(name, topo):
    n = len(topo)
    V = TW.vertex_matrices(3, n, seed=1, stream=n)
    want = T.trace_bruteforce(topo, V)
    got = E.evaluate(topo, V)
    assert rel_err(got, want) < 1e-12, name
    # plan made for charge-conserving vertices: structurally zero tile products are skipped
    assert rel_err(E.evaluate(topo, V, charge=True), want) < 1e-12, name
    Vd = TW.vertex_matrices(2, n, seed=1, stream=50 + n, dense=True)
    assert rel_err(E.evaluate(topo, Vd), T.trace_bruteforce(topo, Vd)) < 1e-12, name
    pc = E.plan(topo, charge=True)
    p = E.plan(topo)
    if n >= 3:
        assert p["dmma_products"] == 64 * (n - 2) and pc["dmma_products"] == 16 * (n - 2), (p, pc)
    assert p["max_open"] <= 4
    if n >= 2:
        assert p["n_sliced"] == 0                                      # chains need no slicing
    if n >= 3:
        # first vertex opens its four lines, the middle ones are 16 x 16 x 16 products, the last closes all four
        assert p["steps"][0] == (1, 256, 1) and p["steps"][-1] == (1, 1, 256), p
        assert all(s == (16, 16, 16) for s in p["steps"][1:-1]), p
        assert p["cmacs"] == 256 + 4096 * (n - 2) + 256


@pytest.mark.parametrize("n,seed", [(n, s) for n in (2, 3, 4, 5) for s in range(6)] + [(6, 0), (6, 1)])
def test_planned_program_equals_the_brute_force_trace_on_random_topologies(n, seed):
    """random closed topologies: self-loops (always sliced), disconnected pieces, frontiers wider than four lines
    (sliced); dense vertices so that no term hides behind a structural zero."""
    topo = TW.random_closed(n, seed)
    p = E.plan(topo)
    assert p is not None, topo
    V = TW.vertex_matrices(2, n, seed=2, stream=10 * n + seed, dense=True)
    want = T.trace_bruteforce(topo, V)
    got = E.evaluate(topo, V)
    assert rel_err(got, want) < 1e-12, (topo, p)
    Vc = V * TW.charge_conserving_mask()
    assert rel_err(E.evaluate(topo, Vc, charge=True), T.trace_bruteforce(topo, Vc)) < 1e-12, (topo, p)
    assert p["max_open"] <= 4 and p["n_sliced"] <= 3
    assert p["n_isospin"] == T.isospin_configs(topo)
    assert sorted(p["order"]) == list(range(n))


def test_complete_graph_topology_needs_slicing_and_is_planned():
    """fifth order, every pair of vertices joined by exactly one line (the widest fifth-order frontier: 6 open lines):
    the planner fixes the labels of two lines in the outer loop."""
    n = 5
    outs = {v: [] for v in range(n)}
    ins = {v: [] for v in range(n)}
    line = 0
    for a in range(n):
        for b in range(a + 1, n):
            src, dst = (a, b) if (a + b) % 2 else (b, a)
            outs[src].append(line); ins[dst].append(line); line += 1
    assert all(len(outs[v]) == 2 and len(ins[v]) == 2 for v in range(n))
    topo = np.array([outs[v] + ins[v] for v in range(n)], dtype=np.int32)
    p = E.plan(topo)
    assert p is not None and p["n_sliced"] >= 1 and p["max_open"] <= 4
    V = TW.vertex_matrices(2, n, seed=3, dense=True)
    assert rel_err(E.evaluate(topo, V), T.trace_bruteforce(topo, V)) < 1e-12


def test_malformed_topologies_are_refused():
    assert E.plan([[0, 1, 0, 0]]) is None
    assert E.plan([[0, 1, 2, 3], [2, 3, 0, 4]]) is None
    assert E.plan(np.zeros((7, 4), dtype=np.int32)) is None


def test_planner_runs_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the product's host planner (no_trace_host.h) as a standalone program under -fsanitize=address,undefined: chains
    of order 1-6 and 300 pseudo-random closed topologies, with and without the charge flag; every tabulated offset
    must stay inside the kernel's shared-memory buffers"""
    import os
    import subprocess
    here = os.path.dirname(__file__)
    exe = str(tmp_path / "trace_plan_sanitized")
    subprocess.run(["g++", "-O1", "-g", "-std=c++17", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                    "-fno-omit-frame-pointer", "-o", exe, os.path.join(here, "trace_plan_sanitize_main.cpp")], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
    assert "plans ok" in r.stdout
