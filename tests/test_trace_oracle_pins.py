"""Pins of the brute-force spin-isospin trace oracle (oracle/trace_oracle.c) against what
the mathematics fixes.  None of these tests touches the CUDA path.  A plausible mistake in the oracle (rows and
columns transposed, slots 1 and 2 confused, spin and isospin bits of the pair index mixed up, a line summed twice or
not at all) fails at least one of them."""
import math

import numpy as np
import pytest

from oracle import trace as T
from paper_2603_24532_b200 import trace_workloads as TW

RNG = np.random.default_rng(20260325)


def rand_vertices(n_sample, n, dense=True):
    V = RNG.normal(size=(n_sample, n, 16, 16)) + 1j * RNG.normal(size=(n_sample, n, 16, 16))
    return V if dense else V * TW.charge_conserving_mask()


def pair(x1, x2):
    """pair index of include/no.h from the line labels x = 2 s + t."""
    return 8 * (x1 >> 1) + 4 * (x2 >> 1) + 2 * (x1 & 1) + (x2 & 1)


def product_vertex(A, B):
    """V[pair(x1',x2'), pair(x1,x2)] = A[x1',x1] B[x2',x2]: a one-body operator on each of the two particles."""
    V = np.zeros((16, 16), dtype=complex)
    for a in range(4):
        for b in range(4):
            for c in range(4):
                for d in range(4):
                    V[pair(a, b), pair(c, d)] = A[a, c] * B[b, d]
    return V


def p12():
    P = np.zeros((16, 16))
    for a in range(4):
        for b in range(4):
            P[pair(b, a), pair(a, b)] = 1.0
    return P


def test_second_order_ladder_is_the_trace_of_a_matrix_product():
    """n = 2: T = sum V_1[o;i] V_0[i;o] = Tr[V_1 V_0], computed with a library matrix product."""
    V = rand_vertices(3, 2)
    got = T.trace_bruteforce(TW.ladder(2), V)
    want = np.array([np.trace(V[s, 1] @ V[s, 0]) for s in range(3)])
    assert np.allclose(got, want, rtol=1e-13, atol=0)


@pytest.mark.parametrize("n", [1, 3, 4, 5])
def test_ladder_is_the_trace_of_the_ordered_matrix_product(n):
    """row = outgoing, column = incoming: the ladder chains to Tr[V_{n-1} ... V_1 V_0] (a transposed convention would
    give the reversed product, which differs for n >= 3)."""
    V = rand_vertices(2, n)
    got = T.trace_bruteforce(TW.ladder(n), V)
    for s in range(2):
        M = np.eye(16, dtype=complex)
        for v in range(n):
            M = V[s, v] @ M
        assert got[s] == pytest.approx(np.trace(M), rel=1e-12)
        if n >= 3:
            Mr = np.eye(16, dtype=complex)
            for v in range(n):
                Mr = Mr @ V[s, v]
            assert abs(got[s] - np.trace(Mr)) > 1e-6 * abs(got[s])


@pytest.mark.parametrize("n", [2, 3, 5])
def test_product_vertices_factorise_into_one_chain_per_fermion_loop(n):
    """With V_v = A_v (x) B_v the ring has two closed loops: slot 1 runs forward through the vertices, slot 2 backward:
    T = Tr[A_{n-1} ... A_0] Tr[B_0 B_1 ... B_{n-1}].  Fixes which slot a line is attached to and the bit layout
    (spin and isospin of one particle form one 4-valued label)."""
    A = RNG.normal(size=(n, 4, 4)) + 1j * RNG.normal(size=(n, 4, 4))
    B = RNG.normal(size=(n, 4, 4)) + 1j * RNG.normal(size=(n, 4, 4))
    V = np.array([[product_vertex(A[v], B[v]) for v in range(n)]])
    got = T.trace_bruteforce(TW.ring(n), V)[0]
    MA = np.eye(4, dtype=complex)
    MB = np.eye(4, dtype=complex)
    for v in range(n):
        MA = A[v] @ MA
        MB = MB @ B[v]
    assert got == pytest.approx(np.trace(MA) * np.trace(MB), rel=1e-12)


def count_loops(topo):
    """closed fermion loops when every vertex passes slot q in to slot q out."""
    topo = np.asarray(topo)
    n = topo.shape[0]
    nxt = {}
    for v in range(n):
        for q in range(2):
            nxt[topo[v, 2 + q]] = topo[v, q]           # the line entering slot q continues as the line leaving slot q
    seen, loops = set(), 0
    for l in range(2 * n):
        if l in seen:
            continue
        loops += 1
        while l not in seen:
            seen.add(l)
            l = nxt[l]
    return loops


@pytest.mark.parametrize("topo", [TW.ladder(4), TW.ring(4), TW.ring(5), TW.exchange_slots(TW.ladder(3), out_mask=0b010),
                                  TW.random_closed(4, 7), TW.random_closed(5, 3), TW.random_closed(3, 11)])
def test_identity_vertices_count_the_closed_loops(topo):
    """V = 1: every line label is copied through the vertices, T = 4^(number of closed loops)."""
    n = len(topo)
    V = np.broadcast_to(np.eye(16, dtype=complex), (1, n, 16, 16)).copy()
    assert T.trace_bruteforce(topo, V)[0] == pytest.approx(4.0 ** count_loops(topo), rel=1e-14)


def test_slot_exchange_is_p12_on_rows_or_columns():
    """exchanging the two outgoing (incoming) slots of a vertex = P12 applied to the rows (columns) of its matrix."""
    n = 4
    V = rand_vertices(1, n)
    P = p12()
    base = T.trace_bruteforce(TW.ring(n), V)[0]
    Vo = V.copy(); Vo[0, 2] = P @ V[0, 2]
    assert T.trace_bruteforce(TW.exchange_slots(TW.ring(n), out_mask=0b0100), Vo)[0] == pytest.approx(base, rel=1e-12)
    Vi = V.copy(); Vi[0, 1] = V[0, 1] @ P
    assert T.trace_bruteforce(TW.exchange_slots(TW.ring(n), in_mask=0b0010), Vi)[0] == pytest.approx(base, rel=1e-12)
    # without compensating the matrix the value changes
    assert abs(T.trace_bruteforce(TW.exchange_slots(TW.ring(n), out_mask=0b0100), V)[0] - base) > 1e-6 * abs(base)


def test_invariance_under_relabelling_of_lines_and_vertices_and_multilinearity():
    n = 4
    topo = TW.exchange_slots(TW.ring(n), out_mask=0b0001)
    V = rand_vertices(2, n)
    base = T.trace_bruteforce(topo, V)
    assert np.allclose(T.trace_bruteforce(TW.relabel(topo, 5), V), base, rtol=1e-12, atol=0)
    perm = [2, 0, 3, 1]                                 # vertices renumbered together with their matrices
    assert np.allclose(T.trace_bruteforce(topo[perm], V[:, perm]), base, rtol=1e-12, atol=0)
    cyc = [1, 2, 3, 0]
    assert np.allclose(T.trace_bruteforce(topo[cyc], V[:, cyc]), base, rtol=1e-12, atol=0)
    # linear in every vertex
    X = rand_vertices(2, n)
    for v in range(n):
        V2 = V.copy(); V2[:, v] = X[:, v]
        V3 = V.copy(); V3[:, v] = 2.0 * V[:, v] - 0.5j * X[:, v]
        assert np.allclose(T.trace_bruteforce(topo, V3), 2.0 * base - 0.5j * T.trace_bruteforce(topo, V2), rtol=1e-11, atol=0)


def test_charge_violating_vertex_gives_zero_and_isospin_subset_counts():
    """A vertex with entries only outside the 96 charge-conserving ones makes every term vanish when
    all other vertices conserve charge.  Charge-conserving isospin assignments: 34 for the fifth-order
    ladder (pp, nn, or one of pn/np between each of the 5 vertex pairs: 1 + 1 + 2^5), within the paper's "maximum
    count of 36 ... across all diagrams at fifth order"; 2^(2n) without the constraint."""
    n = 3
    V = rand_vertices(1, n, dense=False)
    bad = RNG.normal(size=(16, 16)) * ~TW.charge_conserving_mask()
    V[0, 1] = bad
    for topo in (TW.ladder(n), TW.ring(n)):
        assert abs(T.trace_bruteforce(topo, V)[0]) < 1e-13
    assert T.isospin_configs(TW.ladder(5)) == 34 <= 36
    assert T.isospin_configs(TW.ladder(6)) == 66 <= 72
    assert T.isospin_configs(TW.ladder(2)) == 1 + 1 + 4
    for n in (2, 3, 4, 5):
        # ring: brute-force count in numpy over all 2^(2n) assignments
        topo = TW.ring(n)
        cnt = 0
        for m in range(1 << (2 * n)):
            t = [(m >> j) & 1 for j in range(2 * n)]
            cnt += all(t[r[0]] + t[r[1]] == t[r[2]] + t[r[3]] for r in topo)
        assert T.isospin_configs(topo) == cnt
    # the sum restricted to charge-conserving assignments equals the full sum for charge-conserving vertices:
    # zeroing the other entries of dense vertices changes nothing in that restricted sum, so
    # T(dense masked) is the same number as summing only the allowed configurations
    Vd = rand_vertices(1, 3)
    full = T.trace_bruteforce(TW.ring(3), Vd * TW.charge_conserving_mask())[0]
    tot = 0.0
    topo = TW.ring(3)
    for m in range(1 << 6):
        t = [(m >> j) & 1 for j in range(6)]
        if not all(t[r[0]] + t[r[1]] == t[r[2]] + t[r[3]] for r in topo):
            continue
        for sm in range(1 << 6):
            s = [(sm >> j) & 1 for j in range(6)]
            x = [2 * s[j] + t[j] for j in range(6)]
            term = 1.0
            for v, r in enumerate(topo):
                term = term * Vd[0, v, pair(x[r[0]], x[r[1]]), pair(x[r[2]], x[r[3]])]
            tot += term
    assert full == pytest.approx(tot, rel=1e-12)


def test_trace_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """SURVEY.md section 5 for the second oracle: oracle/trace_oracle.c (included verbatim by
    tests/trace_oracle_sanitize_main.c) under -fsanitize=address,undefined, no report, every check held."""
    import os
    import subprocess
    here = os.path.dirname(__file__)
    exe = str(tmp_path / "trace_oracle_sanitized")
    subprocess.run(["gcc", "-O1", "-g", "-std=c99", "-fsanitize=address,undefined", "-fno-sanitize-recover=all",
                    "-fno-omit-frame-pointer", "-o", exe, os.path.join(here, "trace_oracle_sanitize_main.c"), "-lm"], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1"))
    assert r.returncode == 0, r.stdout + r.stderr
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr and "LeakSanitizer" not in r.stderr
    assert "trace oracle sanitized: ok" in r.stdout
