"""Seeded synthetic inputs of the spin-isospin trace kernel: diagram topologies and vertex
matrices.  Shared by the CUDA path's callers and by the oracle's callers; holds NO arithmetic of the method (it only
lists which line leaves / enters which vertex and draws random matrix entries).

The paper's diagram tables live in its companion repository and are not in this container; the
topologies below are generated: particle-particle / hole-hole ladders and particle-hole rings of any order (the two
chain families of two-body MBPT diagrams), their slot-exchanged variants, relabelled copies, and random closed
topologies.  A topology is [n][4] line ids (out 1, out 2, in 1, in 2) per vertex (include/no_trace.h).

Vertex matrices stand in for the effective interactions the normal-ordering kernel produces: complex 16 x 16 with the
charge-conserving sparsity pattern of PAPER.md:174 (96 possibly non-zero entries), entries drawn from the SplitMix64
stream of workloads.py, uniform in [-1, 1) for the real and the imaginary part.
"""
from __future__ import annotations

import numpy as np

from .workloads import splitmix64_doubles


def ladder(n: int) -> np.ndarray:
    """n-th order ladder: both lines leaving vertex v enter vertex v + 1 (cyclically): T = Tr[V_{n-1} ... V_0]."""
    return np.array([[2 * v, 2 * v + 1, 2 * ((v - 1) % n), 2 * ((v - 1) % n) + 1] for v in range(n)], dtype=np.int32)


def ring(n: int) -> np.ndarray:
    """n-th order ring: slot 1 of vertex v is connected forward (to slot 1 of v + 1), slot 2 backward (to slot 2 of v - 1)."""
    return np.array([[2 * v, 2 * v + 1, 2 * ((v - 1) % n), 2 * ((v + 1) % n) + 1] for v in range(n)], dtype=np.int32)


def exchange_slots(topo: np.ndarray, out_mask: int = 0, in_mask: int = 0) -> np.ndarray:
    """swap the two outgoing (incoming) slots of every vertex whose bit is set in out_mask (in_mask)."""
    t = np.array(topo, dtype=np.int32).copy()
    for v in range(t.shape[0]):
        if out_mask >> v & 1:
            t[v, [0, 1]] = t[v, [1, 0]]
        if in_mask >> v & 1:
            t[v, [2, 3]] = t[v, [3, 2]]
    return t


def relabel(topo: np.ndarray, seed: int) -> np.ndarray:
    """the same diagram with the line ids permuted (seeded)."""
    t = np.array(topo, dtype=np.int32)
    n_lines = 2 * t.shape[0]
    perm = np.argsort(splitmix64_doubles(seed, 901, 0, n_lines), kind="stable").astype(np.int32)
    return perm[t]


def random_closed(n: int, seed: int) -> np.ndarray:
    """a random closed topology: the 2 n lines are dealt to the outgoing slots and, independently, to the incoming
    slots (may contain lines that start and end on the same vertex, and disconnected pieces)."""
    u = splitmix64_doubles(seed, 902, 0, 4 * n)
    outs = np.argsort(u[:2 * n], kind="stable").reshape(n, 2)
    ins = np.argsort(u[2 * n:], kind="stable").reshape(n, 2)
    return np.concatenate([outs, ins], axis=1).astype(np.int32)


def charge_conserving_mask() -> np.ndarray:
    """[16,16] bool: entries allowed by charge conservation, t1' + t2' = t1 + t2."""
    idx = np.arange(16)
    q = ((idx >> 1) & 1) + (idx & 1)
    return q[:, None] == q[None, :]


def vertex_matrices(n_sample: int, n_vertex: int, seed: int = 0, stream: int = 0, dense: bool = False) -> np.ndarray:
    """[n_sample, n_vertex, 16, 16] complex128, seeded; charge-conserving sparsity unless dense."""
    count = n_sample * n_vertex * 512
    u = 2.0 * splitmix64_doubles(seed, 1000 + stream, 0, count) - 1.0
    V = u.reshape(n_sample, n_vertex, 16, 16, 2)
    V = V[..., 0] + 1j * V[..., 1]
    if not dense:
        V = V * charge_conserving_mask()[None, None]
    return np.ascontiguousarray(V)


def pack_charge(V: np.ndarray) -> np.ndarray:
    """[..., 16, 16] -> [..., 96]: the NO_PACK_CHARGE layout of include/no.h (an index map, no arithmetic):
    entry 6 sp + nb, sp = 4 (2 s1' + s2') + (2 s1 + s2), nb over (pp,pp) (pn,pn) (np,np) (nn,nn) (pn,np) (np,pn)."""
    blocks = ((0, 0), (1, 1), (2, 2), (3, 3), (1, 2), (2, 1))
    rows = np.array([4 * (sp >> 2) + to for sp in range(16) for to, _ in blocks])
    cols = np.array([4 * (sp & 3) + ti for sp in range(16) for _, ti in blocks])
    return np.ascontiguousarray(np.asarray(V)[..., rows, cols])
