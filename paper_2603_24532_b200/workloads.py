"""Seeded synthetic inputs and the five BASELINE.json workloads.

This module is the ONE piece shared by the CUDA path, the oracle's tests and
bench.py.  It holds no arithmetic of the method (no operator, regulator,
quadrature or trace): only

  * a counter-based SplitMix64 generator and the "uniform in a ball" sampler
    that draws the external momentum configurations (p, p', P), and
  * the table of workloads (Fermi momenta, low-energy constants, regulator,
    k3 grid orders, number of configurations) that BASELINE.json's `configs`
    and SURVEY.md section 8(d) spell out.

The paper measures on no public data set: in production the configurations are
Monte-Carlo-sampled vertex momenta of MBPT diagrams (PAPER.md:139-141, 186,
Sec. III).  The synthetic recipe below stands in for them.

Recipe:
  stream(seed, run)  : SplitMix64 with state0 = mix64(seed) + GOLDEN*mix64(run+1)
  double             : (x >> 11) * 2^-53  in [0, 1)
  vector in a ball   : candidate u = 2*(d0, d1, d2) - 1, accepted iff |u|^2 < 1
                       (three doubles are consumed per candidate, accepted or not);
                       the k-th accepted candidate is vector k of the stream
  configuration i    : vectors 3i, 3i+1, 3i+2 scaled by R_p, R_p, R_P  ->  p, p', P
                       with R_p = 4 fm^-1 and R_P = 2 max(kF_n, kF_p)   (R14)
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List

import numpy as np

_MASK = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15


def _mix64_int(z: int) -> int:
    z &= _MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return z ^ (z >> 31)


def _mix64(z: np.ndarray) -> np.ndarray:
    z = z.astype(np.uint64, copy=True)
    z ^= z >> np.uint64(30)
    z *= np.uint64(0xBF58476D1CE4E5B9)
    z ^= z >> np.uint64(27)
    z *= np.uint64(0x94D049BB133111EB)
    z ^= z >> np.uint64(31)
    return z


def splitmix64_doubles(seed: int, run: int, start: int, count: int) -> np.ndarray:
    """Doubles number start .. start+count-1 of stream (seed, run); each in [0, 1)."""
    state0 = (_mix64_int(seed) + _GOLDEN * _mix64_int(run + 1)) & _MASK
    idx = np.arange(start + 1, start + count + 1, dtype=np.uint64)
    with np.errstate(over="ignore"):
        state = np.uint64(state0) + idx * np.uint64(_GOLDEN)
        bits = _mix64(state)
    return (bits >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def unit_ball_vectors(seed: int, run: int, n_vec: int) -> np.ndarray:
    """First n_vec accepted candidates of stream (seed, run): points uniform in the unit ball."""
    out = np.empty((n_vec, 3), dtype=np.float64)
    have = 0
    consumed = 0  # candidates consumed so far
    while have < n_vec:
        want = n_vec - have
        n_cand = max(64, int(want * 2.05) + 16)  # acceptance is pi/6 = 0.5236
        d = splitmix64_doubles(seed, run, 3 * consumed, 3 * n_cand).reshape(n_cand, 3)
        u = 2.0 * d - 1.0
        ok = np.flatnonzero((u * u).sum(axis=1) < 1.0)
        if ok.size >= want:
            # stop exactly at the candidate that completed the request so that a
            # later, longer request walks the same stream
            ok = ok[:want]
        out[have:have + ok.size] = u[ok]
        have += ok.size
        consumed += n_cand
    return out


def momentum_configurations(seed: int, run: int, n_cfg: int, r_p: float, r_P: float) -> np.ndarray:
    """[n_cfg][9] doubles: p(xyz), p'(xyz), P(xyz) in fm^-1 (layout of no_eval's d_cfg)."""
    v = unit_ball_vectors(seed, run, 3 * n_cfg).reshape(n_cfg, 3, 3)
    v[:, 0, :] *= r_p
    v[:, 1, :] *= r_p
    v[:, 2, :] *= r_P
    return np.ascontiguousarray(v.reshape(n_cfg, 9))


def fermi_momentum(density: float) -> float:
    """kF = (3 pi^2 n_tau)^(1/3), Eq. (7); density of ONE species in fm^-3."""
    return (3.0 * math.pi ** 2 * density) ** (1.0 / 3.0) if density > 0.0 else 0.0


@dataclass(frozen=True)
class Run:
    """One no_init + no_eval call: one parameter set, one batch of configurations."""
    name: str
    kf_n: float
    kf_p: float
    n_cfg: int
    n_quad: int                  # k3 grid is n_quad^3 Gauss-Legendre (radial x cos x phi)
    Lambda: float = 500.0        # MeV
    n_reg: int = 4
    c1: float = -0.81            # GeV^-1
    c3: float = -3.2             # GeV^-1
    c4: float = 0.0              # GeV^-1 (R2: zero in all BASELINE configs)
    cD: float = 1.0
    cE: float = -0.5
    gA: float = 1.27
    fpi: float = 92.4            # MeV
    mpi: float = 138.04          # MeV
    lambda_chi: float = 700.0    # MeV (R3)
    seed: int = 0
    stream: int = 0              # run index of the sweep
    r_p: float = 4.0             # fm^-1
    angular_degree: int = 0      # > 0: n_quad radial points x the octahedral rule of that degree

    @property
    def n_sph(self) -> int:
        """Number of distinct non-zero Fermi momenta."""
        ks = {k for k in (self.kf_n, self.kf_p) if k > 0.0}
        return len(ks)

    @property
    def nodes_per_cfg(self) -> int:
        if self.angular_degree:
            return self.n_quad * len(self.angular()) * self.n_sph
        return self.n_quad ** 3 * self.n_sph

    def angular(self):
        """Direction list [n,4] for no_init_angular / the oracle's `dirs`, or None for the product grid."""
        if not self.angular_degree:
            return None
        from . import angular_rules
        return angular_rules.octahedral_rule(self.angular_degree)

    @property
    def evals(self) -> int:
        return self.n_cfg * self.nodes_per_cfg

    def params(self) -> dict:
        """Keyword arguments of no_init / the oracle (same names as include/no.h)."""
        return dict(kf_n=self.kf_n, kf_p=self.kf_p, c1=self.c1, c3=self.c3, c4=self.c4,
                    cD=self.cD, cE=self.cE, gA=self.gA, fpi=self.fpi, mpi=self.mpi,
                    lambda_chi=self.lambda_chi, Lambda=self.Lambda, n_reg=self.n_reg,
                    n_r=self.n_quad, n_cos=self.n_quad, n_phi=self.n_quad)

    def configurations(self, n: int | None = None) -> np.ndarray:
        n = self.n_cfg if n is None else n
        return momentum_configurations(self.seed, self.stream, n, self.r_p,
                                       2.0 * max(self.kf_n, self.kf_p))

    def shrunk(self, n_cfg: int, n_quad: int | None = None) -> "Run":
        return replace(self, n_cfg=n_cfg, n_quad=self.n_quad if n_quad is None else n_quad)


@dataclass(frozen=True)
class Workload:
    name: str
    description: str
    runs: List[Run] = field(default_factory=list)

    @property
    def evals(self) -> int:
        return sum(r.evals for r in self.runs)

    @property
    def n_cfg(self) -> int:
        return sum(r.n_cfg for r in self.runs)


def _asym(total_density: float, x: float):
    return fermi_momentum((1.0 - x) * total_density), fermi_momentum(x * total_density)


def workload(name: str) -> Workload:
    """The five BASELINE.json configs ("cfg1" .. "cfg5") and the extra c4 case ("c4")."""
    if name == "cfg1":
        return Workload(name, "PNM kF_n=1.0, 256 configurations, 16^3 grid",
                        [Run("pnm_kf1.0", 1.0, 0.0, 256, 16)])
    if name == "cfg2":
        runs = []
        i = 0
        for kf in (1.0, 1.2, 1.4, 1.6, 1.8, 2.0):
            for lam in (450.0, 500.0):
                runs.append(Run(f"pnm_kf{kf:.1f}_L{int(lam)}", kf, 0.0, 8192, 32, Lambda=lam, stream=i))
                i += 1
        return Workload(name, "PNM density sweep kF_n in {1.0..2.0} x Lambda in {450,500}, "
                              "8192 configurations each, 32^3 grid", runs)
    if name == "cfg3":
        return Workload(name, "SNM kF=1.33, 65536 configurations, 40^3 grid",
                        [Run("snm_kf1.33", 1.33, 1.33, 65536, 40)])
    if name == "cfg4":
        kn, kp = _asym(0.16, 0.1)
        return Workload(name, "asymmetric matter x=0.1 at n=0.16 fm^-3, 131072 configurations, "
                              "48^3 grid x 2 spheres, Lambda=450, n_reg=3",
                        [Run("asym_x0.1_n0.16", kn, kp, 131072, 48, Lambda=450.0, n_reg=3)])
    if name == "cfg5":
        runs = [Run("snm_kf1.6", 1.6, 1.6, 1 << 20, 64, stream=0)]
        for i, x in enumerate((0.0, 0.05, 0.1, 0.2, 0.5)):
            kn, kp = _asym(0.32, x)
            if x == 0.5:
                kp = kn  # exact SNM: one fused sphere (cube roots of equal densities)
            runs.append(Run(f"nsm_x{x:g}_n0.32", kn, kp, 1 << 18, 64, stream=i + 1))
        return Workload(name, "SNM kF=1.6 with 2^20 configurations + n=0.32 fm^-3 at "
                              "x in {0,.05,.1,.2,.5} with 2^18 each, 64^3 grid", runs)
    if name == "c4":
        # R2: the c4 part of the two-pion-exchange topology, exercised in one extra SNM case
        return Workload(name, "SNM kF=1.33 with c4=+5.4 GeV^-1 (extra parity case, R2)",
                        [Run("snm_kf1.33_c4", 1.33, 1.33, 1024, 24, c4=5.4, stream=7)])
    if name == "paper":
        # the paper's own production quadrature: 16 Gauss-Legendre radial points x the
        # order-15, 86-point Lebedev-type angular rule; SNM at n = 0.16 fm^-3
        return Workload(name, "SNM kF=1.33, 2^20 configurations, 16 radial x 86-point degree-15 angular rule "
                              "(the paper's quadrature)",
                        [Run("snm_kf1.33_leb15", 1.33, 1.33, 1 << 20, 16, angular_degree=15, stream=9)])
    raise KeyError(name)


WORKLOAD_NAMES = ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "c4", "paper")
