"""Convenience wrapper: a handle plus torch tensors (device memory and streams only)."""
from __future__ import annotations

import torch

from . import binding


class NormalOrdering:
    """`NormalOrdering(**no_params fields)`; `__call__(cfg)` -> complex128 [n,16,16] on the device.

    cfg: float64 tensor [n, 9] = (p, p', P) in fm^-1.  A CUDA tensor goes through no_eval on the
    current stream (asynchronous); a CPU tensor goes through no_eval_host (copies inside, blocks).
    angular: optional [n_dir, 4] array (ux, uy, uz, w) replacing the cos x phi grid (no_init_angular),
    e.g. `angular_rules.octahedral_rule(15)` for the paper's 86-point Lebedev-type rule.
    """

    def __init__(self, device: int = 0, angular=None, layout: int = 0, **params):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2603_24532_b200 needs a CUDA device (no CPU fallback)")
        self.device = device
        self.params = dict(params)
        self._h = binding.no_init(device=device, angular=angular, **params)
        if layout:
            binding.no_set_layout(self._h, layout)

    def close(self):
        if getattr(self, "_h", None) is not None:
            binding.no_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def evals_per_cfg(self) -> int:
        return binding.no_evals_per_cfg(self._h)

    def kernel_info(self) -> dict:
        return binding.no_kernel_info(self._h)

    def eval_into(self, cfg: torch.Tensor, out: torch.Tensor, stream: torch.cuda.Stream | None = None) -> None:
        """Enqueue no_eval: cfg [n,9] float64 CUDA, out [n,16,16,2] float64 CUDA (both contiguous)."""
        assert cfg.is_cuda and out.is_cuda and cfg.dtype == torch.float64 and out.dtype == torch.float64
        assert cfg.is_contiguous() and out.is_contiguous()
        n = cfg.shape[0]
        assert cfg.numel() == 9 * n and out.numel() == 512 * n
        s = stream if stream is not None else torch.cuda.current_stream(cfg.device)
        binding.no_eval(self._h, cfg.data_ptr(), n, out.data_ptr(), s.cuda_stream)

    def diag(self, cfg: torch.Tensor) -> torch.Tensor:
        """no_eval_diag: spin-traced diagonal per isospin pair, float64 [n, 4] (pp, pn, np, nn) on the device."""
        assert cfg.is_cuda
        cfg = cfg.to(torch.float64).contiguous().reshape(-1, 9)
        n = cfg.shape[0]
        out = torch.empty((n, 4), dtype=torch.float64, device=cfg.device)
        binding.no_eval_diag(self._h, cfg.data_ptr(), n, out.data_ptr(), torch.cuda.current_stream(cfg.device).cuda_stream)
        return out

    def packed(self, cfg: torch.Tensor, fmt: int = binding.NO_PACK_CHARGE) -> torch.Tensor:
        """no_eval_packed (CUDA cfg) or no_eval_host_packed (CPU cfg): complex128 [n, 96] (fmt 1: the charge-conserving
        entries) or [n, 32] (fmt 2: isospin-symmetric matter only), on the device of cfg."""
        cfg = cfg.to(torch.float64).contiguous().reshape(-1, 9)
        n = cfg.shape[0]
        pd = binding.no_packed_doubles(self._h, fmt)
        if pd == 0:
            raise ValueError("packed format does not apply to this handle (NO_PACK_ISOSPIN needs kF_n == kF_p)")
        out = torch.empty((n, pd // 2, 2), dtype=torch.float64, device=cfg.device)
        s = torch.cuda.current_stream(self.device).cuda_stream
        if cfg.is_cuda:
            binding.no_eval_packed(self._h, fmt, cfg.data_ptr(), n, out.data_ptr(), s)
        elif n:
            if fmt & binding.NO_PACK_FORWARD:
                raise ValueError("NO_PACK_FORWARD applies to device configurations (no_eval_packed) only")
            binding.no_eval_host_packed(self._h, fmt, cfg.data_ptr(), n, out.data_ptr(), s)
        return torch.view_as_complex(out)

    @staticmethod
    def unpack(packed: torch.Tensor, fmt: int = binding.NO_PACK_CHARGE) -> torch.Tensor:
        """no_unpack: packed complex128 CUDA tensor [n, 96 or 32] -> complex128 [n, 16, 16] on the same device."""
        assert packed.is_cuda and packed.dtype == torch.complex128 and packed.is_contiguous()
        n = packed.shape[0]
        out = torch.empty((n, 16, 16, 2), dtype=torch.float64, device=packed.device)
        with torch.cuda.device(packed.device):
            binding.no_unpack(fmt, packed.data_ptr(), n, out.data_ptr(), torch.cuda.current_stream(packed.device).cuda_stream)
        return torch.view_as_complex(out)

    def hf_energy(self, n_r: int, n_cos: int, n_phi: int) -> float:
        """no_hf_energy: 3N Hartree-Fock energy per volume (fm^-4) on the given grids for particles 1 and 2."""
        return binding.no_hf_energy(self._h, n_r, n_cos, n_phi, torch.cuda.current_stream(self.device).cuda_stream)

    def hf_energy_static(self, n_r: int, n_cos: int, n_phi: int) -> float:
        """no_hf_energy_static: hf_energy for callers that must not allocate GPU memory (workers sharing a GPU, hosts
        whose own pool owns all of HBM): intermediates in the library's fixed device array, n_r n_cos n_phi <= 4096."""
        return binding.no_hf_energy_static(self._h, n_r, n_cos, n_phi,
                                           torch.cuda.current_stream(self.device).cuda_stream)

    def sp_energy(self, k1, n_r: int, n_cos: int, n_phi: int):
        """no_sp_energy: 3N Hartree-Fock self-energy Sigma[n, 2] (proton, neutron; fm^-1) at momenta k1[n, 3]."""
        return binding.no_sp_energy(self._h, k1, n_r, n_cos, n_phi, torch.cuda.current_stream(self.device).cuda_stream)

    def __call__(self, cfg: torch.Tensor) -> torch.Tensor:
        cfg = cfg.to(torch.float64).contiguous().reshape(-1, 9)
        n = cfg.shape[0]
        if cfg.is_cuda:
            out = torch.empty((n, 16, 16, 2), dtype=torch.float64, device=cfg.device)
            self.eval_into(cfg, out)
        else:
            out = torch.empty((n, 16, 16, 2), dtype=torch.float64)
            if n:
                binding.no_eval_host(self._h, cfg.data_ptr(), n, out.data_ptr(),
                                     torch.cuda.current_stream(self.device).cuda_stream)
        return torch.view_as_complex(out)


class SpinIsospinTrace:
    """`SpinIsospinTrace(topo)`; `__call__(vertices)` -> complex128 [n_sample] on the device.

    topo: int array [n_vertex, 4] = line ids (out 1, out 2, in 1, in 2) of every vertex (include/no_trace.h).
    vertices: complex128 CUDA tensor [n_sample, n_vertex, 16, 16] (e.g. NormalOrdering output reshaped), contiguous.
    """

    def __init__(self, topo, device: int = 0, charge_conserving: bool = False):
        """charge_conserving: the vertex matrices are exactly zero outside the 96 charge-conserving entries (true for
        NormalOrdering output): structurally zero blocks are skipped (NO_TRACE_CHARGE_CONSERVING)."""
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2603_24532_b200 needs a CUDA device (no CPU fallback)")
        self.device = device
        self._p = binding.no_trace_init(topo, device, binding.NO_TRACE_CHARGE_CONSERVING if charge_conserving else 0)
        self.n_vertex = len(topo)

    def info(self) -> dict:
        return binding.no_trace_info(self._p, self.n_vertex)

    def eval_into(self, vertices: torch.Tensor, out: torch.Tensor, stream: torch.cuda.Stream | None = None) -> None:
        assert vertices.is_cuda and out.is_cuda and vertices.is_contiguous() and out.is_contiguous()
        assert vertices.dtype == torch.complex128 and out.dtype == torch.complex128
        n = out.numel()
        assert vertices.numel() == n * self.n_vertex * 256
        s = stream if stream is not None else torch.cuda.current_stream(vertices.device)
        binding.no_trace_eval(self._p, vertices.data_ptr(), n, out.data_ptr(), s.cuda_stream)

    def from_packed(self, packed: torch.Tensor, fmt: int = binding.NO_PACK_CHARGE) -> torch.Tensor:
        """no_trace_eval_packed: packed complex128 CUDA tensor [n_sample, n_vertex, 96] (fmt 1) or [n_sample, n_vertex, 32]
        (fmt 2, isospin-symmetric matter), i.e. NormalOrdering.packed(cfg, fmt) reshaped -> complex128 [n_sample]."""
        assert packed.is_cuda and packed.dtype == torch.complex128
        packed = packed.contiguous()
        per = 96 if fmt == binding.NO_PACK_CHARGE else 32
        n = packed.numel() // (self.n_vertex * per)
        assert packed.numel() == n * self.n_vertex * per
        out = torch.empty((n,), dtype=torch.complex128, device=packed.device)
        binding.no_trace_eval_packed(self._p, fmt, packed.data_ptr(), n, out.data_ptr(),
                                     torch.cuda.current_stream(packed.device).cuda_stream)
        return out

    def __call__(self, vertices: torch.Tensor) -> torch.Tensor:
        vertices = vertices.contiguous()
        n = vertices.numel() // (self.n_vertex * 256)
        out = torch.empty((n,), dtype=torch.complex128, device=vertices.device)
        self.eval_into(vertices, out)
        return out

    def close(self):
        if getattr(self, "_p", None) is not None:
            binding.no_trace_free(self._p)
            self._p = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
