"""paper_1806_04801_b200 -- B200-native (sm_100a) hot path of the harmonic surface mapping algorithm
(HSMA, arXiv 1806.04801): the fp64 direct Coulomb sums at the monitoring points, at all sources over
the near image cells, and at all sources from the sphere nodes (charge + dipole), joined by the
device least-squares solve and the harmonic-to-surface mapping.  See DESIGN.md and include/hsma.h.

The arithmetic lives in libhsma_b200.so (csrc/); `binding` marshals arguments; `Plan` is a small
convenience wrapper that owns a plan handle and allocates outputs with torch."""
from __future__ import annotations

from typing import Optional

import numpy as np
import torch

from . import binding
from .binding import *  # noqa: F401,F403  (the C entry points, same names)
from .binding import HsmaError


class Plan:
    """Owns an hsma_plan (preparation step).  evaluate() is the update step."""

    def __init__(self, *, kind: int, L, near_shell, R_aux: float, p: int, M: int, K: int, gamma: float = 1.0,
                 check_xyz=None, closure: int = 0, far_shell=(0, 0, 0), quad_rule: int = 0,
                 rsqrt_refine: int = 0, near_mode: int = 0, dipole_mode: int = 0, fd_dr_rel: float = 0.0,
                 near_algorithm: int = 0, fmm_order: int = 0, fmm_levels: int = 0, stream=None):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1806_04801_b200 needs a CUDA device (no CPU fallback)")
        self.handle = None
        # the stream the plan's kernels run on (the current torch stream unless given): shard.evaluate_distributed
        # orders its collectives against it
        self.torch_stream = stream if stream is not None else torch.cuda.current_stream()
        self.stream = int(self.torch_stream.cuda_stream)
        self.handle = binding.hsma_plan_create_ex(kind=kind, L=L, near_shell=near_shell, gamma=gamma, R_aux=R_aux,
                                                  p=p, M=M, K=K, check_xyz=check_xyz, closure=closure,
                                                  far_shell=far_shell, quad_rule=quad_rule,
                                                  rsqrt_refine=rsqrt_refine, near_mode=near_mode,
                                                  dipole_mode=dipole_mode, fd_dr_rel=fd_dr_rel,
                                                  near_algorithm=near_algorithm, fmm_order=fmm_order,
                                                  fmm_levels=fmm_levels, stream=stream)
        self.info = binding.hsma_plan_info(self.handle)

    @classmethod
    def from_workload(cls, w, **overrides) -> "Plan":
        """w: an hsma_workloads.Workload (plain parameters + inputs; holds none of the method's arithmetic)."""
        kw = dict(kind=w.kind, L=w.L, near_shell=w.near_shell, R_aux=w.R_aux, p=w.p, M=w.M, K=w.K, gamma=w.gamma,
                  check_xyz=w.check_xyz, closure=w.closure, far_shell=w.far_shell, quad_rule=w.quad_rule,
                  near_mode=getattr(w, "near_mode", 0), dipole_mode=getattr(w, "dipole_mode", 0),
                  fd_dr_rel=getattr(w, "fd_dr_rel", 0.0))
        kw.update(overrides)
        return cls(**kw)

    def close(self):
        if self.handle is not None:
            binding.hsma_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    # -- update step ---------------------------------------------------------------------------
    def evaluate(self, xyz: torch.Tensor, q: torch.Tensor, phi_out: Optional[torch.Tensor] = None,
                 energy_out: Optional[torch.Tensor] = None, sync: bool = False):
        N = q.numel()
        phi = phi_out if phi_out is not None else torch.empty(N, dtype=torch.float64, device=q.device)
        U = energy_out if energy_out is not None else torch.empty(1, dtype=torch.float64, device=q.device)
        binding.hsma_evaluate(self.handle, xyz, q, phi, U)
        if sync:
            binding.hsma_plan_sync(self.handle)
        return phi, U

    def evaluate_forces(self, xyz: torch.Tensor, q: torch.Tensor, sync: bool = False):
        """phi [N], F [N,3] = -q grad Phi, U [1]."""
        N = q.numel()
        phi = torch.empty(N, dtype=torch.float64, device=q.device)
        F = torch.empty(N, 3, dtype=torch.float64, device=q.device)
        U = torch.empty(1, dtype=torch.float64, device=q.device)
        binding.hsma_evaluate_forces(self.handle, xyz, q, phi, F, U)
        if sync:
            binding.hsma_plan_sync(self.handle)
        return phi, F, U

    def evaluate_forces_shard(self, xyz: torch.Tensor, q: torch.Tensor, t0: int, t1: int, sync: bool = False):
        T = max(t1 - t0, 0)
        phi = torch.empty(T, dtype=torch.float64, device=q.device)
        F = torch.empty(T, 3, dtype=torch.float64, device=q.device)
        U = torch.empty(1, dtype=torch.float64, device=q.device)
        binding.hsma_evaluate_forces_shard(self.handle, xyz, q, t0, t1, phi, F, U)
        if sync:
            binding.hsma_plan_sync(self.handle)
        return phi, F, U

    def evaluate_shard(self, xyz: torch.Tensor, q: torch.Tensor, t0: int, t1: int, sync: bool = False):
        phi = torch.empty(max(t1 - t0, 0), dtype=torch.float64, device=q.device)
        U = torch.empty(1, dtype=torch.float64, device=q.device)
        binding.hsma_evaluate_shard(self.handle, xyz, q, t0, t1, phi, U)
        if sync:
            binding.hsma_plan_sync(self.handle)
        return phi, U

    def evaluate_host(self, xyz: np.ndarray, q: np.ndarray, phi_out: Optional[np.ndarray] = None,
                      want_phi: bool = True):
        N = q.shape[0]
        phi = phi_out if phi_out is not None else (np.empty(N, dtype=np.float64) if want_phi else None)
        U = np.empty(1, dtype=np.float64)
        binding.hsma_evaluate_host(self.handle, xyz, q, phi, U)
        return phi, float(U[0])

    def sync(self):
        binding.hsma_plan_sync(self.handle)

    def set_timing(self, enable: bool = True):
        binding.hsma_plan_set_timing(self.handle, enable)

    def timing(self) -> dict:
        return binding.hsma_plan_get_timing(self.handle)

    def set_pair_form(self, form: int):
        """0: automatic; 1: ordered pairs always; 2: symmetric form of step (b) wherever it applies (forces too)."""
        binding.hsma_plan_set_pair_form(self.handle, form)

    def set_sym_scratch_cap(self, nbytes: int):
        """Bytes of column-sum scratch per wave of the symmetric form (0: default 64 MiB)."""
        binding.hsma_plan_set_sym_scratch_cap(self.handle, nbytes)

    def set_image_factoring(self, on: bool):
        """Lattice-factored image sums on (default) / off."""
        binding.hsma_plan_set_image_factoring(self.handle, on)

    @property
    def image_factoring(self) -> bool:
        return binding.hsma_plan_image_factoring(self.handle)

    @property
    def scratch_bytes(self) -> int:
        return binding.hsma_plan_scratch_bytes(self.handle)

    @property
    def last_pair_form(self) -> int:
        return binding.hsma_plan_last_pair_form(self.handle)

    # -- introspection (device tensors) ----------------------------------------------------------
    def _new(self, *shape):
        return torch.empty(*shape, dtype=torch.float64, device="cuda")

    def coeffs(self):
        A = self._new(self.info["p"] ** 2)
        binding.hsma_get_coeffs(self.handle, A)
        return A

    def rhs(self):
        r = self._new(self.info["rows"])
        binding.hsma_get_rhs(self.handle, r)
        return r

    def check_targets(self):
        x = self._new(self.info["check_targets"], 3)
        binding.hsma_get_check_targets(self.handle, x)
        return x

    def nodes(self):
        x, w = self._new(self.info["M"], 3), self._new(self.info["M"])
        binding.hsma_get_nodes(self.handle, x, w)
        return x, w

    def surface(self):
        Q, P = self._new(self.info["M"]), self._new(self.info["M"], 3)
        binding.hsma_get_surface(self.handle, Q, P)
        return Q, P

    def fit_residual(self) -> float:
        return binding.hsma_get_fit_residual(self.handle)

    def near_images_last_evaluate(self) -> int:
        return binding.hsma_plan_info(self.handle)["near_images_last_evaluate"]

    def launches_last_evaluate(self) -> int:
        return binding.hsma_plan_info(self.handle)["launches_last_evaluate"]
