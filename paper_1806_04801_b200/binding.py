"""ctypes binding of include/hsma.h -- argument marshalling only.

Every function has the name of the C entry point it calls; torch tensors are used for device
memory (their data_ptr() is passed through) and for the CUDA stream.  Nothing of the method is
computed here, and nothing here imports oracle/.  If libhsma_b200.so is missing and cannot be
built the import fails loudly: there is no CPU fallback."""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

from . import build as _build

c_double_p = ctypes.POINTER(ctypes.c_double)

HSMA_OK = 0
HSMA_ERR_INVALID_ARG, HSMA_ERR_GEOMETRY, HSMA_ERR_NOT_NEUTRAL = -1, -2, -3
HSMA_ERR_CUDA, HSMA_ERR_ALLOC, HSMA_ERR_RANK_DEFICIENT = -4, -5, -6
HSMA_ERR_TOO_LARGE = -7
HSMA_BC_PERIODIC, HSMA_BC_MIRROR_CAVITY, HSMA_BC_SLAB_XY_PERIODIC_Z_MIRROR = 0, 1, 2
HSMA_CLOSURE_BOUNDARY, HSMA_CLOSURE_FAR_DATA, HSMA_CLOSURE_FACE_PAIRS = 0, 1, 2
HSMA_QUAD_SPIRAL, HSMA_QUAD_LATTICE = 0, 1
HSMA_NEAR_WHOLE_CELLS, HSMA_NEAR_SPHERE = 0, 1
HSMA_DIPOLE_EXACT, HSMA_DIPOLE_FD3 = 0, 1


class hsma_plan_desc(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_size_t), ("kind", ctypes.c_int), ("L", ctypes.c_double * 3),
                ("near_shell", ctypes.c_int * 3), ("gamma", ctypes.c_double), ("R_aux", ctypes.c_double),
                ("p", ctypes.c_int), ("M", ctypes.c_int), ("K", ctypes.c_int), ("check_xyz", c_double_p),
                ("closure", ctypes.c_int), ("far_shell", ctypes.c_int * 3), ("quad_rule", ctypes.c_int),
                ("rsqrt_refine", ctypes.c_int), ("near_mode", ctypes.c_int), ("dipole_mode", ctypes.c_int),
                ("fd_dr_rel", ctypes.c_double), ("near_algorithm", ctypes.c_int), ("fmm_order", ctypes.c_int),
                ("fmm_levels", ctypes.c_int)]


class HsmaError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {hsma_status_string(status)} ({status})")


_lib = None

_SIGNATURES = {
    "hsma_plan_create": (ctypes.c_int, [ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int,
                                        ctypes.c_int, ctypes.c_void_p, ctypes.POINTER(ctypes.c_void_p)]),
    "hsma_plan_create_ex": (ctypes.c_int, [ctypes.POINTER(hsma_plan_desc), ctypes.c_void_p,
                                           ctypes.POINTER(ctypes.c_void_p)]),
    "hsma_plan_destroy": (ctypes.c_int, [ctypes.c_void_p]),
    "hsma_evaluate": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                     ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_evaluate_shard": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                           ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_evaluate_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                          ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_evaluate_shard_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                                ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p,
                                                ctypes.c_void_p]),
    "hsma_evaluate_forces": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_evaluate_forces_shard": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                                  ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p,
                                                  ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_evaluate_forces_host": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                                 ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_check_sums_shard": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                             ctypes.c_longlong, ctypes.c_longlong]),
    "hsma_get_check_sums": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p,
                                           ctypes.c_void_p]),
    "hsma_set_check_sums": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p,
                                           ctypes.c_void_p]),
    "hsma_evaluate_rest_shard": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                                ctypes.c_longlong, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                                ctypes.c_void_p]),
    "hsma_plan_sync": (ctypes.c_int, [ctypes.c_void_p]),
    "hsma_status_string": (ctypes.c_char_p, [ctypes.c_int]),
    "hsma_plan_info": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_longlong)]),
    "hsma_get_coeffs": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_get_rhs": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_get_check_targets": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_get_nodes": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_get_surface": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_get_fit_residual": (ctypes.c_int, [ctypes.c_void_p, c_double_p]),
    "hsma_direct_sum": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                       ctypes.c_longlong, c_double_p, c_double_p, c_double_p, ctypes.c_int,
                                       ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_void_p,
                                       ctypes.c_void_p]),
    "hsma_direct_sum_static": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                              ctypes.c_longlong, c_double_p, c_double_p, c_double_p, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_void_p,
                                              ctypes.c_void_p]),
    "hsma_static_scratch_setup": (ctypes.c_int, []),
    "hsma_static_scratch_bytes": (ctypes.c_longlong, []),
    "hsma_static_scratch_fill": (ctypes.c_int, [ctypes.c_int, ctypes.c_void_p]),
    "hsma_node_sum": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                     ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_direct_field": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                         ctypes.c_longlong, c_double_p, c_double_p, c_double_p, ctypes.c_int,
                                         ctypes.c_int, ctypes.c_longlong, ctypes.c_int, ctypes.c_void_p,
                                         ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_node_field": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                       ctypes.c_void_p, ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
                                       ctypes.c_void_p]),
    "hsma_fp64_peak": (ctypes.c_int, [ctypes.c_double, c_double_p, c_double_p]),
    "hsma_evaluate_rest_part": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong,
                                               ctypes.c_int, ctypes.c_int, ctypes.c_longlong, ctypes.c_longlong,
                                               ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]),
    "hsma_plan_part_form_applies": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong]),
    "hsma_plan_set_timing": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "hsma_plan_set_pair_form": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "hsma_plan_last_pair_form": (ctypes.c_int, [ctypes.c_void_p]),
    "hsma_plan_set_sym_scratch_cap": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_longlong]),
    "hsma_plan_scratch_bytes": (ctypes.c_longlong, [ctypes.c_void_p]),
    "hsma_plan_set_image_factoring": (ctypes.c_int, [ctypes.c_void_p, ctypes.c_int]),
    "hsma_plan_image_factoring": (ctypes.c_int, [ctypes.c_void_p]),
    "hsma_plan_fmm_info": (ctypes.c_int, [ctypes.c_void_p, ctypes.POINTER(ctypes.c_longlong)]),
    "hsma_plan_get_timing": (ctypes.c_int, [ctypes.c_void_p, c_double_p]),
    "hsma_launch_count": (ctypes.c_longlong, []),
}
EXPORTS = tuple(_SIGNATURES)


def library_path() -> str:
    return _build.LIB


def load_library() -> ctypes.CDLL:
    """Load (building first if stale) libhsma_b200.so.  Raises if it cannot be had."""
    global _lib
    if _lib is None:
        path = _build.build()
        if not os.path.exists(path):
            raise RuntimeError("libhsma_b200.so missing: the CUDA extension is required (no CPU fallback)")
        lib = ctypes.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def hsma_status_string(status: int) -> str:
    return load_library().hsma_status_string(int(status)).decode()


def _check(status: int, where: str):
    if status != HSMA_OK:
        raise HsmaError(status, where)


def _dev(t: Optional[torch.Tensor], n: Optional[int] = None, name: str = "tensor") -> Optional[int]:
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name}: need a contiguous float64 CUDA tensor")
    if n is not None and t.numel() < n:
        raise ValueError(f"{name}: {t.numel()} elements, need {n}")
    return t.data_ptr()


def _host(a, name="array") -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def _hp(a: np.ndarray):
    return a.ctypes.data_as(c_double_p)


def _stream_ptr(stream) -> Optional[int]:
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream or None


def hsma_plan_create(L: float, boundary_kind: int, near_shell: int, R_aux: float, p: int, M_fib: int,
                     stream=None) -> int:
    h = ctypes.c_void_p()
    _check(load_library().hsma_plan_create(L, boundary_kind, near_shell, R_aux, p, M_fib, _stream_ptr(stream),
                                           ctypes.byref(h)), "hsma_plan_create")
    return h.value


def hsma_plan_create_ex(*, kind: int, L: Sequence[float], near_shell: Sequence[int], gamma: float, R_aux: float,
                        p: int, M: int, K: int, check_xyz=None, closure: int = 0, far_shell=(0, 0, 0),
                        quad_rule: int = 0, rsqrt_refine: int = 0, near_mode: int = 0, dipole_mode: int = 0,
                        fd_dr_rel: float = 0.0, near_algorithm: int = 0, fmm_order: int = 0, fmm_levels: int = 0,
                        stream=None) -> int:
    d = hsma_plan_desc()
    d.struct_size = ctypes.sizeof(hsma_plan_desc)
    d.kind = kind
    d.L[:] = [float(v) for v in L]
    d.near_shell[:] = [int(v) for v in near_shell]
    d.gamma, d.R_aux, d.p, d.M, d.K = float(gamma), float(R_aux), int(p), int(M), int(K)
    keep = None
    if check_xyz is not None:
        keep = _host(check_xyz)
        if keep.shape != (K, 3):
            raise ValueError("check_xyz must be [K,3]")
        d.check_xyz = _hp(keep)
    d.closure = closure
    d.far_shell[:] = [int(v) for v in far_shell]
    d.quad_rule, d.rsqrt_refine = int(quad_rule), int(rsqrt_refine)
    d.near_mode, d.dipole_mode, d.fd_dr_rel = int(near_mode), int(dipole_mode), float(fd_dr_rel)
    d.near_algorithm, d.fmm_order, d.fmm_levels = int(near_algorithm), int(fmm_order), int(fmm_levels)
    h = ctypes.c_void_p()
    _check(load_library().hsma_plan_create_ex(ctypes.byref(d), _stream_ptr(stream), ctypes.byref(h)),
           "hsma_plan_create_ex")
    return h.value


def hsma_plan_destroy(plan: int):
    _check(load_library().hsma_plan_destroy(plan), "hsma_plan_destroy")


def hsma_evaluate(plan: int, xyz: torch.Tensor, q: torch.Tensor, phi_out: torch.Tensor,
                  energy_out: Optional[torch.Tensor] = None):
    N = q.numel()
    _check(load_library().hsma_evaluate(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N, _dev(phi_out, N, "phi_out"),
                                        _dev(energy_out, 1, "energy_out")), "hsma_evaluate")


def hsma_evaluate_shard(plan: int, xyz: torch.Tensor, q: torch.Tensor, t0: int, t1: int, phi_out: torch.Tensor,
                        energy_out: Optional[torch.Tensor] = None):
    N = q.numel()
    _check(load_library().hsma_evaluate_shard(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N, t0, t1,
                                              _dev(phi_out, max(t1 - t0, 0), "phi_out"),
                                              _dev(energy_out, 1, "energy_out")), "hsma_evaluate_shard")


def hsma_evaluate_host(plan: int, xyz: np.ndarray, q: np.ndarray, phi_out: Optional[np.ndarray],
                       energy_out: Optional[np.ndarray]):
    """xyz [N,3], q [N], phi_out [N], energy_out [1]: C-contiguous float64 HOST arrays (pinned or not)."""
    for a in (xyz, q, phi_out, energy_out):
        if a is not None and not (a.dtype == np.float64 and a.flags.c_contiguous):
            raise TypeError("host buffers must be C-contiguous float64")
    N = q.shape[0]
    _check(load_library().hsma_evaluate_host(plan, xyz.ctypes.data, q.ctypes.data, N,
                                             None if phi_out is None else phi_out.ctypes.data,
                                             None if energy_out is None else energy_out.ctypes.data),
           "hsma_evaluate_host")


def hsma_evaluate_shard_host(plan: int, xyz: np.ndarray, q: np.ndarray, t0: int, t1: int,
                             phi_out: Optional[np.ndarray], energy_out: Optional[np.ndarray]):
    """As hsma_evaluate_host for the targets t0 <= i < t1: phi_out [t1-t0]."""
    for a in (xyz, q, phi_out, energy_out):
        if a is not None and not (a.dtype == np.float64 and a.flags.c_contiguous):
            raise TypeError("host buffers must be C-contiguous float64")
    if phi_out is not None and phi_out.shape[0] < t1 - t0:
        raise ValueError("phi_out too small")
    N = q.shape[0]
    _check(load_library().hsma_evaluate_shard_host(plan, xyz.ctypes.data, q.ctypes.data, N, t0, t1,
                                                   None if phi_out is None else phi_out.ctypes.data,
                                                   None if energy_out is None else energy_out.ctypes.data),
           "hsma_evaluate_shard_host")


def hsma_evaluate_forces(plan: int, xyz: torch.Tensor, q: torch.Tensor, phi_out: Optional[torch.Tensor],
                         force_out: torch.Tensor, energy_out: Optional[torch.Tensor] = None):
    N = q.numel()
    _check(load_library().hsma_evaluate_forces(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N,
                                               _dev(phi_out, N, "phi_out"), _dev(force_out, 3 * N, "force_out"),
                                               _dev(energy_out, 1, "energy_out")), "hsma_evaluate_forces")


def hsma_evaluate_forces_shard(plan: int, xyz: torch.Tensor, q: torch.Tensor, t0: int, t1: int,
                               phi_out: Optional[torch.Tensor], force_out: torch.Tensor,
                               energy_out: Optional[torch.Tensor] = None):
    N, T = q.numel(), max(t1 - t0, 0)
    _check(load_library().hsma_evaluate_forces_shard(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N, t0, t1,
                                                     _dev(phi_out, T, "phi_out"), _dev(force_out, 3 * T, "force_out"),
                                                     _dev(energy_out, 1, "energy_out")), "hsma_evaluate_forces_shard")


def hsma_evaluate_forces_host(plan: int, xyz: np.ndarray, q: np.ndarray, phi_out: Optional[np.ndarray],
                              force_out: np.ndarray, energy_out: Optional[np.ndarray]):
    """HOST arrays: xyz [N,3], q [N], phi_out [N] or None, force_out [N,3], energy_out [1] or None."""
    for a in (xyz, q, phi_out, force_out, energy_out):
        if a is not None and not (a.dtype == np.float64 and a.flags.c_contiguous):
            raise TypeError("host buffers must be C-contiguous float64")
    N = q.shape[0]
    if force_out.size < 3 * N:
        raise ValueError("force_out too small")
    _check(load_library().hsma_evaluate_forces_host(plan, xyz.ctypes.data, q.ctypes.data, N,
                                                    None if phi_out is None else phi_out.ctypes.data,
                                                    force_out.ctypes.data,
                                                    None if energy_out is None else energy_out.ctypes.data),
           "hsma_evaluate_forces_host")


def hsma_check_sums_shard(plan: int, xyz: torch.Tensor, q: torch.Tensor, c0: int, c1: int):
    N = q.numel()
    _check(load_library().hsma_check_sums_shard(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N, c0, c1),
           "hsma_check_sums_shard")


def hsma_get_check_sums(plan: int, c0: int, c1: int, pc_out: torch.Tensor, pcg_out: Optional[torch.Tensor] = None):
    _check(load_library().hsma_get_check_sums(plan, c0, c1, _dev(pc_out, c1 - c0, "pc_out"),
                                              _dev(pcg_out, 3 * (c1 - c0), "pcg_out")), "hsma_get_check_sums")


def hsma_set_check_sums(plan: int, c0: int, c1: int, pc_in: torch.Tensor, pcg_in: Optional[torch.Tensor] = None):
    _check(load_library().hsma_set_check_sums(plan, c0, c1, _dev(pc_in, c1 - c0, "pc_in"),
                                              _dev(pcg_in, 3 * (c1 - c0), "pcg_in")), "hsma_set_check_sums")


def hsma_evaluate_rest_shard(plan: int, xyz: torch.Tensor, q: torch.Tensor, t0: int, t1: int,
                             phi_out: Optional[torch.Tensor], force_out: Optional[torch.Tensor],
                             energy_out: Optional[torch.Tensor] = None):
    N, T = q.numel(), max(t1 - t0, 0)
    _check(load_library().hsma_evaluate_rest_shard(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N, t0, t1,
                                                   _dev(phi_out, T, "phi_out"), _dev(force_out, 3 * T, "force_out"),
                                                   _dev(energy_out, 1, "energy_out")), "hsma_evaluate_rest_shard")


def hsma_evaluate_rest_part(plan: int, xyz: torch.Tensor, q: torch.Tensor, part: int, n_parts: int, t0: int, t1: int,
                            phi_part_out: Optional[torch.Tensor], force_part_out: Optional[torch.Tensor] = None,
                            energy_part_out: Optional[torch.Tensor] = None):
    """PART form of the last multi-GPU step: partial phi (and F) over all N targets and partial U (sums over the
    parts = the result)."""
    N = q.numel()
    _check(load_library().hsma_evaluate_rest_part(plan, _dev(xyz, 3 * N, "xyz"), _dev(q, N, "q"), N, int(part), int(n_parts),
                                                  t0, t1, _dev(phi_part_out, N, "phi_part_out"),
                                                  _dev(force_part_out, 3 * N, "force_part_out"),
                                                  _dev(energy_part_out, 1, "energy_part_out")), "hsma_evaluate_rest_part")


def hsma_plan_part_form_applies(plan: int, N: int) -> bool:
    return bool(load_library().hsma_plan_part_form_applies(plan, int(N)))


def hsma_plan_sync(plan: int):
    _check(load_library().hsma_plan_sync(plan), "hsma_plan_sync")


def hsma_plan_info(plan: int) -> dict:
    w = (ctypes.c_longlong * 12)()
    _check(load_library().hsma_plan_info(plan, w), "hsma_plan_info")
    keys = ("rows", "cols", "check_targets", "near_cells", "rhs_cells", "M", "p", "launches_last_evaluate",
            "near_images_last_evaluate", "node_records", "check_gradient", "graph_replays")
    return dict(zip(keys, [int(v) for v in w]))


def hsma_plan_needs_check_gradient(plan: int) -> bool:
    """True if the fit has derivative rows (Neumann walls, face-pair closure): hsma_get/set_check_sums then also move pcg."""
    return bool(hsma_plan_info(plan)["check_gradient"])


def hsma_get_coeffs(plan: int, A_out: torch.Tensor):
    _check(load_library().hsma_get_coeffs(plan, _dev(A_out)), "hsma_get_coeffs")


def hsma_get_rhs(plan: int, rhs_out: torch.Tensor):
    _check(load_library().hsma_get_rhs(plan, _dev(rhs_out)), "hsma_get_rhs")


def hsma_get_check_targets(plan: int, xyz_out: torch.Tensor):
    _check(load_library().hsma_get_check_targets(plan, _dev(xyz_out)), "hsma_get_check_targets")


def hsma_get_nodes(plan: int, xyz_out: Optional[torch.Tensor], w_out: Optional[torch.Tensor]):
    _check(load_library().hsma_get_nodes(plan, _dev(xyz_out), _dev(w_out)), "hsma_get_nodes")


def hsma_get_surface(plan: int, Q_out: Optional[torch.Tensor], P_out: Optional[torch.Tensor]):
    _check(load_library().hsma_get_surface(plan, _dev(Q_out), _dev(P_out)), "hsma_get_surface")


def hsma_get_fit_residual(plan: int) -> float:
    v = ctypes.c_double()
    _check(load_library().hsma_get_fit_residual(plan, ctypes.byref(v)), "hsma_get_fit_residual")
    return v.value


def hsma_direct_sum(tgt: torch.Tensor, src: torch.Tensor, q: torch.Tensor, shift, sign, w, central_cell: int,
                    self_offset: int, refine: int, phi_out: torch.Tensor, stream=None):
    shift, sign, w = _host(shift), _host(sign), _host(w)
    T, N, C = tgt.shape[0], q.numel(), w.shape[0]
    _check(load_library().hsma_direct_sum(_dev(tgt, 3 * T, "tgt"), T, _dev(src, 3 * N, "src"), _dev(q, N, "q"), N,
                                          _hp(shift), _hp(sign), _hp(w), C, central_cell, self_offset, refine,
                                          _dev(phi_out, T, "phi_out"), _stream_ptr(stream)), "hsma_direct_sum")


def hsma_direct_sum_static(tgt: torch.Tensor, src: torch.Tensor, q: torch.Tensor, shift, sign, w, central_cell: int,
                           self_offset: int, refine: int, phi_out: torch.Tensor, stream=None):
    """hsma_direct_sum without any device allocation: scratch in the library's fixed 16 MiB device array (N, T <= 65,536,
    C <= 32; HSMA_ERR_TOO_LARGE beyond).  Asynchronous on `stream`; overlapping calls race on the scratch.  include/hsma.h."""
    shift, sign, w = _host(shift), _host(sign), _host(w)
    T, N, C = tgt.shape[0], q.numel(), w.shape[0]
    _check(load_library().hsma_direct_sum_static(_dev(tgt, 3 * T, "tgt"), T, _dev(src, 3 * N, "src"), _dev(q, N, "q"), N,
                                                 _hp(shift), _hp(sign), _hp(w), C, central_cell, self_offset, refine,
                                                 _dev(phi_out, T, "phi_out"), _stream_ptr(stream)), "hsma_direct_sum_static")


def hsma_static_scratch_setup():
    """Look up the fixed scratch array's address on the current device (once per device; e.g. before a graph capture)."""
    _check(load_library().hsma_static_scratch_setup(), "hsma_static_scratch_setup")


def hsma_static_scratch_bytes() -> int:
    return int(load_library().hsma_static_scratch_bytes())


def hsma_static_scratch_fill(byte: int, stream=None):
    """Test hook: overwrite the fixed scratch array with `byte` (0xFF: NaNs) on `stream`."""
    _check(load_library().hsma_static_scratch_fill(int(byte), _stream_ptr(stream)), "hsma_static_scratch_fill")


def hsma_node_sum(tgt: torch.Tensor, R: torch.Tensor, Q: torch.Tensor, P: torch.Tensor, phi_out: torch.Tensor,
                  stream=None):
    T, M = tgt.shape[0], Q.numel()
    _check(load_library().hsma_node_sum(_dev(tgt, 3 * T, "tgt"), T, _dev(R, 3 * M, "R"), _dev(Q, M, "Q"),
                                        _dev(P, 3 * M, "P"), M, _dev(phi_out, T, "phi_out"), _stream_ptr(stream)),
           "hsma_node_sum")


def hsma_direct_field(tgt: torch.Tensor, src: torch.Tensor, q: torch.Tensor, shift, sign, w, central_cell: int,
                      self_offset: int, refine: int, phi_out: Optional[torch.Tensor], grad_out: torch.Tensor, stream=None):
    shift, sign, w = _host(shift), _host(sign), _host(w)
    T, N, C = tgt.shape[0], q.numel(), w.shape[0]
    _check(load_library().hsma_direct_field(_dev(tgt, 3 * T, "tgt"), T, _dev(src, 3 * N, "src"), _dev(q, N, "q"), N,
                                            _hp(shift), _hp(sign), _hp(w), C, central_cell, self_offset, refine,
                                            _dev(phi_out, T, "phi_out"), _dev(grad_out, 3 * T, "grad_out"),
                                            _stream_ptr(stream)), "hsma_direct_field")


def hsma_node_field(tgt: torch.Tensor, R: torch.Tensor, Q: torch.Tensor, P: torch.Tensor,
                    phi_out: Optional[torch.Tensor], grad_out: torch.Tensor, stream=None):
    T, M = tgt.shape[0], Q.numel()
    _check(load_library().hsma_node_field(_dev(tgt, 3 * T, "tgt"), T, _dev(R, 3 * M, "R"), _dev(Q, M, "Q"),
                                          _dev(P, 3 * M, "P"), M, _dev(phi_out, T, "phi_out"),
                                          _dev(grad_out, 3 * T, "grad_out"), _stream_ptr(stream)), "hsma_node_field")


def hsma_fp64_peak(seconds: float = 1.0):
    t, c = ctypes.c_double(), ctypes.c_double()
    _check(load_library().hsma_fp64_peak(seconds, ctypes.byref(t), ctypes.byref(c)), "hsma_fp64_peak")
    return t.value, c.value


TIMING_KEYS = ("prepass", "near_check_kernel", "fit_map", "near_source_kernel", "node_kernel", "finish", "total", "fmm_far_field")


def hsma_plan_set_timing(plan: int, enable: bool):
    _check(load_library().hsma_plan_set_timing(plan, 1 if enable else 0), "hsma_plan_set_timing")


PAIR_FORM_AUTO, PAIR_FORM_ORDERED, PAIR_FORM_SYMMETRIC = 0, 1, 2
PAIR_FORM_FMM = 3               # reported by hsma_plan_last_pair_form when step (b) ran as the FMM
NEAR_ALG_DIRECT, NEAR_ALG_FMM, NEAR_ALG_AUTO = 0, 1, 2


def hsma_plan_set_pair_form(plan: int, form: int):
    """Step (b): 0 = automatic, 1 = ordered pairs always, 2 = symmetric form wherever it applies (include/hsma.h)."""
    _check(load_library().hsma_plan_set_pair_form(plan, int(form)), "hsma_plan_set_pair_form")


def hsma_plan_last_pair_form(plan: int) -> int:
    """What the last evaluate used for step (b): 1 ordered pairs, 2 symmetric (each unordered pair once)."""
    return int(load_library().hsma_plan_last_pair_form(plan))


def hsma_plan_set_sym_scratch_cap(plan: int, nbytes: int):
    """Column-sum scratch per wave of the symmetric form, bytes (0: the default 64 MiB); include/hsma.h."""
    _check(load_library().hsma_plan_set_sym_scratch_cap(plan, int(nbytes)), "hsma_plan_set_sym_scratch_cap")


def hsma_plan_set_image_factoring(plan: int, on: bool):
    """Lattice-factored image sums on (default) / off; include/hsma.h."""
    _check(load_library().hsma_plan_set_image_factoring(plan, 1 if on else 0), "hsma_plan_set_image_factoring")


def hsma_plan_image_factoring(plan: int) -> bool:
    """True if the lattice-factored kernels are in use for this plan."""
    return bool(load_library().hsma_plan_image_factoring(plan))


def hsma_plan_fmm_info(plan: int) -> dict:
    """near_algorithm = FMM: expansion order, leaf level and leaf count of the last evaluate, whether step (a) uses the multipoles."""
    w = (ctypes.c_longlong * 4)()
    _check(load_library().hsma_plan_fmm_info(plan, w), "hsma_plan_fmm_info")
    return dict(zip(("order", "leaf_level", "leaves", "check_points_by_m2p"), [int(v) for v in w]))


def hsma_plan_scratch_bytes(plan: int) -> int:
    return int(load_library().hsma_plan_scratch_bytes(plan))


def hsma_plan_get_timing(plan: int) -> dict:
    """Stage durations (ms) of the last evaluate; synchronises the plan's stream."""
    ms = (ctypes.c_double * 8)()
    _check(load_library().hsma_plan_get_timing(plan, ms), "hsma_plan_get_timing")
    return dict(zip(TIMING_KEYS, [float(v) for v in ms]))


def hsma_launch_count() -> int:
    return int(load_library().hsma_launch_count())
