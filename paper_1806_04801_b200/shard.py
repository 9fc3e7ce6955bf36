"""Multi-GPU plumbing ("Multi-GPU"): one process per GPU, the sources (N x 32 B) and the plan replicated.
`evaluate_distributed` is one HSMA evaluation over all ranks:
  * step (a): every rank sums its slice of the K_t check targets; ONE all-gather of the check sums (32 KB; x4 with
    derivative rows) before the fit -- the fit needs all of them;
  * steps (b)+(c): when the symmetric form applies (one evaluation per UNORDERED pair), rank r walks its 1/R share of the
    unordered pairs for all targets (PART form) and the result is the SUM over ranks: one all-reduce of phi [N] (and of
    F [N,3]) and of U.  That sum over ranks is part of the method's arithmetic; it is done by the collective (NCCL's
    or gloo's reduction), nothing else of the method is computed here.  Otherwise (small N, sphere-culled near set)
    the N targets are split into contiguous shards and the result is assembled by an all-gather of phi (F) and an
    all-reduce of U.
Collectives go through torch.distributed: nccl on GPUs; a gloo group is staged through host memory (CPU tests, and the
two-processes-on-one-GPU test, where NCCL refuses to put two ranks on one device).  Stream ordering: the library
enqueues on the plan's stream, torch collectives on torch's current stream; evaluate_distributed makes the plan's
stream current for its duration and orders it after the caller's stream on entry and before it on exit, so the
result is correct whatever stream the caller is on.
Verified: world = 2 on one B200 (two processes sharing cuda:0, gloo group, tests/test_gpu_distributed.py) and
world = 2 gloo on CPU (tests/test_shard_gloo.py).  The NCCL path with world > 1 has not run on hardware: only one
GPU is available to this build."""
from __future__ import annotations

from typing import List, Tuple

import torch
import torch.distributed as dist

ALIGN = 256  # shard boundaries on source-tile boundaries (csrc/common.cuh kTile) when N allows it


def shard_bounds(N: int, world: int, align: int = ALIGN) -> List[Tuple[int, int]]:
    """Contiguous [t0, t1) per rank covering 0..N exactly once; sizes differ by at most one `align`
    block (by at most 1 when N < align * world)."""
    if N < 0 or world < 1:
        raise ValueError("need N >= 0 and world >= 1")
    if N < align * world:
        align = 1
    blocks = (N + align - 1) // align
    cuts = [min(N, ((blocks * r) // world) * align) for r in range(world)] + [N]
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def _is_gloo(group) -> bool:
    return dist.is_initialized() and str(dist.get_backend(group)).lower() == "gloo"


def _all_gather_into(recv: torch.Tensor, send: torch.Tensor, group) -> torch.Tensor:
    """dist.all_gather_into_tensor; a gloo group with CUDA tensors is staged through host memory."""
    if _is_gloo(group) and send.is_cuda:
        world = dist.get_world_size(group)
        parts = [torch.empty(send.shape, dtype=send.dtype) for _ in range(world)]
        dist.all_gather(parts, send.cpu(), group=group)
        recv.copy_(torch.cat(parts).reshape(recv.shape))
    elif _is_gloo(group):
        parts = list(recv.reshape((dist.get_world_size(group),) + tuple(send.shape)).unbind(0))
        dist.all_gather(parts, send, group=group)
    else:
        dist.all_gather_into_tensor(recv, send, group=group)
    return recv


def _all_reduce_sum(t: torch.Tensor, group) -> torch.Tensor:
    """In-place sum over the ranks; a gloo group with a CUDA tensor is staged through host memory."""
    if _is_gloo(group) and t.is_cuda:
        h = t.cpu()
        dist.all_reduce(h, op=dist.ReduceOp.SUM, group=group)
        t.copy_(h)
    else:
        dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t


def all_gather_phi(phi_local: torch.Tensor, N: int, group=None) -> torch.Tensor:
    """Assemble phi [N] on every rank from the per-rank shards (shards padded to a common length for
    the equal-size all_gather; the padding is cut away again)."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        return phi_local
    bounds = shard_bounds(N, world)
    width = max(b - a for a, b in bounds)
    send = torch.zeros(width, dtype=phi_local.dtype, device=phi_local.device)
    send[: phi_local.numel()] = phi_local
    recv = torch.empty(world * width, dtype=phi_local.dtype, device=phi_local.device)
    _all_gather_into(recv, send, group)
    return torch.cat([recv[r * width: r * width + (b - a)] for r, (a, b) in enumerate(bounds)])


def all_reduce_energy(U_local: torch.Tensor, group=None) -> torch.Tensor:
    """U = sum over ranks of the shard energies 1/2 sum_{i in shard} q_i phi_i (in place)."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        _all_reduce_sum(U_local, group)
    return U_local


def all_reduce_phi(phi_part: torch.Tensor, group=None) -> torch.Tensor:
    """phi = sum over ranks of the partial potentials of the PART form (in place; [N] doubles, 2 MB at N = 262,144)."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        _all_reduce_sum(phi_part, group)
    return phi_part


def all_gather_slices(local: torch.Tensor, total: int, group=None) -> torch.Tensor:
    """Concatenate per-rank slices along dim 0 (rank r owns shard_bounds(total, world, align=1)[r]); slices are
    padded to a common length for the equal-size all_gather."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    if world == 1:
        return local
    bounds = shard_bounds(total, world, align=1)
    width = max(b - a for a, b in bounds)
    tail = tuple(local.shape[1:])
    send = torch.zeros((width,) + tail, dtype=local.dtype, device=local.device)
    send[: local.shape[0]] = local
    recv = torch.empty((world * width,) + tail, dtype=local.dtype, device=local.device)
    _all_gather_into(recv, send, group)
    return torch.cat([recv[r * width: r * width + (b - a)] for r, (a, b) in enumerate(bounds)])


def evaluate_distributed(plan, xyz: torch.Tensor, q: torch.Tensor, forces: bool = False, group=None):
    """One HSMA evaluation over all ranks of `group` (every rank holds all N sources and an identical plan):
      1. this rank's slice of the check-point sums of step (a)      hsma_check_sums_shard
      2. all-gather of the K_t check sums (one small message)       the only data-path collective before the fit
      3. fit, mapping and steps (b), (c) for this rank's targets    hsma_evaluate_rest_shard
      4. all-gather of phi (and F), all-reduce of U                 assembly of the result
    or, when the symmetric form of step (b) applies (DESIGN.md 6.12 / 8):
      3'. fit, mapping, this rank's share of the UNORDERED pairs of (b), (c) for its targets    hsma_evaluate_rest_part
      4'. all-reduce of the partial phi [N] (and F [N,3]) and of the partial U
    Returns (phi [N], F [N,3] or None, U [1]) on every rank.  `plan` is a paper_1806_04801_b200.Plan.
    The library calls run on the plan's stream and the collectives on torch's current stream: the plan's stream is made
    current here, ordered after the caller's stream on entry and before it on exit."""
    if not q.is_cuda:
        raise RuntimeError("evaluate_distributed needs device tensors (the CUDA path has no CPU fallback)")
    caller = torch.cuda.current_stream(q.device)
    ps = plan.torch_stream
    if ps.cuda_stream == caller.cuda_stream:
        return _evaluate_distributed(plan, xyz, q, forces, group)
    ps.wait_stream(caller)
    with torch.cuda.stream(ps):
        out = _evaluate_distributed(plan, xyz, q, forces, group)
    caller.wait_stream(ps)
    for t in out:
        if t is not None:
            t.record_stream(caller)
    return out


def _evaluate_distributed(plan, xyz: torch.Tensor, q: torch.Tensor, forces: bool, group):
    from . import binding
    N = q.numel()
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    Kt = plan.info["check_targets"]
    c0, c1 = shard_bounds(Kt, world, align=1)[rank]
    t0, t1 = shard_bounds(N, world)[rank]
    need_grad = bool(binding.hsma_plan_needs_check_gradient(plan.handle))
    binding.hsma_check_sums_shard(plan.handle, xyz, q, c0, c1)
    pc = torch.empty(c1 - c0, dtype=torch.float64, device=q.device)
    pcg = torch.empty(c1 - c0, 3, dtype=torch.float64, device=q.device) if need_grad else None
    binding.hsma_get_check_sums(plan.handle, c0, c1, pc, pcg)
    if world > 1:
        pc_all = all_gather_slices(pc, Kt, group)
        pcg_all = all_gather_slices(pcg, Kt, group) if need_grad else None
        binding.hsma_set_check_sums(plan.handle, 0, Kt, pc_all.contiguous(), pcg_all.contiguous() if need_grad else None)
    if binding.hsma_plan_part_form_applies(plan.handle, N):
        # PART form: this rank's share of the unordered pairs of (b) for all targets + (c) for its own targets;
        # phi, F and U are sums over the ranks (one all-reduce each)
        phi_part = torch.empty(N, dtype=torch.float64, device=q.device)
        F_part = torch.empty(N, 3, dtype=torch.float64, device=q.device) if forces else None
        U = torch.empty(1, dtype=torch.float64, device=q.device)
        binding.hsma_evaluate_rest_part(plan.handle, xyz, q, rank, world, t0, t1, phi_part, F_part, U)
        all_reduce_phi(phi_part, group)
        if forces:
            all_reduce_phi(F_part, group)
        all_reduce_energy(U, group)
        return phi_part, F_part, U
    T = t1 - t0
    phi = torch.empty(T, dtype=torch.float64, device=q.device)
    F = torch.empty(T, 3, dtype=torch.float64, device=q.device) if forces else None
    U = torch.empty(1, dtype=torch.float64, device=q.device)
    binding.hsma_evaluate_rest_shard(plan.handle, xyz, q, t0, t1, phi, F, U)
    phi_all = all_gather_phi(phi, N, group)
    F_all = None
    if forces:
        F_all = F if world == 1 else torch.cat([f for f in _gather_rows(F, N, group)])
    all_reduce_energy(U, group)
    return phi_all, F_all, U


def _gather_rows(local: torch.Tensor, N: int, group=None):
    """Per-rank [T_r, 3] blocks in rank order (the shards of shard_bounds(N, world))."""
    world = dist.get_world_size(group)
    bounds = shard_bounds(N, world)
    width = max(b - a for a, b in bounds)
    send = torch.zeros(width, local.shape[1], dtype=local.dtype, device=local.device)
    send[: local.shape[0]] = local
    recv = torch.empty(world * width, local.shape[1], dtype=local.dtype, device=local.device)
    _all_gather_into(recv, send, group)
    return [recv[r * width: r * width + (b - a)] for r, (a, b) in enumerate(bounds)]
