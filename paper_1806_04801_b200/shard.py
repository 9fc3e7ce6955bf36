"""Multi-GPU plumbing: the N targets of steps (b)/(c) are split into
contiguous shards, one per rank; the sources (N x 32 B) and the plan are replicated; step (a) and
the fit are computed redundantly by every rank (no data-path collective).  The only exchange is the
assembly of the result: an all-gather of phi and a 1-double all-reduce of U, through
torch.distributed (nccl on GPUs; gloo in the CPU tests).  No arithmetic of the method lives here."""
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
    dist.all_gather_into_tensor(recv, send, group=group)
    return torch.cat([recv[r * width: r * width + (b - a)] for r, (a, b) in enumerate(bounds)])


def all_reduce_energy(U_local: torch.Tensor, group=None) -> torch.Tensor:
    """U = sum over ranks of the shard energies 1/2 sum_{i in shard} q_i phi_i (in place)."""
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(U_local, op=dist.ReduceOp.SUM, group=group)
    return U_local
