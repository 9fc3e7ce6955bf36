"""The N > 1 path on CPU: world_size-2 `gloo` processes run the host-side sharding of DESIGN.md
"Multi-GPU" (contiguous target shards, replicated sources, all-gather of phi, all-reduce of U), with the
oracle standing in for the per-rank evaluation (tests may call oracle/).  `-m "not gpu"`."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1806_04801_b200 import shard  # noqa: E402


@pytest.mark.parametrize("N,world", [(0, 1), (1, 2), (5, 8), (255, 2), (1000, 2), (1000, 3), (262144, 8), (262145, 7)])
def test_shard_bounds_cover_exactly_once(N, world):
    b = shard.shard_bounds(N, world)
    assert len(b) == world and b[0][0] == 0 and b[-1][1] == N
    for (a0, a1), (b0, b1) in zip(b[:-1], b[1:]):
        assert a1 == b0 and a0 <= a1
    sizes = [y - x for x, y in b]
    assert max(sizes) - min(sizes) <= (shard.ALIGN if N >= shard.ALIGN * world else 1)
    if N >= shard.ALIGN * world:
        assert all(x % shard.ALIGN == 0 for x, _ in b)


def _worker(rank, world, port, N, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import hsma_workloads as W
        from oracle import hsma_oracle as O
        w = W.config(2, N=N)
        t0, t1 = shard.shard_bounds(N, world)[rank]
        r = O.hsma(w, targets_slice=slice(t0, t1))      # this rank's shard: phi[t0:t1], U over the shard
        phi = shard.all_gather_phi(torch.from_numpy(r.phi.copy()), N)
        U = shard.all_reduce_energy(torch.tensor([r.U], dtype=torch.float64))
        np.save(os.path.join(out_dir, f"phi{rank}.npy"), phi.numpy())
        np.save(os.path.join(out_dir, f"U{rank}.npy"), U.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("N", [600, 257 * 2])
def test_two_ranks_assemble_the_single_rank_result(tmp_path, N):
    import hsma_workloads as W
    from oracle import hsma_oracle as O
    world, port = 2, 29500 + (os.getpid() + N) % 2000
    mp.spawn(_worker, args=(world, port, N, str(tmp_path)), nprocs=world, join=True)
    ref = O.hsma(W.config(2, N=N))
    for r in range(world):
        phi = np.load(tmp_path / f"phi{r}.npy")
        U = float(np.load(tmp_path / f"U{r}.npy")[0])
        assert phi.shape == (N,)
        assert np.array_equal(phi, ref.phi)             # same per-target arithmetic: bit-identical
        assert abs(U - ref.U) <= 1e-14 * abs(ref.U)


def _slices_worker(rank, world, port, total, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        a, b = shard.shard_bounds(total, world, align=1)[rank]
        vec = torch.arange(a, b, dtype=torch.float64)
        mat = torch.stack([vec, 2 * vec, -vec], dim=1)
        np.save(os.path.join(out_dir, f"v{rank}.npy"), shard.all_gather_slices(vec, total).numpy())
        np.save(os.path.join(out_dir, f"m{rank}.npy"), shard.all_gather_slices(mat, total).numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("total", [7, 4000])
def test_all_gather_slices_reassembles_in_order(tmp_path, total):
    """The check-point sums of step (a) are sharded with align = 1 and gathered before the fit."""
    world, port = 2, 31500 + (os.getpid() + total) % 2000
    mp.spawn(_slices_worker, args=(world, port, total, str(tmp_path)), nprocs=world, join=True)
    want = np.arange(total, dtype=np.float64)
    for r in range(world):
        assert np.array_equal(np.load(tmp_path / f"v{r}.npy"), want)
        assert np.array_equal(np.load(tmp_path / f"m{r}.npy"), np.stack([want, 2 * want, -want], axis=1))


def _parts_worker(rank, world, port, N, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import hsma_workloads as W
        from oracle import hsma_oracle as O
        w = W.config(2, N=N)
        cells = O.cell_table(w.kind, w.L, w.near_shell, w.gamma)
        # stand-in for hsma_evaluate_rest_part: a share of the PAIR work for ALL targets (here: the sources a..b-1;
        # the self term is left out where the targets are those sources)
        a, b = shard.shard_bounds(N, world, align=1)[rank]
        phi_part = np.empty(N)
        phi_part[a:b] = O.near_sum(w.xyz[a:b], w.xyz[a:b], w.q[a:b], cells, self_offset=0)
        rest = np.r_[0:a, b:N]
        phi_part[rest] = O.near_sum(w.xyz[rest], w.xyz[a:b], w.q[a:b], cells)
        U_part = 0.5 * float(np.dot(w.q, phi_part))
        phi = shard.all_reduce_phi(torch.from_numpy(phi_part))
        U = shard.all_reduce_energy(torch.tensor([U_part], dtype=torch.float64))
        np.save(os.path.join(out_dir, f"p{rank}.npy"), phi.numpy())
        np.save(os.path.join(out_dir, f"u{rank}.npy"), U.numpy())
    finally:
        dist.destroy_process_group()


def test_part_form_all_reduce_assembles_the_near_sum(tmp_path):
    """PART form of the multi-GPU path: every rank computes a share of the pair work for all targets;
    one all-reduce of the partial potentials (and of the partial energies) leaves the full sums on every rank."""
    import hsma_workloads as W
    from oracle import hsma_oracle as O
    N, world, port = 601, 2, 33500 + os.getpid() % 2000
    mp.spawn(_parts_worker, args=(world, port, N, str(tmp_path)), nprocs=world, join=True)
    w = W.config(2, N=N)
    cells = O.cell_table(w.kind, w.L, w.near_shell, w.gamma)
    want = O.near_sum(w.xyz, w.xyz, w.q, cells, self_offset=0)
    p0, p1 = np.load(tmp_path / "p0.npy"), np.load(tmp_path / "p1.npy")
    assert np.array_equal(p0, p1)                                   # the all-reduce gives every rank the same bits
    assert np.max(np.abs(p0 - want)) <= 1e-13 * np.max(np.abs(want))  # = the unsplit sum up to the order of addition
    u0, u1 = float(np.load(tmp_path / "u0.npy")[0]), float(np.load(tmp_path / "u1.npy")[0])
    assert u0 == u1 and abs(u0 - 0.5 * float(np.dot(w.q, want))) <= 1e-12 * abs(u0)


def test_single_process_is_a_no_op():
    x = torch.arange(5, dtype=torch.float64)
    assert shard.all_gather_phi(x, 5) is x
    u = torch.tensor([1.5], dtype=torch.float64)
    assert shard.all_reduce_energy(u) is u
    assert shard.all_reduce_phi(x) is x
