"""Seeded random sweep of the raw kernels and of whole evaluates against the oracle: sizes around the tile (256),
block (256 R) and grid boundaries of the persistent decomposition, every boundary kind / closure / mode.  `-m gpu`."""
import math

import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def H():
    import torch
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    import paper_1806_04801_b200 as H
    H.binding.load_library()
    return H


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a, dtype=np.float64), device="cuda")


def rel_inf(a, b):
    return float(np.max(np.abs(a - b)) / max(np.max(np.abs(b)), 1e-300))


SIZES = [1, 2, 31, 255, 256, 257, 511, 512, 513, 1023, 1024, 1025, 2047, 2048, 2049, 3000, 4095, 4097, 9001]
KINDS = [(W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0), (W.BC_PERIODIC, (1.0, 0.8, 1.3), (2, 2, 1), 1.0),
         (W.BC_MIRROR_CAVITY, (1.0, 1.5, 0.7), (1, 1, 1), -1.0), (W.BC_MIRROR_CAVITY, (1.0, 1.0, 1.0), (1, 1, 1), 1.0),
         (W.BC_SLAB_XY_PERIODIC_Z_MIRROR, (1.0, 1.0, 0.5), (1, 1, 2), 0.5)]


@pytest.mark.parametrize("case", range(60))
def test_raw_sums_random_shapes(H, case):
    import torch
    rng = np.random.default_rng(1000 + case)
    N = int(rng.choice(SIZES))
    kind, L, shell, gamma = KINDS[case % len(KINDS)]
    refine = 1 + case % 2
    Lh = np.asarray(L)
    src = (rng.random((N, 3)) - 0.5) * Lh
    pattern = case % 4
    q = [rng.standard_normal(N), W.alternating_charges(N), np.full(N, -0.5),
         np.where(rng.random(N) < 0.3, 1.0, -1.0)][pattern]
    cells = O.cell_table(kind, L, shell, gamma)
    self_mode = case % 3 == 0
    if self_mode:
        t0 = int(rng.integers(0, N))
        T = int(rng.integers(1, N - t0 + 1))
        tgt = src[t0:t0 + T]
        so = t0
    else:
        T = int(rng.choice(SIZES[:14]))
        tgt = (rng.random((T, 3)) - 0.5) * Lh * 1.1
        so = -1
    ref = O.near_sum(tgt, src, q, cells, self_offset=so)
    refg = O.near_grad(tgt, src, q, cells, self_offset=so)
    out = torch.empty(T, dtype=torch.float64, device="cuda")
    H.hsma_direct_sum(dev(tgt), dev(src), dev(q), cells.shift, cells.sign, cells.w, cells.central, so, refine, out)
    scale = max(np.max(np.abs(ref)), np.max(np.abs(q)))          # image terms may cancel: the size of one term counts too
    tol = 5e-11 if refine == 1 else 1e-12
    got = out.cpu().numpy()
    assert np.all(np.isfinite(got)) and np.max(np.abs(got - ref)) <= tol * scale
    phi = torch.empty(T, dtype=torch.float64, device="cuda")
    g = torch.empty(T, 3, dtype=torch.float64, device="cuda")
    H.hsma_direct_field(dev(tgt), dev(src), dev(q), cells.shift, cells.sign, cells.w, cells.central, so, refine, phi, g)
    assert np.max(np.abs(phi.cpu().numpy() - ref)) <= tol * scale
    gscale = max(np.max(np.abs(refg)), np.max(np.abs(q)))
    assert np.max(np.abs(g.cpu().numpy() - refg)) <= 3 * tol * gscale


@pytest.mark.parametrize("case", range(24))
def test_whole_evaluates_random_configurations(H, case):
    rng = np.random.default_rng(5000 + case)
    N = 2 * int(rng.integers(1, 1800))
    which = case % 6
    p = int(rng.integers(4, 13))
    M = int(rng.integers(300, 3000))
    K = int(2 * p * p + rng.integers(20, 300))
    s32 = math.sqrt(3.0) / 2.0
    if which == 0:
        w = W.Workload("f", W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0, float(rng.uniform(1.05, 1.7)) * s32, p, M, K,
                       rng.random((N, 3)), W.alternating_charges(N))
    elif which == 1:
        w = W.Workload("f", W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0, 1.5 * s32, p, M, K, rng.random((N, 3)),
                       W.alternating_charges(N), closure=W.CLOSURE_FACE_PAIRS)
    elif which == 2:
        L = (1.0, 1.0, 1.0)
        w = W.Workload("f", W.BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0, 1.5 * s32, p, M, K, 0.02 + 0.96 * rng.random((N, 3)),
                       rng.standard_normal(N), check_xyz=W.seeded_face_points(K, L, W.ALL_FACES, seed=case))
    elif which == 3:
        L = (1.0, 1.0, 1.0)
        q = rng.standard_normal(N)
        w = W.Workload("f", W.BC_MIRROR_CAVITY, L, (1, 1, 1), 1.0, 1.5 * s32, p, M, K, 0.02 + 0.96 * rng.random((N, 3)),
                       q - q.mean(), check_xyz=W.seeded_face_points(K, L, W.ALL_FACES, seed=case))
    elif which == 4:
        L = (1.0, 1.0, 0.5)
        xyz = rng.random((N, 3)) * np.asarray(L)
        xyz[:, 2] = 0.02 + 0.92 * xyz[:, 2]
        w = W.Workload("f", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), -1.0, 1.1, p, M, K, xyz, rng.standard_normal(N),
                       closure=W.CLOSURE_BOUNDARY)
    else:
        w = W.Workload("f", W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0, 1.3 * s32, p, M, K, rng.random((N, 3)),
                       W.alternating_charges(N), near_mode=W.NEAR_SPHERE)
    refine = case % 3
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w, rsqrt_refine=refine) as plan:
        phi, F, U = plan.evaluate_forces(dev(w.xyz), dev(w.q), sync=True)
        phi0, U0 = plan.evaluate(dev(w.xyz), dev(w.q), sync=True)
    assert rel_inf(phi.cpu().numpy(), r.phi) <= 1e-10 and rel_inf(phi0.cpu().numpy(), r.phi) <= 1e-10
    # Energy bar: |dU| <= 1e-11 |U| -- unless the random-magnitude charges of this fuzz case make
    # U = 1/2 sum q_i phi_i cancel to less than 1 % of S = 1/2 sum |q_i phi_i|.  Then |U| is no scale for the rounding of
    # the sum (each side carries ~eps S of it) and the bar is 1e-13 S: the phi bar (1e-10) applied to the terms, with
    # three more digits because their errors do not add coherently.  No additive slack otherwise.
    S = 0.5 * float(np.sum(np.abs(w.q * r.phi)))
    assert abs(float(U) - r.U) <= (1e-11 * abs(r.U) if abs(r.U) >= 0.01 * S else 1e-13 * S)
    assert rel_inf(F.cpu().numpy(), r.F) <= 1e-10


@pytest.mark.parametrize("case", range(12))
def test_symmetric_and_part_forms_random_sizes(H, case):
    """DESIGN.md 6.12 / 8: random sizes between the smallest case the symmetric form takes and 60,000, random cell
    table, charges, refinement and part count.  The symmetric potential and gradient kernels and the sum over the
    parts of the multi-GPU PART form must agree with the ordered-pair kernels (which the other tests hold to the
    oracle) to rounding: these sizes are too large for the oracle in a test, and what is checked here is the work
    decomposition (visits, chunks, rows, column sums), which does not depend on it."""
    import torch
    from paper_1806_04801_b200 import shard
    rng = np.random.default_rng(7000 + case)
    idx = int(rng.choice([2, 3, 4, 5]))
    N = 2 * int(rng.integers(3969, 30000))
    w = W.config(idx, N=N)
    if rng.random() < 0.4:
        q = rng.standard_normal(N)
        w = w.with_(q=q - q.mean())
    with H.Plan.from_workload(w, rsqrt_refine=int(rng.choice([1, 2]))) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi, U = plan.evaluate(xyz, q, sync=True)
        assert plan.last_pair_form == 2
        pf, F, Uf = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == 2
        plan.set_pair_form(1)
        phi1, U1 = plan.evaluate(xyz, q, sync=True)
        _, F1, _ = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == 1
        plan.set_pair_form(0)
        n_parts = int(rng.integers(1, 9))
        H.binding.hsma_check_sums_shard(plan.handle, xyz, q, 0, plan.info["check_targets"])
        ps = torch.zeros(N, dtype=torch.float64, device="cuda")
        Fs = torch.zeros(N, 3, dtype=torch.float64, device="cuda")
        Us = torch.zeros(1, dtype=torch.float64, device="cuda")
        for part, (t0, t1) in enumerate(shard.shard_bounds(N, n_parts)):
            a = torch.empty(N, dtype=torch.float64, device="cuda")
            b = torch.empty(N, 3, dtype=torch.float64, device="cuda")
            c = torch.empty(1, dtype=torch.float64, device="cuda")
            H.binding.hsma_evaluate_rest_part(plan.handle, xyz, q, part, n_parts, t0, t1, a, b, c)
            plan.sync()
            ps += a
            Fs += b
            Us += c
    sc = float(phi1.abs().max())
    fs = max(float(F1.abs().max()), float(np.max(np.abs(w.q))) * sc / max(w.L))
    tol = 2e-11
    assert float((phi - phi1).abs().max()) <= tol * sc and float((pf - phi1).abs().max()) <= tol * sc
    assert float((F - F1).abs().max()) <= tol * fs
    assert float((ps - phi1).abs().max()) <= tol * sc and float((Fs - F1).abs().max()) <= tol * fs
    assert abs(float(U) - float(U1)) <= 1e-11 * abs(float(U1)) and abs(float(Us) - float(U1)) <= 1e-11 * abs(float(U1))


@pytest.mark.parametrize("case", range(12))
def test_fmm_random_configurations(H, case):
    """near_algorithm = FMM on random sizes, box shapes the FMM can tile (cubic, 2:1:1, 1:1:0.5, 2x2x1
    boxes per cell), cell tables (periodic; Dirichlet, Neumann and dielectric mirrors; grounded slab), shells, leaf
    levels, charges of any magnitude and box scales far from 1: potentials, forces and U against the oracle at the bars."""
    rng = np.random.default_rng(9100 + case)
    N = 2 * int(rng.integers(50, 9000))
    p = int(rng.integers(5, 12))
    M = int(rng.integers(400, 2500))
    K = int(2 * p * p + rng.integers(20, 300))
    scale = float(10.0 ** rng.uniform(-2, 2))          # box size 0.01 .. 100: the FMM works in box units at every level
    which = case % 6
    levels = int(rng.integers(0, 4))
    if which == 0:
        L = (scale, scale, scale)
        R0 = 0.5 * math.sqrt(3.0) * scale
        w = W.Workload("f", W.BC_PERIODIC, L, (1, 1, 1), 1.0, float(rng.uniform(1.05, 1.7)) * R0, p, M, K,
                       rng.random((N, 3)) * scale, W.alternating_charges(N))
    elif which == 1:                                   # non-cubic cell, cubic FMM boxes: 2 x 1 x 1 per cell
        L = (2.0 * scale, scale, scale)
        R0 = 0.5 * math.sqrt(6.0) * scale
        q = rng.standard_normal(N)
        w = W.Workload("f", W.BC_PERIODIC, L, (1, 1, 1), 1.0, 1.15 * R0, p, M, K, rng.random((N, 3)) * np.asarray(L), q - q.mean())
    elif which == 2:
        L = (scale, scale, scale)
        R0 = 0.5 * math.sqrt(3.0) * scale
        w = W.Workload("f", W.BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0, 1.5 * R0, p, M, K, (0.02 + 0.96 * rng.random((N, 3))) * scale,
                       rng.standard_normal(N), check_xyz=W.seeded_face_points(K, L, W.ALL_FACES, seed=case))
    elif which == 3:                                   # Neumann cavity: derivative rows -> step (a) keeps its direct FIELD form
        L = (scale, scale, scale)
        R0 = 0.5 * math.sqrt(3.0) * scale
        q = rng.standard_normal(N)
        w = W.Workload("f", W.BC_MIRROR_CAVITY, L, (1, 1, 1), 1.0, 1.5 * R0, p, M, K, (0.02 + 0.96 * rng.random((N, 3))) * scale,
                       q - q.mean(), check_xyz=W.seeded_face_points(K, L, W.ALL_FACES, seed=case))
    elif which == 4:                                   # grounded slab, boundary closure, 2 x 2 x 1 boxes per cell
        L = (scale, scale, 0.5 * scale)
        xyz = rng.random((N, 3)) * np.asarray(L)
        xyz[:, 2] = (0.02 + 0.92 * xyz[:, 2] / L[2]) * L[2]
        w = W.Workload("f", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), -1.0, 1.1 * scale, p, M, K, xyz, rng.standard_normal(N),
                       closure=W.CLOSURE_BOUNDARY)
    else:                                              # dielectric slab, far-data closure (step (a) over the far table: direct)
        L = (scale, scale, 0.5 * scale)
        q = rng.standard_normal(N)
        w = W.Workload("f", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), float(rng.uniform(-0.9, 0.9)), 1.1 * scale, p, M, K,
                       rng.random((N, 3)) * np.asarray(L), q - q.mean(), closure=W.CLOSURE_FAR_DATA, far_shell=(2, 2, 3),
                       check_xyz=W.seeded_face_points(K, L, W.ALL_FACES, seed=case))
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w, near_algorithm=H.binding.NEAR_ALG_FMM, fmm_levels=levels) as plan:
        phi, F, U = plan.evaluate_forces(dev(w.xyz), dev(w.q), sync=True)
        assert plan.last_pair_form == 3
        phi0, U0 = plan.evaluate(dev(w.xyz), dev(w.q), sync=True)
        assert plan.last_pair_form == 3
    assert rel_inf(phi.cpu().numpy(), r.phi) <= 1e-10 and rel_inf(phi0.cpu().numpy(), r.phi) <= 1e-10
    S = 0.5 * float(np.sum(np.abs(w.q * r.phi)))
    for u in (float(U), float(U0)):
        assert abs(u - r.U) <= (1e-11 * abs(r.U) if abs(r.U) >= 0.01 * S else 1e-13 * S)
    assert rel_inf(F.cpu().numpy(), r.F) <= 1e-10
