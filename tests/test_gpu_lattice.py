"""Lattice-factored image sums (csrc/lattice_kernels.cuh: |r_i - img_k(r_j)|^2 = X[k_x] + Y[k_y] + Z[k_z]
for the full box of image cells of PAPER.md:40-50 Eq.(3)/(4); one add per image for r^2, charges and cell weights once
per pair) against the CPU oracle and against the cell-by-cell kernels they replace, through the C-ABI.  Every shape that
is instantiated -- 27 periodic cells, 27 reflected cells (gamma = -1 and +1), 45 slab cells (3 x 3 periodic x 5 reflected,
gamma = 0.5 and -1), 27 slab cells (3 x 3 periodic x 3 reflected) -- in the ordered form (small N, target shards, step (a)), the symmetric form (N >= 7,937) and their
gradient forms; both refinements; and the geometries that must keep the cell-by-cell kernels.  Bars as in
test_gpu_parity (north_star).  All `-m gpu`."""
import math

import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O

pytestmark = pytest.mark.gpu

PHI_TOL, U_TOL, F_TOL = 1e-10, 1e-11, 1e-10
AGREE = 2e-12          # the two kernel families differ only in the rounding of r^2 and of the sums


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
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def on_and_off(H, w, forces, **plan_kw):
    """Results with the factored kernels (default) and with the cell-by-cell ones, from ONE plan."""
    out = []
    with H.Plan.from_workload(w, **plan_kw) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        assert plan.image_factoring
        for on in (True, False):
            plan.set_image_factoring(on)
            assert plan.image_factoring == on
            if forces:
                phi, F, U = plan.evaluate_forces(xyz, q, sync=True)
                out.append((phi.cpu().numpy(), F.cpu().numpy(), float(U), plan.last_pair_form))
            else:
                phi, U = plan.evaluate(xyz, q, sync=True)
                out.append((phi.cpu().numpy(), None, float(U), plan.last_pair_form))
    return out


def check(w, r, got, forces):
    (phi, F, U, form), (phi0, F0, U0, form0) = got
    assert form == form0
    for p, f, u in ((phi, F, U), (phi0, F0, U0)):
        assert rel_inf(p, r.phi) <= PHI_TOL and abs(u - r.U) <= U_TOL * abs(r.U)
        if forces:
            assert np.max(np.abs(f - r.F)) <= F_TOL * np.max(np.abs(r.F))
    assert rel_inf(phi, phi0) <= AGREE and abs(U - U0) <= AGREE * abs(U0)
    if forces:
        assert np.max(np.abs(F - F0)) <= AGREE * np.max(np.abs(F0))
    return form


# (config, N): 2 / 5 = 27 periodic cells, 3 = 27 reflected cells gamma = -1, 4 = 45 slab cells gamma = 0.5 with the far-data
# closure (step (a) keeps the cell-by-cell kernel there: its table is the 396 far cells).  N < 7,937: ordered pairs
# (R = 1 and 2 targets per thread, ragged last block and tile); N >= 7,937: symmetric form, ragged last block.
CASES = [(2, 700), (2, 3000), (3, 1501), (4, 2500), (5, 9000), (3, 9001), (4, 8210)]


@pytest.mark.parametrize("forces", [False, True])
@pytest.mark.parametrize("refine", [1, 2])
@pytest.mark.parametrize("idx,N", CASES)
def test_factored_kernels_match_oracle_and_cell_by_cell(H, idx, N, refine, forces):
    w = W.config(idx, N=N)
    r = O.hsma(w, forces=forces)
    form = check(w, r, on_and_off(H, w, forces, rsqrt_refine=refine), forces)
    assert form == (2 if N >= 7937 else 1)


@pytest.mark.parametrize("forces", [False, True])
def test_generic_charges_and_weights(H, forces):
    """Charges of any magnitude (the factored kernels multiply by q once per pair) with the weighted slab images."""
    w = W.config(4, N=3001)
    q = np.random.default_rng(5).standard_normal(w.N)
    w = w.with_(q=q - q.mean())
    check(w, O.hsma(w, forces=forces), on_and_off(H, w, forces), forces)


@pytest.mark.parametrize("closure", ["walls", "slab_boundary", "face_pairs"])
def test_other_closures(H, closure):
    """Neumann walls (27 reflected cells with gamma = +1: every weight class has weight 1), the grounded slab by its own
    boundary conditions (gamma = -1 on the 45-cell table) and the face-pair closure, whose derivative rows take
    step (a) in its gradient form (near_lat_sum_kernel<.., FIELD> at the check targets)."""
    rng = np.random.default_rng(8)
    if closure == "walls":
        N, L = 1200, (1.0, 1.0, 1.0)
        w = W.Workload("neumann_cavity", W.BC_MIRROR_CAVITY, L, (1, 1, 1), 1.0, 1.5 * math.sqrt(3) / 2, 12, 4000, 900,
                       0.03 + 0.94 * rng.random((N, 3)), W.alternating_charges(N),
                       check_xyz=W.seeded_face_points(900, L, W.ALL_FACES, seed=9))
    elif closure == "slab_boundary":
        N, L = 1500, (1.0, 1.0, 0.5)
        xyz = rng.random((N, 3)) * np.asarray(L)
        xyz[:, 2] = 0.02 + 0.92 * xyz[:, 2]
        w = W.Workload("slab_grounded", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), -1.0, 1.1, 12, 6000, 1000, xyz,
                       rng.standard_normal(N) + 0.2, closure=W.CLOSURE_BOUNDARY)
    else:
        w = W.config(2, N=1100)
        w = w.with_(closure=W.CLOSURE_FACE_PAIRS, check_xyz=W.seeded_face_points(w.K, w.L, W.LOWER_FACES, seed=3))
    check(w, O.hsma(w, forces=True), on_and_off(H, w, True), True)


@pytest.mark.parametrize("forces", [False, True])
@pytest.mark.parametrize("N", [2501, 9003])
def test_slab_with_one_shell(H, N, forces):
    """The slab kind with near shell (1,1,1) -- what hsma_plan_create(L, SLAB, near_shell = 1, ...) builds: 27 cells, z
    reflecting (weights gamma^|k_z|), grounded plates closed by their own boundary conditions.  Ordered and symmetric forms."""
    rng = np.random.default_rng(17)
    L = (1.0, 1.0, 0.8)
    xyz = rng.random((N, 3)) * np.asarray(L)
    xyz[:, 2] = 0.02 * L[2] + 0.96 * xyz[:, 2]
    w = W.Workload("slab_one_shell", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 1), -1.0, 1.0, 10, 3000, 700, xyz,
                   rng.standard_normal(N) + 0.1, closure=W.CLOSURE_BOUNDARY)
    form = check(w, O.hsma(w, forces=forces), on_and_off(H, w, forces), forces)
    assert form == (2 if N >= 7937 else 1)


def test_target_shards(H):
    """Target shards (ordered pairs, self term found by slot) with the factored kernels: the pieces add up to the one-call
    evaluate (symmetric form).  The PART form runs in tests/test_gpu_distributed.py."""
    import torch
    w = W.config(5, N=9000)
    xyz, q = dev(w.xyz), dev(w.q)
    with H.Plan.from_workload(w) as plan:
        phi, U = plan.evaluate(xyz, q, sync=True)
        cuts = [0, 2999, 3000, 7000, w.N]
        pieces = [plan.evaluate_shard(xyz, q, a, b, sync=True)[0] for a, b in zip(cuts[:-1], cuts[1:])]
        assert plan.last_pair_form == 1
        got = torch.cat(pieces)
        assert float((got - phi).abs().max() / phi.abs().max()) <= AGREE


def test_where_the_cell_by_cell_kernels_stay(H):
    """Shell 2 (config 1: 125 cells) and the sphere-culled near set are not instantiated / not a full box."""
    with H.Plan.from_workload(W.config(1)) as plan:
        assert not plan.image_factoring
    w = W.config(2, N=800).with_(near_mode=W.NEAR_SPHERE)
    with H.Plan.from_workload(w) as plan:
        assert not plan.image_factoring


@pytest.mark.parametrize("idx,N", [(5, 30010), (4, 20500)])
def test_both_families_over_many_blocks_and_waves(H, idx, N):
    """Many target blocks and several waves (column scratch capped at 4 MiB): the factored kernels against the oracle, and the
    cell-by-cell kernels -- now only the fallback for cell tables that are not instantiated -- against them, potentials and
    forces, every element."""
    w = W.config(idx, N=N)
    r = O.hsma(w, forces=True)
    res = []
    with H.Plan.from_workload(w) as plan:
        plan.set_sym_scratch_cap(4 << 20)
        xyz, q = dev(w.xyz), dev(w.q)
        for on in (True, False):
            plan.set_image_factoring(on)
            phi, F, U = plan.evaluate_forces(xyz, q, sync=True)
            phi2, U2 = plan.evaluate(xyz, q, sync=True)
            assert plan.last_pair_form == 2
            res.append((phi.cpu().numpy(), F.cpu().numpy(), float(U), phi2.cpu().numpy(), float(U2)))
    for phi, F, U, phi2, U2 in res:
        assert rel_inf(phi, r.phi) <= PHI_TOL and rel_inf(phi2, r.phi) <= PHI_TOL
        assert abs(U - r.U) <= U_TOL * abs(r.U) and abs(U2 - r.U) <= U_TOL * abs(r.U)
        assert np.max(np.abs(F - r.F)) <= F_TOL * np.max(np.abs(r.F))
    assert rel_inf(res[0][0], res[1][0]) <= AGREE and rel_inf(res[0][3], res[1][3]) <= AGREE
    assert np.max(np.abs(res[0][1] - res[1][1])) <= AGREE * np.max(np.abs(res[1][1]))


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_fuzz_both_families_agree(H, seed):
    """40 random cases per seed -- boundary kind, box, N from 1 to 40,000 (ordered and symmetric forms, ragged tiles, phantom
    targets of a last block), charges (alternating, scaled, random), refinement, potentials or forces, column-scratch cap
    (waves) -- evaluated by the factored and by the cell-by-cell kernels from one plan: finite and equal to rounding.  (The
    oracle comparisons are the tests above; this one hunts index errors at sizes no fixed case names.)"""
    rng = np.random.default_rng(seed)
    for case in range(40):
        kind = int(rng.integers(0, 3))
        N = int(rng.integers(7937, 40000)) if rng.random() < 0.6 else int(rng.integers(1, 7937))
        if kind == 0:
            L = (1.0, 1.0, 1.0) if rng.random() < 0.5 else (1.0, 1.1, 0.9)
            N += N % 2
            q = W.alternating_charges(N) * (1.0 if rng.random() < 0.5 else 0.37)
            if rng.random() < 0.4:
                q = rng.standard_normal(N)
                q -= q.mean()
            R = min(1.3 * 0.5 * math.sqrt(sum(x * x for x in L)), 1.45 * min(L))
            w = W.Workload("f", W.BC_PERIODIC, L, (1, 1, 1), 1.0, R, 8, 1500, 400, rng.random((N, 3)) * np.asarray(L), q)
        elif kind == 1:
            q = rng.standard_normal(N) if rng.random() < 0.5 else W.alternating_charges(N + N % 2)[:N]
            w = W.Workload("f", W.BC_MIRROR_CAVITY, (1.0, 1.0, 1.0), (1, 1, 1), -1.0, 1.5 * math.sqrt(3) / 2, 8, 1500, 400,
                           0.02 + 0.96 * rng.random((N, 3)), q)
        else:
            L = (1.0, 1.0, 0.5)
            xyz = rng.random((N, 3)) * np.asarray(L)
            xyz[:, 2] = 0.02 + 0.92 * xyz[:, 2]
            w = W.Workload("f", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), -1.0, 1.1, 8, 2000, 500, xyz, rng.standard_normal(N),
                           closure=W.CLOSURE_BOUNDARY)
        refine, forces = int(rng.integers(0, 3)), bool(rng.random() < 0.5)
        res = []
        with H.Plan.from_workload(w, rsqrt_refine=refine) as plan:
            if rng.random() < 0.3:
                plan.set_sym_scratch_cap(int(rng.integers(1, 16)) << 20)
            xyz, q = dev(w.xyz), dev(w.q)
            for on in (True, False):
                plan.set_image_factoring(on)
                if forces:
                    phi, F, U = plan.evaluate_forces(xyz, q, sync=True)
                    res.append((phi.cpu().numpy(), F.cpu().numpy()))
                else:
                    phi, U = plan.evaluate(xyz, q, sync=True)
                    res.append((phi.cpu().numpy(), None))
        tag = f"seed {seed} case {case}: kind {kind} N {N} refine {refine} forces {forces}"
        assert np.all(np.isfinite(res[0][0])), tag
        assert rel_inf(res[0][0], res[1][0]) <= AGREE, tag
        if forces:
            assert np.max(np.abs(res[0][1] - res[1][1])) <= AGREE * np.max(np.abs(res[1][1])), tag
