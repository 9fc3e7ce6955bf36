"""The symmetric form of step (b) (near_sym_kernel: each unordered source pair evaluated once,
PAPER.md:64 Eq.(5) with the image cells of PAPER.md:40-50) against the CPU oracle and against the ordered-pair
kernel, through the C-ABI.  Bars as in test_gpu_parity.  All `-m gpu`."""
import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O

pytestmark = pytest.mark.gpu

PHI_TOL = 1e-10
U_TOL = 1e-11
ORDERED, SYMMETRIC = 1, 2     # also the values of hsma_plan_set_pair_form (0 = automatic)


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


def both_forms(H, w, **plan_kw):
    """(phi, U) of the automatic form and of the ordered form, and which form each evaluate used."""
    with H.Plan.from_workload(w, **plan_kw) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi, U = plan.evaluate(xyz, q, sync=True)
        form = plan.last_pair_form
        plan.set_pair_form(ORDERED)
        phi1, U1 = plan.evaluate(xyz, q, sync=True)
        form1 = plan.last_pair_form
    return phi.cpu().numpy(), float(U), form, phi1.cpu().numpy(), float(U1), form1


# N: 7938 = 32 tiles with a two-source last tile (the smallest case the symmetric form takes); 9000 = 36 tiles, the
# last block holds 4 tiles (phantom targets) and a ragged tile; 12288 = whole blocks only
@pytest.mark.parametrize("refine", [1, 2])
@pytest.mark.parametrize("idx,N", [(2, 7938), (2, 9000), (3, 9000), (4, 9000), (5, 12288)])
def test_symmetric_form_matches_oracle(H, idx, N, refine):
    """Periodic, mirror-cavity (reflected images, gamma = -1) and slab (reflected + weighted images, gamma = 0.5)
    cell tables: every potential and U against the oracle; the ordered kernel agrees to rounding."""
    w = W.config(idx, N=N)
    r = O.hsma(w)
    phi, U, form, phi1, U1, form1 = both_forms(H, w, rsqrt_refine=refine)
    assert (form, form1) == (SYMMETRIC, ORDERED)
    assert rel_inf(phi, r.phi) <= PHI_TOL and abs(U - r.U) <= U_TOL * abs(r.U)
    assert rel_inf(phi1, r.phi) <= PHI_TOL and abs(U1 - r.U) <= U_TOL * abs(r.U)
    assert rel_inf(phi, phi1) <= 2e-11


@pytest.mark.parametrize("refine", [1, 2])
def test_symmetric_form_random_magnitudes(H, refine):
    """Charges of any magnitude and sign (the symmetric kernel always multiplies by q): slab table, ragged N."""
    w = W.config(4, N=8209)
    q = np.random.default_rng(77).standard_normal(w.N)
    q -= q.mean()
    w = w.with_(q=q)
    r = O.hsma(w)
    phi, U, form, phi1, U1, form1 = both_forms(H, w, rsqrt_refine=refine)
    assert (form, form1) == (SYMMETRIC, ORDERED)
    assert rel_inf(phi, r.phi) <= PHI_TOL and abs(U - r.U) <= U_TOL * abs(r.U)
    assert rel_inf(phi, phi1) <= 2e-11


def test_when_the_symmetric_form_applies(H):
    """All N targets, >= 32 source tiles: symmetric (potentials and forces).  Shards, small N: ordered.  The form
    is not a property of the result: every variant agrees with the full evaluate."""
    import torch
    w = W.config(5, N=8192)
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi, U = plan.evaluate(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
        ref = phi.cpu().numpy()
        a, _ = plan.evaluate_shard(xyz, q, 0, 5000, sync=True)
        assert plan.last_pair_form == ORDERED
        b, _ = plan.evaluate_shard(xyz, q, 5000, w.N, sync=True)
        assert np.max(np.abs(np.concatenate([a.cpu().numpy(), b.cpu().numpy()]) - ref)) <= 2e-11 * np.max(np.abs(ref))
        phi_f, F, U_f = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC                      # forces over all targets: the gradient form
        assert rel_inf(phi_f.cpu().numpy(), ref) <= 2e-11 and abs(float(U_f) - float(U)) <= 1e-11 * abs(float(U))
        _, Fs, _ = plan.evaluate_forces_shard(xyz, q, 100, 7000, sync=True)
        assert plan.last_pair_form == ORDERED
        Fh = F.cpu().numpy()
        assert np.max(np.abs(Fs.cpu().numpy() - Fh[100:7000])) <= 2e-11 * np.max(np.abs(Fh))
        phi2, U2 = plan.evaluate(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
        assert torch.equal(phi2, phi) and float(U2) == float(U)     # deterministic: fixed summation order
        with pytest.raises(Exception):
            plan.set_pair_form(3)
    w_small = W.config(5, N=7936)   # 31 tiles
    with H.Plan.from_workload(w_small) as plan:
        plan.evaluate(dev(w_small.xyz), dev(w_small.q), sync=True)
        assert plan.last_pair_form == ORDERED


def test_symmetric_form_in_a_replayed_graph(H):
    """The whole-evaluate CUDA graph (captured on the second identical call on a side stream) holds the symmetric
    launches; switching the form drops the graph."""
    import torch
    w = W.config(5, N=8192)
    r = O.hsma(w)
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with H.Plan.from_workload(w) as plan:
            xyz, q = dev(w.xyz), dev(w.q)
            phi = torch.empty(w.N, dtype=torch.float64, device="cuda")
            U = torch.empty(1, dtype=torch.float64, device="cuda")
            outs = []
            for _ in range(4):
                H.hsma_evaluate(plan.handle, xyz, q, phi, U)
                plan.sync()
                outs.append((phi.cpu().numpy().copy(), float(U)))
            assert H.binding.hsma_plan_info(plan.handle)["graph_replays"] >= 1 and plan.last_pair_form == SYMMETRIC
            for o in outs[1:]:
                assert np.array_equal(o[0], outs[0][0]) and o[1] == outs[0][1]
            assert rel_inf(outs[0][0], r.phi) <= PHI_TOL and abs(outs[0][1] - r.U) <= U_TOL * abs(r.U)
            # the gradient form (64 KB + 32 KB of dynamic shared memory) inside a replayed graph
            rf = O.hsma(w, forces=True)
            F = torch.empty(w.N, 3, dtype=torch.float64, device="cuda")
            before = H.binding.hsma_plan_info(plan.handle)["graph_replays"]
            Fs = []
            for _ in range(3):
                H.hsma_evaluate_forces(plan.handle, xyz, q, phi, F, U)
                plan.sync()
                Fs.append(F.cpu().numpy().copy())
            assert H.binding.hsma_plan_info(plan.handle)["graph_replays"] == before + 2 and plan.last_pair_form == SYMMETRIC
            assert np.array_equal(Fs[0], Fs[1]) and np.array_equal(Fs[0], Fs[2])
            assert rel_inf(Fs[0], rf.F) <= 1e-10
            plan.set_pair_form(ORDERED)
            H.hsma_evaluate(plan.handle, xyz, q, phi, U)
            plan.sync()
            assert plan.last_pair_form == ORDERED
            assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL


@pytest.mark.parametrize("idx,N", [(5, 8192), (4, 9000), (3, 8200)])
@pytest.mark.parametrize("n_parts", [1, 2, 3, 7])
def test_part_form_adds_up_to_the_evaluate(H, idx, N, n_parts):
    """Multi-GPU PART form with the "ranks" run one after the other on one device: the partial
    potentials and energies of the parts add up to the one-rank result, for every part count."""
    import torch
    from paper_1806_04801_b200 import shard
    w = W.config(idx, N=N)
    r = O.hsma(w)
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        assert H.binding.hsma_plan_part_form_applies(plan.handle, w.N)
        phi_ref, U_ref = plan.evaluate(xyz, q, sync=True)
        Kt = plan.info["check_targets"]
        H.binding.hsma_check_sums_shard(plan.handle, xyz, q, 0, Kt)
        phi = torch.zeros(w.N, dtype=torch.float64, device="cuda")
        U = torch.zeros(1, dtype=torch.float64, device="cuda")
        for part, (t0, t1) in enumerate(shard.shard_bounds(w.N, n_parts)):
            pp = torch.empty(w.N, dtype=torch.float64, device="cuda")
            up = torch.empty(1, dtype=torch.float64, device="cuda")
            H.binding.hsma_evaluate_rest_part(plan.handle, xyz, q, part, n_parts, t0, t1, pp, None, up)
            plan.sync()
            phi += pp
            U += up
        assert rel_inf(phi.cpu().numpy(), phi_ref.cpu().numpy()) <= 1e-12
        assert abs(float(U) - float(U_ref)) <= 1e-12 * abs(float(U_ref))
        assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL and abs(float(U) - r.U) <= U_TOL * abs(r.U)
        # bad part index: refused
        with pytest.raises(Exception):
            H.binding.hsma_evaluate_rest_part(plan.handle, xyz, q, n_parts, n_parts, 0, w.N, phi, None, U)
        # the same with forces: partial phi, F and U add up
        phi_r, F_ref, U_r = plan.evaluate_forces(xyz, q, sync=True)
        H.binding.hsma_check_sums_shard(plan.handle, xyz, q, 0, Kt)
        phi.zero_(); U.zero_()
        F = torch.zeros(w.N, 3, dtype=torch.float64, device="cuda")
        for part, (t0, t1) in enumerate(shard.shard_bounds(w.N, n_parts)):
            pp = torch.empty(w.N, dtype=torch.float64, device="cuda")
            fp = torch.empty(w.N, 3, dtype=torch.float64, device="cuda")
            up = torch.empty(1, dtype=torch.float64, device="cuda")
            H.binding.hsma_evaluate_rest_part(plan.handle, xyz, q, part, n_parts, t0, t1, pp, fp, up)
            plan.sync()
            phi += pp
            F += fp
            U += up
        assert rel_inf(phi.cpu().numpy(), phi_r.cpu().numpy()) <= 1e-12
        assert np.max(np.abs((F - F_ref).cpu().numpy())) <= 1e-12 * max(float(F_ref.abs().max()), float(phi_r.abs().max()))
        assert abs(float(U) - float(U_r)) <= 1e-12 * abs(float(U_r))


def test_evaluate_distributed_single_process_uses_the_part_form(H):
    """shard.evaluate_distributed without a process group (world = 1): part 0 of 1 = the whole evaluate."""
    from paper_1806_04801_b200 import shard
    w = W.config(5, N=8192)
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi_ref, U_ref = plan.evaluate(xyz, q, sync=True)
        phi, F, U = shard.evaluate_distributed(plan, xyz, q)
        plan.sync()
        assert F is None and plan.last_pair_form == SYMMETRIC
        plan.set_pair_form(ORDERED)             # forced ordered pairs: the distributed call takes the target-shard path
        assert not H.binding.hsma_plan_part_form_applies(plan.handle, w.N)
        phi_o, _, U_o = shard.evaluate_distributed(plan, xyz, q)
        plan.sync()
        assert plan.last_pair_form == ORDERED and rel_inf(phi_o.cpu().numpy(), phi_ref.cpu().numpy()) <= 2e-11
        plan.set_pair_form(0)
        phi_f, F_f, U_f = shard.evaluate_distributed(plan, xyz, q, forces=True)
        plan.sync()
        _, F_ref, _ = plan.evaluate_forces(xyz, q, sync=True)
        assert float((F_f - F_ref).abs().max()) <= 1e-12 * float(F_ref.abs().max())
        assert rel_inf(phi.cpu().numpy(), phi_ref.cpu().numpy()) <= 1e-13 and abs(float(U) - float(U_ref)) <= 1e-13 * abs(float(U_ref))
        # small systems keep the target-shard path
        ws = W.config(2)
        with H.Plan.from_workload(ws) as plan_s:
            assert not H.binding.hsma_plan_part_form_applies(plan_s.handle, ws.N)
            ps, _, Us = shard.evaluate_distributed(plan_s, dev(ws.xyz), dev(ws.q))
            pr, Ur = plan_s.evaluate(dev(ws.xyz), dev(ws.q), sync=True)
            assert rel_inf(ps.cpu().numpy(), pr.cpu().numpy()) <= 1e-13


@pytest.mark.parametrize("refine", [1, 2])
@pytest.mark.parametrize("idx,N", [(2, 7938), (3, 9000), (4, 9000), (5, 12288)])
def test_symmetric_forces_match_oracle(H, idx, N, refine):
    """The gradient form of the symmetric kernel (near_sym_field_kernel): forces, potentials and U against the oracle
    for the periodic, mirror-cavity and slab cell tables (reflected axes flip the column gradient), and against the
    ordered potential+gradient kernel."""
    w = W.config(idx, N=N)
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w, rsqrt_refine=refine) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        plan.set_pair_form(SYMMETRIC)
        phi, F, U = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
        plan.set_pair_form(ORDERED)
        phi1, F1, U1 = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == ORDERED
    F, F1, phi = F.cpu().numpy(), F1.cpu().numpy(), phi.cpu().numpy()
    scale = max(float(np.max(np.abs(r.F))), float(np.max(np.abs(w.q)) * np.max(np.abs(r.phi)) / max(w.L)))
    assert np.max(np.abs(F - r.F)) <= 1e-10 * scale
    assert np.max(np.abs(F1 - r.F)) <= 1e-10 * scale
    assert np.max(np.abs(F - F1)) <= 2e-11 * scale
    assert rel_inf(phi, r.phi) <= PHI_TOL and abs(float(U) - r.U) <= U_TOL * abs(r.U)


def test_symmetric_forces_random_magnitudes_and_momentum(H):
    """Random-magnitude charges in the periodic box: forces against the oracle; the net force of the near sum
    vanishes identically in the symmetric form (every pair contributes +f and -f), so the total is at the level of
    the far field's truncation."""
    w = W.config(5, N=8300)
    q = np.random.default_rng(5).standard_normal(w.N)
    q -= q.mean()
    w = w.with_(q=q)
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w) as plan:
        plan.set_pair_form(SYMMETRIC)
        phi, F, U = plan.evaluate_forces(dev(w.xyz), dev(w.q), sync=True)
        assert plan.last_pair_form == SYMMETRIC
    F = F.cpu().numpy()
    assert rel_inf(F, r.F) <= 1e-10
    assert np.abs(F.sum(0)).max() < 1e-3 * np.abs(F).max()


def test_cell_table_sizes_at_the_limit_of_the_symmetric_form(H):
    """125 near cells (shell 2,2,2) fit the symmetric kernel's shared-memory table (128 entries); 175 (shell 2,2,3) do
    not and fall back to the ordered kernel.  Both against the oracle."""
    for shell, cells, form in (((2, 2, 2), 125, SYMMETRIC), ((2, 2, 3), 175, ORDERED)):
        w = W.config(2, N=8000).with_(near_shell=shell)
        r = O.hsma(w)
        with H.Plan.from_workload(w) as plan:
            phi, U = plan.evaluate(dev(w.xyz), dev(w.q), sync=True)
            assert plan.info["near_cells"] == cells and plan.last_pair_form == form
        assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL and abs(float(U) - r.U) <= U_TOL * abs(r.U)


# ------------------------------------------------------------------ all-element comparisons at sizes where one CTA of
# the persistent grid walks many (block, tile) visits and crosses block boundaries (the launch regime of config 5)
def test_symmetric_every_potential_and_force_at_65536(H):
    """Config-5 recipe at N = 65,536 (256 tiles, 32 blocks, ~28 visits per CTA of each launch, block boundaries
    crossed inside a CTA): EVERY potential and EVERY force component of the symmetric potential and gradient kernels
    against the oracle (1.2e11 pairs on the host cores), default refinement (Newton) and the cubic step."""
    w = W.config(5, N=65536)
    r = O.hsma(w, forces=True)
    fscale = float(np.max(np.abs(r.F)))
    for refine in (0, 2):
        with H.Plan.from_workload(w, rsqrt_refine=refine) as plan:
            xyz, q = dev(w.xyz), dev(w.q)
            phi, U = plan.evaluate(xyz, q, sync=True)
            assert plan.last_pair_form == SYMMETRIC
            phi_f, F, U_f = plan.evaluate_forces(xyz, q, sync=True)
            assert plan.last_pair_form == SYMMETRIC
        assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL and abs(float(U) - r.U) <= U_TOL * abs(r.U)
        assert rel_inf(phi_f.cpu().numpy(), r.phi) <= PHI_TOL and abs(float(U_f) - r.U) <= U_TOL * abs(r.U)
        assert np.max(np.abs(F.cpu().numpy() - r.F)) <= 1e-10 * fscale


@pytest.mark.parametrize("idx,N", [(3, 40961), (4, 43010)])
def test_symmetric_every_potential_ragged_mirror_and_slab_tables(H, idx, N):
    """Mirror-cavity (27 reflected cells, gamma = -1) and slab (45 cells, reflected + weighted) tables at ragged sizes
    above 40k (161 / 169 tiles: a partly filled last tile and a partly filled last block): every potential, every
    force component and U against the oracle."""
    w = W.config(idx, N=N)
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi, U = plan.evaluate(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
        phi_f, F, U_f = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
    assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL and abs(float(U) - r.U) <= U_TOL * abs(r.U)
    assert rel_inf(phi_f.cpu().numpy(), r.phi) <= PHI_TOL and abs(float(U_f) - r.U) <= U_TOL * abs(r.U)
    assert np.max(np.abs(F.cpu().numpy() - r.F)) <= 1e-10 * float(np.max(np.abs(r.F)))


# ------------------------------------------------------------------ bounded scratch: the pairs are walked in waves
@pytest.mark.parametrize("idx,N", [(5, 12288), (4, 9000), (3, 20011)])
def test_waves_of_the_symmetric_form(H, idx, N):
    """hsma_plan_set_sym_scratch_cap: with a tiny cap the unordered pairs are walked in many waves (launch + gather
    each, wave boundaries inside visits and inside blocks); potentials, forces and the PART form agree with the
    single-wave result to rounding, meet the oracle bars and stay deterministic."""
    import torch
    w = W.config(idx, N=N)
    r = O.hsma(w, forces=True)
    fscale = float(np.max(np.abs(r.F)))
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi0, U0 = plan.evaluate(xyz, q, sync=True)
        _, F0, _ = plan.evaluate_forces(xyz, q, sync=True)
        launches_one_wave = plan.launches_last_evaluate()
    for cap in (2 * 2048, 37 * 2048, 301 * 8192):     # 2 / 37 visits per potential wave, 9 / 301 per force wave
        with H.Plan.from_workload(w) as plan:
            plan.set_sym_scratch_cap(cap)
            xyz, q = dev(w.xyz), dev(w.q)
            phi, U = plan.evaluate(xyz, q, sync=True)
            assert plan.last_pair_form == SYMMETRIC
            phi_f, F, U_f = plan.evaluate_forces(xyz, q, sync=True)
            assert plan.last_pair_form == SYMMETRIC
            if cap < 100000:
                assert plan.launches_last_evaluate() > launches_one_wave      # one launch + one gather per wave
            phi2, U2 = plan.evaluate(xyz, q, sync=True)
            assert torch.equal(phi2, phi) and float(U2) == float(U)
            # PART form on top of the waves: three "ranks" one after the other
            tot = torch.zeros(w.N, dtype=torch.float64, device="cuda")
            Ut = 0.0
            for part in range(3):
                t0, t1 = part * w.N // 3, (part + 1) * w.N // 3
                pp = torch.empty(w.N, dtype=torch.float64, device="cuda")
                Up = torch.empty(1, dtype=torch.float64, device="cuda")
                H.hsma_check_sums_shard(plan.handle, xyz, q, 0, plan.info["check_targets"])
                H.hsma_evaluate_rest_part(plan.handle, xyz, q, part, 3, t0, t1, pp, None, Up)
                plan.sync()
                tot += pp
                Ut += float(Up)
        for got in (phi, phi_f, tot):
            assert rel_inf(got.cpu().numpy(), r.phi) <= PHI_TOL
            assert rel_inf(got.cpu().numpy(), phi0.cpu().numpy()) <= 1e-12
        for u in (float(U), float(U_f), Ut):
            assert abs(u - r.U) <= U_TOL * abs(r.U)
        assert np.max(np.abs(F.cpu().numpy() - r.F)) <= 1e-10 * fscale
        assert np.max(np.abs((F - F0).cpu().numpy())) <= 1e-12 * fscale


def test_scratch_stays_linear_in_N_at_one_million(H):
    """N = 2^20 (config-5 recipe), potentials and forces in the symmetric form: the column scratch of a single launch
    would be 2.1 GB (8.6 GB with forces); walked in waves the whole per-evaluate scratch of the plan stays below
    0.5 GB, and a slice of potentials and forces straddling a block boundary meets the oracle at the bars."""
    w = W.config(5, N=1 << 20)
    sl = slice(524288 - 32, 524288 + 32)
    r = O.hsma(w, targets_slice=sl, forces=True)
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi, U = plan.evaluate(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
        phi_f, F, U_f = plan.evaluate_forces(xyz, q, sync=True)
        assert plan.last_pair_form == SYMMETRIC
        assert plan.scratch_bytes < 500e6
    phi, phi_f, F = phi.cpu().numpy(), phi_f.cpu().numpy(), F.cpu().numpy()
    scale = float(np.max(np.abs(phi)))
    assert np.max(np.abs(phi[sl] - r.phi)) <= PHI_TOL * scale and np.max(np.abs(phi_f[sl] - r.phi)) <= PHI_TOL * scale
    assert np.max(np.abs(F[sl] - r.F)) <= 1e-10 * float(np.max(np.abs(F)))
    assert abs(float(U) - float(U_f)) <= U_TOL * abs(float(U))
    Uself = 0.5 * float(np.sum(np.asarray(w.q, dtype=np.longdouble) * phi.astype(np.longdouble)))
    assert abs(float(U) - Uself) <= U_TOL * abs(Uself)
