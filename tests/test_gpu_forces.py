"""Parity of the CUDA potential+gradient path (forces, Eq.(9)) against the CPU oracle,
through the C-ABI.  Bars: max|dF|/max|F| <= 1e-10 (the north_star bar for phi, applied to the forces),
phi and U as in test_gpu_parity.  All `-m gpu`."""
import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O

pytestmark = pytest.mark.gpu

F_TOL = 1e-10
PHI_TOL = 1e-10
U_TOL = 1e-11


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


# ------------------------------------------------------------------ raw kernels
@pytest.mark.parametrize("kind,L,shell,gamma", [
    (W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0),
    (W.BC_MIRROR_CAVITY, (1.0, 1.5, 0.7), (1, 1, 1), -1.0),
    (W.BC_SLAB_XY_PERIODIC_Z_MIRROR, (1.0, 1.0, 0.5), (1, 1, 2), 0.5),
])
@pytest.mark.parametrize("refine", [1, 2])
@pytest.mark.parametrize("charges", ["normal", "pm1"])
@pytest.mark.parametrize("N,T", [(1, 1), (255, 257), (1000, 1029), (2311, 77)])
def test_direct_field_matches_oracle(H, kind, L, shell, gamma, refine, charges, N, T):
    """Gradient of the near sum for all three cell tables (reflected axes flip the component back),
    generic and uniform-|q| loops, ragged sizes."""
    import torch
    rng = np.random.default_rng(200 + N + T)
    Lh = np.asarray(L)
    src = (rng.random((N, 3)) - 0.5) * Lh
    q = rng.standard_normal(N) if charges == "normal" else W.alternating_charges(N)
    tgt = (rng.random((T, 3)) - 0.5) * Lh * 1.2
    cells = O.cell_table(kind, L, shell, gamma)
    ref_phi = O.near_sum(tgt, src, q, cells)
    ref_g = O.near_grad(tgt, src, q, cells)
    phi = torch.empty(T, dtype=torch.float64, device="cuda")
    g = torch.empty(T, 3, dtype=torch.float64, device="cuda")
    H.hsma_direct_field(dev(tgt), dev(src), dev(q), cells.shift, cells.sign, cells.w, cells.central, -1, refine, phi, g)
    # Newton form: per-pair error <= 1.2e-12 (3.6e-12 on y^3), amplified where image terms of opposite sign cancel
    tol = 3e-11 if refine == 1 else 2e-12
    assert rel_inf(phi.cpu().numpy(), ref_phi) < tol
    assert rel_inf(g.cpu().numpy(), ref_g) < tol


@pytest.mark.parametrize("refine", [1, 2])
@pytest.mark.parametrize("N,t0,T", [(300, 0, 300), (1500, 700, 555), (5000, 4990, 10)])
def test_direct_field_self_exclusion(H, refine, N, t0, T):
    import torch
    rng = np.random.default_rng(17 + N)
    src = rng.random((N, 3)) - 0.5
    q = W.alternating_charges(N)
    cells = O.cell_table(W.BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0)
    ref_g = O.near_grad(src[t0:t0 + T], src, q, cells, self_offset=t0)
    g = torch.empty(T, 3, dtype=torch.float64, device="cuda")
    H.hsma_direct_field(dev(src[t0:t0 + T]), dev(src), dev(q), cells.shift, cells.sign, cells.w, cells.central, t0,
                        refine, None, g)
    got = g.cpu().numpy()
    assert np.all(np.isfinite(got))
    assert rel_inf(got, ref_g) < (3e-11 if refine == 1 else 2e-12)


@pytest.mark.parametrize("T,M", [(1, 8), (300, 127), (1029, 128), (513, 2000)])
def test_node_field_matches_oracle(H, T, M):
    import torch
    rng = np.random.default_rng(T + M + 1)
    nodes, nrm, w = O.nodes_spiral(M, 1.3)
    Q, D = rng.standard_normal(M), rng.standard_normal(M)
    tgt = rng.random((T, 3)) - 0.5
    ref_phi = O.node_sum(tgt, nodes, nrm, Q, D)
    ref_g = O.node_grad(tgt, nodes, nrm, Q, D)
    phi = torch.empty(T, dtype=torch.float64, device="cuda")
    g = torch.empty(T, 3, dtype=torch.float64, device="cuda")
    H.hsma_node_field(dev(tgt), dev(nodes), dev(Q), dev(D[:, None] * nrm), phi, g)
    assert rel_inf(phi.cpu().numpy(), ref_phi) < 1e-13
    assert rel_inf(g.cpu().numpy(), ref_g) < 1e-12


# ------------------------------------------------------------------ full path
def run_forces(H, w, **plan_kw):
    import torch
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w, **plan_kw) as plan:
        phi, F, U = plan.evaluate_forces(dev(w.xyz), dev(w.q), sync=True)
        phi0, U0 = plan.evaluate(dev(w.xyz), dev(w.q), sync=True)
        torch.cuda.synchronize()
    return r, phi.cpu().numpy(), F.cpu().numpy(), float(U), phi0.cpu().numpy(), float(U0)


def force_scale(r, w):
    """max|F|, but never below max|q| max|phi| / L: in a perfect crystal (config 1) every force vanishes by
    symmetry and what is left is the rounding of O(1) terms, so max|F| itself is no scale."""
    return max(float(np.max(np.abs(r.F))), float(np.max(np.abs(w.q)) * np.max(np.abs(r.phi)) / max(w.L)))


def check(r, phi, F, U, phi0, U0, w):
    assert np.max(np.abs(F - r.F)) <= F_TOL * force_scale(r, w)
    assert rel_inf(phi, r.phi) <= PHI_TOL
    assert abs(U - r.U) <= U_TOL * abs(r.U)
    # the potential of the force path and of the plain path agree to rounding (different kernels)
    assert rel_inf(phi, phi0) <= 1e-11 and abs(U - U0) <= 1e-11 * abs(U0)


@pytest.mark.parametrize("refine", [0, 1, 2])
@pytest.mark.parametrize("idx", [1, 2, 3, 4])
def test_config_forces(H, idx, refine):
    """BASELINE.json configs 1-4 at full size: every force component compared with the oracle."""
    w = W.config(idx)
    check(*run_forces(H, w, rsqrt_refine=refine), w)


def test_paper_example2_forces(H):
    """PAPER.md:167 geometry (charges +2, -1, -1: the generic multiply-by-q loops)."""
    w = W.paper_example2()
    check(*run_forces(H, w), w)


def test_config3_random_magnitude_forces(H):
    w = W.config(3)
    w = w.with_(q=np.random.default_rng(34).standard_normal(w.N))
    check(*run_forces(H, w), w)


def test_config5_reduced_forces_shards_and_host(H):
    """Config 5 recipe at N = 20,012: full forces; shards reassemble to rounding (the split points of the
    partial sums move with the shard); host form agrees bit for bit;
    the periodic net force vanishes to truncation accuracy."""
    import torch
    w = W.config(5, N=20012)
    r = O.hsma(w, forces=True)
    with H.Plan.from_workload(w) as plan:
        xyz, q = dev(w.xyz), dev(w.q)
        phi, F, U = plan.evaluate_forces(xyz, q, sync=True)
        Fh = F.cpu().numpy()
        assert rel_inf(Fh, r.F) <= F_TOL
        assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL
        assert abs(float(U) - r.U) <= U_TOL * abs(r.U)
        parts = []
        for a, b in ((0, 4096), (4096, 4097), (4097, 20012)):
            _, Fs, _ = plan.evaluate_forces_shard(xyz, q, a, b, sync=True)
            parts.append(Fs.cpu().numpy())
        assert np.max(np.abs(np.concatenate(parts) - Fh)) <= 1e-13 * np.max(np.abs(Fh))
        F_host = np.empty((w.N, 3))
        phi_host = np.empty(w.N)
        U_host = np.empty(1)
        H.hsma_evaluate_forces_host(plan.handle, np.ascontiguousarray(w.xyz), np.ascontiguousarray(w.q), phi_host,
                                    F_host, U_host)
        assert np.array_equal(F_host, Fh) and U_host[0] == float(U)
    assert np.abs(Fh.sum(0)).max() < 1e-3 * np.abs(Fh).max()


def test_config5_full_size_forces_sampled(H):
    """Config 5 at N = 262,144: forces on a 64-target slice straddling a tile boundary against the oracle."""
    w = W.config(5)
    sl = slice(131072 - 24, 131072 + 40)
    r = O.hsma(w, targets_slice=sl, forces=True)
    with H.Plan.from_workload(w) as plan:
        i0, i1, _ = sl.indices(w.N)
        phi, F, U = plan.evaluate_forces_shard(dev(w.xyz), dev(w.q), i0, i1, sync=True)
    assert rel_inf(F.cpu().numpy(), r.F) <= F_TOL
    assert rel_inf(phi.cpu().numpy(), r.phi) <= PHI_TOL
