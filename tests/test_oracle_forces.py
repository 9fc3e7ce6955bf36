"""Pins of the oracle's gradient / force routines (Eq.(9)).
All `-m "not gpu"`.  The gradient routines are separate C loops (oracle_near_grad, oracle_node_grad);
they are pinned against numerical differentiation of the (independently pinned) potential routines,
closed forms, the textbook Ewald force and physical properties."""
import math

import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins


def central_difference(f, x, h):
    g = np.zeros_like(x)
    for a in range(3):
        e = np.zeros(3)
        e[a] = h
        g[:, a] = (f(x + e) - f(x - e)) / (2 * h)
    return g


@pytest.mark.parametrize("kind,shell,gamma,L", [
    (O.BC_PERIODIC, (1, 1, 1), 1.0, (1.0, 1.0, 1.0)),
    (O.BC_MIRROR_CAVITY, (1, 1, 1), -1.0, (1.0, 1.3, 0.8)),
    (O.BC_SLAB, (1, 1, 2), 0.5, (1.0, 1.0, 0.5)),
])
def test_near_grad_is_the_derivative_of_near_sum(kind, shell, gamma, L):
    rng = np.random.default_rng(3)
    Lh = np.asarray(L)
    src = (rng.random((40, 3)) - 0.5) * Lh
    q = rng.standard_normal(40)
    tgt = (rng.random((25, 3)) - 0.5) * Lh
    cells = O.cell_table(kind, L, shell, gamma)
    g = O.near_grad(tgt, src, q, cells)
    fd = central_difference(lambda x: O.near_sum(x, src, q, cells), tgt, 1e-5)
    assert np.abs(g - fd).max() < 2e-7 * np.abs(g).max()      # O(h^2) of the difference quotient
    # Richardson: halving h must cut the discrepancy ~4x (it is the FD error, not the gradient's)
    fd2 = central_difference(lambda x: O.near_sum(x, src, q, cells), tgt, 2e-5)
    assert np.abs(g - fd).max() < 0.5 * np.abs(g - fd2).max()


def test_near_grad_self_exclusion_and_closed_form():
    """Two charges, one cell: grad at charge 0 is q1 (r1 - r0)/|r1 - r0|^3 (self skipped)."""
    src = np.array([[0.1, -0.2, 0.05], [-0.3, 0.25, 0.4]])
    q = np.array([1.5, -2.0])
    one = O.CellTable(np.zeros((1, 3), dtype=np.int64), np.zeros((1, 3)), np.ones((1, 3)), np.ones(1), 0)
    g = O.near_grad(src, src, q, one, self_offset=0)
    d = src[1] - src[0]
    r3 = np.linalg.norm(d) ** 3
    assert np.allclose(g[0], q[1] * d / r3, rtol=1e-14)
    assert np.allclose(g[1], -q[0] * d / r3, rtol=1e-14)
    # Newton's third law for the pair forces F = -q grad
    F = -q[:, None] * g
    assert np.abs(F.sum(0)).max() < 1e-15 * np.abs(F).max()


def test_node_grad_closed_forms_and_derivative():
    R = np.array([[0.0, 0.0, 2.0]])
    n = np.array([[0.0, 0.0, 1.0]])
    t = np.array([[0.3, -0.4, 0.5]])
    d = t[0] - R[0]
    rho = np.linalg.norm(d)
    gQ = O.node_grad(t, R, n, np.array([1.7]), np.array([0.0]))
    assert np.allclose(gQ[0], -1.7 * d / rho ** 3, rtol=1e-14)
    gD = O.node_grad(t, R, n, np.array([0.0]), np.array([0.9]))
    nd = n[0] @ d
    assert np.allclose(gD[0], -0.9 * n[0] / rho ** 3 + 3 * 0.9 * nd * d / rho ** 5, rtol=1e-13)
    rng = np.random.default_rng(4)
    nodes, nrm, w = O.nodes_spiral(300, 1.4)
    Q, D = rng.standard_normal(300), rng.standard_normal(300)
    tg = rng.random((20, 3)) - 0.5
    g = O.node_grad(tg, nodes, nrm, Q, D)
    fd = central_difference(lambda x: O.node_sum(x, nodes, nrm, Q, D), tg, 1e-5)
    assert np.abs(g - fd).max() < 2e-7 * np.abs(g).max()


@pytest.fixture(scope="module")
def ewald_force_case():
    w = W.config(2, N=120)
    L = np.array(w.L)
    f1 = pins.ewald_forces(w.xyz, w.q, L, alpha=6.0, rcut_cells=1, kmax=9)
    f2 = pins.ewald_forces(w.xyz, w.q, L, alpha=8.0, rcut_cells=1, kmax=12)
    assert np.abs(f1 - f2).max() < 1e-10 * np.abs(f1).max()
    return w, f2


def test_ewald_force_pin_is_the_derivative_of_the_ewald_energy():
    w = W.config(2, N=16)
    L = np.array(w.L)
    F = pins.ewald_forces(w.xyz, w.q, L, 6.0, 1, 9)
    h = 1e-6
    for i, a in ((0, 0), (5, 2), (11, 1)):
        xp, xm = w.xyz.copy(), w.xyz.copy()
        xp[i, a] += h
        xm[i, a] -= h
        U = lambda x: 0.5 * float(w.q @ pins.ewald_potentials(x, w.q, L, 6.0, 1, 9))
        assert abs(F[i, a] + (U(xp) - U(xm)) / (2 * h)) < 1e-7 * np.abs(F).max()


def test_periodic_forces_match_ewald(ewald_force_case):
    """forces converge like the potential, with an error about 10x larger."""
    w, F_e = ewald_force_case
    scale = np.abs(F_e).max()
    errs = []
    for p, M in ((10, 2000), (16, 6000), (22, 2 * 988 * 2)):
        r = O.hsma(w.with_(p=p, M=M, K=max(w.K, 2 * p * p)), forces=True)
        errs.append(np.abs(r.F - F_e).max() / scale)
    assert errs[0] < 5e-3 and errs[1] < 5e-5 and errs[2] < 5e-7
    assert errs[2] < errs[1] < errs[0]


def test_periodic_net_force_vanishes(ewald_force_case):
    w, F_e = ewald_force_case
    r = O.hsma(w.with_(p=16, M=6000, K=600), forces=True)
    assert np.abs(r.F.sum(0)).max() < 1e-4 * np.abs(r.F).max()


def test_charge_near_a_grounded_wall_is_attracted_with_the_image_force():
    """One charge at distance a << L from the wall x = 0 of the grounded unit cube: the force is
    dominated by its nearest image, F_x ~ -q^2/(2a)^2 (towards the wall)."""
    a = 0.02
    L = (1.0, 1.0, 1.0)
    chk = W.seeded_face_points(1200, L, W.ALL_FACES, seed=9)
    w = W.Workload("wall", W.BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0, 1.5 * math.sqrt(3) / 2, 16, 4000, 1200,
                   np.array([[a, 0.5, 0.5]]), np.array([1.0]), check_xyz=chk)
    r = O.hsma(w, forces=True)
    assert r.F[0, 0] < 0
    assert abs(r.F[0, 0] + 1.0 / (2 * a) ** 2) < 0.01 / (2 * a) ** 2   # other images are O(1) vs 625
    assert abs(r.F[0, 1]) < 1e-6 and abs(r.F[0, 2]) < 1e-6           # symmetric in y and z


def test_forces_are_minus_the_gradient_of_the_energy_in_the_cavity():
    """Grounded cavity, 3 charges (PAPER.md:167 geometry): F_i = -dU/dr_i with U = 1/2 sum q phi,
    checked by moving one charge (the fit is redone for each displaced configuration)."""
    w = W.paper_example2().with_(p=20, M=6000)
    r = O.hsma(w, forces=True)
    h = 1e-5
    for i, a in ((0, 0), (1, 2)):
        xp, xm = w.xyz.copy(), w.xyz.copy()
        xp[i, a] += h
        xm[i, a] -= h
        dU = (O.hsma(w.with_(xyz=xp)).U - O.hsma(w.with_(xyz=xm)).U) / (2 * h)
        assert abs(r.F[i, a] + dU) < 2e-6 * np.abs(r.F).max()
