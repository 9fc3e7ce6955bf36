"""Pins of the CPU oracle against things other than itself (all `-m "not gpu"`).

Each test names the part of oracle/hsma_oracle.py it pins and the mistake it is meant to catch.
Tolerances are the method's truncation accuracy at the stated (p, M, shell), not rounding.
"""
import math

import numpy as np
import pytest
from scipy.special import eval_legendre

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins
from tests.conftest import golden

MADELUNG = -golden("madelung_nacl.txt")[0][0]          # PAPER.md:165, positive constant


# ---------------------------------------------------------------------------------------------
# cell table + near sum (oracle/direct_sum.c)  <- explicit image lists, pure Python
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,reflecting,shell,gamma,L", [
    (O.BC_PERIODIC, (False, False, False), (1, 1, 1), 1.0, (1.0, 1.0, 1.0)),
    (O.BC_PERIODIC, (False, False, False), (2, 1, 2), 1.0, (1.0, 1.3, 0.7)),
    (O.BC_MIRROR_CAVITY, (True, True, True), (1, 1, 1), -1.0, (1.0, 1.0, 1.0)),
    (O.BC_MIRROR_CAVITY, (True, True, True), (2, 2, 1), 0.3, (2.0, 1.0, 1.5)),
    (O.BC_SLAB, (False, False, True), (1, 1, 2), 0.5, (1.0, 1.0, 0.5)),
])
def test_near_sum_matches_explicit_images(kind, reflecting, shell, gamma, L):
    rng = np.random.default_rng(11)
    N = 7
    src = (rng.random((N, 3)) - 0.5) * np.array(L)
    q = rng.normal(size=N)
    cells = O.cell_table(kind, L, shell, gamma)
    # potentials at the sources themselves (self term of the central cell dropped)
    got = O.near_sum(src, src, q, cells, self_offset=0)
    want = pins.brute_image_sum(src, src, q, L, reflecting, shell, gamma, skip_self=True)
    np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-13)
    # potentials at other points, nothing dropped; and a slice with an offset
    tg = (rng.random((5, 3)) - 0.5) * np.array(L) * 1.4
    got = O.near_sum(tg, src, q, cells)
    want = pins.brute_image_sum(tg, src, q, L, reflecting, shell, gamma)
    np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-13)
    got = O.near_sum(src[3:6], src, q, cells, self_offset=3)
    want = pins.brute_image_sum(src, src, q, L, reflecting, shell, gamma, skip_self=True)[3:6]
    np.testing.assert_allclose(got, want, rtol=1e-13, atol=1e-13)


def test_far_cell_table_is_block_minus_near():
    L, gamma = (1.0, 1.0, 0.5), 0.5
    rng = np.random.default_rng(5)
    src = (rng.random((4, 3)) - 0.5) * np.array(L)
    q = np.array([1.0, -1.0, 1.0, -1.0])
    tg = (rng.random((3, 3)) - 0.5) * np.array(L)
    far = O.cell_table(O.BC_SLAB, L, (2, 2, 3), gamma, exclude_shell=(1, 1, 2))
    assert far.w.shape[0] == 5 * 5 * 7 - 3 * 3 * 5 and far.central == -1
    got = O.near_sum(tg, src, q, far)
    want = pins.brute_image_sum(tg, src, q, L, (False, False, True), (2, 2, 3), gamma,
                                exclude_shell=(1, 1, 2))
    np.testing.assert_allclose(got, want, rtol=1e-12, atol=1e-13)


def test_rock_salt_shell_sums_approach_madelung():
    """Brute-force image sums over many shells (north_star pin): the 8-ion rock-salt cell has no
    dipole and no quadrupole, so cubic shell sums converge quickly to the Madelung constant."""
    xyz, q, L = W.rock_salt(1)
    src = xyz - L / 2
    errs = []
    for S in (2, 4, 8):
        cells = O.cell_table(O.BC_PERIODIC, (L, L, L), (S, S, S), 1.0)
        phi = O.near_sum(src, src, q, cells, self_offset=0)
        M = O.madelung_constant(O.energy(q, phi), len(q), 1.0)
        errs.append(abs(M - MADELUNG))
    assert errs[2] < errs[1] < errs[0]
    assert errs[2] < 2e-5


# ---------------------------------------------------------------------------------------------
# node sum (charge + exact dipole)  <- closed forms
# ---------------------------------------------------------------------------------------------
def test_node_sum_single_node_closed_form():
    R = np.array([[0.3, -0.2, 2.0]])
    n = np.array([[0.0, 0.0, 1.0]])
    tg = np.array([[0.1, 0.4, -0.5], [0.0, 0.0, 0.0]])
    got = O.node_sum(tg, R, n, np.array([2.0]), np.array([0.7]))
    for t in range(2):
        d = tg[t] - R[0]
        rho = np.linalg.norm(d)
        want = 2.0 / rho - 0.7 * d[2] / rho ** 3
        assert abs(got[t] - want) < 1e-15
    # the dipole term is the directional derivative of 1/rho along +n at the node (finite difference)
    h = 1e-6
    fd = (1.0 / np.linalg.norm(tg[0] - (R[0] + h * n[0])) - 1.0 / np.linalg.norm(tg[0] - (R[0] - h * n[0]))) / (2 * h)
    only_dip = O.node_sum(tg[:1], R, n, np.array([0.0]), np.array([1.0]))[0]
    assert abs(only_dip - (-fd)) < 1e-9


def test_energy_closed_form():
    q = np.array([1.0, -2.0, 0.5])
    phi = np.array([0.25, 4.0, -8.0])
    assert O.energy(q, phi) == 0.5 * (0.25 - 8.0 - 4.0)


# ---------------------------------------------------------------------------------------------
# basis (real solid harmonics)  <- addition theorem, harmonicity, orthonormality
# ---------------------------------------------------------------------------------------------
def test_harmonics_addition_theorem():
    """sum_m Y_nm(a) Y_nm(b) = (2n+1)/(4 pi) P_n(a.b): pins normalisation, the Legendre
    recurrences and the cos/sin pairing, for every degree."""
    rng = np.random.default_rng(2)
    p = 14
    a = rng.normal(size=(6, 3)); a /= np.linalg.norm(a, axis=1)[:, None]
    b = rng.normal(size=(6, 3)); b /= np.linalg.norm(b, axis=1)[:, None]
    Ya = O.real_solid_harmonics(a, p, 1.0)
    Yb = O.real_solid_harmonics(b, p, 1.0)
    for n in range(p):
        lo, hi = n * n, (n + 1) * (n + 1)
        got = (Ya[:, lo:hi] * Yb[:, lo:hi]).sum(1)
        want = (2 * n + 1) / (4 * math.pi) * eval_legendre(n, (a * b).sum(1))
        np.testing.assert_allclose(got, want, atol=2e-13)


def test_harmonics_radial_scaling_and_laplacian():
    rng = np.random.default_rng(3)
    p, a = 9, 1.7
    x = rng.normal(size=(4, 3))
    B1 = O.real_solid_harmonics(x, p, a)
    B2 = O.real_solid_harmonics(2.0 * x, p, a)
    np.testing.assert_allclose(B2, B1 * 2.0 ** O.degree_of_column(p), rtol=1e-12, atol=1e-14)
    # harmonic: 7-point Laplacian vanishes to O(h^2)
    h = 1e-3
    lap = -6.0 * B1
    for ax in range(3):
        e = np.zeros(3); e[ax] = h
        lap = lap + O.real_solid_harmonics(x + e, p, a) + O.real_solid_harmonics(x - e, p, a)
    assert np.abs(lap / h ** 2).max() < 1e-3 * np.abs(B1).max() / 1e-1
    # column order: n^2 + n + m; the (1, m) block is proportional to (y, z, x)
    c = math.sqrt(3 / (4 * math.pi)) / a
    np.testing.assert_allclose(B1[:, 1:4], c * x[:, [1, 2, 0]], rtol=1e-12)
    np.testing.assert_allclose(B1[:, 0], 1 / math.sqrt(4 * math.pi))


def test_harmonics_orthonormal_under_paper_quadrature():
    """Y_nm orthonormal on the sphere, integrated with the paper's lattice rule;
    also pins the rule itself (weights, warp)."""
    F2, R = 987, 1.3
    nodes, nrm, w = O.nodes_lattice(F2, R)
    p = 10
    Y = O.real_solid_harmonics(nodes, p, R)
    G = (Y * (w / R ** 2)[:, None]).T @ Y
    assert np.abs(G - np.eye(p * p)).max() < 1e-9


# ---------------------------------------------------------------------------------------------
# nodes and check points  <- counts printed in the paper, closed-form totals
# ---------------------------------------------------------------------------------------------
def test_node_counts_and_weight_sums():
    for F2, No in golden("node_counts.txt"):
        nodes, nrm, w = O.nodes_lattice(int(F2), 2.0)
        assert 3 * nodes.shape[0] == int(No)                      # three spheres
        assert abs(w.sum() - 4 * math.pi * 4.0) < 1e-11
        np.testing.assert_allclose(np.linalg.norm(nodes, axis=1), 2.0, rtol=1e-14)
        np.testing.assert_allclose(np.linalg.norm(nrm, axis=1), 1.0, rtol=1e-14)
    for M in (400, 2000, 20000):
        nodes, nrm, w = O.nodes_spiral(M, 1.5)
        assert nodes.shape == (M, 3)
        assert abs(w.sum() - 4 * math.pi * 2.25) < 1e-10
        # quadrature of z^2 over the sphere: (4 pi R^2) R^2 / 3
        assert abs((w * nodes[:, 2] ** 2).sum() - 4 * math.pi * 1.5 ** 4 / 3) < 1e-8


def test_checkpoint_spiral_geometry():
    K, R0 = 200, math.sqrt(3.0)
    x = O.fibonacci_sphere_checkpoints(K, R0)
    np.testing.assert_allclose(np.linalg.norm(x, axis=1), R0, rtol=1e-14)
    z = x[:, 2] / R0
    np.testing.assert_allclose(z, (2 * np.arange(1, K + 1) - 1) / K - 1, atol=1e-15)
    np.testing.assert_allclose(np.diff(z), 2.0 / K, atol=1e-14)                          # equal-area bands
    xt = O.wrap_into_box(x, (2.0, 2.0, 2.0))
    assert np.abs(xt).max() <= 1.0 + 1e-15
    k = (x - xt) / 2.0
    np.testing.assert_allclose(k, np.round(k), atol=1e-14)


# ---------------------------------------------------------------------------------------------
# mapping + quadrature  <- Green's identity: surface images reproduce the harmonic series inside
# ---------------------------------------------------------------------------------------------
def test_surface_images_reproduce_series_inside():
    """Eq.(10): for any interior point the node sum equals sum A_nm B_nm(r).
    A sign error in the dipole layer, a missing 1/(4 pi), or n vs n+1 in Eq.(11) breaks it."""
    w = W.config(2, N=60).with_(p=10, M=2 * 988, quad_rule=W.QUAD_LATTICE)
    r = O.hsma(w)
    rng = np.random.default_rng(0)
    pts = (rng.random((20, 3)) - 0.5)
    series = O.series_at(pts, r.A, w.p, 0.5 * math.sqrt(3.0))
    images = O.node_sum(pts, r.nodes, r.normals, r.Q, r.D)
    assert np.abs(images - series).max() < 1e-10 * max(1.0, np.abs(series).max())
    # the spiral rule with the config's M is good to the truncation level as well
    r2 = O.hsma(w.with_(M=2000, quad_rule=W.QUAD_SPIRAL))
    images2 = O.node_sum(pts, r2.nodes, r2.normals, r2.Q, r2.D)
    assert np.abs(images2 - series).max() < 1e-7 * max(1.0, np.abs(series).max())


def test_fd_three_sphere_form_matches_exact_dipole():
    """Eq.(12)-(14) PAPER.md:107-120 (the paper's all-Coulomb form) vs the exact dipole (S9)."""
    w = W.config(2, N=60).with_(p=10, M=2000)
    a = O.hsma(w, dipole="exact")
    b = O.hsma(w, dipole="fd3", dr_rel=1e-4)
    assert np.abs(a.phi_out - b.phi_out).max() < 1e-7 * np.abs(a.phi_out).max()
    c = O.hsma(w, dipole="fd3", dr_rel=1e-3)     # truncation error is O(dr^2)
    e_b = np.abs(a.phi_out - b.phi_out).max()
    e_c = np.abs(a.phi_out - c.phi_out).max()
    assert 30 < e_c / e_b < 300
