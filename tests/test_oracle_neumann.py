"""Pins of the Neumann (gamma = +1) wall rows of the boundary closure and of
the gradient of the basis they need.  A box with even-reflection walls is one octant of a fully periodic cell of twice
the size that holds the mirror copies of every charge, so the textbook Ewald sum pins it.  `-m "not gpu"`."""
import math

import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins


def test_basis_gradient_is_the_derivative_of_the_basis():
    rng = np.random.default_rng(1)
    x = rng.standard_normal((9, 3)) * 0.6
    p, a = 12, 0.8
    G = O.real_solid_harmonics_grad(x, p, a)

    def fd(h):
        out = np.zeros_like(G)
        for k in range(3):
            e = np.zeros(3)
            e[k] = h
            out[:, :, k] = (O.real_solid_harmonics(x + e, p, a) - O.real_solid_harmonics(x - e, p, a)) / (2 * h)
        return out
    e1, e2 = np.abs(G - fd(1e-4)).max(), np.abs(G - fd(2e-4)).max()
    assert e1 < 1e-5 * np.abs(G).max() and e1 < 0.3 * e2          # O(h^2): it is the difference quotient's error
    # Euler's identity for homogeneous polynomials, r . grad B = n B, and harmonicity via the z-derivative identity
    B = O.real_solid_harmonics(x, p, a)
    n = O.degree_of_column(p)
    assert np.abs(np.einsum("tk,tck->tc", x, G) - n * B).max() < 1e-12 * np.abs(B).max()
    # d/dz (r^n Y_nm) = sqrt((2n+1)(n^2-m^2)/(2n-1)) r^(n-1) Y_(n-1)m   (textbook ladder relation)
    for nn, m in ((3, 1), (5, 0), (7, -4), (11, 6)):
        c = math.sqrt((2 * nn + 1) * (nn * nn - m * m) / (2 * nn - 1)) / a
        assert np.allclose(G[:, O.basis_index(nn, m), 2], c * B[:, O.basis_index(nn - 1, m)], rtol=1e-11, atol=1e-13)
    with pytest.raises(ValueError):
        O.real_solid_harmonics_grad(np.array([[0.0, 0.0, 0.7]]), 4, 1.0)


def mirrored_copies(xyz, q, L, axes):
    """All even reflections of the charges about the lower walls of the listed axes: the contents of the periodic
    cell of size 2 L_a along those axes."""
    pts, chg = [np.asarray(xyz, float)], [np.asarray(q, float)]
    for a in axes:
        more = [p.copy() for p in pts]
        for p_ in more:
            p_[:, a] = -p_[:, a]
        pts += more
        chg += [c.copy() for c in chg]
    return np.concatenate(pts), np.concatenate(chg)


def test_neumann_cavity_is_an_octant_of_a_periodic_cell():
    rng = np.random.default_rng(6)
    N = 12
    xyz = 0.1 + 0.8 * rng.random((N, 3))
    q = W.alternating_charges(N) * (1.0 + rng.random(N))
    q -= q.mean()
    L = (1.0, 1.0, 1.0)
    big_xyz, big_q = mirrored_copies(xyz, q, L, (0, 1, 2))
    phi_e = pins.ewald_potentials(big_xyz, big_q, np.array([2.0, 2.0, 2.0]), alpha=4.0, rcut_cells=1, kmax=10)[:N]
    U_e = 0.5 * float(q @ phi_e)
    errs = []
    for p in (10, 16, 22):
        chk = W.seeded_face_points(max(900, 2 * p * p), L, W.ALL_FACES, seed=12)
        w = W.Workload("neumann_box", W.BC_MIRROR_CAVITY, L, (1, 1, 1), 1.0, 1.5 * math.sqrt(3) / 2, p, 6000,
                       chk.shape[0], xyz, q, check_xyz=chk)
        r = O.hsma(w)
        assert r.A[0] == 0.0
        errs.append(abs(r.U - U_e) / abs(U_e))
        d = r.phi - phi_e
        assert np.abs(d - d.mean()).max() < 100 * max(errs[-1], 1e-11) * np.abs(phi_e).max()   # same up to the gauge
    assert errs[0] < 2e-3 and errs[1] < 2e-5 and errs[2] < 5e-7 and errs[2] < errs[1] < errs[0]


def test_neumann_slab_is_half_of_a_periodic_cell():
    rng = np.random.default_rng(7)
    N = 14
    L = (1.0, 1.0, 0.5)
    xyz = rng.random((N, 3)) * np.array(L)
    xyz[:, 2] = 0.05 + 0.8 * xyz[:, 2]
    q = W.alternating_charges(N)
    big_xyz, big_q = mirrored_copies(xyz, q, L, (2,))
    phi_e = pins.ewald_potentials(big_xyz, big_q, np.array([1.0, 1.0, 1.0]), alpha=7.0, rcut_cells=1, kmax=11)[:N]
    U_e = 0.5 * float(q @ phi_e)
    errs = []
    for p in (10, 18):
        w = W.Workload("neumann_slab", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), 1.0, 1.1, p, 6000,
                       max(700, 2 * p * p), xyz, q, closure=W.CLOSURE_BOUNDARY)
        r = O.hsma(w)
        errs.append(abs(r.U - U_e) / abs(U_e))
    assert errs[0] < 5e-4 and errs[1] < 1e-6 and errs[1] < errs[0]


def test_neumann_needs_a_neutral_system():
    w = W.Workload("bad", W.BC_MIRROR_CAVITY, (1.0, 1.0, 1.0), (1, 1, 1), 1.0, 1.2, 6, 500, 300,
                   np.array([[0.3, 0.4, 0.5]]), np.array([1.0]))
    with pytest.raises(ValueError):
        O.hsma(w)
