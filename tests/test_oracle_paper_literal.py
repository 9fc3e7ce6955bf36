"""Pins of the oracle's paper-literal variants: the sphere-culled near set of PAPER.md:62
and the three-sphere central-difference dipole of Eq.(12)-(14), at the paper's own operating points.  `-m "not gpu"`."""
import math

import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins
from tests.conftest import golden

MADELUNG = -golden("madelung_nacl.txt")[0][0]


@pytest.mark.parametrize("kind,shell,gamma", [(O.BC_PERIODIC, (1, 1, 1), 1.0), (O.BC_MIRROR_CAVITY, (1, 1, 1), -1.0),
                                              (O.BC_SLAB, (1, 1, 2), 0.5)])
def test_images_inside_sphere_matches_a_plain_loop(kind, shell, gamma):
    rng = np.random.default_rng(8)
    L = (1.0, 1.0, 0.5) if kind == O.BC_SLAB else (1.0, 1.0, 1.0)
    src = (rng.random((13, 3)) - 0.5) * np.array(L)
    q = rng.standard_normal(13)
    R = 1.2
    cells = O.cell_table(kind, L, shell, gamma)
    pos, chg = O.images_inside_sphere(src, q, cells, R)
    assert np.allclose(pos[:13], src) and np.allclose(chg[:13], q)       # the sources come first, in order
    refl = {O.BC_PERIODIC: (0, 0, 0), O.BC_MIRROR_CAVITY: (1, 1, 1), O.BC_SLAB: (0, 0, 1)}[kind]
    want = []
    for kx in range(-shell[0], shell[0] + 1):
        for ky in range(-shell[1], shell[1] + 1):
            for kz in range(-shell[2], shell[2] + 1):
                k = (kx, ky, kz)
                for j in range(13):
                    p, wt = [], q[j]
                    for a in range(3):
                        sgn = -1.0 if (refl[a] and k[a] % 2) else 1.0
                        p.append(sgn * src[j, a] + k[a] * L[a])
                        if refl[a]:
                            wt *= gamma ** abs(k[a])
                    if p[0] ** 2 + p[1] ** 2 + p[2] ** 2 <= R * R:
                        want.append((round(p[0], 12), round(p[1], 12), round(p[2], 12), round(wt, 12)))
    got = sorted((round(a, 12), round(b, 12), round(c, 12), round(d, 12)) for (a, b, c), d in zip(pos, chg))
    assert got == sorted(want)
    assert len(got) < 13 * cells.w.shape[0]                               # something was culled


def test_madelung_with_the_papers_near_set_and_three_spheres():
    """64 unit charges on a lattice in the L = 2 box, PBC, alpha = 2, N_o = 5928 (F2 = 987):
    the error falls with P and the printed constant is reached to ~1e-9 at P = 23."""
    xyz, q, _ = W.rock_salt(2)
    errs = {}
    for P in (7, 15, 23):
        w = W.Workload("nacl64", W.BC_PERIODIC, (2.0, 2.0, 2.0), (2, 2, 2), 1.0, 2.0 * math.sqrt(3.0), P + 1,
                       2 * 988, 2 * P * P, xyz * 0.5, q, quad_rule=W.QUAD_LATTICE, near_mode=W.NEAR_SPHERE,
                       dipole_mode=W.DIPOLE_FD3)
        r = O.hsma(w)
        errs[P] = abs(O.madelung_constant(r.U, w.N, 0.5) - MADELUNG)
    assert errs[23] < errs[15] < errs[7]
    assert errs[23] < 5e-9 and errs[15] < 1e-6
    # the exact dipole layer gives the same constant to the accuracy of the central difference (dr = 1e-5 R_s)
    w_exact = w.with_(dipole_mode=W.DIPOLE_EXACT)
    assert abs(O.hsma(w_exact).U - r.U) < 1e-8 * abs(r.U)


def test_paper_timing_workload_against_ewald():
    """random-sign lattice-site charges, alpha = 1.3, P = 25, N_o = 5928, N_m = 2 P^2.
    Energy against the textbook Ewald sum; alpha = 2 (two shells) is much more accurate, as in Fig.4."""
    w = W.paper_timing(216)
    assert w.M * 3 == 5928 and w.K == 1250 and w.p == 26
    L = np.array(w.L)
    phi_e = pins.ewald_potentials(w.xyz, w.q, L, alpha=8.0, rcut_cells=1, kmax=12)
    U_e = 0.5 * float(w.q @ phi_e)
    r13 = O.hsma(w)
    n_images = r13.pairs["b"] // w.N
    assert 5.0 * w.N < n_images < 7.5 * w.N                     # (4 pi/3)(1.3 sqrt3/2)^3 = 5.97 images per source
    e13 = abs(r13.U - U_e) / abs(U_e)
    r20 = O.hsma(w.with_(R_aux=2.0 * math.sqrt(3.0) / 2.0, near_shell=(2, 2, 2)))
    e20 = abs(r20.U - U_e) / abs(U_e)
    assert e13 < 2e-3 and e20 < 1e-6 and e20 < 0.01 * e13


def test_sphere_mode_rejections():
    w = W.paper_timing(64).with_(R_aux=1.6)                       # sphere pokes out of the 3^3 cell block
    with pytest.raises(ValueError):
        O.hsma(w)
