"""Pin of the grounded-slab boundary closure: x,y periodic, conducting plates
at z = 0, H (gamma = -1), closed by wrapped circumsphere pairs in x,y plus Dirichlet rows on the plates.
Against the in-plane Fourier series of the textbook parallel-plate Green function.  `-m "not gpu"`."""
import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins

L = (1.0, 1.0, 0.5)


def slab(p, xyz, q, K=None, M=6000):
    return W.Workload("slab_grounded", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), -1.0, 1.1, p, M,
                      K or max(700, 2 * p * p), np.asarray(xyz, float), np.asarray(q, float), closure=W.CLOSURE_BOUNDARY)


def test_green_function_of_the_grounded_slab():
    A = np.array([[0.32, 0.58, 0.13]])
    Bs = np.array([[0.61, 0.41, 0.37], [0.2, 0.8, 0.4], [0.5, 0.5, 0.3]])
    g = np.array([pins.grounded_slab_green(b, A[0], 1.0, 1.0, 0.5) for b in Bs])
    cells = O.cell_table(O.BC_SLAB, L, (1, 1, 2), -1.0)
    half, R0 = 0.5 * np.array(L), 0.5 * np.linalg.norm(L)
    errs = []
    for p in (10, 16, 22):
        r = O.hsma(slab(p, A, [1.0]))
        tot = O.near_sum(Bs - half, A - half, np.array([1.0]), cells) + O.series_at(Bs - half, r.A, p, R0)
        errs.append(np.abs(tot - g).max())
    assert errs[0] < 5e-5 and errs[1] < 1e-7 and errs[2] < 5e-10
    assert errs[2] < errs[1] < errs[0]


def test_pin_is_symmetric_periodic_and_vanishes_on_the_plates():
    a, b = np.array([0.1, 0.7, 0.2]), np.array([0.8, 0.3, 0.35])
    g = pins.grounded_slab_green(a, b, 1.0, 1.0, 0.5)
    assert abs(g - pins.grounded_slab_green(b, a, 1.0, 1.0, 0.5)) < 1e-13
    assert abs(g - pins.grounded_slab_green(a + np.array([1.0, -2.0, 0.0]), b, 1.0, 1.0, 0.5)) < 1e-12
    assert abs(pins.grounded_slab_green(np.array([0.3, 0.3, 0.0]), b, 1.0, 1.0, 0.5)) < 1e-13
    assert abs(pins.grounded_slab_green(np.array([0.3, 0.3, 0.5]), b, 1.0, 1.0, 0.5)) < 1e-13
    # close to the source it is the bare Coulomb potential plus a smooth part
    c = b + np.array([0.0, 0.0, -0.02])
    assert abs(pins.grounded_slab_green(c, b, 1.0, 1.0, 0.5, mmax=120) * 0.02 - 1.0) < 0.1


def test_two_particle_energy_and_non_neutral_input():
    """U = 1/2 sum q phi of two charges = q1 q2 G(1,2) + self-image terms; the cross term is pinned by the Green
    function through the difference of three energies.  Grounded plates do not need a neutral system."""
    x1, x2 = [0.3, 0.6, 0.15], [0.7, 0.2, 0.38]
    p = 20
    U12 = O.hsma(slab(p, [x1, x2], [1.0, 2.0])).U
    U1 = O.hsma(slab(p, [x1], [1.0])).U
    U2 = O.hsma(slab(p, [x2], [2.0])).U
    g = pins.grounded_slab_green(np.array(x1), np.array(x2), 1.0, 1.0, 0.5)
    assert abs((U12 - U1 - U2) - 2.0 * g) < 2e-8
    assert U1 < 0 and U2 < 0            # a charge is attracted by its own induced charge


def test_rejections():
    with pytest.raises(ValueError):
        O.hsma(slab(8, [[0.5, 0.5, 0.2]], [1.0]).with_(gamma=0.5))
