"""Pins of the face-pair closure of the periodic kind (reading S15):
BASELINE.json's "check-point pairs on opposite faces", with value AND normal-derivative rows.  `-m "not gpu"`."""
import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins
from tests.conftest import golden

MADELUNG = -golden("madelung_nacl.txt")[0][0]


@pytest.fixture(scope="module")
def case():
    w = W.config(2, N=120)
    L = np.array(w.L)
    phi_e = pins.ewald_potentials(w.xyz, w.q, L, alpha=8.0, rcut_cells=1, kmax=12)
    return w, phi_e, 0.5 * float(w.q @ phi_e)


def test_value_rows_alone_are_rank_deficient_and_derivative_rows_complete_them(case):
    """Reading S15, now a test: harmonics even in x, y and z are invisible to value matching across opposite faces."""
    w, _, _ = case
    L = np.array(w.L)
    R0 = 0.5 * np.linalg.norm(L)
    p, K = 10, 500
    x = W.seeded_face_points(K, w.L, W.LOWER_FACES, seed=3)
    ax = np.argmax(np.isclose(x, -0.5 * L), axis=1)
    xt = x.copy()
    xt[np.arange(K), ax] += L[ax]
    Fv = (O.real_solid_harmonics(x, p, R0) - O.real_solid_harmonics(xt, p, R0))[:, 1:]
    sv = np.linalg.svd(Fv, compute_uv=False)
    assert int((sv > 1e-10 * sv[0]).sum()) == 85                       # of 99 unknowns (85/99)
    r = O.hsma(w.with_(p=p, K=K, M=6000, closure=W.CLOSURE_FACE_PAIRS, check_xyz=x))
    assert r.rhs.shape[0] == 2 * K and r.cond < 200


def test_face_pair_closure_converges_to_ewald(case):
    w, phi_e, U_e = case
    errs = []
    for p, K in ((10, 500), (16, 800), (22, 1500)):
        chk = W.seeded_face_points(K, w.L, W.LOWER_FACES, seed=3)
        r = O.hsma(w.with_(p=p, K=K, M=2 * 988 * 2 if p > 16 else 6000, closure=W.CLOSURE_FACE_PAIRS, check_xyz=chk))
        assert r.A[0] == 0.0
        errs.append(abs(r.U - U_e) / abs(U_e))
        d = r.phi - phi_e
        assert np.abs(d - d.mean()).max() < 100 * max(errs[-1], 1e-11) * np.abs(phi_e).max()
    assert errs[0] < 2e-6 and errs[1] < 2e-8 and errs[2] < 2e-9 and errs[2] < errs[1] < errs[0]
    # the library's own lattice on the lower faces works too
    r = O.hsma(w.with_(p=10, K=500, M=6000, closure=W.CLOSURE_FACE_PAIRS))
    assert abs(r.U - U_e) / abs(U_e) < 2e-5


def test_config1_as_literally_written_reaches_the_madelung_constant():
    """BASELINE.json config 1: "200 random check-point pairs on opposite faces (seed 0)", p = 8, M = 400 -- with the
    derivative rows this reading is well posed (shell 2 and R = sqrt3 L as in reading S7)."""
    w = W.config(1)
    chk = W.seeded_face_points(200, w.L, W.LOWER_FACES, seed=0)
    r = O.hsma(w.with_(closure=W.CLOSURE_FACE_PAIRS, check_xyz=chk))
    assert abs(O.madelung_constant(r.U, w.N, 1.0) - MADELUNG) < 5e-7
    r = O.hsma(w.with_(closure=W.CLOSURE_FACE_PAIRS, check_xyz=chk, p=16, M=2 * 988, quad_rule=W.QUAD_LATTICE,
                       K=600).with_(check_xyz=W.seeded_face_points(600, w.L, W.LOWER_FACES, seed=0)))
    assert abs(O.madelung_constant(r.U, w.N, 1.0) - MADELUNG) < 1e-8


def test_rejections():
    w = W.config(2, N=20)
    bad = W.seeded_face_points(50, w.L, W.ALL_FACES, seed=1)       # some points on upper faces / none on lower
    bad[:, :] = 0.1
    with pytest.raises(ValueError):
        O.hsma(w.with_(closure=W.CLOSURE_FACE_PAIRS, K=50, check_xyz=bad))
