"""End-to-end pins of the oracle's HSMA (fit + mapping + sums) against exact answers:
the Madelung constant printed in the paper, a textbook Ewald sum, the grounded-box Green
function, and brute force over the finite image block of config 4.  All `-m "not gpu"`."""
import math

import numpy as np
import pytest

import hsma_workloads as W
from oracle import hsma_oracle as O
from tests import pins
from tests.conftest import golden

MADELUNG = -golden("madelung_nacl.txt")[0][0]


# ------------------------------------------------------------------ periodic: Madelung
def test_madelung_config1_as_configured():
    """BASELINE.json config 1 (p=8, M=400, K=200; shell 2, reading S7): ~8 digits."""
    w = W.config(1)
    r = O.hsma(w)
    M = O.madelung_constant(r.U, w.N, w.meta["a_nn"])
    assert abs(M - MADELUNG) < 5e-8
    assert abs(M - 1.7475645946) < 5e-8            # the value BASELINE.json quotes


def test_madelung_converges_to_printed_value():
    """the error falls with p and reaches ~1e-12 at p=24, M=5928 (F2=987)."""
    errs = {}
    for p in (8, 16, 24):
        w = W.config(1).with_(p=p, M=2 * 988, quad_rule=W.QUAD_LATTICE, K=2 * p * p)
        r = O.hsma(w)
        errs[p] = abs(O.madelung_constant(r.U, w.N, 1.0) - MADELUNG)
    assert errs[24] < 5e-12 and errs[16] < 1e-8 and errs[8] < 1e-7
    assert errs[24] < errs[16] < errs[8]


def test_madelung_translation_invariance():
    """Shifting the lattice by (1/2,1/2,1/2) (no ion on a face any more) gives the same constant."""
    xyz, q, L = W.rock_salt(1, shift=(0.5, 0.5, 0.5))
    w = W.config(1).with_(xyz=xyz, q=q, p=16, M=2 * 988, quad_rule=W.QUAD_LATTICE, K=512)
    r = O.hsma(w)
    assert abs(O.madelung_constant(r.U, w.N, 1.0) - MADELUNG) < 1e-8
    # every ion sees the same |phi| in a perfect crystal (up to the gauge constant, S2)
    per_ion = -q * r.phi
    assert per_ion.max() - per_ion.min() < 1e-3
    assert abs(per_ion.mean() - MADELUNG) < 1e-8


def test_madelung_64_ion_cell_of_the_paper():
    """PAPER.md:165 uses 64 ions at spacing 1/2 in the L=2 box; same constant (a_nn = 1/2)."""
    xyz, q, L = W.rock_salt(2)
    w = W.config(1).with_(xyz=xyz * 0.5, q=q, p=16, M=2 * 988, quad_rule=W.QUAD_LATTICE, K=512)
    r = O.hsma(w)
    assert abs(O.madelung_constant(r.U, w.N, 0.5) - MADELUNG) < 2e-8


# ------------------------------------------------------------------ periodic: Ewald
@pytest.fixture(scope="module")
def ewald_case():
    w = W.config(2, N=120)
    L = np.array(w.L)
    e1 = pins.ewald_potentials(w.xyz, w.q, L, alpha=6.0, rcut_cells=1, kmax=9)
    e2 = pins.ewald_potentials(w.xyz, w.q, L, alpha=8.0, rcut_cells=1, kmax=12)
    assert np.abs(e1 - e2).max() < 1e-11 * np.abs(e1).max()      # the pin agrees with itself
    return w, e2


def test_periodic_hsma_matches_ewald(ewald_case):
    """HSMA -> Ewald.  A system with a large cell dipole: the periodic residual
    picks the tin-foil solution (reading S3).  phi differs by the gauge constant only (S2)."""
    w, phi_e = ewald_case
    U_e = 0.5 * float(w.q @ phi_e)
    errs = []
    for p, M in ((10, 2000), (16, 6000), (22, 2 * 988 * 2)):
        r = O.hsma(w.with_(p=p, M=M, K=max(w.K, 2 * p * p)))
        errs.append(abs(r.U - U_e) / abs(U_e))
        d = r.phi - phi_e
        spread = (d - d.mean())
        assert np.abs(spread).max() < 50 * max(errs[-1], 1e-12) * np.abs(phi_e).max() + 1e-9
    assert errs[0] < 5e-4 and errs[1] < 2e-6 and errs[2] < 2e-8
    assert errs[2] < errs[1] < errs[0]


def test_shell2_is_more_accurate_than_shell1(ewald_case):
    """Reading S7: with whole cells the truncation error is set by the shell."""
    w, phi_e = ewald_case
    U_e = 0.5 * float(w.q @ phi_e)
    r1 = O.hsma(w.with_(p=14, M=6000, K=600))
    r2 = O.hsma(w.with_(p=14, M=6000, K=600, near_shell=(2, 2, 2), R_aux=2.4))
    assert abs(r2.U - U_e) < 0.05 * abs(r1.U - U_e)


# ------------------------------------------------------------------ grounded cavity: Jackson
def test_grounded_cube_matches_green_function():
    """One unit charge at A in the grounded cube; total potential at B (different height) =
    near images + harmonic series, against the Green-function series.  Pins the mirror cell table
    (sign (-1)^(i+j+k)), the Dirichlet rows, the fit and the basis, end to end."""
    L = (1.0, 1.0, 1.0)
    A = np.array([[0.32, 0.58, 0.27]])
    chk = W.seeded_face_points(1500, L, W.ALL_FACES, seed=7)
    w = W.Workload("green", W.BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0, 1.5 * math.sqrt(3) / 2, 24, 6000,
                   1500, A, np.array([1.0]), check_xyz=chk)
    r = O.hsma(w)
    cells = O.cell_table(O.BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0)
    Bs = np.array([[0.61, 0.41, 0.72], [0.2, 0.8, 0.9], [0.5, 0.5, 0.6]])
    tot = O.near_sum(Bs - 0.5, A - 0.5, w.q, cells) + O.series_at(Bs - 0.5, r.A, w.p, 0.5 * math.sqrt(3))
    for b in range(len(Bs)):
        g = pins.grounded_box_green(Bs[b], A[0], L, nmax=70)
        assert abs(tot[b] - g) < 2e-9 * max(1.0, abs(g))
    # maximum principle: the total potential on held-out wall points bounds the interior error
    held = W.seeded_face_points(300, L, W.ALL_FACES, seed=8)
    wall = O.near_sum(held, A - 0.5, w.q, cells) + O.series_at(held, r.A, w.p, 0.5 * math.sqrt(3))
    assert np.abs(wall).max() < 1e-6


def test_paper_example2_energy_converges():
    """PAPER.md:167 geometry (tests/golden/paper_example2.txt).  No value is printed in the
    paper; the pin is self-convergence in p plus the Green-function cross term."""
    rows = golden("paper_example2.txt")
    w = W.paper_example2()
    assert rows[0][0] == w.L[0]
    np.testing.assert_allclose(np.array([r[1:] for r in rows[1:]]) + 1.0, w.xyz)
    np.testing.assert_allclose([r[0] for r in rows[1:]], w.q)
    U = {p: O.hsma(w.with_(p=p, M=8000)).U for p in (8, 16, 24)}
    assert abs(U[24] - U[16]) < 1e-7 and abs(U[16] - U[8]) < 1e-4
    assert abs(U[16] - U[8]) > abs(U[24] - U[16])
    # induced potential at charge 0 due to charge 1 alone, against the Green function
    one = w.with_(xyz=w.xyz[1:2], q=w.q[1:2], p=24, M=8000)
    r = O.hsma(one)
    cells = O.cell_table(O.BC_MIRROR_CAVITY, w.L, (1, 1, 1), -1.0)
    B = w.xyz[0:1] - 1.0
    tot = O.near_sum(B, one.xyz - 1.0, one.q, cells) + O.series_at(B, r.A, 24, math.sqrt(3.0))
    g = one.q[0] * pins.grounded_box_green(w.xyz[0], w.xyz[1], w.L, nmax=70)
    assert abs(tot[0] - g) < 1e-9


# ------------------------------------------------------------------ config 4 finite model
def test_slab_far_data_closure_matches_block_brute_force():
    """Reading S16: config 4 computes the finite 7x7x9 image block (weights 0.5^|kz|); HSMA
    compresses the 396 far cells.  Exact brute force over the whole block is the pin."""
    w = W.config(4, N=24).with_(p=20, M=8000)
    r = O.hsma(w)
    src = w.xyz - 0.5 * np.array(w.L)
    want = pins.brute_image_sum(src, src, w.q, w.L, (False, False, True), w.far_shell, w.gamma,
                                skip_self=True)
    assert np.abs(r.phi - want).max() < 1e-10 * np.abs(want).max()
    r14 = O.hsma(w.with_(p=14))
    assert np.abs(r14.phi - want).max() < 1e-6 * np.abs(want).max()


# ------------------------------------------------------------------ convergence + invariants
def test_fit_residual_decays_exponentially_in_p():
    """Eq.(8): spectral convergence.  Whole-cell shell 1: ratio per degree
    about R0/(1.5 L) = 0.577; allow a band around it."""
    w = W.config(2, N=200)
    ps = (6, 10, 14, 18)
    rms = [O.hsma(w.with_(p=p, M=4000, K=1200)).fit_rms for p in ps]
    for a, b in zip(rms[:-1], rms[1:]):
        rate = (b / a) ** (1.0 / 4.0)
        assert 0.35 < rate < 0.75
    assert rms[-1] < 1e-2 * rms[0]


def test_invariants():
    w = W.config(2, N=150)
    r = O.hsma(w)
    # permutation of the particles permutes phi
    perm = np.random.default_rng(0).permutation(w.N)
    rp = O.hsma(w.with_(xyz=w.xyz[perm], q=w.q[perm]))
    np.testing.assert_allclose(rp.phi, r.phi[perm], rtol=0, atol=1e-11 * np.abs(r.phi).max())
    # linear in the charges
    r2 = O.hsma(w.with_(q=2.5 * w.q))
    np.testing.assert_allclose(r2.phi, 2.5 * r.phi, rtol=1e-12, atol=1e-12)
    assert abs(r2.U - 6.25 * r.U) < 1e-11 * abs(r.U)
    # periodic gauge (S2): A00 = 0; energy unaffected by adding a constant to phi (neutral)
    assert r.A[0] == 0.0
    assert abs(O.energy(w.q, r.phi + 3.0) - r.U) < 1e-10 * abs(r.U)
    # translation of all particles (re-wrapped): U unchanged to truncation accuracy
    sh = np.mod(w.xyz + np.array([0.31, 0.12, 0.77]), 1.0)
    rs = O.hsma(w.with_(xyz=sh))
    assert abs(rs.U - r.U) < 2e-3 * abs(r.U)
    rs16 = O.hsma(w.with_(xyz=sh, p=16, M=6000, K=600))
    r16 = O.hsma(w.with_(p=16, M=6000, K=600))
    assert abs(rs16.U - r16.U) < 0.05 * abs(rs.U - r.U) + 1e-7 * abs(r.U)
    # a slice of targets gives the same potentials
    rsl = O.hsma(w, targets_slice=slice(40, 90))
    np.testing.assert_array_equal(rsl.phi, r.phi[40:90])


def test_rejections():
    w = W.config(2, N=50)
    with pytest.raises(ValueError):
        O.hsma(w.with_(q=np.ones(50)))                      # not neutral (S17)
    with pytest.raises(ValueError):
        O.hsma(w.with_(R_aux=1.6))                          # sphere pokes out of the 3^3 block (S7)
    with pytest.raises(ValueError):
        O.hsma(w.with_(R_aux=0.8))                          # inside the circumsphere


def test_stored_config5_values_are_the_oracles():
    """tests/golden/config5_oracle.txt (used by the GPU parity test at full size) is what the oracle computes:
    two of its stored potentials are recomputed here (the fit needs the full step (a): 2.8e10 pairs), and the stored
    indices follow the rule stated in its header (a sample that reaches every thread position of the CUDA kernels)."""
    import importlib.util
    import os
    spec = importlib.util.spec_from_file_location(
        "make_config5_golden", os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "make_config5_golden.py"))
    gen = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(gen)
    rows = golden("config5_oracle.txt")
    w = W.config(5)
    idx = np.array([int(a) for a, _ in rows[1:]])
    assert np.array_equal(idx, gen.sample_indices(w.N))
    assert set(idx % 256) == set(range(256)) and set(idx // 2048) == set(range(w.N // 2048))
    r = O.hsma(w, targets_slice=slice(0, 252))
    stored = {int(a): b for a, b in rows[1:]}
    assert abs(r.phi[0] - stored[0]) <= 1e-13 * rows[0][1]
    assert abs(r.phi[251] - stored[251]) <= 1e-13 * rows[0][1]
    assert abs(r.fit_rms - rows[0][2]) <= 1e-9 * rows[0][2]


def test_non_cubic_periodic_box_matches_ewald():
    """A box with three different sides (the paper's tests are cubic): both closures of the periodic kind."""
    L = (1.0, 1.2, 0.9)
    rng = np.random.default_rng(12)
    N = 100
    xyz = rng.random((N, 3)) * np.array(L)
    q = W.alternating_charges(N)
    U_e = 0.5 * float(q @ pins.ewald_potentials(xyz, q, np.array(L), alpha=7.0, rcut_cells=1, kmax=12))
    w = W.Workload("box", W.BC_PERIODIC, L, (1, 1, 1), 1.0, 1.3, 16, 6000, 900, xyz, q)
    assert abs(O.hsma(w).U - U_e) < 2e-6 * abs(U_e)
    assert abs(O.hsma(w.with_(closure=W.CLOSURE_FACE_PAIRS)).U - U_e) < 4e-6 * abs(U_e)
    assert abs(O.hsma(w.with_(p=10, K=500)).U - U_e) < 2e-3 * abs(U_e)
