"""Host-side accounting of bench.py (no GPU): the unit counts its roofline figures are built from.  `-m "not gpu"`."""
import importlib.util
import os

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bench():
    spec = importlib.util.spec_from_file_location("bench_module", os.path.join(ROOT, "bench.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


@pytest.mark.parametrize("N,C", [(7937, 27), (8192, 27), (9000, 45), (20012, 27), (65536, 27), (262144, 27), (1048876, 125)])
def test_sym_evaluations_counts_the_visits_of_the_symmetric_kernel(bench, N, C):
    """block I (8 tiles of 256 packed sources) visits the tiles J >= 8 I; every visit is
    256 x 2048 x C pair evaluations.  bench.sym_evaluations is the closed form of this walk."""
    n_tiles = -(-N // 256)
    n_blocks = -(-n_tiles // 8)
    visits = sum(1 for I in range(n_blocks) for J in range(n_tiles) if J >= 8 * I)
    assert bench.sym_evaluations(N, C) == visits * 256 * 2048 * C
    # every ordered pair interaction is covered: evaluations >= N (N - 1) C / 2, and the excess is the diagonal
    # visits (done as ordered pairs) plus the padding of the last tile and block
    assert bench.sym_evaluations(N, C) >= N * (N - 1) * C // 2
    assert bench.sym_evaluations(N, C) <= (n_blocks * 2048) * (n_tiles * 256) * C // 2 + n_blocks * 8 * 256 * 2048 * C


def test_executed_instruction_tables_are_consistent(bench):
    """Per-unit figures quoted in DESIGN.md 6.1 / 6.6 / 6.12 (FP64-pipe instructions, flops with fma = 2)."""
    assert bench.EXEC_PAIR[(1, True)] == (9.0, 13.0) and bench.EXEC_PAIR[(2, False)] == (12.0, 18.0)
    assert bench.EXEC_EVAL_SYM[1] == (11.625, 17.125) and bench.EXEC_EVAL_SYM[2] == (13.625, 21.125)
    assert bench.EXEC_EVAL_SYM_FIELD[1] == (22.375, 35.25)
    assert bench.FLOPS_EVAL_SYM == bench.FLOPS_PAIR_CHARGE + 2 and bench.FLOPS_EVAL_SYM_FIELD == bench.FLOPS_PAIR_CHARGE_FIELD + 9


def test_lattice_factored_counts(bench):
    """DESIGN.md 6.14 / csrc/lattice_kernels.cuh: FP64-pipe instructions and flops per image-pair evaluation of the
    lattice-factored kernels, counted from the formulation (per image: r^2 DFMA, y0^2 DMUL, Newton DFMA, accumulate DFMA;
    per pair: offsets, x squares, x^2 + y^2, weight classes, row/column accumulation).  The SASS of the 27-cell periodic
    inner loop has 533 FP64 instructions for 108 images = 4.935 (profiles/r02c_ncu_lat_sym_N262144.md)."""
    p = (False, False, False)
    i, f = bench.lat_counts((1, 1, 1), p, 1, False, True)
    assert abs(i - (4 + (9 + 4 + 11 + 1.25) / 27)) < 1e-12 and abs(f - (7 + (9 + 4 + 22 + 1.25) / 27)) < 1e-12
    assert abs(i - 533 / 108) < 1e-3          # SASS of the inner loop, profiles/r02c_ncu_lat_sym_N262144.md
    # cubic refinement: two more DFMA per image; ordered pairs: one accumulation less per pair
    i2, f2 = bench.lat_counts((1, 1, 1), p, 2, False, True)
    assert abs(i2 - i - 2) < 1e-12 and abs(f2 - f - 4) < 1e-12
    io, fo = bench.lat_counts((1, 1, 1), p, 1, False, False)
    assert abs(i - io - 2.25 / 27) < 1e-12 and abs(f - fo - 3.25 / 27) < 1e-12
    # reflecting axes: one more offset per axis (x_i + x_j) and one DFMA per further weight class
    im, _ = bench.lat_counts((1, 1, 1), (True, True, True), 1, False, True)
    assert abs(im - i - (3 + 3) / 27) < 1e-12
    # the 45-cell slab table spreads the per-pair part over more images
    isl, _ = bench.lat_counts((1, 1, 2), (False, False, True), 1, False, True)
    assert isl < i
    # every count stays below SURVEY 8(d)'s 18 flops per pair: the factoring removes work
    assert f < bench.FLOPS_PAIR_CHARGE and bench.lat_counts((1, 1, 1), p, 1, True, True)[1] < bench.FLOPS_PAIR_CHARGE_FIELD
