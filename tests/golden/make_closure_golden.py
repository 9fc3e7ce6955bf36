"""Writes tests/golden/closure_results.txt: results of oracle.hsma() for one small workload per closure / near mode /
dipole mode, as hexadecimal floats (bit-exact).  Written ONCE with the single-function hsma() of round 1, before that
function was split into one routine per closure (round 2): tests/test_oracle_closures.py asserts that
the split oracle reproduces every stored number bit for bit.  Calls only oracle/ and the seeded input generator.
Run from the repo root:  python tests/golden/make_closure_golden.py"""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import hsma_workloads as W  # noqa: E402
from oracle import hsma_oracle as O  # noqa: E402


def cases():
    """name -> (workload, hsma keyword arguments)"""
    rng = np.random.default_rng(2718)
    out = {}
    out["periodic_circumsphere_cfg1"] = (W.config(1), {})
    out["periodic_circumsphere_cfg2"] = (W.config(2, N=150), {})
    out["cavity_dirichlet_cfg3"] = (W.config(3, N=140), {})
    out["far_data_cfg4"] = (W.config(4, N=120), {})
    out["paper_example2"] = (W.paper_example2(), {})
    w2 = W.config(2, N=120)
    out["face_pairs_seeded"] = (w2.with_(p=8, K=300, M=1500, closure=W.CLOSURE_FACE_PAIRS,
                                         check_xyz=W.seeded_face_points(300, w2.L, W.LOWER_FACES, seed=3)), {})
    out["face_pairs_default_points"] = (w2.with_(p=8, K=300, M=1500, closure=W.CLOSURE_FACE_PAIRS), {})
    L = (1.0, 1.0, 0.5)
    xyz = rng.random((90, 3)) * np.asarray(L)
    out["slab_grounded"] = (W.Workload("slab_grounded", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), -1.0, 1.1, 9, 1500, 300,
                                       xyz, rng.standard_normal(90)), {})
    out["slab_neumann"] = (W.Workload("slab_neumann", W.BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), 1.0, 1.1, 9, 1500, 300,
                                      xyz, W.alternating_charges(90)), {})
    Lc = (1.0, 1.0, 1.0)
    xc = 0.05 + 0.9 * rng.random((80, 3))
    out["cavity_neumann"] = (W.Workload("cavity_neumann", W.BC_MIRROR_CAVITY, Lc, (1, 1, 1), 1.0, 1.5 * math.sqrt(3) / 2, 8,
                                        1500, 400, xc, W.alternating_charges(80)), {})
    out["cavity_dirichlet_default_points"] = (W.Workload("cavity_default", W.BC_MIRROR_CAVITY, Lc, (1, 1, 1), -1.0,
                                                         1.5 * math.sqrt(3) / 2, 8, 1500, 400, xc, rng.standard_normal(80)), {})
    out["sphere_culled_paper_timing"] = (W.paper_timing(64).with_(p=9, K=200), {})
    out["fd3_dipole"] = (W.config(2, N=100).with_(dipole_mode=W.DIPOLE_FD3), {})
    out["forces_and_slice"] = (W.config(2, N=130), {"forces": True, "targets_slice": slice(17, 101)})
    out["forces_cavity"] = (W.config(3, N=100), {"forces": True})
    out["forces_face_pairs"] = (w2.with_(p=8, K=200, M=1500, closure=W.CLOSURE_FACE_PAIRS), {"forces": True})
    return out


def digest(r):
    """The numbers that are stored: every scalar, and sums / extreme entries of every array."""
    vals = {"U": r.U, "fit_rms": r.fit_rms, "cond": r.cond}
    for name in ("phi", "A", "rhs", "phi_near", "phi_out", "phi_check", "Q", "D"):
        a = np.asarray(getattr(r, name), dtype=np.float64).ravel()
        vals[name + "_sum"] = float(a.sum())
        vals[name + "_first"] = float(a[0])
        vals[name + "_last"] = float(a[-1])
        vals[name + "_absmax"] = float(np.abs(a).max())
    if r.F is not None:
        vals["F_sum"] = float(np.asarray(r.F).sum())
        vals["F_absmax"] = float(np.abs(r.F).max())
    vals["rows"] = float(r.rhs.shape[0])
    vals["check_targets"] = float(r.check_targets.shape[0])
    return vals


def main():
    out = os.path.join(ROOT, "tests", "golden", "closure_results.txt")
    with open(out, "w") as f:
        f.write("# oracle.hsma() per closure, hexadecimal floats; written by tests/golden/make_closure_golden.py with the\n")
        f.write("# single-function hsma() of round 1 (before the per-closure split); format: case key value\n")
        for name, (w, kw) in cases().items():
            for k, v in digest(O.hsma(w, **kw)).items():
                f.write(f"{name} {k} {float(v).hex()}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
