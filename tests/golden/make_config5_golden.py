"""Writes tests/golden/config5_oracle.txt: the oracle's total energy and every 256th potential of BASELINE.json
config 5 (N = 262,144) -- 1.9e12 pairs, minutes of CPU time, hence stored.  Calls only oracle/ and the seeded input
generator; nothing from the CUDA path.  Run from the repo root:  python tests/golden/make_config5_golden.py"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import hsma_workloads as W  # noqa: E402
from oracle import hsma_oracle as O  # noqa: E402

STRIDE = 256


def main():
    w = W.config(5)
    t = time.time()
    r = O.hsma(w)
    dt = time.time() - t
    out = os.path.join(ROOT, "tests", "golden", "config5_oracle.txt")
    with open(out, "w") as f:
        f.write("# oracle/hsma_oracle.py hsma(hsma_workloads.config(5)): BASELINE.json config 5, N = 262144, periodic,\n")
        f.write("# 27 cells, p = 16, M = 20000, K = 2000 circumsphere pairs (PAPER.md:62-82, 99-105, 142; DESIGN.md readings)\n")
        f.write(f"# written by tests/golden/make_config5_golden.py in {dt:.0f} s on {O.num_threads()} threads\n")
        f.write("# line 1: U  max|phi|  fit_rms ; then: index phi_index for every 256th source\n")
        f.write(f"{r.U!r} {float(np.max(np.abs(r.phi)))!r} {r.fit_rms!r}\n")
        for i in range(0, w.N, STRIDE):
            f.write(f"{i} {float(r.phi[i])!r}\n")
    print("wrote", out, "U =", r.U, "in", round(dt), "s")


if __name__ == "__main__":
    main()
