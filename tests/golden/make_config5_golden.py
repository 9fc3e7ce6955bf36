"""Writes tests/golden/config5_oracle.txt: the oracle's total energy and a sample of the potentials of BASELINE.json
config 5 (N = 262,144) -- 1.9e12 pairs, minutes of CPU time, hence stored.  Calls only oracle/ and the seeded input
generator; nothing from the CUDA path.  Run from the repo root:  python tests/golden/make_config5_golden.py

Index rule of the sample (`sample_indices`, also used by the CPU test that recomputes some of the stored values):
the first 8,192 entries of numpy.random.default_rng(20250).permutation(N), plus every 251st index (251 is prime, so
i mod 256 runs through every residue), sorted, duplicates removed.  The CUDA path stores a source at a packed slot that
depends on (i mod 256, the signs of the charges before it in its tile), works on it in thread (slot mod 256) of the
block that owns tile i // 256, eight tiles per block: a sample must reach every thread position and every block, which
a stride of 256 does not (it only ever hits the first source of a tile)."""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import hsma_workloads as W  # noqa: E402
from oracle import hsma_oracle as O  # noqa: E402

N_RANDOM = 8192
STRIDE = 251
SEED = 20250


def sample_indices(N):
    perm = np.random.default_rng(SEED).permutation(N)[:N_RANDOM]
    return np.unique(np.concatenate([perm, np.arange(0, N, STRIDE)]))


def main():
    w = W.config(5)
    t = time.time()
    r = O.hsma(w)
    dt = time.time() - t
    idx = sample_indices(w.N)
    out = os.path.join(ROOT, "tests", "golden", "config5_oracle.txt")
    with open(out, "w") as f:
        f.write("# oracle/hsma_oracle.py hsma(hsma_workloads.config(5)): BASELINE.json config 5, N = 262144, periodic,\n")
        f.write("# 27 cells, p = 16, M = 20000, K = 2000 circumsphere pairs (PAPER.md:62-82, 99-105, 142; DESIGN.md readings)\n")
        f.write(f"# written by tests/golden/make_config5_golden.py in {dt:.0f} s on {O.num_threads()} threads\n")
        f.write(f"# index rule: first {N_RANDOM} of default_rng({SEED}).permutation(N) + every {STRIDE}th index, sorted, unique\n")
        f.write(f"# ({idx.shape[0]} potentials; every residue mod 256 and every block of 2048 sources is sampled)\n")
        f.write("# line 1: U  max|phi|  fit_rms ; then: index phi_index\n")
        f.write(f"{r.U!r} {float(np.max(np.abs(r.phi)))!r} {r.fit_rms!r}\n")
        for i in idx:
            f.write(f"{int(i)} {float(r.phi[i])!r}\n")
    print("wrote", out, "U =", r.U, "in", round(dt), "s")


if __name__ == "__main__":
    main()
