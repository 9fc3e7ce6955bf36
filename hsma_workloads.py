"""Seeded synthetic workloads shared by the CPU oracle (tests) and the CUDA path.

This module holds NO arithmetic of the method (no image cells, harmonics, fits,
nodes or sums): only the particle coordinates/charges of BASELINE.json's five
configs, the plain parameters that describe each config, and the seeded random
face check points that are *inputs* to both implementations.  Both `oracle/`
and `paper_1806_04801_b200/` receive exactly these arrays; neither imports the
other.

Recipes; the paper's own workloads
are synthetic lattices / random-sign systems:
  cfg1  8 ions at {0,1}^3, q=(-1)^(x+y+z), L=2           (stands in for PAPER.md:165)
  cfg2  default_rng(1).random((1000,3)),   q=+1 even/-1 odd (stands in for PAPER.md:171)
  cfg3  0.05+0.9*default_rng(2).random((4000,3)), same charge rule (scaled-up PAPER.md:167)
  cfg4  default_rng(3).random((16384,3))*(1,1,0.5), same charge rule
  cfg5  default_rng(4).random((262144,3)), same charge rule   (stands in for PAPER.md:171)
Coordinates are box coordinates in [0, L_a]; the implementations centre them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

# boundary kinds (values match include/hsma.h)
BC_PERIODIC = 0
BC_MIRROR_CAVITY = 1
BC_SLAB_XY_PERIODIC_Z_MIRROR = 2

# closures (values match include/hsma.h)
CLOSURE_BOUNDARY = 0   # residual of the boundary condition at the check points
CLOSURE_FAR_DATA = 1   # explicit far-cell data at the check points (reading S16)
CLOSURE_FACE_PAIRS = 2 # periodic: value + normal-derivative pairs on opposite faces (reading S15)
LOWER_FACES = [(0, -1), (1, -1), (2, -1)]   # the faces x_a = -L_a/2 (their partners are on the opposite faces)

# quadrature rules (values match include/hsma.h)
QUAD_SPIRAL = 0        # exactly M nodes (reading S10)
QUAD_LATTICE = 1       # the paper's F1/F2 lattice, M = 2(F2+1)

# near set (values match include/hsma.h)
NEAR_WHOLE_CELLS = 0   # every image of the neighbour cells (reading S7, north_star)
NEAR_SPHERE = 1        # paper-literal: only the images inside the auxiliary sphere

# dipole layer (values match include/hsma.h)
DIPOLE_EXACT = 0       # exact normal dipole on M nodes (reading S9)
DIPOLE_FD3 = 1         # paper-literal: central difference over three spheres, 3M charges (Eq.12-14)


@dataclass
class Workload:
    name: str
    kind: int
    L: tuple            # (Lx, Ly, Lz)
    near_shell: tuple   # (sx, sy, sz)
    gamma: float        # reflection factor on mirror axes (unused for periodic axes)
    R_aux: float
    p: int
    M: int
    K: int              # check points (periodic: K points + K wrapped partners)
    xyz: np.ndarray     # [N,3] box coordinates in [0, L_a]
    q: np.ndarray       # [N]
    check_xyz: Optional[np.ndarray] = None  # [K,3] CENTRED coords; None -> implementation's rule
    far_shell: tuple = (0, 0, 0)
    closure: int = CLOSURE_BOUNDARY
    quad_rule: int = QUAD_SPIRAL
    near_mode: int = NEAR_WHOLE_CELLS
    dipole_mode: int = DIPOLE_EXACT
    fd_dr_rel: float = 1e-5   # Delta r / R_s of the three-sphere form
    meta: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.xyz.shape[0])

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


def alternating_charges(n: int) -> np.ndarray:
    """q_i = +1 for even i, -1 for odd i (neutral for even n)."""
    q = np.ones(n, dtype=np.float64)
    q[1::2] = -1.0
    return q


def seeded_face_points(K: int, L, faces, seed: int) -> np.ndarray:
    """K points drawn uniformly on the listed box faces, a face chosen with
    probability proportional to its area.  `faces` is a list of (axis, side)
    with side in {-1,+1}.  Returned in CENTRED coordinates (box = prod [-L_a/2, L_a/2]).
    These are inputs handed identically to the oracle and to the library."""
    L = np.asarray(L, dtype=np.float64)
    rng = np.random.default_rng(seed)
    areas = np.array([np.prod(np.delete(L, ax)) for ax, _ in faces])
    which = rng.choice(len(faces), size=K, p=areas / areas.sum())
    uvw = rng.random((K, 3))
    pts = (uvw - 0.5) * L
    for i in range(K):
        ax, side = faces[which[i]]
        pts[i, ax] = 0.5 * side * L[ax]
    return pts


ALL_FACES = [(0, -1), (0, 1), (1, -1), (1, 1), (2, -1), (2, 1)]


def rock_salt(cells_per_axis: int = 1, shift=(0.0, 0.0, 0.0)):
    """Rock-salt ions at integer coordinates {0..2c-1}^3 with q=(-1)^(x+y+z), box side 2c.
    `shift` translates all ions (wrapped back into the box)."""
    n = 2 * cells_per_axis
    g = np.arange(n)
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    xyz = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1).astype(np.float64)
    q = np.where((X + Y + Z).ravel() % 2 == 0, 1.0, -1.0)
    xyz = np.mod(xyz + np.asarray(shift, dtype=np.float64), float(n))
    return xyz, q, float(n)


def config(idx: int, N: Optional[int] = None, **overrides) -> Workload:
    """BASELINE.json configs[idx-1].  `N` overrides the particle count (same generator,
    same seed) for reduced-size parity cases.  Readings of unspecified values follow
    SURVEY.md 8(c) (S6, S7, S8, S15, S16) and are listed in DESIGN.md."""
    s3 = math.sqrt(3.0)
    if idx == 1:
        xyz, q, L = rock_salt(1)
        w = Workload("cfg1_madelung", BC_PERIODIC, (L, L, L), (2, 2, 2), 1.0, s3 * L, 8, 400, 200,
                     xyz, q, meta={"a_nn": 1.0})
    elif idx == 2:
        n = N or 1000
        xyz = np.random.default_rng(1).random((n, 3))
        w = Workload("cfg2_random_periodic", BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0,
                     1.5 * s3 / 2.0, 10, 2000, 500, xyz, alternating_charges(n))
    elif idx == 3:
        n = N or 4000
        xyz = 0.05 + 0.9 * np.random.default_rng(2).random((n, 3))
        L = (1.0, 1.0, 1.0)
        chk = seeded_face_points(1000, L, ALL_FACES, seed=1003)
        w = Workload("cfg3_metallic_cavity", BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0,
                     1.5 * s3 / 2.0, 12, 4000, 1000, xyz, alternating_charges(n), check_xyz=chk)
    elif idx == 4:
        n = N or 16384
        L = (1.0, 1.0, 0.5)
        xyz = np.random.default_rng(3).random((n, 3)) * np.asarray(L)
        chk = seeded_face_points(1500, L, ALL_FACES, seed=1004)
        w = Workload("cfg4_slab", BC_SLAB_XY_PERIODIC_Z_MIRROR, L, (1, 1, 2), 0.5, 1.1, 14, 8000, 1500,
                     xyz, alternating_charges(n), check_xyz=chk, far_shell=(3, 3, 4),
                     closure=CLOSURE_FAR_DATA)
    elif idx == 5:
        n = N or 262144
        xyz = np.random.default_rng(4).random((n, 3))
        w = Workload("cfg5_large_periodic", BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0,
                     1.5 * s3 / 2.0, 16, 20000, 2000, xyz, alternating_charges(n))
    else:
        raise ValueError(f"no config {idx}")
    if N is not None:
        w.name += f"_N{N}"
    return w.with_(**overrides) if overrides else w


def paper_timing(N: int, seed: int = 5, alpha: float = 1.3, P: int = 25, F2: int = 987) -> Workload:
    """The paper's timing workload: N unit charges of random sign on the sites of a uniformly
    spaced lattice in the unit cube (neutral), PBC, alpha = 1.3, P = 25 (p = 26 degrees), N_o = 3 x 2(F2+1) = 5928
    images on three spheres, N_m = 2 P^2 monitoring points, near set = the images inside the sphere.
    N must be a perfect cube with an even number of sites."""
    n = round(N ** (1.0 / 3.0))
    if n ** 3 != N or N % 2:
        raise ValueError("N must be an even perfect cube")
    g = (np.arange(n) + 0.5) / n
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    xyz = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    q = np.ones(N)
    q[np.random.default_rng(seed).permutation(N)[: N // 2]] = -1.0
    return Workload(f"paper_timing_N{N}", BC_PERIODIC, (1.0, 1.0, 1.0), (1, 1, 1), 1.0, alpha * math.sqrt(3.0) / 2.0,
                    P + 1, 2 * (F2 + 1), 2 * P * P, xyz, q, quad_rule=QUAD_LATTICE, near_mode=NEAR_SPHERE,
                    dipole_mode=DIPOLE_FD3)


def paper_example2() -> Workload:
    """L=2 grounded cube (DBC), +2 at (0.1,0,0), -1 at (0.8,0.8,0.8),
    -1 at (-0.9,-0.9,-0.9) in centred Cartesian coordinates (box coords = centred + 1)."""
    c = np.array([[0.1, 0.0, 0.0], [0.8, 0.8, 0.8], [-0.9, -0.9, -0.9]])
    q = np.array([2.0, -1.0, -1.0])
    L = (2.0, 2.0, 2.0)
    return Workload("paper_example2", BC_MIRROR_CAVITY, L, (1, 1, 1), -1.0, 1.5 * math.sqrt(3.0),
                    12, 4000, 1000, c + 1.0, q,
                    check_xyz=seeded_face_points(1000, L, ALL_FACES, seed=1102))
