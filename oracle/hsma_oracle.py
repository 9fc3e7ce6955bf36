"""ORACLE -- TEST INFRASTRUCTURE ONLY.

Plain, slow CPU implementation of the harmonic surface mapping algorithm (HSMA,
arxiv 1806.04801), written step by step from the paper (PAPER.md line numbers are cited on
every function) with the readings listed in DESIGN.md ("Readings of the paper").  fp64 numpy;
the O(N^2) pairwise sums are the plain C loops of oracle/direct_sum.c.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_1806_04801_b200/ and imports nothing from
it; the only common module is hsma_workloads.py (seeded inputs, no arithmetic of the method).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): rock-salt Madelung constant printed at
PAPER.md:165; textbook Ewald sum; Jackson's grounded-box Green function; brute force over
explicitly materialised images; quadrature/mapping identities; exponential residual decay in p;
invariants.  The true infinite dielectric slab behind config 4 has no pin: "parity unpinned"
for that physics -- the finite 441-cell model config 4 actually computes IS pinned by brute force.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess
from dataclasses import dataclass
from typing import Callable, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None

BC_PERIODIC, BC_MIRROR_CAVITY, BC_SLAB = 0, 1, 2
CLOSURE_BOUNDARY, CLOSURE_FAR_DATA, CLOSURE_FACE_PAIRS = 0, 1, 2
QUAD_SPIRAL, QUAD_LATTICE = 0, 1
NEAR_WHOLE_CELLS, NEAR_SPHERE = 0, 1
DIPOLE_EXACT, DIPOLE_FD3 = 0, 1


# --------------------------------------------------------------------------------------
# C loops (oracle/direct_sum.c)
# --------------------------------------------------------------------------------------
def build_c(force: bool = False) -> str:
    """Compile oracle/direct_sum.c -> oracle/liboracle.so (gcc -O3 -fopenmp, no fast-math)."""
    src = os.path.join(_HERE, "direct_sum.c")
    out = os.path.join(_HERE, "liboracle.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        cmd = ["gcc", "-O3", "-march=native", "-fopenmp", "-fno-fast-math", "-shared", "-fPIC",
               "-o", out, src, "-lm"]
        subprocess.check_call(cmd)
    return out


def _lib():
    global _LIB
    if _LIB is None:
        # always rebuilt for the host it runs on (-march=native objects do not travel)
        marker = os.path.join(_HERE, ".liboracle.host")
        host = open("/proc/cpuinfo").read().split("model name")[1].split("\n")[0] if os.path.exists("/proc/cpuinfo") else ""
        stale = not os.path.exists(marker) or open(marker).read() != host
        path = build_c(force=stale)
        with open(marker, "w") as f:
            f.write(host)
        lib = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_near_sum.argtypes = [dp, ctypes.c_long, dp, dp, ctypes.c_long, dp, dp, dp,
                                        ctypes.c_long, ctypes.c_long, ctypes.c_long, dp]
        lib.oracle_near_sum.restype = None
        lib.oracle_node_sum.argtypes = [dp, ctypes.c_long, dp, dp, dp, dp, ctypes.c_long, dp]
        lib.oracle_node_sum.restype = None
        lib.oracle_near_grad.argtypes = lib.oracle_near_sum.argtypes
        lib.oracle_near_grad.restype = None
        lib.oracle_node_grad.argtypes = lib.oracle_node_sum.argtypes
        lib.oracle_node_grad.restype = None
        lib.oracle_energy.argtypes = [dp, dp, ctypes.c_long]
        lib.oracle_energy.restype = ctypes.c_double
        lib.oracle_num_threads.restype = ctypes.c_int
        _LIB = lib
    return _LIB


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _c(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.float64)


def num_threads() -> int:
    return int(_lib().oracle_num_threads())


@dataclass
class CellTable:
    k: np.ndarray       # [C,3] integer cell indices
    shift: np.ndarray   # [C,3] k o L
    sign: np.ndarray    # [C,3] per-axis sign of the source coordinates
    w: np.ndarray       # [C]   weight
    central: int        # index of k = 0 (or -1 if absent)


def cell_table(kind: int, L, shell, gamma: float, exclude_shell=None) -> CellTable:
    """Near (or far) image cells.  PAPER.md:40-50.
    Periodic axis (Eq.3): image = r_j + k L, weight 1.
    Reflecting axis (Eq.4): image = (-1)^k r_j + k L, weight gamma^|k| with |k| summed over the
    reflecting axes only (reading G11).  Whole cells |k_a| <= shell_a (reading S7).
    `exclude_shell`: drop the cells with all |k_a| <= exclude_shell_a (the far table of S16)."""
    L = np.asarray(L, dtype=np.float64)
    if kind == BC_PERIODIC:
        reflecting = (False, False, False)
    elif kind == BC_MIRROR_CAVITY:
        reflecting = (True, True, True)
    elif kind == BC_SLAB:
        reflecting = (False, False, True)
    else:
        raise ValueError("unknown boundary kind")
    ks, shifts, signs, ws = [], [], [], []
    for kx in range(-shell[0], shell[0] + 1):
        for ky in range(-shell[1], shell[1] + 1):
            for kz in range(-shell[2], shell[2] + 1):
                k = (kx, ky, kz)
                if exclude_shell is not None and all(abs(k[a]) <= exclude_shell[a] for a in range(3)):
                    continue
                sgn = [(-1.0) ** abs(k[a]) if reflecting[a] else 1.0 for a in range(3)]
                order = sum(abs(k[a]) for a in range(3) if reflecting[a])
                ks.append(k)
                shifts.append([k[a] * L[a] for a in range(3)])
                signs.append(sgn)
                ws.append(float(gamma) ** order if order > 0 else 1.0)
    ks = np.array(ks, dtype=np.int64).reshape(-1, 3)
    central = -1
    for c in range(len(ks)):
        if not ks[c].any():
            central = c
    return CellTable(ks, _c(np.array(shifts).reshape(-1, 3)), _c(np.array(signs).reshape(-1, 3)),
                     _c(np.array(ws)), central)


def near_sum(tgt, src, q, cells: CellTable, self_offset: int = -1) -> np.ndarray:
    """Phi_in at the targets, Eq.(5), over the cells of `cells`."""
    tgt, src, q = _c(tgt), _c(src), _c(q)
    phi = np.zeros(tgt.shape[0])
    if tgt.shape[0] == 0:
        return phi
    _lib().oracle_near_sum(_p(tgt), tgt.shape[0], _p(src), _p(q), src.shape[0], _p(cells.shift),
                           _p(cells.sign), _p(cells.w), cells.w.shape[0], cells.central,
                           self_offset, _p(phi))
    return phi


def node_sum(tgt, R, nrm, Q, D) -> np.ndarray:
    """Phi_out at the targets from the surface nodes: Eq.(10) PAPER.md:101 discretised,
    exact normal dipole (reading S9)."""
    tgt, R, nrm, Q, D = _c(tgt), _c(R), _c(nrm), _c(Q), _c(D)
    phi = np.zeros(tgt.shape[0])
    if tgt.shape[0] == 0:
        return phi
    _lib().oracle_node_sum(_p(tgt), tgt.shape[0], _p(R), _p(nrm), _p(Q), _p(D), R.shape[0], _p(phi))
    return phi


def near_grad(tgt, src, q, cells: CellTable, self_offset: int = -1) -> np.ndarray:
    """Gradient of Phi_in (Eq.5) with respect to the target position, [T,3].
    The force on source i is -q_i grad Phi(r_i)."""
    tgt, src, q = _c(tgt), _c(src), _c(q)
    g = np.zeros((tgt.shape[0], 3))
    if tgt.shape[0] == 0:
        return g
    _lib().oracle_near_grad(_p(tgt), tgt.shape[0], _p(src), _p(q), src.shape[0], _p(cells.shift),
                            _p(cells.sign), _p(cells.w), cells.w.shape[0], cells.central,
                            self_offset, _p(g))
    return g


def node_grad(tgt, R, nrm, Q, D) -> np.ndarray:
    """Gradient of Phi_out (Eq.10 PAPER.md:101 on the nodes, exact normal dipole) at the targets, [T,3]."""
    tgt, R, nrm, Q, D = _c(tgt), _c(R), _c(nrm), _c(Q), _c(D)
    g = np.zeros((tgt.shape[0], 3))
    if tgt.shape[0] == 0:
        return g
    _lib().oracle_node_grad(_p(tgt), tgt.shape[0], _p(R), _p(nrm), _p(Q), _p(D), R.shape[0], _p(g))
    return g


def images_inside_sphere(src, q, cells: CellTable, R: float):
    """Paper-literal near set: "the set of those charges within the sphere, where the first N
    charges are the sources and the remaining N_s - N are the images near the central box".  Every image
    sign o r_j + k L of the cell table with |image| <= R, carrying charge w_c q_j; the central cell comes first
    and in source order (the box lies inside the sphere), so image i < N is source i."""
    src, q = _c(src), _c(q)
    order = [cells.central] + [c for c in range(cells.w.shape[0]) if c != cells.central]
    pos, chg = [], []
    for c in order:
        p = cells.sign[c] * src + cells.shift[c]
        keep = (p * p).sum(axis=1) <= R * R
        if c == cells.central and not keep.all():
            raise ValueError("a source lies outside the auxiliary sphere")
        pos.append(p[keep])
        chg.append(cells.w[c] * q[keep])
    return np.concatenate(pos, axis=0), np.concatenate(chg)


def identity_cell() -> CellTable:
    return CellTable(np.zeros((1, 3), dtype=np.int64), np.zeros((1, 3)), np.ones((1, 3)), np.ones(1), 0)


def energy(q, phi) -> float:
    """U = 1/2 sum q_i phi_i, PAPER.md:142, 165 (reading S11)."""
    q, phi = _c(q), _c(phi)
    return float(_lib().oracle_energy(_p(q), _p(phi), q.shape[0]))


# --------------------------------------------------------------------------------------
# Basis: real solid harmonics (r/a)^n Y_nm, PAPER.md:68-72 (Eq.6), real form PAPER.md:140
# --------------------------------------------------------------------------------------
def basis_index(n: int, m: int) -> int:
    """Column of (n, m): n^2 + n + m, n = 0..p-1, m = -n..n (reading S1: p degrees, N_b = p^2)."""
    return n * n + n + m


def real_solid_harmonics(xyz, p: int, a: float) -> np.ndarray:
    """B[t, n^2+n+m] = (r/a)^n Y_nm(theta, phi) with Y_nm the real orthonormal spherical
    harmonics (reading S4):
        Y_n0  = N_n0 P_n(cos th)
        Y_nm  = sqrt2 N_nm P_n^m(cos th) cos(m ph)      (m > 0)
        Y_n-m = sqrt2 N_nm P_n^m(cos th) sin(m ph)      (m > 0)
    N_nm = sqrt((2n+1)/(4 pi) (n-m)!/(n+m)!), P_n^m the associated Legendre function WITHOUT the
    Condon-Shortley phase, from its textbook recurrences:
        P_m^m = (2m-1)!! sin^m,  P_{m+1}^m = (2m+1) cos P_m^m,
        (n-m) P_n^m = (2n-1) cos P_{n-1}^m - (n+m-1) P_{n-2}^m."""
    xyz = np.atleast_2d(np.asarray(xyz, dtype=np.float64))
    T = xyz.shape[0]
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    r = np.sqrt(x * x + y * y + z * z)
    safe = np.where(r > 0, r, 1.0)
    ct = np.where(r > 0, z / safe, 1.0)
    st = np.where(r > 0, np.sqrt(x * x + y * y) / safe, 0.0)
    ph = np.arctan2(y, x)
    B = np.zeros((T, p * p))
    # associated Legendre table P[n][m]
    P = [[None] * (n + 1) for n in range(p)]
    for m in range(p):
        dfact = 1.0
        for k in range(1, 2 * m, 2):
            dfact *= k
        P[m][m] = dfact * st ** m
        if m + 1 < p:
            P[m + 1][m] = (2 * m + 1) * ct * P[m][m]
        for n in range(m + 2, p):
            P[n][m] = ((2 * n - 1) * ct * P[n - 1][m] - (n + m - 1) * P[n - 2][m]) / (n - m)
    rho = r / a
    for n in range(p):
        rn = rho ** n
        for m in range(0, n + 1):
            Nnm = math.sqrt((2 * n + 1) / (4 * math.pi) * math.factorial(n - m) / math.factorial(n + m))
            if m == 0:
                B[:, basis_index(n, 0)] = rn * Nnm * P[n][0]
            else:
                B[:, basis_index(n, m)] = rn * math.sqrt(2.0) * Nnm * P[n][m] * np.cos(m * ph)
                B[:, basis_index(n, -m)] = rn * math.sqrt(2.0) * Nnm * P[n][m] * np.sin(m * ph)
    return B


def real_solid_harmonics_grad(xyz, p: int, a: float) -> np.ndarray:
    """Cartesian gradient of the same basis, G[t, n^2+n+m, :] = grad B_nm(r_t), written out in spherical
    components and rotated (needed by the Neumann rows, d Phi/d n = 0):
        d/dr      B = n B / r
        d/dtheta  B = (r/a)^n N_nm dP_n^m/dtheta {cos, sin}(m phi),
                      dP_n^m/dtheta = [n cos(th) P_n^m - (n+m) P_{n-1}^m] / sin(th)       (textbook identity)
        d/dphi    B = m (r/a)^n N_nm P_n^m {-sin, cos}(m phi)
        grad = r^ d/dr + th^ (1/r) d/dtheta + ph^ (1/(r sin th)) d/dphi.
    Points on the z axis (sin th = 0) are refused: the formulas divide by sin th."""
    xyz = np.atleast_2d(np.asarray(xyz, dtype=np.float64))
    T = xyz.shape[0]
    x, y, z = xyz[:, 0], xyz[:, 1], xyz[:, 2]
    r = np.sqrt(x * x + y * y + z * z)
    st = np.sqrt(x * x + y * y) / r
    ct = z / r
    if np.any(st < 1e-9):
        raise ValueError("gradient of the basis requested on the z axis")
    ph = np.arctan2(y, x)
    cp, sp = np.cos(ph), np.sin(ph)
    rhat = np.stack([st * cp, st * sp, ct], axis=1)
    that = np.stack([ct * cp, ct * sp, -st], axis=1)
    phat = np.stack([-sp, cp, np.zeros(T)], axis=1)
    P = [[None] * (n + 1) for n in range(p)]
    for m in range(p):
        dfact = 1.0
        for k in range(1, 2 * m, 2):
            dfact *= k
        P[m][m] = dfact * st ** m
        if m + 1 < p:
            P[m + 1][m] = (2 * m + 1) * ct * P[m][m]
        for n in range(m + 2, p):
            P[n][m] = ((2 * n - 1) * ct * P[n - 1][m] - (n + m - 1) * P[n - 2][m]) / (n - m)
    G = np.zeros((T, p * p, 3))
    rho = r / a
    for n in range(1, p):
        rn = rho ** n
        for m in range(0, n + 1):
            Nnm = math.sqrt((2 * n + 1) / (4 * math.pi) * math.factorial(n - m) / math.factorial(n + m))
            Pnm = P[n][m]
            Pn1m = P[n - 1][m] if m <= n - 1 else 0.0
            dP = (n * ct * Pnm - (n + m) * Pn1m) / st
            # members: m = 0 has the cosine one only (trig = 1); m > 0 has cos(m phi) [column +m] and sin(m phi) [column -m]
            members = [(np.ones(T), np.zeros(T), 0)] if m == 0 else \
                      [(np.cos(m * ph), -np.sin(m * ph), m), (np.sin(m * ph), np.cos(m * ph), -m)]
            c = (1.0 if m == 0 else math.sqrt(2.0)) * Nnm * rn
            for trig, dtrig, mm in members:
                d_r = n * c * Pnm * trig / r
                d_t = c * dP * trig / r
                d_p = c * Pnm * m * dtrig / (r * st)
                G[:, basis_index(n, mm), :] = d_r[:, None] * rhat + d_t[:, None] * that + d_p[:, None] * phat
    return G


def degree_of_column(p: int) -> np.ndarray:
    return np.array([n for n in range(p) for _ in range(2 * n + 1)], dtype=np.float64)


# --------------------------------------------------------------------------------------
# Monitoring (check) points
# --------------------------------------------------------------------------------------
def fibonacci_sphere_checkpoints(K: int, R0: float) -> np.ndarray:
    """latitude sin(theta_i) = (2i-1)/K - 1, azimuth 2 i pi omega, omega=(sqrt5-1)/2,
    i = 1..K (reading G7: theta_i is the latitude), on the circumsphere |x| = R0."""
    i = np.arange(1, K + 1, dtype=np.float64)
    s = (2.0 * i - 1.0) / K - 1.0
    c = np.sqrt(1.0 - s * s)
    om = (math.sqrt(5.0) - 1.0) / 2.0
    az = 2.0 * i * math.pi * om
    return np.stack([R0 * c * np.cos(az), R0 * c * np.sin(az), R0 * s], axis=1)


def wrap_into_box(x, L, periodic_axes=(True, True, True)) -> np.ndarray:
    """x~ = x - k L with k the index vector that puts x~ inside the central box."""
    x = np.array(x, dtype=np.float64, copy=True)
    L = np.asarray(L, dtype=np.float64)
    for a in range(3):
        if periodic_axes[a]:
            x[:, a] = x[:, a] - L[a] * np.round(x[:, a] / L[a])
    return x


PLASTIC = 1.32471795724474602596


def default_face_points(K: int, L, axes) -> np.ndarray:
    """Deterministic 'nearly uniformly distributed' points on the faces normal to `axes`
    (reading S5b): faces ordered (-x,+x,-y,+y,-z,+z); face f gets
    floor(K a_f / sum a) points, leftovers go one each to the first faces; point number n
    (global counter, 0-based) has in-face coordinates ((frac(1/2+(n+1) g1) - 1/2) L_u,
    (frac(1/2+(n+1) g2) - 1/2) L_v), g1 = 1/rho, g2 = 1/rho^2, rho the plastic number."""
    L = np.asarray(L, dtype=np.float64)
    faces = [(a, s) for a in range(3) if a in axes for s in (-1, 1)]
    areas = np.array([np.prod(np.delete(L, a)) for a, _ in faces])
    cnt = np.floor(K * areas / areas.sum()).astype(int)
    for f in range(K - int(cnt.sum())):
        cnt[f] += 1
    g1, g2 = 1.0 / PLASTIC, 1.0 / (PLASTIC * PLASTIC)
    pts = np.zeros((K, 3))
    n = 0
    for f, (a, s) in enumerate(faces):
        u_ax, v_ax = [b for b in range(3) if b != a]
        for _ in range(cnt[f]):
            u = math.fmod(0.5 + (n + 1) * g1, 1.0)
            v = math.fmod(0.5 + (n + 1) * g2, 1.0)
            pts[n, a] = 0.5 * s * L[a]
            pts[n, u_ax] = (u - 0.5) * L[u_ax]
            pts[n, v_ax] = (v - 0.5) * L[v_ax]
            n += 1
    return pts


# --------------------------------------------------------------------------------------
# Integration nodes on the auxiliary sphere
# --------------------------------------------------------------------------------------
def default_lower_face_points(K: int, L) -> np.ndarray:
    """The face-pair closure's default points: the same lattice rule as default_face_points, on the three lower
    faces x_a = -L_a/2 only (face f gets floor(K a_f / sum a) points, leftovers one each to the first faces)."""
    L = np.asarray(L, dtype=np.float64)
    areas = np.array([np.prod(np.delete(L, a)) for a in range(3)])
    cnt = np.floor(K * areas / areas.sum()).astype(int)
    for f in range(K - int(cnt.sum())):
        cnt[f] += 1
    g1, g2 = 1.0 / PLASTIC, 1.0 / (PLASTIC * PLASTIC)
    pts = np.zeros((K, 3))
    n = 0
    for a in range(3):
        u_ax, v_ax = [b for b in range(3) if b != a]
        for _ in range(cnt[a]):
            pts[n, a] = -0.5 * L[a]
            pts[n, u_ax] = (math.fmod(0.5 + (n + 1) * g1, 1.0) - 0.5) * L[u_ax]
            pts[n, v_ax] = (math.fmod(0.5 + (n + 1) * g2, 1.0) - 0.5) * L[v_ax]
            n += 1
    return pts


def fibonacci_pair(F2: int):
    a, b = 1, 1
    while b < F2:
        a, b = b, a + b
    if b != F2:
        raise ValueError(f"{F2} is not a Fibonacci number")
    return a, b


def nodes_lattice(F2: int, R: float):
    """The paper's rule (reading G4): z_j = -1 + 2j/F2, j = 0..F2,
    cos(theta_j) = z_j + sin(pi z_j)/pi, phi_j = pi j F1/F2, two nodes per j at phi_j and
    phi_j + pi, each with weight (2 pi R^2/F2)(1 + cos(pi z_j)).  2(F2+1) nodes."""
    F1, _ = fibonacci_pair(F2)
    j = np.arange(0, F2 + 1, dtype=np.float64)
    z = -1.0 + 2.0 * j / F2
    ct = np.clip(z + np.sin(math.pi * z) / math.pi, -1.0, 1.0)
    st = np.sqrt(1.0 - ct * ct)
    ph = math.pi * j * F1 / F2
    wj = (2.0 * math.pi * R * R / F2) * (1.0 + np.cos(math.pi * z))
    n1 = np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)
    n2 = np.stack([st * np.cos(ph + math.pi), st * np.sin(ph + math.pi), ct], axis=1)
    nrm = np.empty((2 * (F2 + 1), 3))
    nrm[0::2], nrm[1::2] = n1, n2
    w = np.repeat(wj, 2)
    return R * nrm, nrm, w


def nodes_spiral(M: int, R: float):
    """Exactly M nodes (reading S10): z_j = -1 + (2j+1)/M, cos(theta_j) = z_j + sin(pi z_j)/pi,
    phi_j = 2 pi j omega, w_j = (4 pi R^2/M)(1 + cos(pi z_j)), j = 0..M-1: the Hannay-Nye warp of
    PAPER.md:124-126 on a golden-angle spiral."""
    j = np.arange(0, M, dtype=np.float64)
    z = -1.0 + (2.0 * j + 1.0) / M
    ct = np.clip(z + np.sin(math.pi * z) / math.pi, -1.0, 1.0)
    st = np.sqrt(1.0 - ct * ct)
    om = (math.sqrt(5.0) - 1.0) / 2.0
    ph = 2.0 * math.pi * j * om
    w = (4.0 * math.pi * R * R / M) * (1.0 + np.cos(math.pi * z))
    nrm = np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)
    return R * nrm, nrm, w


def make_nodes(M: int, R: float, rule: int):
    if rule == QUAD_LATTICE:
        if M % 2 or M < 4:
            raise ValueError("lattice rule needs M = 2(F2+1)")
        return nodes_lattice(M // 2 - 1, R)
    return nodes_spiral(M, R)


# --------------------------------------------------------------------------------------
# The algorithm, PAPER.md:136-146 (preparation + update), Table I
# --------------------------------------------------------------------------------------
@dataclass
class OracleResult:
    phi: np.ndarray            # [N] potential at the sources (periodic: gauge A00 = 0, reading S2)
    U: float                   # 1/2 sum q phi
    A: np.ndarray              # [p^2] coefficients in the R0-scaled basis (A00 = 0 if periodic)
    rhs: np.ndarray            # [rows]
    fit_rms: float             # ||F A - rhs||_2 / sqrt(rows)
    cond: float                # 2-norm condition number of the fitting matrix
    phi_near: np.ndarray       # [N] part (b)
    phi_out: np.ndarray        # [N] part (c)
    check_targets: np.ndarray  # [K_t,3] points where Phi_in was summed for the rhs
    phi_check: np.ndarray      # [K_t]
    Q: np.ndarray
    D: np.ndarray
    nodes: np.ndarray
    normals: np.ndarray
    pairs: dict                # pair counts per call site
    grad: Optional[np.ndarray] = None   # [N,3] grad Phi at the sources (forces=True)
    F: Optional[np.ndarray] = None      # [N,3] forces -q_i grad Phi(r_i)


def validate_geometry(L, shell, R_aux):
    """Reading S7: whole-cell near set is valid iff R0 < R_aux <= min_a (s_a + 1/2) L_a."""
    L = np.asarray(L, dtype=np.float64)
    R0 = 0.5 * float(np.linalg.norm(L))
    bound = min((shell[a] + 0.5) * L[a] for a in range(3))
    if not (R_aux > R0 and R_aux <= bound * (1 + 1e-14)):
        raise ValueError(f"R_aux={R_aux} must lie in (R0={R0}, {bound}]")
    return R0


# ---- the fit of Eq.(7), one routine per closure --------------------------------------------------------------------
# A closure says WHERE Phi_in is sampled (check_targets), WHICH linear functionals of the harmonic series are matched
# there (the rows of the fitting matrix F) and WHAT they are matched to (the right-hand side, built from the sums of
# Phi_in -- and, for derivative rows, of grad Phi_in -- at the check targets).  hsma() below is the same for all of them.
@dataclass
class Closure:
    F: np.ndarray                  # [rows, unknowns] fitting matrix, Eq.(7)
    check_targets: np.ndarray      # [K_t, 3] where Phi_in is summed
    drop_constant: bool            # no row sees the constant harmonic: column (0,0) dropped, A00 = 0 (reading S2)
    rhs: Callable                  # rhs(phi_check [K_t], grad_check() -> [K_t, 3]) -> [rows]
    far_cells: Optional["CellTable"] = None   # far-data closure: the cells whose field is fitted (else the near set)


def _wall_axes(xf, L, kind):
    """The reflecting axis whose face each wall point lies on (cavity: any axis; slab: z)."""
    return np.argmax(np.isclose(np.abs(xf), 0.5 * L, rtol=0, atol=1e-12 * L.max()) &
                     np.array([kind == BC_MIRROR_CAVITY, kind == BC_MIRROR_CAVITY, True]), axis=1)


def closure_periodic_circumsphere(w, L, R0, p) -> Closure:
    """K points x_i on the circumsphere |x| = R0 (Fibonacci grid) and their partners x~_i wrapped into
    the box; v_i = Phi(x_i) - Phi(x~_i) = 0.  Rows B(x_i) - B(x~_i); the constant cancels (reading S2)."""
    x = fibonacci_sphere_checkpoints(w.K, R0) if w.check_xyz is None else np.asarray(w.check_xyz, float)
    xt = wrap_into_box(x, L)
    keep = np.any(np.abs(x - xt) > 0, axis=1)       # rows with x~ = x carry no information
    x, xt = x[keep], xt[keep]
    Bx = real_solid_harmonics(x, p, R0)
    Bt = real_solid_harmonics(xt, p, R0)
    K = x.shape[0]
    return Closure((Bx - Bt)[:, 1:], np.concatenate([x, xt], axis=0), True,
                   lambda phi, grad: -(phi[:K] - phi[K:]))


def closure_periodic_face_pairs(w, L, R0, p) -> Closure:
    """BASELINE.json: "check-point pairs on opposite faces".  Matching the values alone is rank deficient (every
    harmonic even in x, y and z is invisible, reading S15); periodicity of Phi AND of its normal derivative across the
    faces is the complete condition: K points on the lower faces x_a = -L_a/2, partners x + L_a e_a, one value row and
    one derivative row per pair.  The constant is dropped (reading S2)."""
    x = default_lower_face_points(w.K, L) if w.check_xyz is None else np.asarray(w.check_xyz, float)
    on = np.isclose(x, -0.5 * L, rtol=0, atol=1e-12 * L.max())
    if not on.any(axis=1).all():
        raise ValueError("face-pair check points must lie on the lower faces x_a = -L_a/2")
    pair_axes = np.argmax(on, axis=1)
    xt = x.copy()
    xt[np.arange(x.shape[0]), pair_axes] += L[pair_axes]
    idx = np.arange(x.shape[0])
    Fv = real_solid_harmonics(x, p, R0) - real_solid_harmonics(xt, p, R0)
    Fd = (real_solid_harmonics_grad(x, p, R0)[idx, :, pair_axes]
          - real_solid_harmonics_grad(xt, p, R0)[idx, :, pair_axes])
    K = x.shape[0]

    def rhs(phi, grad):
        g = grad()[np.arange(2 * K), np.tile(pair_axes, 2)]
        return np.concatenate([-(phi[:K] - phi[K:]), -(g[:K] - g[K:])])

    return Closure(np.concatenate([Fv, Fd], axis=0)[:, 1:], np.concatenate([x, xt], axis=0), True, rhs)


def closure_slab_boundary(w, L, R0, p, neumann) -> Closure:
    """Slab closed by its own boundary conditions: two families of rows ("boundary
    conditions", 80-82 for the periodic directions):
      pairs    K Fibonacci points on the circumsphere and their partners wrapped in x and y only,
               Phi(x_i) - Phi(x~_i) = 0 (the image system is xy-periodic at every height, also beyond the plates);
      plates   K points on the two faces z = +-H/2: Phi = 0 for gamma = -1 ("DBC"), d Phi/dz = 0
               for gamma = +1.
    Dirichlet plate rows see the constant harmonic (no column dropped); Neumann rows do not (A00 = 0)."""
    xs = fibonacci_sphere_checkpoints(w.K, R0)
    xt = wrap_into_box(xs, L, periodic_axes=(True, True, False))
    keep = np.any(np.abs(xs - xt) > 0, axis=1)
    xs, xt = xs[keep], xt[keep]
    xf = default_face_points(w.K, L, (2,)) if w.check_xyz is None else np.asarray(w.check_xyz, float)
    n_pair = xs.shape[0]
    if neumann:
        axes = _wall_axes(xf, L, w.kind)
        Fw = real_solid_harmonics_grad(xf, p, R0)[np.arange(xf.shape[0]), :, axes]
    else:
        axes, Fw = None, real_solid_harmonics(xf, p, R0)
    F = np.concatenate([real_solid_harmonics(xs, p, R0) - real_solid_harmonics(xt, p, R0), Fw], axis=0)

    def rhs(phi, grad):
        if neumann:
            wall = -grad()[2 * n_pair:][np.arange(xf.shape[0]), axes]
        else:
            wall = -phi[2 * n_pair:]
        return np.concatenate([-(phi[:n_pair] - phi[n_pair:2 * n_pair]), wall])

    return Closure(F[:, 1:] if neumann else F, np.concatenate([xs, xt, xf], axis=0), neumann, rhs)


def closure_walls(w, L, R0, p, neumann) -> Closure:
    """Reflecting walls closed by the wall condition at K wall points: gamma = -1 is a conductor,
    Phi_in + Phi_out = 0 (Dirichlet rows B(x), "DBC"); gamma = +1 the insulating / symmetric wall,
    d(Phi_in + Phi_out)/d x_a = 0 with a the axis of the wall the point lies on (Neumann rows)."""
    if w.check_xyz is not None:
        x = np.asarray(w.check_xyz, float)
    else:
        x = default_face_points(w.K, L, (0, 1, 2) if w.kind == BC_MIRROR_CAVITY else (2,))
    if neumann:
        axes = _wall_axes(x, L, w.kind)
        F = real_solid_harmonics_grad(x, p, R0)[np.arange(x.shape[0]), :, axes][:, 1:]
        return Closure(F, x, True, lambda phi, grad: -grad()[np.arange(x.shape[0]), axes])
    return Closure(real_solid_harmonics(x, p, R0), x, False, lambda phi, grad: -phi)


def closure_far_data(w, L, R0, p) -> Closure:
    """Reading S16 (config 4): Phi_out := the field of the far cells (far_shell minus near_shell), fitted from its
    directly summed values at K points on the six faces.  Rows B(x), right-hand side +Phi_far(x)."""
    x = np.asarray(w.check_xyz, float) if w.check_xyz is not None else default_face_points(w.K, L, (0, 1, 2))
    far = cell_table(w.kind, L, w.far_shell, w.gamma, exclude_shell=w.near_shell)
    return Closure(real_solid_harmonics(x, p, R0), x, False, lambda phi, grad: phi.copy(), far_cells=far)


def make_closure(w, L, R0, p) -> Closure:
    periodic = w.kind == BC_PERIODIC
    if periodic:
        if w.closure == CLOSURE_FACE_PAIRS:
            return closure_periodic_face_pairs(w, L, R0, p)
        if w.closure != CLOSURE_BOUNDARY:
            raise ValueError("periodic kind uses the boundary or the face-pair closure")
        return closure_periodic_circumsphere(w, L, R0, p)
    if w.closure == CLOSURE_FAR_DATA:
        return closure_far_data(w, L, R0, p)
    # wall rows of the boundary closure on reflecting axes
    if w.gamma not in (-1.0, 1.0):
        raise ValueError("the boundary closure on reflecting walls is defined for gamma = -1 (Dirichlet) or +1 (Neumann)")
    neumann = w.gamma == 1.0
    if w.kind == BC_SLAB:
        return closure_slab_boundary(w, L, R0, p, neumann)
    return closure_walls(w, L, R0, p, neumann)


def must_be_neutral(w) -> bool:
    """Periodic axes without a screening conductor, and Neumann walls, admit no solution for a net charge (S17)."""
    slab_bc = w.kind == BC_SLAB and w.closure == CLOSURE_BOUNDARY
    neumann = w.kind != BC_PERIODIC and w.closure == CLOSURE_BOUNDARY and w.gamma == 1.0
    return w.kind == BC_PERIODIC or (w.kind == BC_SLAB and not slab_bc) or neumann


def hsma(w, targets_slice: Optional[slice] = None, dipole: str = "exact", dr_rel: float = 1e-5,
         p: Optional[int] = None, M: Optional[int] = None, forces: bool = False) -> OracleResult:
    """One HSMA evaluation of workload `w` (an hsma_workloads.Workload), PAPER.md:140-142 in order:
    cells -> closure (check points, fitting matrix) -> nodes -> Phi_in at the check points -> least squares ->
    surface mapping -> sums at the sources -> energy.
    `targets_slice`: evaluate phi only at that slice of the sources (sampled parity at full size);
    U is then the partial sum over the slice.  `dipole`: "exact" (reading S9, primary) or "fd3"
    (the paper's three-sphere central difference, Eq.12-14, cross-check)."""
    p = int(p if p is not None else w.p)
    M = int(M if M is not None else w.M)
    if getattr(w, "dipole_mode", DIPOLE_EXACT) == DIPOLE_FD3 and dipole == "exact":
        dipole, dr_rel = "fd3", float(getattr(w, "fd_dr_rel", dr_rel))
    L = np.asarray(w.L, dtype=np.float64)
    R0 = validate_geometry(L, w.near_shell, w.R_aux)
    # -- centre the box at the origin ("same center at the origin"; reading G10)
    src = np.asarray(w.xyz, dtype=np.float64) - 0.5 * L
    q = np.asarray(w.q, dtype=np.float64)
    N = src.shape[0]
    if w.kind != BC_PERIODIC and w.closure == CLOSURE_BOUNDARY and w.gamma not in (-1.0, 1.0):
        raise ValueError("the boundary closure on reflecting walls is defined for gamma = -1 (Dirichlet) or +1 (Neumann)")
    if must_be_neutral(w) and abs(q.sum()) > 1e-12 * np.abs(q).sum():
        raise ValueError("periodic / Neumann system must be neutral (reading S17)")

    # -- preparation step, PAPER.md:140 ----------------------------------------------------
    near = cell_table(w.kind, L, w.near_shell, w.gamma)
    # paper-literal near set: the images inside the sphere, as an explicit list summed with the
    # identity cell; otherwise the whole cells of the table (reading S7)
    sphere = getattr(w, "near_mode", NEAR_WHOLE_CELLS) == NEAR_SPHERE
    if sphere:
        if w.closure == CLOSURE_FAR_DATA:
            raise ValueError("the sphere-culled near set is defined for the boundary closures")
        near_src, near_q, near_cells = (*images_inside_sphere(src, q, near, w.R_aux), identity_cell())
    else:
        near_src, near_q, near_cells = src, q, near
    cl = make_closure(w, L, R0, p)
    F, check_targets = cl.F, cl.check_targets
    nodes, nrm, wq = make_nodes(M, w.R_aux, w.quad_rule)
    Ynodes = real_solid_harmonics(nodes, p, w.R_aux)      # = Y_nm at the node directions (r = a)

    # -- update step, PAPER.md:142 ---------------------------------------------------------
    # right-hand side: Phi_in at the monitoring points, Eq.(5), cost O(N_s N_m) PAPER.md:78
    if cl.far_cells is not None:
        phi_check = near_sum(check_targets, src, q, cl.far_cells)   # Phi_out := field of the far cells (S16)
        n_check_cells = cl.far_cells.w.shape[0]
        rhs = cl.rhs(phi_check, None)
    else:
        phi_check = near_sum(check_targets, near_src, near_q, near_cells)
        n_check_cells = near.w.shape[0]
        rhs = cl.rhs(phi_check, lambda: near_grad(check_targets, near_src, near_q, near_cells))
    # least squares, Eq.(7)
    sol, *_ = np.linalg.lstsq(F, rhs, rcond=None)
    sv = np.linalg.svd(F, compute_uv=False)
    A = np.concatenate([[0.0], sol]) if cl.drop_constant else sol
    fit_rms = float(np.linalg.norm(F @ sol - rhs) / math.sqrt(F.shape[0]))

    # harmonic surface mapping, Eq.(10),(11) PAPER.md:99-105: on |r'| = R_aux
    n_of = degree_of_column(p)
    A_aux = A * (w.R_aux / R0) ** n_of                    # same series in the R_aux-scaled basis
    S = Ynodes @ A_aux                                    # Phi_out(R_j)
    Nrm = Ynodes @ (n_of * A_aux) / w.R_aux               # sigma(R_j) = d/dr Phi_out, Eq.(11)
    Q = wq * Nrm / (4.0 * math.pi)
    D = wq * S / (4.0 * math.pi)

    # potential at the sources
    sl = targets_slice if targets_slice is not None else slice(0, N)
    i0, i1, _ = sl.indices(N)
    tg = src[i0:i1]
    phi_near = near_sum(tg, near_src, near_q, near_cells, self_offset=i0)
    if dipole == "exact":
        phi_out = node_sum(tg, nodes, nrm, Q, D)
    elif dipole == "fd3":
        # Eq.(12)-(14): charges sigma on R_s, +mu^- on R_s - dr/2, -mu^+ on R_s + dr/2; with the
        # area factor of Eq.(13) the point charges are -/+ w_j Phi_out(R_j) / (4 pi dr).
        dr = dr_rel * w.R_aux
        zero = np.zeros_like(Q)
        phi_out = (node_sum(tg, nodes, nrm, Q, zero)
                   + node_sum(tg, (w.R_aux - dr / 2) * nrm, nrm, D / dr, zero)
                   - node_sum(tg, (w.R_aux + dr / 2) * nrm, nrm, D / dr, zero))
    else:
        raise ValueError(dipole)
    phi = phi_near + phi_out
    U = energy(q[i0:i1], phi)
    n_near = int(near_src.shape[0]) if sphere else N * int(near.w.shape[0])
    pairs = {"a": int(check_targets.shape[0]) * (n_near if sphere else N * int(n_check_cells)),
             "b": int(i1 - i0) * n_near,
             "c": int(i1 - i0) * int(nodes.shape[0]) * (3 if dipole == "fd3" else 1)}
    res = OracleResult(phi, U, A, rhs, fit_rms, float(sv[0] / sv[-1]), phi_near, phi_out,
                       check_targets, phi_check, Q, D, nodes, nrm, pairs)
    if forces:
        # PAPER.md:89-93 (Eq.9): F_i = -q_i grad [Phi_in + Phi_out](r_i), bare self term excluded,
        # coefficients A_nm held fixed; the image gradient uses the exact dipole layer (reading S9)
        if dipole == "exact":
            g_out = node_grad(tg, nodes, nrm, Q, D)
        else:   # the three charged spheres of Eq.(14): gradients of pure charges
            zero = np.zeros_like(Q)
            g_out = (node_grad(tg, nodes, nrm, Q, zero)
                     + node_grad(tg, (w.R_aux - dr / 2) * nrm, nrm, D / dr, zero)
                     - node_grad(tg, (w.R_aux + dr / 2) * nrm, nrm, D / dr, zero))
        res.grad = near_grad(tg, near_src, near_q, near_cells, self_offset=i0) + g_out
        res.F = -q[i0:i1, None] * res.grad
    return res


def series_at(points_centred, A, p: int, R0: float) -> np.ndarray:
    """Phi_out(r) = sum A_nm B_nm(r), Eq.(6), in the R0-scaled basis."""
    return real_solid_harmonics(points_centred, p, R0) @ A


def madelung_constant(U: float, N: int, a_nn: float) -> float:
    """PAPER.md:165 (reading S11): U = -N M / (2 a_nn) for unit charges."""
    return -2.0 * U * a_nn / N
