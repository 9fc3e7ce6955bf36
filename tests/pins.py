"""Independent textbook routines the oracle is pinned against (test-only; nothing here is used
by the oracle or by the CUDA path, and nothing here imports either).

  ewald_potentials      classical Ewald sum, tin-foil boundary (the paper's "exact" reference for
                        periodic systems, ref. [44])
  grounded_box_green    Green function of a grounded rectangular box (Dirichlet), double sine
                        series x sinh in z (Jackson, Classical Electrodynamics, sec. 3.12)
  brute_image_sum       explicit image lists, pure-Python double loop: Eq.(3)/(4) PAPER.md:40-50
"""
import math

import numpy as np
from scipy.special import erfc


def ewald_potentials(xyz, q, L, alpha, rcut_cells, kmax):
    """phi_i (self excluded) for the fully periodic system, Gaussian units, tin-foil.
    xyz [N,3] in any frame, L (3,), real-space images |n_a| <= rcut_cells, |m_a| <= kmax."""
    xyz = np.asarray(xyz, float)
    q = np.asarray(q, float)
    L = np.asarray(L, float)
    N = len(q)
    V = float(np.prod(L))
    phi = np.zeros(N)
    d = xyz[:, None, :] - xyz[None, :, :]
    rng = range(-rcut_cells, rcut_cells + 1)
    for nx in rng:
        for ny in rng:
            for nz in rng:
                s = np.array([nx, ny, nz]) * L
                r = np.sqrt(((d + s) ** 2).sum(-1))
                if nx == 0 and ny == 0 and nz == 0:
                    np.fill_diagonal(r, np.inf)
                phi += (erfc(alpha * r) / r) @ q
    ms = np.arange(-kmax, kmax + 1)
    MX, MY, MZ = np.meshgrid(ms, ms, ms, indexing="ij")
    m = np.stack([MX.ravel(), MY.ravel(), MZ.ravel()], 1)
    m = m[(m != 0).any(1)]
    k = 2 * math.pi * m / L
    k2 = (k * k).sum(1)
    ph = xyz @ k.T                                   # [N, nk]
    S = (q[:, None] * np.exp(1j * ph)).sum(0)        # structure factor
    coef = (4 * math.pi / V) * np.exp(-k2 / (4 * alpha * alpha)) / k2
    phi += (np.exp(-1j * ph) * (coef * S)[None, :]).sum(1).real
    phi -= 2 * alpha / math.sqrt(math.pi) * q
    return phi


def ewald_forces(xyz, q, L, alpha, rcut_cells, kmax):
    """F_i = -dU/dr_i of the same Ewald sum (tin-foil), textbook form:
    real space  q_i q_j [erfc(a r)/r + 2a/sqrt(pi) exp(-a^2 r^2)] r_vec/r^2,
    reciprocal  -q_i (4 pi/V) sum_k k exp(-k^2/4a^2)/k^2 Im[exp(-i k.r_i) S(k)] with S = sum q exp(i k.r)."""
    xyz = np.asarray(xyz, float)
    q = np.asarray(q, float)
    L = np.asarray(L, float)
    N = len(q)
    V = float(np.prod(L))
    F = np.zeros((N, 3))
    d = xyz[:, None, :] - xyz[None, :, :]
    rng = range(-rcut_cells, rcut_cells + 1)
    for nx in rng:
        for ny in rng:
            for nz in rng:
                dv = d + np.array([nx, ny, nz]) * L
                r2 = (dv ** 2).sum(-1)
                if nx == 0 and ny == 0 and nz == 0:
                    np.fill_diagonal(r2, np.inf)
                r = np.sqrt(r2)
                c = (erfc(alpha * r) / r + 2 * alpha / math.sqrt(math.pi) * np.exp(-alpha * alpha * r2)) / r2
                F += q[:, None] * np.einsum("ij,ijk->ik", c * q[None, :], dv)
    ms = np.arange(-kmax, kmax + 1)
    MX, MY, MZ = np.meshgrid(ms, ms, ms, indexing="ij")
    m = np.stack([MX.ravel(), MY.ravel(), MZ.ravel()], 1)
    m = m[(m != 0).any(1)]
    k = 2 * math.pi * m / L
    k2 = (k * k).sum(1)
    ph = xyz @ k.T
    S = (q[:, None] * np.exp(1j * ph)).sum(0)
    coef = (4 * math.pi / V) * np.exp(-k2 / (4 * alpha * alpha)) / k2
    im = (np.exp(-1j * ph) * S[None, :]).imag                  # [N, nk]
    F += -q[:, None] * ((im * coef[None, :]) @ k)
    return F


def grounded_box_green(x, xp, box, nmax=80):
    """G(x, x') with G = 0 on the walls of [0,a]x[0,b]x[0,c], normalised so that
    G -> 1/|x-x'| near x' (Gaussian units).  Converges like exp(-K |z - z'|): use |z-z'| > 0."""
    a, b, c = box
    zl, zg = (x[2], xp[2]) if x[2] < xp[2] else (xp[2], x[2])
    total = 0.0
    for l in range(1, nmax + 1):
        sx = math.sin(l * math.pi * x[0] / a) * math.sin(l * math.pi * xp[0] / a)
        for m in range(1, nmax + 1):
            K = math.pi * math.sqrt((l / a) ** 2 + (m / b) ** 2)
            sy = math.sin(m * math.pi * x[1] / b) * math.sin(m * math.pi * xp[1] / b)
            # sinh(K zl) sinh(K (c - zg)) / sinh(K c), written with decaying exponentials
            num = (1 - math.exp(-2 * K * zl)) * (1 - math.exp(-2 * K * (c - zg)))
            den = 1 - math.exp(-2 * K * c)
            ratio = 0.5 * math.exp(-K * (zg - zl)) * num / den
            total += sx * sy * ratio / K
    return 16 * math.pi / (a * b) * total


def grounded_slab_green(x, xp, Lx, Ly, H, mmax=40):
    """G(x, x') between two grounded plates z = 0 and z = H, periodic in x and y with cell Lx x Ly, normalised so
    that G -> 1/|x - x'| near x' (Gaussian units): the in-plane Fourier series of the textbook parallel-plate
    Green function,  G = (4 pi/A) [ z<(H - z>)/H + sum_{k != 0} cos(k.drho) sinh(k z<) sinh(k (H - z>)) / (k sinh kH) ].
    Converges like exp(-k |z - z'|): use z != z'."""
    A = Lx * Ly
    zl, zg = (x[2], xp[2]) if x[2] < xp[2] else (xp[2], x[2])
    total = zl * (H - zg) / H
    dx, dy = x[0] - xp[0], x[1] - xp[1]
    for m in range(-mmax, mmax + 1):
        for n in range(-mmax, mmax + 1):
            if m == 0 and n == 0:
                continue
            kx, ky = 2 * math.pi * m / Lx, 2 * math.pi * n / Ly
            k = math.hypot(kx, ky)
            num = (1 - math.exp(-2 * k * zl)) * (1 - math.exp(-2 * k * (H - zg)))
            den = 1 - math.exp(-2 * k * H)
            total += math.cos(kx * dx + ky * dy) * 0.5 * math.exp(-k * (zg - zl)) * num / den / k
    return 4 * math.pi / A * total


def brute_image_sum(targets, src_c, q, L, reflecting, shell, gamma, skip_self=False,
                    exclude_shell=None):
    """Explicit images, pure Python.  src_c: CENTRED source coordinates.  For every cell k with
    |k_a| <= shell_a: image coordinate on a periodic axis x + k L (Eq.3); on a reflecting axis
    (-1)^k x + k L (Eq.4) and a factor gamma per reflection.  If skip_self, target t is source t
    and its own k=0 term is dropped."""
    imgs = []
    for kx in range(-shell[0], shell[0] + 1):
        for ky in range(-shell[1], shell[1] + 1):
            for kz in range(-shell[2], shell[2] + 1):
                kk = (kx, ky, kz)
                if exclude_shell is not None and all(abs(kk[a]) <= exclude_shell[a] for a in range(3)):
                    continue
                for j in range(len(q)):
                    pos = []
                    wt = q[j]
                    for a in range(3):
                        if reflecting[a]:
                            pos.append((src_c[j][a] if kk[a] % 2 == 0 else -src_c[j][a]) + kk[a] * L[a])
                            wt *= gamma ** abs(kk[a])
                        else:
                            pos.append(src_c[j][a] + kk[a] * L[a])
                    imgs.append((pos[0], pos[1], pos[2], wt, j, kk == (0, 0, 0)))
    out = []
    for t, tg in enumerate(targets):
        terms = []
        for (x, y, z, wt, j, central) in imgs:
            if skip_self and central and j == t:
                continue
            terms.append(wt / math.sqrt((x - tg[0]) ** 2 + (y - tg[1]) ** 2 + (z - tg[2]) ** 2))
        out.append(math.fsum(terms))
    return np.array(out)
