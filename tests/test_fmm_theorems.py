"""The mathematics the FMM kernels of csrc/fmm_kernels.cuh rest on, checked on CPU with an independent
numpy transcription of the recurrences: the three addition theorems of the solid harmonics in the normalisation
R_n^m = r^n P_n^m e^{i m phi} / (n+m)!,  S_n^m = (n-m)! P_n^m e^{i m phi} / r^{n+1}  (no Condon-Shortley phase), the
reflection rules used for image boxes, the derivative ladder used for forces, the (m, -m) fold of the M2L kernel and the
box-unit scalings of M2M / L2L.  `-m "not gpu"`; nothing here is used by the product."""
import numpy as np
import pytest


def fid(n, m):
    return n * n + n + m


def regular(r, p):
    """R_n^m(r) for 0 <= n <= p, -n <= m <= n by the three-term recurrence in n (the one p2m_kernel runs per lane)."""
    x, y, z = r
    r2 = x * x + y * y + z * z
    R = np.zeros((p + 1) ** 2, dtype=complex)
    R[0] = 1.0
    for m in range(p + 1):
        if m > 0:
            R[fid(m, m)] = (x + 1j * y) / (2 * m) * R[fid(m - 1, m - 1)]
        for n in range(m + 1, p + 1):
            prev2 = R[fid(n - 2, m)] if n - 2 >= m else 0.0
            R[fid(n, m)] = ((2 * n - 1) * z * R[fid(n - 1, m)] - r2 * prev2) / ((n + m) * (n - m))
    for n in range(p + 1):
        for m in range(1, n + 1):
            R[fid(n, -m)] = (-1) ** m * np.conj(R[fid(n, m)])
    return R


def singular(r, p):
    """S_n^m(r) (the recurrence of tables_kernel / m2p_points_kernel)."""
    x, y, z = r
    r2 = x * x + y * y + z * z
    S = np.zeros((p + 1) ** 2, dtype=complex)
    S[0] = 1.0 / np.sqrt(r2)
    for m in range(p + 1):
        if m > 0:
            S[fid(m, m)] = (2 * m - 1) * (x + 1j * y) / r2 * S[fid(m - 1, m - 1)]
        for n in range(m + 1, p + 1):
            prev2 = S[fid(n - 2, m)] if n - 2 >= m else 0.0
            S[fid(n, m)] = ((2 * n - 1) * z * S[fid(n - 1, m)] - (n - 1 + m) * (n - 1 - m) * prev2) / r2
    for n in range(p + 1):
        for m in range(1, n + 1):
            S[fid(n, -m)] = (-1) ** m * np.conj(S[fid(n, m)])
    return S


def get(A, n, m):
    return A[fid(n, m)] if (n >= 0 and abs(m) <= n) else 0.0


RNG = np.random.default_rng(1806)


def test_closed_forms_of_the_lowest_orders():
    r = RNG.standard_normal(3)
    x, y, z = r
    R, S = regular(r, 2), singular(r, 2)
    rr = np.linalg.norm(r)
    assert np.isclose(R[fid(1, 0)], z) and np.isclose(R[fid(1, 1)], (x + 1j * y) / 2)
    assert np.isclose(R[fid(2, 0)], (3 * z * z - rr ** 2) / 4)               # r^2 P_2(cos) / 2!
    assert np.isclose(S[fid(0, 0)], 1 / rr) and np.isclose(S[fid(1, 0)], z / rr ** 3)
    assert np.isclose(S[fid(1, 1)], (x + 1j * y) / rr ** 3)


def test_expansion_of_the_coulomb_kernel():
    """1/|a - b| = sum conj R_n^m(a) S_n^m(b), |a| < |b|: P2M followed by M2P."""
    p = 40
    a = RNG.standard_normal(3) * 0.2
    b = RNG.standard_normal(3)
    b *= 1.7 / np.linalg.norm(b)
    tot = np.sum(np.conj(regular(a, p)) * singular(b, p))
    assert abs(tot.imag) < 1e-15 and abs(tot.real - 1 / np.linalg.norm(a - b)) < 1e-14


def test_addition_theorem_of_the_regular_harmonics():
    """R_n^m(a + b) = sum_{k,l} R_k^l(a) R_{n-k}^{m-l}(b): M2M and L2L, no coefficients in this normalisation."""
    p = 9
    a, b = RNG.standard_normal(3) * 0.4, RNG.standard_normal(3) * 0.3
    Ra, Rb, Rab = regular(a, p), regular(b, p), regular(a + b, p)
    for n in range(p + 1):
        for m in range(-n, n + 1):
            t = sum(get(Ra, k, l) * get(Rb, n - k, m - l) for k in range(n + 1) for l in range(-k, k + 1))
            assert abs(t - Rab[fid(n, m)]) < 1e-14 * max(1.0, abs(t))


def test_addition_theorem_of_the_singular_harmonics():
    """S_n^m(a + b) = sum_{k,l} (-1)^k conj R_k^l(a) S_{n+k}^{m+l}(b), |a| < |b|: M2L."""
    p, q = 6, 44
    a = RNG.standard_normal(3) * 0.15
    b = RNG.standard_normal(3)
    b *= 2.0 / np.linalg.norm(b)
    Ra, Sb, Sab = regular(a, q), singular(b, p + q), singular(a + b, p)
    for n in range(p + 1):
        for m in range(-n, n + 1):
            t = sum((-1) ** k * np.conj(get(Ra, k, l)) * get(Sb, n + k, m + l) for k in range(q + 1) for l in range(-k, k + 1))
            assert abs(t - Sab[fid(n, m)]) < 1e-12 * abs(Sab[fid(n, m)])


def test_reflection_rules_of_image_boxes():
    """Mirrored sources: x -> -x gives R_n^{-m} (= (-1)^m conj R_n^m), y -> -y gives conj, z -> -z gives (-1)^{n+m}."""
    p = 8
    r = RNG.standard_normal(3)
    R = regular(r, p)
    for n in range(p + 1):
        for m in range(0, n + 1):
            assert np.isclose(regular(r * [-1, 1, 1], p)[fid(n, m)], (-1) ** m * np.conj(R[fid(n, m)]))
            assert np.isclose(regular(r * [1, -1, 1], p)[fid(n, m)], np.conj(R[fid(n, m)]))
            assert np.isclose(regular(r * [1, 1, -1], p)[fid(n, m)], (-1) ** (n + m) * R[fid(n, m)])


def test_derivative_ladder_and_the_gradient_of_a_local_expansion():
    """d/dz R_n^m = R_{n-1}^m, (d/dx - i d/dy) R_n^m = R_{n-1}^{m-1}, (d/dx + i d/dy) R_n^m = -R_{n-1}^{m+1}; hence the
    gradient formulas of leaf_kernel<.,true> for Psi = Re sum conj R_k^l L_k^l."""
    p, h = 7, 1e-6
    r = RNG.standard_normal(3) * 0.5
    R0 = regular(r, p)
    d = [(regular(r + h * e, p) - regular(r - h * e, p)) / (2 * h) for e in np.eye(3)]
    for n in range(1, p + 1):
        for m in range(-n, n + 1):
            i = fid(n, m)
            assert abs(d[2][i] - get(R0, n - 1, m)) < 1e-8
            assert abs(d[0][i] - 1j * d[1][i] - get(R0, n - 1, m - 1)) < 1e-8
            assert abs(d[0][i] + 1j * d[1][i] + get(R0, n - 1, m + 1)) < 1e-8
    L = RNG.standard_normal((p + 1) ** 2) + 1j * RNG.standard_normal((p + 1) ** 2)
    for n in range(p + 1):
        L[fid(n, 0)] = L[fid(n, 0)].real
        for m in range(1, n + 1):
            L[fid(n, -m)] = (-1) ** m * np.conj(L[fid(n, m)])
    psi = lambda v: float(np.real(np.conj(regular(v, p)) @ L))          # noqa: E731
    g_fd = np.array([(psi(r + h * e) - psi(r - h * e)) / (2 * h) for e in np.eye(3)])
    gp, gz = 0.0, 0.0
    for k in range(p):
        for j in range(k + 1):
            gp += np.conj(R0[fid(k, j)]) * L[fid(k + 1, j + 1)]
            if j >= 1:
                gp -= R0[fid(k, j)] * np.conj(L[fid(k + 1, j - 1)])
            gz += (1 if j == 0 else 2) * np.real(np.conj(R0[fid(k, j)]) * L[fid(k + 1, j)])
    assert np.allclose([gp.real, gp.imag, gz], g_fd, rtol=0, atol=1e-7 * np.abs(g_fd).max())


def test_m2l_fold_of_the_orders_m_and_minus_m():
    """conj(M_n^m) S^{l+m} + conj(M_n^{-m}) S^{l-m} = a P + b Q with M_n^m = a + ib, P = S^{l+m} + (-1)^m S^{l-m},
    Q = -i (S^{l+m} - (-1)^m S^{l-m}): what m2l_inner computes with 4 real FMA per sibling and term pair."""
    p = 6
    src = RNG.standard_normal((5, 3)) * 0.3
    q = RNG.standard_normal(5)
    M = sum(qi * regular(s, p) for qi, s in zip(q, src))
    S = singular(np.array([2.0, -3.0, 4.0]), 2 * p)
    for k in range(p + 1):
        for l in range(k + 1):
            full = sum(np.conj(get(M, n, m)) * get(S, n + k, m + l) for n in range(p + 1) for m in range(-n, n + 1))
            fold = 0.0
            for n in range(p + 1):
                fold += M[fid(n, 0)].real * get(S, n + k, l)
                for m in range(1, n + 1):
                    a, b = M[fid(n, m)].real, M[fid(n, m)].imag
                    up, dn, sg = get(S, n + k, l + m), get(S, n + k, l - m), (-1) ** m
                    fold += a * (up + sg * dn) + b * (-1j) * (up - sg * dn)
            assert abs(full - fold) < 1e-13 * max(1.0, abs(full))


def test_box_unit_scalings_of_m2m_and_l2l():
    """In units of the box side a of each level (M~ = M / a^n, phi = (1/a) sum conj R(x/a) L~): M2M carries 2^{-(n-k)},
    L2L carries 2^{-(n+1)} -- the factors in m2m_kernel / l2l_kernel."""
    p, a = 8, 0.37
    src = (RNG.random((6, 3)) - 0.5) * a / 2          # inside a child box of side a/2
    q = RNG.standard_normal(6)
    shift = np.array([0.25, -0.25, 0.25]) * a         # child centre - parent centre
    Mc = sum(qi * regular(s / (a / 2), p) for qi, s in zip(q, src))                 # child moments, child units
    Mp_direct = sum(qi * regular((s + shift) / a, p) for qi, s in zip(q, src))      # parent moments, parent units
    Rs = regular(shift / a, p)
    for n in range(p + 1):
        for m in range(-n, n + 1):
            t = sum(get(Rs, k, l) * get(Mc, n - k, m - l) * 0.5 ** (n - k) for k in range(n + 1) for l in range(-k, k + 1))
            assert abs(t - Mp_direct[fid(n, m)]) < 1e-14 * max(1e-3, abs(t))
    # a local expansion about the parent's centre (one unit charge far away), shifted to the child's centre
    far = np.array([3.1, -2.2, 2.7]) * a

    def local(c, u, order):
        """phi(x) = 1/|x - far| = (1/u) sum conj R_k^l((x - c)/u) L~_k^l with L~_k^l = (-1)^k S_k^l((c - far)/u)."""
        S = singular((c - far) / u, order)
        return np.array([(-1) ** n * S[fid(n, m)] for n in range(order + 1) for m in range(-n, n + 1)])

    P = p + 22
    Lpar, Lchild, RsP = local(np.zeros(3), a, P), local(shift, a / 2, p), regular(shift / a, P)
    x = shift + (RNG.random(3) - 0.5) * a / 2                                       # a point of the child box
    assert abs(np.real(np.conj(regular((x - shift) / (a / 2), p)) @ Lchild) / (a / 2) - 1 / np.linalg.norm(x - far)) < 1e-9
    for n in range(p + 1):
        for m in range(-n, n + 1):
            t = 0.5 ** (n + 1) * sum(np.conj(get(RsP, k - n, l - m)) * Lpar[fid(k, l)] for k in range(n, P + 1) for l in range(-k, k + 1))
            assert abs(t - Lchild[fid(n, m)]) < 1e-12 * max(1e-3, abs(Lchild[fid(n, m)]))
