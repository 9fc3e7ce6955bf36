// The small dense steps that connect the pair sums: fitting matrix, Householder QR (plan time),
// Q^T b + back-substitution (H3), harmonic-to-surface mapping (H4).  DESIGN.md "Kernels".
#pragma once
#include "common.cuh"

namespace hsma {

constexpr int kMaxP = 32;
constexpr double kInv4Pi = 0.07957747154594767280;   // 1/(4 pi)
constexpr double kSqrtInv4Pi = 0.28209479177387814347;  // sqrt(1/(4 pi))

// Real orthonormal solid harmonics (r/a)^n Y_nm, n < p (Eq.6; real form PAPER.md:140;
// reading S4), evaluated without trigonometry or division by rho:
//   xi = (x + i y)/a, zeta = z/a, rho2 = |r|^2/a^2
//   V_m^m     = K_m xi^m,  K_0 = sqrt(1/4pi), K_m = K_{m-1} sqrt((2m+1)/(2m))
//   V_{m+1}^m = sqrt(2m+3) zeta V_m^m
//   V_n^m     = a_nm (zeta V_{n-1}^m - b_nm rho2 V_{n-2}^m),
//               a_nm = sqrt((4n^2-1)/(n^2-m^2)),  b_nm = sqrt(((n-1)^2-m^2)/(4(n-1)^2-1))
// (the fully normalised associated-Legendre recurrences with (r/a)^n folded in).  Column n^2+n+m:
// m = 0: Re V_n^0;  m > 0: sqrt2 Re V_n^m (cos);  -m: sqrt2 Im V_n^m (sin).
// f(n, m, vc, vs) is called once per (n, m >= 0) with vc/vs the cos/sin members already scaled.
template <class F>
__device__ __forceinline__ void solid_harmonics(double x, double y, double z, double inv_a, int p, F f) {
    const double xr = x * inv_a, xi = y * inv_a, zeta = z * inv_a;
    const double rho2 = xr * xr + xi * xi + zeta * zeta;
    double er = kSqrtInv4Pi, ei = 0.0;  // K_m xi^m
    for (int m = 0; m < p; ++m) {
        if (m > 0) {
            const double k = sqrt((2.0 * m + 1.0) / (2.0 * m));
            const double nr = k * (er * xr - ei * xi), ni = k * (er * xi + ei * xr);
            er = nr; ei = ni;
        }
        const double s = m == 0 ? 1.0 : 1.4142135623730951;
        double c2 = 0.0, s2 = 0.0;            // V_{n-2}^m
        double c1 = er, s1 = ei;              // V_{n-1}^m (starts at n-1 = m)
        f(m, m, s * c1, s * s1);
        for (int n = m + 1; n < p; ++n) {
            const double nn = (double)n, mm = (double)m;
            const double anm = sqrt((4.0 * nn * nn - 1.0) / (nn * nn - mm * mm));
            const double bnm = n == m + 1 ? 0.0 : sqrt(((nn - 1.0) * (nn - 1.0) - mm * mm) / (4.0 * (nn - 1.0) * (nn - 1.0) - 1.0));
            const double c0 = anm * (zeta * c1 - bnm * rho2 * c2);
            const double s0 = anm * (zeta * s1 - bnm * rho2 * s2);
            f(n, m, s * c0, s * s0);
            c2 = c1; s2 = s1; c1 = c0; s1 = s0;
        }
    }
}

// The same recurrences carried in forward mode: value and Cartesian gradient of every basis function (plan time
// only: the Neumann rows d Phi/d n = 0 of DESIGN.md 6.9).  g(n, m, vc, vs) receives the cos/sin members as D4.
struct D4 { double v, x, y, z; };
__device__ __forceinline__ D4 operator+(D4 a, D4 b) { return {a.v + b.v, a.x + b.x, a.y + b.y, a.z + b.z}; }
__device__ __forceinline__ D4 operator-(D4 a, D4 b) { return {a.v - b.v, a.x - b.x, a.y - b.y, a.z - b.z}; }
__device__ __forceinline__ D4 operator*(D4 a, D4 b) {
    return {a.v * b.v, a.x * b.v + a.v * b.x, a.y * b.v + a.v * b.y, a.z * b.v + a.v * b.z};
}
__device__ __forceinline__ D4 operator*(double k, D4 a) { return {k * a.v, k * a.x, k * a.y, k * a.z}; }
template <class F>
__device__ __forceinline__ void solid_harmonics_grad(double x, double y, double z, double inv_a, int p, F f) {
    const D4 xr{x * inv_a, inv_a, 0.0, 0.0}, xi{y * inv_a, 0.0, inv_a, 0.0}, zeta{z * inv_a, 0.0, 0.0, inv_a};
    const D4 rho2 = xr * xr + xi * xi + zeta * zeta;
    D4 er{kSqrtInv4Pi, 0.0, 0.0, 0.0}, ei{0.0, 0.0, 0.0, 0.0};
    for (int m = 0; m < p; ++m) {
        if (m > 0) {
            const double k = sqrt((2.0 * m + 1.0) / (2.0 * m));
            const D4 nr = k * (er * xr - ei * xi), ni = k * (er * xi + ei * xr);
            er = nr; ei = ni;
        }
        const double s = m == 0 ? 1.0 : 1.4142135623730951;
        D4 c2{0.0, 0.0, 0.0, 0.0}, s2{0.0, 0.0, 0.0, 0.0};
        D4 c1 = er, s1 = ei;
        f(m, m, s * c1, s * s1);
        for (int n = m + 1; n < p; ++n) {
            const double nn = (double)n, mm = (double)m;
            const double anm = sqrt((4.0 * nn * nn - 1.0) / (nn * nn - mm * mm));
            const double bnm = n == m + 1 ? 0.0 : sqrt(((nn - 1.0) * (nn - 1.0) - mm * mm) / (4.0 * (nn - 1.0) * (nn - 1.0) - 1.0));
            const D4 c0 = anm * (zeta * c1 - bnm * (rho2 * c2));
            const D4 s0 = anm * (zeta * s1 - bnm * (rho2 * s2));
            f(n, m, s * c0, s * s0);
            c2 = c1; s2 = s1; c1 = c0; s1 = s0;
        }
    }
}

// One row of the least-squares problem: the residual of a boundary condition,
//   row = D B(chk[i1]) - D B(chk[i2]),   rhs = -(D Phi_in(chk[i1]) - D Phi_in(chk[i2]))      (i2 < 0: no second point)
// with D = identity (axis < 0) or d/dx_axis.  Pair rows express periodicity (and for the face-pair
// closure also of the normal derivative); single value rows a grounded wall or given data; single derivative rows a
// Neumann wall.
struct RowDesc { int i1, i2, axis, pad; };

// Fitting matrix, column-major [rows x ncol] (ld = rows).  drop = 1: the constant column is dropped because no row
// sees it (periodic kinds, reading S2; Neumann walls): col = idx - 1.
__global__ void build_fit_matrix_kernel(const double* __restrict__ chk, const RowDesc* __restrict__ desc, int rows,
                                        int drop, int p, double inv_R0, double* __restrict__ Fm) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows) return;
    const RowDesc d = desc[i];
    for (int k = 0; k < 2; ++k) {
        const int idx = k == 0 ? d.i1 : d.i2;
        if (idx < 0) continue;
        const double sgn = k == 0 ? 1.0 : -1.0;
        const double* a = chk + 3 * (size_t)idx;
        if (d.axis >= 0) {
            solid_harmonics_grad(a[0], a[1], a[2], inv_R0, p, [&](int n, int m, D4 vc, D4 vs) {
                const int cc = n * n + n + m - drop, cs = n * n + n - m - drop;
                const double gc = d.axis == 0 ? vc.x : (d.axis == 1 ? vc.y : vc.z);
                const double gs = d.axis == 0 ? vs.x : (d.axis == 1 ? vs.y : vs.z);
                if (cc >= 0) Fm[(size_t)cc * rows + i] = (k == 0 ? 0.0 : Fm[(size_t)cc * rows + i]) + sgn * gc;
                if (m > 0) Fm[(size_t)cs * rows + i] = (k == 0 ? 0.0 : Fm[(size_t)cs * rows + i]) + sgn * gs;
            });
        } else {
            solid_harmonics(a[0], a[1], a[2], inv_R0, p, [&](int n, int m, double vc, double vs) {
                const int cc = n * n + n + m - drop, cs = n * n + n - m - drop;
                if (cc >= 0) Fm[(size_t)cc * rows + i] = (k == 0 ? 0.0 : Fm[(size_t)cc * rows + i]) + sgn * vc;
                if (m > 0) Fm[(size_t)cs * rows + i] = (k == 0 ? 0.0 : Fm[(size_t)cs * rows + i]) + sgn * vs;
            });
        }
    }
}

// ---- block-wide helpers (blockDim.x = 1024) --------------------------------------------------
__device__ __forceinline__ double warp_sum(double a) {
    for (int o = 16; o; o >>= 1) a += __shfl_xor_sync(0xffffffffu, a, o);
    return a;
}
__device__ __forceinline__ double block_sum(double a, double* sh /* [32] */) {
    a = warp_sum(a);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = a;
    __syncthreads();
    double b = l < (int)(blockDim.x >> 5) ? sh[l] : 0.0;
    return warp_sum(b);  // every thread gets the same value, same order
}

// apply H = I - tau v v^T (v[0] = 1 implicit, v stored in col k of A below the diagonal) to the
// columns j0..j1-1 of B (rows k..m-1); one warp per column.
__device__ __forceinline__ void apply_reflector(const double* __restrict__ v, double tau, int k, int m, double* B,
                                                int ldb, int j0, int j1) {
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = blockDim.x >> 5;
    for (int j = j0 + w; j < j1; j += nw) {
        double* col = B + (size_t)j * ldb;
        double s = 0.0;
        for (int i = k + 1 + l; i < m; i += 32) s += v[i] * col[i];
        s = warp_sum(s) + col[k];
        const double ts = tau * s;
        for (int i = k + 1 + l; i < m; i += 32) col[i] -= ts * v[i];
        __syncwarp();
        if (l == 0) col[k] -= ts;
    }
}

// Householder QR of A [m x n] column-major in place (LAPACK dgeqr2 convention): R in the upper
// triangle, reflector vectors below the diagonal, tau[n].  Then the thin Q [m x n] is formed
// explicitly in Qm (dorg2r) and R copied to Rm [n x n] column-major.  Single block.  Eq.(7) PAPER.md:76-78,
// preparation step PAPER.md:140.  flag[0] = 1 if |R_kk| <= 1e-13 max|R_jj| (rank deficient).
__global__ void __launch_bounds__(1024) householder_qr_kernel(double* __restrict__ A, int m, int n,
                                                              double* __restrict__ tau, double* __restrict__ Qm,
                                                              double* __restrict__ Rm, int* __restrict__ flag) {
    __shared__ double sh[32];
    __shared__ double s_tau;
    for (int k = 0; k < n; ++k) {
        double* x = A + (size_t)k * m;
        double ss = 0.0;
        for (int i = k + 1 + threadIdx.x; i < m; i += blockDim.x) ss += x[i] * x[i];
        ss = block_sum(ss, sh);
        const double alpha = x[k];
        __syncthreads();
        const double beta = -copysign(sqrt(alpha * alpha + ss), alpha);
        const double t = (ss == 0.0) ? 0.0 : (beta - alpha) / beta;
        const double inv = (ss == 0.0) ? 0.0 : 1.0 / (alpha - beta);
        for (int i = k + 1 + threadIdx.x; i < m; i += blockDim.x) x[i] *= inv;
        if (threadIdx.x == 0) { x[k] = (ss == 0.0) ? alpha : beta; tau[k] = t; s_tau = t; }
        __syncthreads();
        apply_reflector(x, s_tau, k, m, A, m, k + 1, n);
        __syncthreads();
    }
    // R, rank check
    for (int idx = threadIdx.x; idx < n * n; idx += blockDim.x) {
        const int i = idx % n, j = idx / n;
        Rm[idx] = i <= j ? A[(size_t)j * m + i] : 0.0;
    }
    if (threadIdx.x == 0) {
        double mx = 0.0, mn = 1e300;
        for (int k = 0; k < n; ++k) { const double d = fabs(A[(size_t)k * m + k]); mx = fmax(mx, d); mn = fmin(mn, d); }
        flag[0] = (mn <= 1e-13 * mx) ? 1 : 0;
    }
    // thin Q = H_0 ... H_{n-1} [I; 0]
    for (size_t idx = threadIdx.x; idx < (size_t)m * n; idx += blockDim.x) {
        const int i = (int)(idx % m), j = (int)(idx / m);
        Qm[idx] = i == j ? 1.0 : 0.0;
    }
    __syncthreads();
    for (int k = n - 1; k >= 0; --k) {
        apply_reflector(A + (size_t)k * m, tau[k], k, m, Qm, m, k, n);
        __syncthreads();
    }
}

// Plan time: Pinv = R^-1 Q^T  [ncol x rows], row j contiguous (Pinv[j*rows + i]).  One thread per row i of F
// (column i of Q^T) back-substitutes R x = Q^T e_i; R is read uniformly (cache broadcast), x lives in Pinv.
// With it the update step solves Eq.(7) PAPER.md:76 as one parallel mat-vec A = Pinv rhs instead of a single-block
// Q^T b + back-substitution (0.1-0.45 ms of pure latency per evaluate).  cond(F) <= 2e3 in every configuration,
// so the explicit pseudo-inverse costs cond * eps ~ 1e-13 relative: far inside the parity bars.
__global__ void pinv_kernel(const double* __restrict__ Qm, const double* __restrict__ Rm, int rows, int ncol,
                            double* __restrict__ Pinv) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= rows) return;
    for (int k = ncol - 1; k >= 0; --k) {
        double s = Qm[(size_t)k * rows + i];
        for (int j = k + 1; j < ncol; ++j) s -= Rm[(size_t)j * ncol + k] * Pinv[(size_t)j * rows + i];
        Pinv[(size_t)k * rows + i] = s / Rm[(size_t)k * ncol + k];
    }
}

// H3 (update step): rhs from the check-point sums, A = Pinv rhs.  One warp per coefficient, 8 warps per block;
// block 0 also stores rhs.  Fixed summation order (lane-strided partial sums, xor-shuffle tree).
__global__ void __launch_bounds__(256) ls_apply_kernel(const double* __restrict__ pc, const double* __restrict__ pcg,
                                                       const RowDesc* __restrict__ desc, int rows, int ncol, int drop,
                                                       double sgn, const double* __restrict__ Pinv,
                                                       double* __restrict__ rhs, double* __restrict__ A_full) {
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    const int j = blockIdx.x * 8 + w;
    // residual of the boundary condition of row i from Phi_in (pc [K_t]) or a component of grad Phi_in (pcg [K_t,3])
    auto rhs_of = [&](int i) {
        const RowDesc d = desc[i];
        const double a = d.axis < 0 ? pc[d.i1] : pcg[3 * (size_t)d.i1 + d.axis];
        const double b = d.i2 < 0 ? 0.0 : (d.axis < 0 ? pc[d.i2] : pcg[3 * (size_t)d.i2 + d.axis]);
        return sgn * (a - b);
    };
    if (blockIdx.x == 0)
        for (int i = threadIdx.x; i < rows; i += blockDim.x) rhs[i] = rhs_of(i);
    if (j < ncol) {
        const double* row = Pinv + (size_t)j * rows;
        double s = 0.0;
        for (int i = l; i < rows; i += 32) s += row[i] * rhs_of(i);
        s = warp_sum(s);
        if (l == 0) A_full[j + drop] = s;
    }
    if (blockIdx.x == 0 && threadIdx.x == 0 && drop) A_full[0] = 0.0;
}

// c = R A (the Q^T rhs of the fitted part), for the residual below.  Single block.
__global__ void r_times_a_kernel(const double* __restrict__ Rm, const double* __restrict__ A_full, int ncol, int drop,
                                 double* __restrict__ cvec) {
    for (int j = threadIdx.x; j < ncol; j += blockDim.x) {
        double s = 0.0;
        for (int k = j; k < ncol; ++k) s += Rm[(size_t)k * ncol + j] * A_full[k + drop];
        cvec[j] = s;
    }
}

// residual of the fit: out[0] = || rhs - Q c ||_2 / sqrt(rows).  Single block.
__global__ void __launch_bounds__(1024) fit_residual_kernel(const double* __restrict__ rhs, int rows, int ncol,
                                                            const double* __restrict__ Qm,
                                                            const double* __restrict__ cvec, double* __restrict__ out) {
    __shared__ double sh[32];
    double ss = 0.0;
    for (int i = threadIdx.x; i < rows; i += blockDim.x) {
        double r = rhs[i];
        for (int j = 0; j < ncol; ++j) r -= Qm[(size_t)j * rows + i] * cvec[j];
        ss += r * r;
    }
    ss = block_sum(ss, sh);
    if (threadIdx.x == 0) out[0] = sqrt(ss / rows);
}

// H4: harmonic surface mapping, Eq.(10),(11) PAPER.md:99-105.  One thread per node j:
//   S_j = sum A'_nm Y_nm(n_j)        (= Phi_out on the sphere),  A'_nm = A_nm (R_aux/R0)^n
//   N_j = (1/R_aux) sum n A'_nm Y_nm (= sigma = d/dr Phi_out, Eq.11)
//   Q_j = w_j N_j / 4pi,  P_j = (w_j S_j / 4pi) n_j   (exact normal dipole, reading S9)
// Writes the packed record (R_j, Q_j | P_j, 0) read by node_sum_kernel.
// fd_dr > 0: the paper's three-sphere form instead (Eq.12-14): three pure charges per node,
//   Q_j on R_s,  +D_j/dr on R_s - dr/2,  -D_j/dr on R_s + dr/2,  D_j = w_j S_j/4pi (the area factors of Eq.(13)
//   cancel against the quadrature weights of the two displaced spheres); records j, M + j, 2M + j.
__global__ void surface_mapping_kernel(const double* __restrict__ A_full, int p, double ratio /* R_aux/R0 */,
                                       double R_aux, const double* __restrict__ nrm /* [M,3] */,
                                       const double* __restrict__ wq /* [M] */, int M, double fd_dr,
                                       Node8* __restrict__ nodes) {
    __shared__ double As[kMaxP * kMaxP];
    for (int idx = threadIdx.x; idx < p * p; idx += blockDim.x) {
        int n = 0;
        while ((n + 1) * (n + 1) <= idx) ++n;
        As[idx] = A_full[idx] * pow(ratio, (double)n);
    }
    __syncthreads();
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    const double nx = nrm[3 * j], ny = nrm[3 * j + 1], nz = nrm[3 * j + 2];
    double S = 0.0, Nn = 0.0;
    solid_harmonics(nx, ny, nz, 1.0, p, [&](int n, int m, double vc, double vs) {
        double t = As[n * n + n + m] * vc;
        if (m > 0) t += As[n * n + n - m] * vs;
        S += t;
        Nn += n * t;
    });
    const double w = wq[j] * kInv4Pi;
    const double D = w * S;
    Node8 o;
    o.x = R_aux * nx; o.y = R_aux * ny; o.z = R_aux * nz; o.q = w * Nn / R_aux;
    o.px = D * nx; o.py = D * ny; o.pz = D * nz; o.pad = 0.0;
    if (fd_dr > 0.0) {
        o.px = 0.0; o.py = 0.0; o.pz = 0.0;
        Node8 in = o, out = o;
        const double ri = R_aux - 0.5 * fd_dr, ro = R_aux + 0.5 * fd_dr;
        in.x = ri * nx; in.y = ri * ny; in.z = ri * nz; in.q = D / fd_dr;
        out.x = ro * nx; out.y = ro * ny; out.z = ro * nz; out.q = -D / fd_dr;
        nodes[M + j] = in;
        nodes[2 * M + j] = out;
    }
    nodes[j] = o;
}

}  // namespace hsma
