/*
 * ORACLE -- TEST INFRASTRUCTURE ONLY.  Plain C restatement of the Coulomb pairwise sums of
 * arxiv 1806.04801 (HSMA).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this library.  It shares no code with the CUDA path.
 *
 * What each function is (citations are PAPER.md lines):
 *   oracle_near_sum   Eq.(5) PAPER.md:64 with the near images of Eq.(3)/(4), PAPER.md:40-50:
 *                       Phi_in(t) = sum_c w_c sum_j q_j / | (s_c o r_j + d_c) - t |
 *                     image position = sign o source + shift, written out exactly as in Eq.(4)
 *                     (r_{j,k} = (-1)^k o r_j, plus kL).  Optionally skips j == self index in
 *                     the one cell flagged as central (the potential at source i
 *                     excludes only its own bare term; its images are kept).
 *   oracle_node_sum   Eq.(10) PAPER.md:101 discretised on the nodes R_j with
 *                     the exact normal dipole instead of the finite difference of Eq.(12)
 *                     (reading S9):
 *                       Phi_out(t) = sum_j [ Q_j / rho - D_j * n_j.(t - R_j) / rho^3 ],  rho = |t - R_j|
 *                     since dG/dn' = n'.(r - r')/|r - r'|^3 for G = 1/|r - r'|.
 *
 * Arithmetic: fp64, correctly rounded sqrt and divide (no fast-math).  Long sums are
 * accumulated in double inside blocks of at most 256 terms and in long double across blocks
 * (SURVEY.md 8(c) step 8), so the summation error stays far below the 1e-10 / 1e-11 parity bars.
 * Parallel over targets with OpenMP; no other blocking, fusion or reordering.
 */
#include <math.h>
#include <stddef.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_BLOCK 256

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * tgt      [T,3]  target points (centred coordinates)
 * src      [N,3]  central-cell sources (centred coordinates), q [N]
 * shift    [C,3]  k o L for each near cell;  sign [C,3] = (-1)^k per axis (or +1);  w [C] weights
 * central_cell    index of the cell with k = 0, or -1
 * self_offset     if >= 0 and central_cell >= 0: target t IS source (self_offset + t) and that one
 *                 term (cell = central_cell, j = self_offset + t) is skipped; -1: nothing skipped
 * phi      [T]    output
 */
void oracle_near_sum(const double *tgt, long T, const double *src, const double *q, long N,
                     const double *shift, const double *sign, const double *w, long C,
                     long central_cell, long self_offset, double *phi)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (long t = 0; t < T; ++t) {
        const double tx = tgt[3 * t], ty = tgt[3 * t + 1], tz = tgt[3 * t + 2];
        long double total = 0.0L;
        for (long c = 0; c < C; ++c) {
            const double ax = sign[3 * c], ay = sign[3 * c + 1], az = sign[3 * c + 2];
            const double bx = shift[3 * c], by = shift[3 * c + 1], bz = shift[3 * c + 2];
            const long skip = (c == central_cell && self_offset >= 0) ? self_offset + t : -1;
            long double cell_sum = 0.0L;
            for (long j0 = 0; j0 < N; j0 += ORACLE_BLOCK) {
                const long j1 = (j0 + ORACLE_BLOCK < N) ? j0 + ORACLE_BLOCK : N;
                double blk = 0.0;
                if (skip >= j0 && skip < j1) {
                    for (long j = j0; j < j1; ++j) {
                        if (j == skip) continue;
                        const double dx = (ax * src[3 * j] + bx) - tx;
                        const double dy = (ay * src[3 * j + 1] + by) - ty;
                        const double dz = (az * src[3 * j + 2] + bz) - tz;
                        blk += q[j] / sqrt(dx * dx + dy * dy + dz * dz);
                    }
                } else {
#pragma omp simd reduction(+ : blk)
                    for (long j = j0; j < j1; ++j) {
                        const double dx = (ax * src[3 * j] + bx) - tx;
                        const double dy = (ay * src[3 * j + 1] + by) - ty;
                        const double dz = (az * src[3 * j + 2] + bz) - tz;
                        blk += q[j] / sqrt(dx * dx + dy * dy + dz * dz);
                    }
                }
                cell_sum += (long double)blk;
            }
            total += (long double)w[c] * cell_sum;
        }
        phi[t] = (double)total;
    }
}

/*
 * tgt [T,3]; nodes R [M,3]; unit outward normals nrm [M,3]; charges Q [M]; dipole strengths D [M].
 * phi [T] output = sum_j Q_j/rho - D_j (n_j . (t - R_j)) / rho^3.
 */
void oracle_node_sum(const double *tgt, long T, const double *R, const double *nrm,
                     const double *Q, const double *D, long M, double *phi)
{
#pragma omp parallel for schedule(static)
    for (long t = 0; t < T; ++t) {
        const double tx = tgt[3 * t], ty = tgt[3 * t + 1], tz = tgt[3 * t + 2];
        long double total = 0.0L;
        for (long j0 = 0; j0 < M; j0 += ORACLE_BLOCK) {
            const long j1 = (j0 + ORACLE_BLOCK < M) ? j0 + ORACLE_BLOCK : M;
            double blk = 0.0;
#pragma omp simd reduction(+ : blk)
            for (long j = j0; j < j1; ++j) {
                const double dx = tx - R[3 * j], dy = ty - R[3 * j + 1], dz = tz - R[3 * j + 2];
                const double rho2 = dx * dx + dy * dy + dz * dz;
                const double rho = sqrt(rho2);
                const double nd = nrm[3 * j] * dx + nrm[3 * j + 1] * dy + nrm[3 * j + 2] * dz;
                blk += Q[j] / rho - D[j] * nd / (rho2 * rho);
            }
            total += (long double)blk;
        }
        phi[t] = (double)total;
    }
}

/*
 * Gradients with respect to the TARGET position (Eq.(9): the force on source i is
 * -q_i grad Phi(r_i)); same arguments and conventions as the two sums above, out [T,3].
 *   d/dt  q/|p - t|                      =  q (p - t)/|p - t|^3                      (p = image position)
 *   d/dt [Q/rho - D n.(t-R)/rho^3]       = -Q d/rho^3 - D n/rho^3 + 3 D (n.d) d/rho^5,   d = t - R
 */
void oracle_near_grad(const double *tgt, long T, const double *src, const double *q, long N,
                      const double *shift, const double *sign, const double *w, long C,
                      long central_cell, long self_offset, double *grad)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (long t = 0; t < T; ++t) {
        const double tx = tgt[3 * t], ty = tgt[3 * t + 1], tz = tgt[3 * t + 2];
        long double gx = 0.0L, gy = 0.0L, gz = 0.0L;
        for (long c = 0; c < C; ++c) {
            const double ax = sign[3 * c], ay = sign[3 * c + 1], az = sign[3 * c + 2];
            const double bx = shift[3 * c], by = shift[3 * c + 1], bz = shift[3 * c + 2];
            const long skip = (c == central_cell && self_offset >= 0) ? self_offset + t : -1;
            long double cx = 0.0L, cy = 0.0L, cz = 0.0L;
            for (long j0 = 0; j0 < N; j0 += ORACLE_BLOCK) {
                const long j1 = (j0 + ORACLE_BLOCK < N) ? j0 + ORACLE_BLOCK : N;
                double sx = 0.0, sy = 0.0, sz = 0.0;
                for (long j = j0; j < j1; ++j) {
                    if (j == skip) continue;
                    const double dx = (ax * src[3 * j] + bx) - tx;
                    const double dy = (ay * src[3 * j + 1] + by) - ty;
                    const double dz = (az * src[3 * j + 2] + bz) - tz;
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    const double f = q[j] / (r2 * sqrt(r2));
                    sx += f * dx; sy += f * dy; sz += f * dz;
                }
                cx += (long double)sx; cy += (long double)sy; cz += (long double)sz;
            }
            gx += (long double)w[c] * cx; gy += (long double)w[c] * cy; gz += (long double)w[c] * cz;
        }
        grad[3 * t] = (double)gx; grad[3 * t + 1] = (double)gy; grad[3 * t + 2] = (double)gz;
    }
}

void oracle_node_grad(const double *tgt, long T, const double *R, const double *nrm,
                      const double *Q, const double *D, long M, double *grad)
{
#pragma omp parallel for schedule(static)
    for (long t = 0; t < T; ++t) {
        const double tx = tgt[3 * t], ty = tgt[3 * t + 1], tz = tgt[3 * t + 2];
        long double gx = 0.0L, gy = 0.0L, gz = 0.0L;
        for (long j0 = 0; j0 < M; j0 += ORACLE_BLOCK) {
            const long j1 = (j0 + ORACLE_BLOCK < M) ? j0 + ORACLE_BLOCK : M;
            double sx = 0.0, sy = 0.0, sz = 0.0;
            for (long j = j0; j < j1; ++j) {
                const double dx = tx - R[3 * j], dy = ty - R[3 * j + 1], dz = tz - R[3 * j + 2];
                const double rho2 = dx * dx + dy * dy + dz * dz;
                const double rho = sqrt(rho2);
                const double i3 = 1.0 / (rho2 * rho), i5 = i3 / rho2;
                const double nd = nrm[3 * j] * dx + nrm[3 * j + 1] * dy + nrm[3 * j + 2] * dz;
                const double a = -Q[j] * i3 + 3.0 * D[j] * nd * i5;   /* multiplies d */
                const double b = -D[j] * i3;                          /* multiplies n */
                sx += a * dx + b * nrm[3 * j];
                sy += a * dy + b * nrm[3 * j + 1];
                sz += a * dz + b * nrm[3 * j + 2];
            }
            gx += (long double)sx; gy += (long double)sy; gz += (long double)sz;
        }
        grad[3 * t] = (double)gx; grad[3 * t + 1] = (double)gy; grad[3 * t + 2] = (double)gz;
    }
}

/* U = 1/2 sum_i q_i phi_i, accumulated in long double. */
double oracle_energy(const double *q, const double *phi, long N)
{
    long double u = 0.0L;
    for (long i = 0; i < N; ++i) u += (long double)q[i] * (long double)phi[i];
    return (double)(0.5L * u);
}
