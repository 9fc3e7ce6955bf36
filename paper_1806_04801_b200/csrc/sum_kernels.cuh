// The all-pairs Coulomb kernels: hot-path steps H2 (a), H5 (b), H6 (c) of DESIGN.md.
//   near_sum_kernel  Eq.(5) PAPER.md:64 over the image cells of Eq.(3)/(4) PAPER.md:40-50
//   node_sum_kernel  Eq.(10) PAPER.md:101 discretised on the sphere nodes, exact dipole
// Each thread owns R targets in registers; source tiles (packed 32-B / 64-B records) are brought into
// shared memory by 1-D bulk async copies (TMA engine) into a 2-stage mbarrier ring; all lanes of a
// warp read the same record (shared-memory broadcast).  Image cells are never materialised: for
// sign s = +-1 per axis, |t - (s o r + kL)| = |s o (t - kL) - r|, so each thread transforms its
// TARGETS once per (tile, cell) and the per-pair work does not know about images.
#pragma once
#include "common.cuh"

namespace hsma {

struct NearArgs {
    const double* tgt;   // targets, `tstride` doubles apart (3 = xyz rows, 4 = packed Src4 rows)
    int tstride;
    long long T;         // number of targets
    long long t_first;   // index of the first target inside tgt (row offset)
    const Src4* src;     // packed, padded to a multiple of kTile with q = 0 records at kFar
    long long n_tiles;   // padded source count / kTile
    const Cell* cells;   // [C]
    int C;
    int n_src_split;     // blockIdx.y = cell_group * n_src_split + src_split
    int tiles_per_split;
    int cells_per_group;
    long long self_offset;  // >= 0: target t is source (self_offset + t); its bare term is skipped
    double scale;        // applied to the cell weights (0.5 for the Newton form, see below)
    double* part;        // [gridDim.y][T] partial sums
};

// One pair: acc += q / |d|.
//  REFINE 1: y0 = seed; q*y = (q*y0) * (kNewton3 - r2*y0^2) / 2  (one Newton step; the 1/2 lives in `scale`)
//            -> 3 DADD + DMUL + 2 DFMA (r2) + MUFU + DMUL + DFMA + DMUL + DFMA = 10 FP64-pipe instructions
//            Plain Newton (constant 3) always lands below 1/sqrt: relative error -1.5 eps^2 for a seed
//            error eps; measured on B200 (MUFU.RSQ64H): |eps| <= 9.2e-7 (2^-20), mean eps^2 = 7.6e-14, i.e.
//            error in [-1.27e-12, 0] with mean -1.14e-13.  kNewton3 = 3 + 2.28e-13 shifts the mean to zero
//            (DESIGN.md "rsqrt"); the per-pair error is then within [-1.16e-12, +1.2e-13], rms 1.6e-13.
//  REFINE 2: cubic step, q*y = (q*y0) * (1 + e (1/2 + 3e/8))                     = 12 FP64-pipe instructions
constexpr double kNewton3 = 3.0 + 2.28e-13;

template <int REFINE>
__device__ __forceinline__ void pair(double tx, double ty, double tz, double sx, double sy, double sz,
                                     double sq, double& acc) {
    const double dx = tx - sx, dy = ty - sy, dz = tz - sz;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double y0 = rsqrt_seed(r2);
    const double t = y0 * y0;
    const double u = sq * y0;
    if (REFINE == 1) {
        const double g = fma(-r2, t, kNewton3);
        acc = fma(u, g, acc);
    } else {
        const double e = fma(-r2, t, 1.0);
        const double h = fma(e, 0.375, 0.5);
        const double k = fma(e, h, 1.0);
        acc = fma(u, k, acc);
    }
}

template <int R, int REFINE>
__global__ void __launch_bounds__(kThreads) near_sum_kernel(const NearArgs a) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    __shared__ Cell cells[kMaxCells];

    const int tid = threadIdx.x;
    const int split = blockIdx.y % a.n_src_split;
    const int group = blockIdx.y / a.n_src_split;
    const int c0 = group * a.cells_per_group;
    const int c1 = min(a.C, c0 + a.cells_per_group);
    const long long tile0 = (long long)split * a.tiles_per_split;
    const long long tile1 = min(a.n_tiles, tile0 + a.tiles_per_split);
    const int nt = (int)(tile1 - tile0);

    for (int c = c0 + tid; c < c1; c += kThreads) cells[c - c0] = a.cells[c];
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0 && nt > 0) {
        mbar_expect_tx(&full[0], kTile * sizeof(Src4));
        bulk_g2s(tile[0], a.src + tile0 * kTile, kTile * sizeof(Src4), &full[0]);
    }

    // targets owned by this thread (tail threads recompute target T-1 and do not store)
    const long long tb = (long long)blockIdx.x * (kThreads * R);
    double ox[R], oy[R], oz[R], tot[R];
    long long ti[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        long long t = tb + r * kThreads + tid;
        ti[r] = t < a.T ? t : a.T - 1;
        const double* p = a.tgt + (a.t_first + ti[r]) * a.tstride;
        ox[r] = p[0]; oy[r] = p[1]; oz[r] = p[2];
        tot[r] = 0.0;
    }
    // block-uniform range of source indices that can be "self" for this block's targets
    const long long self_lo = a.self_offset + tb;
    const long long self_hi = a.self_offset + min(a.T, tb + (long long)kThreads * R);  // exclusive

    for (int it = 0; it < nt; ++it) {
        const int st = it & 1;
        if (tid == 0 && it + 1 < nt) {  // buffer st^1 was released by the barrier that ended iteration it-1
            mbar_expect_tx(&full[st ^ 1], kTile * sizeof(Src4));
            bulk_g2s(tile[st ^ 1], a.src + (tile0 + it + 1) * kTile, kTile * sizeof(Src4), &full[st ^ 1]);
        }
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        const long long j0 = (tile0 + it) * kTile;
        const bool tile_has_self = a.self_offset >= 0 && j0 < self_hi && j0 + kTile > self_lo;

        for (int c = 0; c < c1 - c0; ++c) {
            const Cell cell = cells[c];
            double tx[R], ty[R], tz[R], acc[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                tx[r] = flip(ox[r] - cell.sx, cell.fx);
                ty[r] = flip(oy[r] - cell.sy, cell.fy);
                tz[r] = flip(oz[r] - cell.sz, cell.fz);
                acc[r] = 0.0;
            }
            if (cell.central && tile_has_self) {
                // masked path: the pair (t, j = self_offset + t) has r2 = 0; give it r2 = 1, q = 0
                for (int j = 0; j < kTile; ++j) {
                    const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                    const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const bool self = (j0 + j) == (a.self_offset + ti[r]);
                        pair<REFINE>(tx[r], ty[r], tz[r], self ? tx[r] + 1.0 : xy.x, self ? ty[r] : xy.y,
                                     self ? tz[r] : zq.x, self ? 0.0 : zq.y, acc[r]);
                    }
                }
            } else {
#pragma unroll 4
                for (int j = 0; j < kTile; ++j) {
                    const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                    const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
#pragma unroll
                    for (int r = 0; r < R; ++r) pair<REFINE>(tx[r], ty[r], tz[r], xy.x, xy.y, zq.x, zq.y, acc[r]);
                }
            }
            const double w = cell.w * a.scale;
#pragma unroll
            for (int r = 0; r < R; ++r) tot[r] = fma(w, acc[r], tot[r]);
        }
        __syncthreads();  // everyone is done with tile[st] before it is refilled
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const long long t = tb + r * kThreads + tid;
        if (t < a.T) a.part[(long long)blockIdx.y * a.T + t] = tot[r];
    }
}

struct NodeArgs {
    const double* tgt;
    int tstride;
    long long T;
    long long t_first;
    const Node8* nodes;  // padded to a multiple of kTile/2 with zero-strength records at kFar
    long long n_tiles;   // tiles of kTile/2 nodes (same 8 KB stage size)
    int tiles_per_split; // blockIdx.y = split over node tiles
    double* part;        // [gridDim.y][T]
};

// phi(t) = sum_j Q_j/rho - P_j.(t - R_j)/rho^3  = sum_j y (Q_j - (P_j.d) y^2),  y = 1/rho,
// with the exact normal dipole P_j = D_j n_j (reading S9).  y by the cubic step (relative ~1e-19
// before rounding).  3 DADD + 3 (r2) + 5 (rsqrt) + 3 (P.d) + DMUL (y^2) + DFMA + DFMA = 17 FP64 instructions.
template <int R>
__global__ void __launch_bounds__(kThreads) node_sum_kernel(const NodeArgs a) {
    constexpr int kNT = kTile / 2;
    __shared__ __align__(128) Node8 tile[kStages][kNT];
    __shared__ __align__(8) uint64_t full[kStages];
    const int tid = threadIdx.x;
    const long long tile0 = (long long)blockIdx.y * a.tiles_per_split;
    const long long tile1 = min(a.n_tiles, tile0 + a.tiles_per_split);
    const int nt = (int)(tile1 - tile0);
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0 && nt > 0) {
        mbar_expect_tx(&full[0], kNT * sizeof(Node8));
        bulk_g2s(tile[0], a.nodes + tile0 * kNT, kNT * sizeof(Node8), &full[0]);
    }
    const long long tb = (long long)blockIdx.x * (kThreads * R);
    double tx[R], ty[R], tz[R], acc[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        long long t = tb + r * kThreads + tid;
        t = t < a.T ? t : a.T - 1;
        const double* p = a.tgt + (a.t_first + t) * a.tstride;
        tx[r] = p[0]; ty[r] = p[1]; tz[r] = p[2];
        acc[r] = 0.0;
    }
    for (int it = 0; it < nt; ++it) {
        const int st = it & 1;
        if (tid == 0 && it + 1 < nt) {
            mbar_expect_tx(&full[st ^ 1], kNT * sizeof(Node8));
            bulk_g2s(tile[st ^ 1], a.nodes + (tile0 + it + 1) * kNT, kNT * sizeof(Node8), &full[st ^ 1]);
        }
        mbar_wait(&full[st], (it >> 1) & 1);
        const Node8* __restrict__ s = tile[st];
#pragma unroll 2
        for (int j = 0; j < kNT; ++j) {
            const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
            const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
            const double2 pxy = *reinterpret_cast<const double2*>(&s[j].px);
            const double pz = s[j].pz;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const double dx = tx[r] - xy.x, dy = ty[r] - xy.y, dz = tz[r] - zq.x;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                const double y = rsqrt_cubic(r2);
                const double pd = fma(pz, dz, fma(pxy.y, dy, pxy.x * dx));
                const double u = fma(-pd, y * y, zq.y);
                acc[r] = fma(y, u, acc[r]);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const long long t = tb + r * kThreads + tid;
        if (t < a.T) a.part[(long long)blockIdx.y * a.T + t] = acc[r];
    }
}

// ---- H1 pre-pass: centre the coordinates and pack (x,y,z,q); pad with q = 0 records ----------
// Also accumulates sum q and sum |q| per block for the neutrality check (reading S17).
__global__ void pack_sources_kernel(const double* __restrict__ xyz, const double* __restrict__ q, long long N,
                                    long long Npad, double hx, double hy, double hz, Src4* __restrict__ out,
                                    double* __restrict__ qsum_part /* [gridDim.x][2] or null */) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double qi = 0.0;
    if (i < Npad) {
        Src4 s;
        if (i < N) {
            s.x = xyz[3 * i] - hx; s.y = xyz[3 * i + 1] - hy; s.z = xyz[3 * i + 2] - hz; s.q = q[i];
            qi = s.q;
        } else {
            s.x = kFar; s.y = kFar; s.z = kFar; s.q = 0.0;
        }
        out[i] = s;
    }
    if (qsum_part) {
        __shared__ double sh[2][32];
        double a = qi, b = fabs(qi);
        for (int o = 16; o; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) { sh[0][w] = a; sh[1][w] = b; }
        __syncthreads();
        if (w == 0) {
            const int nw = blockDim.x >> 5;
            a = l < nw ? sh[0][l] : 0.0; b = l < nw ? sh[1][l] : 0.0;
            for (int o = 16; o; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
            if (l == 0) { qsum_part[2 * blockIdx.x] = a; qsum_part[2 * blockIdx.x + 1] = b; }
        }
    }
}

// ---- H7: phi = sum over partial rows (fixed order), U block partials --------------------------
// part_b [nb][T], part_c [nc][T] (either may have 0 rows).  q read from the packed sources.
__global__ void finish_phi_kernel(const double* __restrict__ part_b, int nb, const double* __restrict__ part_c,
                                  int nc, long long T, const Src4* __restrict__ src, long long t_first,
                                  double* __restrict__ phi, double* __restrict__ u_part /* [gridDim.x] or null */) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (t < T) {
        double sb = 0.0, sc = 0.0;
        for (int k = 0; k < nb; ++k) sb += part_b[(long long)k * T + t];
        for (int k = 0; k < nc; ++k) sc += part_c[(long long)k * T + t];
        const double v = sb + sc;
        phi[t] = v;
        if (src) e = src[t_first + t].q * v;
    }
    if (u_part) {
        __shared__ double sh[32];
        for (int o = 16; o; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) sh[w] = e;
        __syncthreads();
        if (w == 0) {
            const int nw = blockDim.x >> 5;
            e = l < nw ? sh[l] : 0.0;
            for (int o = 16; o; o >>= 1) e += __shfl_down_sync(0xffffffffu, e, o);
            if (l == 0) u_part[blockIdx.x] = e;
        }
    }
}

// second level of the deterministic reductions: out[k] = scale * sum_i in[i*stride + k], one block
__global__ void reduce_rows_kernel(const double* __restrict__ in, long long n, int stride, int ncomp, double scale,
                                   double* __restrict__ out) {
    __shared__ double sh[32];
    for (int k = 0; k < ncomp; ++k) {
        double a = 0.0;
        for (long long i = threadIdx.x; i < n; i += blockDim.x) a += in[i * stride + k];
        for (int o = 16; o; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
        const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
        if (l == 0) sh[w] = a;
        __syncthreads();
        if (w == 0) {
            const int nw = blockDim.x >> 5;
            a = l < nw ? sh[l] : 0.0;
            for (int o = 16; o; o >>= 1) a += __shfl_down_sync(0xffffffffu, a, o);
            if (l == 0) out[k] = scale * a;
        }
        __syncthreads();
    }
}

}  // namespace hsma
