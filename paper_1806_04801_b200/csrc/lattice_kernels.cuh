// Lattice-factored image sums: the near set of steps (a) and (b) is a FULL box of image cells
// k in prod_a {-s_a .. s_a} (Eq.(3)/(4); whole cells, reading S7), so for one target i and one source j the
// squared distance to the image in cell k separates over the axes:
//     |r_i - img_k(r_j)|^2 = X[k_x] + Y[k_y] + Z[k_z],     X[k] = (x_i - (-1)^{k rho_x} x_j - k L_x)^2   (rho_a = 1: reflecting)
// The (2 s_a + 1) squares per axis are made once per (i, j) -- 5 instructions per axis at s = 1 -- and every image then
// costs ONE add for its r^2 (plus a third of one for X + Y), against 3 subtractions and 3 multiply-adds when each cell
// is walked as a separate source.  All images of a pair share q_i q_j and, within a weight class m = sum over the
// reflecting axes of |k_a| (weight gamma^m, Eq.(4)), the weight, so the reciprocal distances are accumulated per class
// with one DFMA (seed * Newton factor, never multiplied out) and the charges enter once per PAIR:
//     S_ij = sum_m gamma^m sum_{k in class m} 1 / |r_i - img_k(r_j)|,     phi_i += q_j S_ij,   phi_j += q_i S_ij.
// Per image (Newton form): DADD (r^2) + MUFU.RSQ64H + DMUL (y0^2) + DFMA (3 - r^2 y0^2) + DFMA (accumulate) = 4 FP64
// instructions + 1/3 + (15 + 3) / 27 per-pair ones = 5.0, against 11 in near_sym_kernel and 9 in near_sum_kernel.
// Instantiated for the shapes the configurations use; any other cell table keeps the cell-by-cell kernels.
#pragma once
#include "sum_kernels.cuh"

namespace hsma {

struct LatGeom {
    double sh[3][5];     // sh[a][k + 2] = k * L_a, k = -2 .. 2
    double wpow[8];      // wpow[m] = scale * gamma^m (scale: 0.5 for the Newton form, whose terms are 2 / r)
};

// X[k + S] = (x_i - img_k(x_j))^2 for one axis
template <int S, bool REFL>
__device__ __forceinline__ void lat_axis(double xi, double xj, const double (&sh)[5], double (&A)[2 * S + 1]) {
    const double d = xi - xj;
    const double sm = REFL ? xi + xj : 0.0;
#pragma unroll
    for (int k = -S; k <= S; ++k) {
        const double e = k == 0 ? d : ((REFL && (k & 1)) ? sm : d) - sh[k + 2];
        A[k + S] = e * e;
    }
}

template <int REFINE>
__device__ __forceinline__ void lat_term(double r2, double& acc) {   // acc += 2 / r (Newton) or 1 / r (cubic)
    const double y0 = rsqrt_seed(r2);
    const double t = y0 * y0;
    if (REFINE == 1) {
        acc = fma(y0, fma(-r2, t, kNewton3), acc);
    } else {
        const double e = fma(-r2, t, 1.0);
        const double h = fma(e, 0.375, 0.5);
        acc = fma(y0, fma(e, h, 1.0), acc);
    }
}

__host__ __device__ constexpr int lat_classes(int SX, int SY, int SZ, int MASK) {
    return ((MASK & 1) ? SX : 0) + ((MASK & 2) ? SY : 0) + ((MASK & 4) ? SZ : 0) + 1;
}

// S_ij (times 2 in the Newton form; the factor sits in wpow).  DIAG: the pair may be a source with itself, whose bare
// term (central cell) is left out while its images stay (Eq.(5): "j = i only in the central cell").
template <int REFINE, int SX, int SY, int SZ, int MASK, bool DIAG>
__device__ __forceinline__ double lat_sum(const LatGeom& g, double xi, double yi, double zi, double xj, double yj, double zj,
                                          bool self) {
    double AX[2 * SX + 1], AY[2 * SY + 1], AZ[2 * SZ + 1];
    lat_axis<SX, (MASK & 1) != 0>(xi, xj, g.sh[0], AX);
    lat_axis<SY, (MASK & 2) != 0>(yi, yj, g.sh[1], AY);
    lat_axis<SZ, (MASK & 4) != 0>(zi, zj, g.sh[2], AZ);
    constexpr int NC = lat_classes(SX, SY, SZ, MASK);
    double acc[NC];
#pragma unroll
    for (int m = 0; m < NC; ++m) acc[m] = 0.0;
    double central = 0.0;
#pragma unroll
    for (int kx = -SX; kx <= SX; ++kx)
#pragma unroll
        for (int ky = -SY; ky <= SY; ++ky) {
            const double axy = AX[kx + SX] + AY[ky + SY];
#pragma unroll
            for (int kz = -SZ; kz <= SZ; ++kz) {
                const int m = ((MASK & 1) ? (kx < 0 ? -kx : kx) : 0) + ((MASK & 2) ? (ky < 0 ? -ky : ky) : 0) +
                              ((MASK & 4) ? (kz < 0 ? -kz : kz) : 0);
                const double r2 = axy + AZ[kz + SZ];
                if (DIAG && kx == 0 && ky == 0 && kz == 0) lat_term<REFINE>(self ? 1.0 : r2, central);
                else lat_term<REFINE>(r2, acc[m]);
            }
        }
    if (DIAG) acc[0] += self ? 0.0 : central;
    double s = g.wpow[0] * acc[0];
#pragma unroll
    for (int m = 1; m < NC; ++m) s = fma(g.wpow[m], acc[m], s);
    return s;
}

// ---- step (b), symmetric form, lattice-factored: same work decomposition, arguments, scratch layout and gathers as
// near_sym_kernel (sum_kernels.cuh; a.cells / a.C are not read), so launch_sym's waves and the PART form carry over.
template <int REFINE, int SX, int SY, int SZ, int MASK>
__global__ void __launch_bounds__(kThreads, 1) near_lat_sym_kernel(const SymArgs a, const LatGeom g) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    __shared__ double colw[kThreads / 32][kTile];

    constexpr int R = kSymR, S = kSymS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, k = blockIdx.x;
    const long long f0 = a.f_begin + unit_start(k, a.fine, G), f1 = a.f_begin + unit_start(k + 1, a.fine, G);
    if (f1 <= f0) return;
    const long long V0 = f0 / kSymChunks, V1 = (f1 - 1) / kSymChunks;
    const int nt = (int)a.n_tiles;
    int I = 0;
    while (sym_visit0(I + 1, nt) <= V0) ++I;
    int J = I * R + (int)(V0 - sym_visit0(I, nt));

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&full[0], kTile * sizeof(Src4));
        bulk_g2s(tile[0], a.src + (long long)J * kTile, kTile * sizeof(Src4), &full[0]);
    }

    double ox[R], oy[R], oz[R], oq[R], tot[R];
    const int nvis = (int)(V1 - V0) + 1;
    const int ch_first = (int)(f0 - V0 * kSymChunks), ch_last = (int)(f1 - 1 - V1 * kSymChunks) + 1;
    const long long Tp = (long long)a.part_blocks * kSymBlock;
    bool fresh = true;
    auto store_block = [&](int blk) {
        const int row = k - cta_of_unit(max(sym_visit0(blk, nt) * kSymChunks, a.f_begin) - a.f_begin, a.fine, G);
#pragma unroll
        for (int r = 0; r < R; ++r) a.part[(long long)row * Tp + (long long)(blk - a.blk_base) * kSymBlock + r * kThreads + tid] = tot[r];
    };

    for (int it = 0; it < nvis; ++it) {
        const int st = it & 1;
        const bool last_of_block = J + 1 == nt;
        if (tid == 0 && it + 1 < nvis) {
            const int Jn = last_of_block ? (I + 1) * R : J + 1;
            mbar_expect_tx(&full[st ^ 1], kTile * sizeof(Src4));
            bulk_g2s(tile[st ^ 1], a.src + (long long)Jn * kTile, kTile * sizeof(Src4), &full[st ^ 1]);
        }
        if (fresh) {
            fresh = false;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int tt = I * R + r;               // tile of these targets; beyond the last tile: phantom, q = 0
                const Src4 t = a.src[(long long)min(tt, nt - 1) * kTile + tid];
                ox[r] = t.x; oy[r] = t.y; oz[r] = t.z; oq[r] = tt < nt ? t.q : 0.0;
                tot[r] = 0.0;
            }
        }
        const int rd = J - I * R;                       // < R: the tile is one of the block's own
        const bool diag = rd < R;
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        const int j_lo = (it == 0 ? ch_first : 0) * S;
        const int j_hi = (it == nvis - 1 ? ch_last : kSymChunks) * S;

        if (diag) {
            // the block's own tile: ordered pairs, row sums only; target (r = rd, tid) IS source j = tid
#pragma unroll 1
            for (int j = j_lo; j < j_hi; ++j) {
                const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
                const bool mine = j == tid;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double v = lat_sum<REFINE, SX, SY, SZ, MASK, true>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, mine && r == rd);
                    tot[r] = fma(zq.y, v, tot[r]);
                }
            }
        } else {
#pragma unroll 1
            for (int j = j_lo; j < j_hi; ++j) {
                const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
                double cj = 0.0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double v = lat_sum<REFINE, SX, SY, SZ, MASK, false>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, false);
                    tot[r] = fma(zq.y, v, tot[r]);
                    cj = fma(oq[r], v, cj);
                }
#pragma unroll
                for (int o = 16; o; o >>= 1) cj += __shfl_xor_sync(0xffffffffu, cj, o);
                if (lane == 0) colw[warp][j] = cj;
            }
        }
        __syncthreads();  // tile[st] may be refilled; colw is complete
        if (!diag) {
            const int j = tid;  // kTile == kThreads
            if (j >= j_lo && j < j_hi) {
                double v = 0.0;
#pragma unroll
                for (int w = 0; w < kThreads / 32; ++w) v += colw[w][j];
                a.col[(V0 + it - a.v_base) * kTile + j] = v;
            }
            __syncthreads();  // colw is rewritten by the next visit
        }
        if (last_of_block) {
            store_block(I);
            ++I; J = I * R; fresh = true;
        } else {
            ++J;
        }
    }
    if (!fresh) store_block(I);
}

}  // namespace hsma
