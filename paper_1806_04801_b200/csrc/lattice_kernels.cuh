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
// Per image (Newton form): DFMA (r^2 = e_z^2 + (X + Y)) + MUFU.RSQ64H + DMUL (y0^2) + DFMA (3 - r^2 y0^2) + DFMA (accumulate)
// = 4 FP64 instructions, + per pair (9 offsets, 3 x-squares, 9 X + Y, scale, row and column sums) / 27 = 0.89: 4.9, against
// 11.6 in near_sym_kernel and 9 in near_sum_kernel (SASS counts: profiles/r02c_ncu_lat_sym_N262144.md).
// Instantiated for the shapes the configurations use; any other cell table keeps the cell-by-cell kernels.
#pragma once
#include "sum_kernels.cuh"

namespace hsma {

struct LatGeom {
    double sh[3][5];     // sh[a][k + 2] = k * L_a, k = -2 .. 2
    double wpow[8];      // wpow[m] = scale * gamma^m (scale: 0.5 for the Newton form, whose terms are 2 / r)
    double wa[3][5];     // gradient forms: wa[a][k + 2] = gamma^|k| on a reflecting axis, 1 on a periodic one
    double wxy[5][5];    // wa[0][kx + 2] * wa[1][ky + 2]
    double cgrad;        // gradient forms: 1/8 (Newton: v = 8 / r^3), 1 (cubic)
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
// 512 threads per CTA and 4 targets per thread (16 warps per SM under a 128-register cap; the image chains of one pair
// are all the instruction-level parallelism a thread needs, so the wider CTA buys latency hiding: 312.4 -> 303.5 ms at
// config 5 against 256 threads x 8 targets, 10-13 % on the reflecting shapes).  Thread t owns the block's targets
// r * 512 + t, r < 4, i.e. tile 2r + (t >> 8), slot t & 255 -- the same linear index as near_sym_kernel's r * 256 + t.
// colw [16][kTile] lives in dynamic shared memory.
constexpr int kSymWideThreads = 512;
constexpr int kSymWideR = kSymBlock / kSymWideThreads;
constexpr int kSymWideDynSmem = (kSymWideThreads / 32) * kTile * (int)sizeof(double);

template <int REFINE, int SX, int SY, int SZ, int MASK>
__global__ void __launch_bounds__(kSymWideThreads, 1) near_lat_sym_kernel(const SymArgs a, const LatGeom g) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    extern __shared__ __align__(16) double colw_dyn[];     // [kSymWideThreads / 32][kTile]

    constexpr int R = kSymWideR, TH = kSymWideThreads, S = kSymS, RB = kSymR;   // RB: tiles per block
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, k = blockIdx.x;
    const long long f0 = a.f_begin + unit_start(k, a.fine, G), f1 = a.f_begin + unit_start(k + 1, a.fine, G);
    if (f1 <= f0) return;
    const long long V0 = f0 / kSymChunks, V1 = (f1 - 1) / kSymChunks;
    const int nt = (int)a.n_tiles;
    int I = 0;
    while (sym_visit0(I + 1, nt) <= V0) ++I;
    int J = I * RB + (int)(V0 - sym_visit0(I, nt));

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
    const int my_tile = tid >> 8, my_slot = tid & (kTile - 1);   // tile (within a pair of tiles) and slot of this thread's targets
    bool fresh = true;
    auto store_block = [&](int blk) {
        const int row = k - cta_of_unit(max(sym_visit0(blk, nt) * kSymChunks, a.f_begin) - a.f_begin, a.fine, G);
#pragma unroll
        for (int r = 0; r < R; ++r) a.part[(long long)row * Tp + (long long)(blk - a.blk_base) * kSymBlock + r * TH + tid] = tot[r];
    };

    for (int it = 0; it < nvis; ++it) {
        const int st = it & 1;
        const bool last_of_block = J + 1 == nt;
        if (tid == 0 && it + 1 < nvis) {
            const int Jn = last_of_block ? (I + 1) * RB : J + 1;
            mbar_expect_tx(&full[st ^ 1], kTile * sizeof(Src4));
            bulk_g2s(tile[st ^ 1], a.src + (long long)Jn * kTile, kTile * sizeof(Src4), &full[st ^ 1]);
        }
        if (fresh) {
            fresh = false;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int tt = I * RB + 2 * r + my_tile;
                const Src4 t = a.src[(long long)min(tt, nt - 1) * kTile + my_slot];
                ox[r] = t.x; oy[r] = t.y; oz[r] = t.z; oq[r] = tt < nt ? t.q : 0.0;
                tot[r] = 0.0;
            }
        }
        const int rd = J - I * RB;                      // < RB: the tile is one of the block's own
        const bool diag = rd < RB;
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        const int j_lo = (it == 0 ? ch_first : 0) * S;
        const int j_hi = (it == nvis - 1 ? ch_last : kSymChunks) * S;

        if (diag) {
            const int r_self = (rd - my_tile) >= 0 && ((rd - my_tile) & 1) == 0 ? (rd - my_tile) >> 1 : -1;   // my target that lives in tile rd
#pragma unroll 1
            for (int j = j_lo; j < j_hi; ++j) {
                const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
                const bool mine = j == my_slot;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const double v = lat_sum<REFINE, SX, SY, SZ, MASK, true>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, mine && r == r_self);
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
                if (lane == 0) colw_dyn[warp * kTile + j] = cj;
            }
        }
        __syncthreads();  // tile[st] may be refilled; colw is complete
        if (!diag) {
            const int j = tid;
            if (j < kTile && j >= j_lo && j < j_hi) {
                double v = 0.0;
#pragma unroll
                for (int w = 0; w < TH / 32; ++w) v += colw_dyn[w * kTile + j];
                a.col[(V0 + it - a.v_base) * kTile + j] = v;
            }
            __syncthreads();  // colw is rewritten by the next visit
        }
        if (last_of_block) {
            store_block(I);
            ++I; J = I * RB; fresh = true;
        } else {
            ++J;
        }
    }
    if (!fresh) store_block(I);
}

// ---- potential + gradient (forces, Eq.(9)) -------------------------------------------------------
// With e_a[k_a] the per-axis offsets (d_k = (e_x[k_x], e_y[k_y], e_z[k_z])), y = 1/|d_k|, v = y^3 and the cell weight
// w_k = wa_x[k_x] wa_y[k_y] wa_z[k_z]:
//     sum_k w_k v_k d_k  =  ( sum_kx e_x[kx] VX[kx],  sum_ky e_y[ky] VY[ky],  sum_kz e_z[kz] VZ[kz] ),
//     VX[kx] = sum_{ky,kz} w v,  VY[ky] = sum_{kx,kz} w v,  VZ[kz] = sum_{kx,ky} w v            (bucket sums),
// so an image costs, beyond its reciprocal distance, y^2, y^3 and two bucket updates (the z bucket and the running sum of
// its (kx, ky) line); the multiplications by the offsets and by the charges happen once per pair and axis.
// grad_i phi_i gets -q_j T, T_a = sum_k e_a VA[k]; grad_j phi_j gets +q_i sum_k sigma_a[k] e_a VA[k], sigma = -1 for an odd
// cell of a reflecting axis (partner cell d' = -sigma o d, see near_sym_field_kernel), +1 otherwise.
struct LatField { double p, tx, ty, tz, ux, uy, uz; };   // p = sum w y; t = row sums; u = column sums (sigma applied)

template <int REFINE>
__device__ __forceinline__ void lat_term_field(double r2, double& y, double& v) {
    const double y0 = rsqrt_seed(r2);
    const double t = y0 * y0;
    if (REFINE == 1) {
        y = y0 * fma(-r2, t, kNewton3);
    } else {
        const double e = fma(-r2, t, 1.0);
        const double h = fma(e, 0.375, 0.5);
        y = y0 * fma(e, h, 1.0);
    }
    v = y * (y * y);
}

template <int S, bool REFL>
__device__ __forceinline__ void lat_axis_field(double xi, double xj, const double (&sh)[5], double (&E)[2 * S + 1], double (&A)[2 * S + 1]) {
    const double d = xi - xj;
    const double sm = REFL ? xi + xj : 0.0;
#pragma unroll
    for (int k = -S; k <= S; ++k) {
        E[k + S] = k == 0 ? d : ((REFL && (k & 1)) ? sm : d) - sh[k + 2];
        A[k + S] = E[k + S] * E[k + S];
    }
}

template <int S, bool REFL>
__device__ __forceinline__ void lat_axis_close(const double (&E)[2 * S + 1], const double (&V)[2 * S + 1], double& t, double& u) {
    double te = 0.0, to = 0.0;    // even and odd cells
#pragma unroll
    for (int k = -S; k <= S; ++k) {
        if (REFL && (k & 1)) to = fma(E[k + S], V[k + S], to);
        else te = fma(E[k + S], V[k + S], te);
    }
    t = te + to; u = te - to;
}

template <int REFINE, int SX, int SY, int SZ, int MASK, bool DIAG>
__device__ __forceinline__ LatField lat_sum_field(const LatGeom& g, double xi, double yi, double zi, double xj, double yj, double zj,
                                                  bool self) {
    double EX[2 * SX + 1], EY[2 * SY + 1], EZ[2 * SZ + 1], AX[2 * SX + 1], AY[2 * SY + 1], AZ[2 * SZ + 1];
    lat_axis_field<SX, (MASK & 1) != 0>(xi, xj, g.sh[0], EX, AX);
    lat_axis_field<SY, (MASK & 2) != 0>(yi, yj, g.sh[1], EY, AY);
    lat_axis_field<SZ, (MASK & 4) != 0>(zi, zj, g.sh[2], EZ, AZ);
    double VX[2 * SX + 1], VY[2 * SY + 1], VZ[2 * SZ + 1];
#pragma unroll
    for (int k = 0; k <= 2 * SY; ++k) VY[k] = 0.0;
#pragma unroll
    for (int k = 0; k <= 2 * SZ; ++k) VZ[k] = 0.0;
    double p = 0.0;
#pragma unroll
    for (int kx = -SX; kx <= SX; ++kx) {
        double sx = 0.0, px = 0.0;
#pragma unroll
        for (int ky = -SY; ky <= SY; ++ky) {
            const double axy = AX[kx + SX] + AY[ky + SY];
            double sxy = 0.0, pxy = 0.0;
#pragma unroll
            for (int kz = -SZ; kz <= SZ; ++kz) {
                const bool c0 = DIAG && kx == 0 && ky == 0 && kz == 0;
                const double r2 = axy + AZ[kz + SZ];
                double y, v;
                lat_term_field<REFINE>(c0 && self ? 1.0 : r2, y, v);
                if (c0) { y = self ? 0.0 : y; v = self ? 0.0 : v; }
                if (MASK & 4) { pxy = fma(g.wa[2][kz + 2], y, pxy); sxy = fma(g.wa[2][kz + 2], v, sxy); }
                else { pxy += y; sxy += v; }
                if (MASK & 3) VZ[kz + SZ] = fma(g.wxy[kx + 2][ky + 2], v, VZ[kz + SZ]);
                else VZ[kz + SZ] += v;
            }
            if (MASK & 1) VY[ky + SY] = fma(g.wa[0][kx + 2], sxy, VY[ky + SY]); else VY[ky + SY] += sxy;
            if (MASK & 2) { sx = fma(g.wa[1][ky + 2], sxy, sx); px = fma(g.wa[1][ky + 2], pxy, px); }
            else { sx += sxy; px += pxy; }
        }
        if (MASK & 1) { VX[kx + SX] = g.wa[0][kx + 2] * sx; p = fma(g.wa[0][kx + 2], px, p); }
        else { VX[kx + SX] = sx; p += px; }
    }
    if (MASK & 4) {
#pragma unroll
        for (int k = -SZ; k <= SZ; ++k) VZ[k + SZ] *= g.wa[2][k + 2];
    }
    if (MASK & 2) {
#pragma unroll
        for (int k = -SY; k <= SY; ++k) VY[k + SY] *= g.wa[1][k + 2];
    }
    LatField f;
    f.p = p;
    lat_axis_close<SX, (MASK & 1) != 0>(EX, VX, f.tx, f.ux);
    lat_axis_close<SY, (MASK & 2) != 0>(EY, VY, f.ty, f.uy);
    lat_axis_close<SZ, (MASK & 4) != 0>(EZ, VZ, f.tz, f.uz);
    return f;
}

// Symmetric gradient form, lattice-factored; arguments, scratch layout (part [rows][4][...], col [visits][4][kTile]) and
// gather as near_sym_field_kernel.  The state of a thread's 8 targets (x, y | z, q | phi, gx | gy, gz: 64 B each) lives in
// shared memory -- one pair is ~320 FP64 instructions, so its 4 loads and 2 stores are noise -- which leaves the
// registers to the 27 independent image chains of a pair.
constexpr int kLatFieldDynSmem = ((kThreads / 32) * 4 * kTile + 8 * kSymR * kThreads) * (int)sizeof(double);

template <int REFINE, int SX, int SY, int SZ, int MASK>
__global__ void __launch_bounds__(kThreads, 1) near_lat_sym_field_kernel(const SymArgs a, const LatGeom g) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    extern __shared__ __align__(16) double colw[];                      // [kThreads / 32][4][kTile]
    double2* tg = reinterpret_cast<double2*>(colw + (kThreads / 32) * 4 * kTile);   // [R][4][kThreads] double2

    constexpr int R = kSymR, S = kSymFS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int G = gridDim.x, k = blockIdx.x;
    const long long f0 = a.f_begin + unit_start(k, a.fine, G), f1 = a.f_begin + unit_start(k + 1, a.fine, G);
    if (f1 <= f0) return;
    const long long V0 = f0 / kSymFChunks, V1 = (f1 - 1) / kSymFChunks;
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

    const int nvis = (int)(V1 - V0) + 1;
    const int ch_first = (int)(f0 - V0 * kSymFChunks), ch_last = (int)(f1 - 1 - V1 * kSymFChunks) + 1;
    const long long Tp = (long long)a.part_blocks * kSymBlock;
    const double cphi = a.scale, cg = g.cgrad;
    bool fresh = true;
    auto slot = [&](int r, int w) -> double2& { return tg[(r * 4 + w) * kThreads + tid]; };   // read and written by thread tid only
    auto store_block = [&](int blk) {
        const int row = k - cta_of_unit(max(sym_visit0(blk, nt) * kSymFChunks, a.f_begin) - a.f_begin, a.fine, G);
        for (int r = 0; r < R; ++r) {
            double* o = a.part + (long long)row * 4 * Tp + (long long)(blk - a.blk_base) * kSymBlock + r * kThreads + tid;
            const double2 a01 = slot(r, 2), a23 = slot(r, 3);
            o[0] = a01.x; o[Tp] = a01.y; o[2 * Tp] = a23.x; o[3 * Tp] = a23.y;
        }
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
            for (int r = 0; r < R; ++r) {
                const int tt = I * R + r;
                const Src4 t = a.src[(long long)min(tt, nt - 1) * kTile + tid];
                slot(r, 0) = make_double2(t.x, t.y);
                slot(r, 1) = make_double2(t.z, tt < nt ? t.q : 0.0);
                slot(r, 2) = make_double2(0.0, 0.0);
                slot(r, 3) = make_double2(0.0, 0.0);
            }
        }
        const int rd = J - I * R;
        const bool diag = rd < R;
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        const int j_lo = (it == 0 ? ch_first : 0) * S;
        const int j_hi = (it == nvis - 1 ? ch_last : kSymFChunks) * S;
        double* colv = a.col + (V0 + it - a.v_base) * 4 * kTile;

#pragma unroll 1
        for (int j = j_lo; j < j_hi; ++j) {
            const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
            const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
            const double qp = zq.y * cphi, qg = -zq.y * cg;
            double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
            if (diag) {
                const bool mine = j == tid;
#pragma unroll 1
                for (int r = 0; r < R; ++r) {
                    const double2 oxy = slot(r, 0), ozq = slot(r, 1);
                    const LatField f = lat_sum_field<REFINE, SX, SY, SZ, MASK, true>(g, oxy.x, oxy.y, ozq.x, xy.x, xy.y, zq.x, mine && r == rd);
                    double2 a01 = slot(r, 2), a23 = slot(r, 3);
                    a01.x = fma(qp, f.p, a01.x); a01.y = fma(qg, f.tx, a01.y);
                    a23.x = fma(qg, f.ty, a23.x); a23.y = fma(qg, f.tz, a23.y);
                    slot(r, 2) = a01; slot(r, 3) = a23;
                }
            } else {
#pragma unroll 2
                for (int r = 0; r < R; ++r) {
                    const double2 oxy = slot(r, 0), ozq = slot(r, 1);
                    const LatField f = lat_sum_field<REFINE, SX, SY, SZ, MASK, false>(g, oxy.x, oxy.y, ozq.x, xy.x, xy.y, zq.x, false);
                    double2 a01 = slot(r, 2), a23 = slot(r, 3);
                    a01.x = fma(qp, f.p, a01.x); a01.y = fma(qg, f.tx, a01.y);
                    a23.x = fma(qg, f.ty, a23.x); a23.y = fma(qg, f.tz, a23.y);
                    slot(r, 2) = a01; slot(r, 3) = a23;
                    c0 = fma(ozq.y, f.p, c0); c1 = fma(ozq.y, f.ux, c1); c2 = fma(ozq.y, f.uy, c2); c3 = fma(ozq.y, f.uz, c3);
                }
#pragma unroll
                for (int o = 16; o; o >>= 1) {
                    c0 += __shfl_xor_sync(0xffffffffu, c0, o); c1 += __shfl_xor_sync(0xffffffffu, c1, o);
                    c2 += __shfl_xor_sync(0xffffffffu, c2, o); c3 += __shfl_xor_sync(0xffffffffu, c3, o);
                }
                if (lane == 0) {
                    double* o = colw + (warp * 4) * kTile + j;
                    o[0] = c0 * cphi; o[kTile] = c1 * cg; o[2 * kTile] = c2 * cg; o[3 * kTile] = c3 * cg;
                }
            }
        }
        __syncthreads();  // tile[st] may be refilled; colw is complete
        if (!diag) {
            const int j = tid;  // kTile == kThreads
            if (j >= j_lo && j < j_hi) {
#pragma unroll
                for (int comp = 0; comp < 4; ++comp) {
                    double v = 0.0;
#pragma unroll
                    for (int w = 0; w < kThreads / 32; ++w) v += colw[(w * 4 + comp) * kTile + j];
                    colv[comp * kTile + j] = v;
                }
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

// ---- ordered pairs (steps (a) and (b) of near_sum_kernel), lattice-factored ---------------------------------------
// Same targets, partial-row layout and grid logic as near_sum_kernel (sum_kernels.cuh), with one difference: a unit is
// (target block, source tile, chunk of kLatChunk sources) -- all cells of the chunk -- instead of (block, tile, cell),
// so the host passes a.C = kLatChunks.  a.cells, a.qinfo and a.tile_np are not read (the charges enter once per pair,
// so there is nothing to gain from the sign-sorted tiles here).
constexpr int kLatChunk = 8;
constexpr int kLatChunks = kTile / kLatChunk;

template <int R, int REFINE, bool FIELD, int SX, int SY, int SZ, int MASK>
__global__ void __launch_bounds__(kThreads, FIELD ? 1 : 2) near_lat_sum_kernel(const NearArgs a, const LatGeom g) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];

    const int tid = threadIdx.x;
    const int G = gridDim.x, k = blockIdx.x;
    const long long u0 = unit_start(k, a.units, G), u1 = unit_start(k + 1, a.units, G);
    if (u1 <= u0) return;
    const long long Ub = a.n_tiles * kLatChunks;
    const long long V0 = u0 / kLatChunks, V1 = (u1 - 1) / kLatChunks;

    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&full[0], kTile * sizeof(Src4));
        bulk_g2s(tile[0], a.src + (V0 % a.n_tiles) * kTile, kTile * sizeof(Src4), &full[0]);
    }

    constexpr int RG = FIELD ? R : 1;
    double ox[R], oy[R], oz[R], tot[R];
    double totx[RG], toty[RG], totz[RG];
    const int nvis = (int)(V1 - V0) + 1;
    const int nt = (int)a.n_tiles;
    int b = (int)(V0 / a.n_tiles), tl = (int)(V0 - (long long)b * a.n_tiles);
    const int c_first = (int)(u0 - V0 * kLatChunks), c_last = (int)(u1 - 1 - V1 * kLatChunks) + 1;
    const double cphi = a.scale, cg = -g.cgrad;
    bool fresh = true;
    auto store_block = [&](int blk) {
        const int row = k - cta_of_unit(blk * Ub, a.units, G);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long t = (long long)blk * (kThreads * R) + r * kThreads + tid;
            if (t < a.T) {
                if (FIELD) {
                    double* o = a.part + (long long)row * 4 * a.T + t;
                    o[0] = cphi * tot[r]; o[a.T] = cg * totx[r % RG]; o[2 * a.T] = cg * toty[r % RG]; o[3 * a.T] = cg * totz[r % RG];
                } else {
                    a.part[(long long)row * a.T + t] = tot[r];
                }
            }
        }
    };

    for (int it = 0; it < nvis; ++it) {
        const int st = it & 1;
        if (tid == 0 && it + 1 < nvis) {
            const int tn = tl + 1 == nt ? 0 : tl + 1;
            mbar_expect_tx(&full[st ^ 1], kTile * sizeof(Src4));
            bulk_g2s(tile[st ^ 1], a.src + (long long)tn * kTile, kTile * sizeof(Src4), &full[st ^ 1]);
        }
        const long long tb = (long long)b * (kThreads * R);
        if (fresh) {
            fresh = false;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                long long t = a.t_first + min(tb + r * kThreads + tid, a.T - 1);
                if (a.tgt_index) t = a.tgt_index[t];
                const double* p = a.tgt + t * a.tstride;
                ox[r] = p[0]; oy[r] = p[1]; oz[r] = p[2];
                tot[r] = 0.0;
                if (FIELD) { totx[r % RG] = 0.0; toty[r % RG] = 0.0; totz[r % RG] = 0.0; }
            }
        }
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        const long long j0 = (long long)tl * kTile;
        const long long self_lo = a.self_offset + tb, self_hi = a.self_offset + min(a.T, tb + (long long)kThreads * R);
        const bool tile_has_self = a.self_offset >= 0 && j0 < self_hi && j0 + kTile > self_lo;
        const int j_lo = (it == 0 ? c_first : 0) * kLatChunk;
        const int j_hi = (it == nvis - 1 ? c_last : kLatChunks) * kLatChunk;

        if (tile_has_self) {
            int sj[R];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const long long i = a.self_offset + min(tb + r * kThreads + tid, a.T - 1);
                const long long slot = a.slot_of ? (long long)a.slot_of[i] : i;
                sj[r] = (int)max(-1LL, min((long long)kTile, slot - j0));
            }
#pragma unroll 1
            for (int j = j_lo; j < j_hi; ++j) {
                const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (FIELD) {
                        const LatField f = lat_sum_field<REFINE, SX, SY, SZ, MASK, true>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, j == sj[r]);
                        tot[r] = fma(zq.y, f.p, tot[r]);
                        totx[r % RG] = fma(zq.y, f.tx, totx[r % RG]); toty[r % RG] = fma(zq.y, f.ty, toty[r % RG]); totz[r % RG] = fma(zq.y, f.tz, totz[r % RG]);
                    } else {
                        tot[r] = fma(zq.y, lat_sum<REFINE, SX, SY, SZ, MASK, true>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, j == sj[r]), tot[r]);
                    }
                }
            }
        } else {
#pragma unroll 1
            for (int j = j_lo; j < j_hi; ++j) {
                const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    if (FIELD) {
                        const LatField f = lat_sum_field<REFINE, SX, SY, SZ, MASK, false>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, false);
                        tot[r] = fma(zq.y, f.p, tot[r]);
                        totx[r % RG] = fma(zq.y, f.tx, totx[r % RG]); toty[r % RG] = fma(zq.y, f.ty, toty[r % RG]); totz[r % RG] = fma(zq.y, f.tz, totz[r % RG]);
                    } else {
                        tot[r] = fma(zq.y, lat_sum<REFINE, SX, SY, SZ, MASK, false>(g, ox[r], oy[r], oz[r], xy.x, xy.y, zq.x, false), tot[r]);
                    }
                }
            }
        }
        __syncthreads();  // everyone is done with tile[st] before it is refilled
        if (++tl == nt) {
            store_block(b);
            tl = 0; ++b; fresh = true;
        }
    }
    if (!fresh) store_block(b);
}

}  // namespace hsma
