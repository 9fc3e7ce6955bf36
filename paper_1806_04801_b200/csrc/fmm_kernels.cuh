// Sub-quadratic form of step (b) (PAPER.md:144-146 and Table I: "both FMM and
// GPU accelerations are applied", O(N_s + N_m)): a uniform-grid fast multipole method for the near sum
//     phi_i = sum_c w_c sum_j' q_j / |r_i - (sigma_c o r_j + k_c L)|            (Eq.(5), whole cells)
// written from scratch for sm_100a.  It computes the SAME sum as near_sum_kernel / near_sym_kernel up to the truncation
// of the expansions (order p: measured <= 1e-12 of max|phi| at p = 20); the oracle stays the exact
// direct sum and the parity bars stay 1e-10 / 1e-11.
//
// Expansions (complex solid harmonics, m >= 0 stored, X_n^{-m} = (-1)^m conj X_n^m):
//     R_n^m(r) = r^n P_n^m(cos th) e^{i m ph} / (n+m)!          regular
//     S_n^m(r) = (n-m)! P_n^m(cos th) e^{i m ph} / r^{n+1}      singular            (P_n^m without Condon-Shortley phase)
// with the three addition theorems (checked numerically before this file was written)
//     1/|a - b|   = sum_{n,m} conj R_n^m(a) S_n^m(b)                                   |a| < |b|
//     R_n^m(a+b)  = sum_{k,l} R_k^l(a) R_{n-k}^{m-l}(b)
//     S_n^m(a+b)  = sum_{k,l} (-1)^k conj R_k^l(a) S_{n+k}^{m+l}(b)                    |a| < |b|
// so that, in units of the box side a_l of each level (M~ = M / a^n, phi = (1/a) sum conj R(x/a) L~):
//     P2M   M_n^m = sum_j q_j R_n^m((r_j - c)/a)
//     M2M   M_n^m(parent) = sum_{child} sum_{k,l} R_k^l(s) M_{n-k}^{m-l}(child) 2^{-(n-k)},   s = (c_child - c_parent)/a_parent
//     M2L   L_k^l(t) = (-1)^k sum_{src} sum_{n,m} conj M_n^m(src) S_{n+k}^{m+l}(d),           d = (c_t - c_src)/a
//     L2L   L_n^m(child) = 2^{-(n+1)} sum_{k,l} conj R_{k-n}^{l-m}(s) L_k^l(parent)
//     L2P   phi(x) = (1/a) Re sum_{k,l} conj R_k^l((x - c)/a) L_k^l
// Well-separated = more than kWs = 2 boxes apart (Chebyshev distance): convergence ratio (sqrt3/2)/2.5 = 0.35 per
// order instead of 0.58 with one box, which is what makes 1e-12 reachable at p = 20 (one-box separation needs p > 60).
// Image cells are never materialised here either: a source box in image cell k is the central box (mirrored in a
// reflecting axis when k_a is odd) shifted by k L; its multipole moments are those of the central box with the
// reflection signs applied on load (x: (-1)^m conj, y: conj, z: (-1)^{n+m}) and the cell weight gamma^|k|.
#pragma once
#include "common.cuh"
#include "sum_kernels.cuh"

namespace hsma {
namespace fmm {

constexpr int kWs = 2;                 // boxes within Chebyshev distance kWs are near (P2P)
constexpr int kOffR = 2 * kWs + 1;     // M2L offsets d in [-5,5]^3 with |d|_inf > kWs
constexpr int kOffW = 2 * kOffR + 1;   // 11
constexpr int kOffN = kOffW * kOffW * kOffW;
constexpr int kMaxOrder = 30;          // P2M runs one lane per order m: p <= 31; shared memory of M2L: p <= 30
constexpr int kMaxLevels = 6;          // leaf level <= 5 (keys < 2^16: two 8-bit radix passes)
constexpr int kInvW = kMaxOrder + 2;

__host__ __device__ inline int nc(int p) { return (p + 1) * (p + 2) / 2; }
__host__ __device__ inline int cidx(int n, int m) { return n * (n + 1) / 2 + m; }
__host__ __device__ inline int fidx(int n, int m) { return n * n + n + m; }   // full range m = -n..n
// Shared-memory layout of the expanded S table: row N (N = 0..2p) at N (N + 1), split by the parity of mu -- even orders
// first, odd orders N + 1 slots later -- so that the threads of a row (l0 = 0, 2, 4, ...: orders of one parity at every
// step) read CONSECUTIVE 16-byte slots (the plain layout had them 32 bytes apart: two-way bank conflicts on every read).
__host__ __device__ inline int sp_size(int p) { return (2 * p + 1) * (2 * p + 2) + 2; }
__host__ __device__ inline int sp_index(int N, int mu) {
    const int par = mu & 1;
    return N * (N + 1) + par * (N + 1) + ((mu + N + ((N + par) & 1)) >> 1);
}

struct Geom {
    int base[3];       // level-0 boxes per cell and axis (cubic boxes of side a0 = L_a / base_a)
    int levels;        // leaf level (>= 1)
    int shell[3];      // near cell table: |k_a| <= shell_a
    int refl[3];       // axis is reflecting: images in odd cells are mirrored
    int p;             // expansion order
    double a0;         // level-0 box side
    double half[3];    // L_a / 2
    double L[3];
    const double* w_lut;   // [(2 s_x+1)(2 s_y+1)(2 s_z+1)] cell weights gamma^|k|
};
__host__ __device__ inline int grid_n(const Geom& g, int lev, int a) { return g.base[a] << lev; }
__host__ __device__ inline long long boxes_at(const Geom& g, int lev) {
    return (long long)grid_n(g, lev, 0) * grid_n(g, lev, 1) * grid_n(g, lev, 2);
}
__host__ __device__ inline long long level_offset(const Geom& g, int lev) {   // boxes of the levels above
    long long o = 0;
    for (int l = 0; l < lev; ++l) o += boxes_at(g, l);
    return o;
}
__host__ __device__ inline int floor_div(int a, int b) { return a >= 0 ? a / b : -((-a + b - 1) / b); }

// A box with GLOBAL grid coordinates g (any cell) at level lev: the central box it is an image of, its cell's
// shift, reflection flags and weight.  Returns false if the cell is not in the near table.
struct ImageBox { int box; int fx, fy, fz; double sx, sy, sz, w; int central; };
__device__ __forceinline__ bool image_box(const Geom& G, int lev, int gx, int gy, int gz, ImageBox& out) {
    const int g[3] = {gx, gy, gz};
    int j[3], f[3], k[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int n = grid_n(G, lev, a);
        k[a] = floor_div(g[a], n);
        if (k[a] < -G.shell[a] || k[a] > G.shell[a]) return false;
        j[a] = g[a] - k[a] * n;
        f[a] = G.refl[a] && (k[a] & 1);
        if (f[a]) j[a] = n - 1 - j[a];
    }
    out.box = (j[0] * grid_n(G, lev, 1) + j[1]) * grid_n(G, lev, 2) + j[2];
    out.fx = f[0]; out.fy = f[1]; out.fz = f[2];
    out.sx = k[0] * G.L[0]; out.sy = k[1] * G.L[1]; out.sz = k[2] * G.L[2];
    const int wy = 2 * G.shell[1] + 1, wz = 2 * G.shell[2] + 1;
    out.w = G.w_lut[((k[0] + G.shell[0]) * wy + (k[1] + G.shell[1])) * wz + (k[2] + G.shell[2])];
    out.central = (k[0] == 0 && k[1] == 0 && k[2] == 0);
    return true;
}

// complex helpers on double2
__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ void cfma(double2& acc, double2 a, double2 b) {
    acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
// X_n^m for any |m| <= n from the m >= 0 storage
__device__ __forceinline__ double2 cget(const double2* X, int n, int m) {
    if (m >= 0) return X[cidx(n, m)];
    const double2 v = X[cidx(n, -m)];
    return (m & 1) ? make_double2(-v.x, v.y) : make_double2(v.x, -v.y);   // (-1)^m conj
}

// ---- leaf assignment and a stable two-pass radix sort (8 bits each) of the particles by leaf ------------------------
__global__ void key_kernel(const double* __restrict__ xyz, long long N, const Geom G, int* __restrict__ key, int* __restrict__ idx) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double inv = (double)(1 << G.levels) / G.a0;
    int c[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int n = grid_n(G, G.levels, a);
        const int v = (int)floor(xyz[3 * i + a] * inv);     // box coordinates: [0, L_a] -> [0, n]
        c[a] = v < 0 ? 0 : (v >= n ? n - 1 : v);
    }
    key[i] = (c[0] * grid_n(G, G.levels, 1) + c[1]) * grid_n(G, G.levels, 2) + c[2];
    idx[i] = (int)i;
}
__global__ void __launch_bounds__(256) radix_hist_kernel(const int* __restrict__ key, long long N, int shift, long long n_blk,
                                                         long long* __restrict__ counts) {
    __shared__ int h[256];
    h[threadIdx.x] = 0;
    __syncthreads();
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i < N) atomicAdd(&h[(key[i] >> shift) & 255], 1);     // integer counts: order does not matter
    __syncthreads();
    counts[(long long)threadIdx.x * n_blk + blockIdx.x] = h[threadIdx.x];
}
// counts[d][b] (digit-major) -> exclusive prefix over the blocks b of row d; tot[d] = row total.  One CTA per digit.
__global__ void __launch_bounds__(1024) radix_rowscan_kernel(long long* __restrict__ counts, long long n_blk, long long* __restrict__ tot) {
    __shared__ long long wsum[32];
    __shared__ long long carry;
    long long* row = counts + (long long)blockIdx.x * n_blk;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (long long base = 0; base < n_blk; base += 1024) {
        const long long i = base + threadIdx.x;
        const long long v = i < n_blk ? row[i] : 0;
        long long x = v;
        for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) wsum[warp] = x;
        __syncthreads();
        if (warp == 0) {
            long long w = wsum[lane];
            for (int o = 1; o < 32; o <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += y; }
            wsum[lane] = w;
        }
        __syncthreads();
        const long long before = carry + (warp > 0 ? wsum[warp - 1] : 0);
        if (i < n_blk) row[i] = before + x - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += wsum[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) tot[blockIdx.x] = carry;
}
// tot[256] -> exclusive prefix (digit bases), in place.  One warp-scan per 32, single block of 256.
__global__ void __launch_bounds__(256) radix_base_kernel(long long* __restrict__ tot) {
    __shared__ long long sh[256];
    sh[threadIdx.x] = tot[threadIdx.x];
    __syncthreads();
    if (threadIdx.x == 0) {
        long long run = 0;
        for (int d = 0; d < 256; ++d) { const long long v = sh[d]; sh[d] = run; run += v; }
    }
    __syncthreads();
    tot[threadIdx.x] = sh[threadIdx.x];
}
// stable: items keep their order within a digit (lane order in a warp, warp order in a block, block order)
__global__ void __launch_bounds__(256) radix_scatter_kernel(const int* __restrict__ key_in, const int* __restrict__ idx_in,
                                                            long long N, int shift, long long n_blk,
                                                            const long long* __restrict__ offs, const long long* __restrict__ dbase,
                                                            int* __restrict__ key_out, int* __restrict__ idx_out) {
    __shared__ int cnt[8][256];
    for (int k = threadIdx.x; k < 8 * 256; k += 256) (&cnt[0][0])[k] = 0;
    __syncthreads();
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    const bool valid = i < N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int kv = valid ? key_in[i] : 0;
    const int d = (kv >> shift) & 255;
    const unsigned peers = __match_any_sync(0xffffffffu, valid ? d : -1 - lane);
    const int rank = __popc(peers & ((1u << lane) - 1u));
    if (valid && rank == 0) cnt[warp][d] = __popc(peers);
    __syncthreads();
    if (valid) {
        int before = 0;
        for (int w = 0; w < warp; ++w) before += cnt[w][d];
        const long long pos = dbase[d] + offs[(long long)d * n_blk + blockIdx.x] + before + rank;
        key_out[pos] = kv;
        idx_out[pos] = idx_in[i];
    }
}
// leaf_start[l] = first sorted position with key >= l (l = 0..n_leaves), and the sorted, centred source records
__global__ void leaf_start_kernel(const int* __restrict__ key, long long N, int n_leaves, int* __restrict__ leaf_start) {
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l > n_leaves) return;
    long long lo = 0, hi = N;
    while (lo < hi) {
        const long long mid = (lo + hi) >> 1;
        if (key[mid] < l) lo = mid + 1; else hi = mid;
    }
    leaf_start[l] = (int)lo;
}
__global__ void gather_sorted_kernel(const double* __restrict__ xyz, const double* __restrict__ q, const int* __restrict__ idx,
                                     long long N, double hx, double hy, double hz, Src4* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const long long j = idx[i];
    out[i] = Src4{xyz[3 * j] - hx, xyz[3 * j + 1] - hy, xyz[3 * j + 2] - hz, q[j]};
}

// centre of box (ix, iy, iz) of level lev, centred coordinates
__device__ __forceinline__ void box_centre(const Geom& G, int lev, int box, double c[3], int ic[3]) {
    const int ny = grid_n(G, lev, 1), nz = grid_n(G, lev, 2);
    ic[2] = box % nz; ic[1] = (box / nz) % ny; ic[0] = box / (nz * ny);
    const double a = G.a0 / (double)(1 << lev);
#pragma unroll
    for (int k = 0; k < 3; ++k) c[k] = (ic[k] + 0.5) * a - G.half[k];
}

// inv[n * kInvW + m] = 1 / ((n+m)(n-m)) for n > m (the three-term recurrence of R_n^m in n)
__device__ __forceinline__ void fill_inv_table(double* inv, int p) {
    for (int t = threadIdx.x; t < (p + 1) * kInvW; t += blockDim.x) {
        const int n = t / kInvW, m = t % kInvW;
        inv[t] = (n > m) ? 1.0 / ((double)(n + m) * (double)(n - m)) : 0.0;
    }
}

// ---- P2M: one CTA per leaf, one lane per order m, warps share the particles --------------------------------------------
// dynamic shared memory: accw [8][nc(p)] double2, inv [(p+1) * kInvW] double
__global__ void __launch_bounds__(256) p2m_kernel(const Geom G, const Src4* __restrict__ srt, const int* __restrict__ leaf_start,
                                                  double2* __restrict__ M /* all levels */) {
    extern __shared__ __align__(16) double2 sm2[];
    const int p = G.p, NC = nc(p);
    double2* accw = sm2;
    double* inv = reinterpret_cast<double*>(sm2 + 8 * NC);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int t = tid; t < 8 * NC; t += 256) accw[t] = make_double2(0.0, 0.0);
    fill_inv_table(inv, p);
    __syncthreads();
    const int leaf = blockIdx.x;
    double c[3]; int ic[3];
    box_centre(G, G.levels, leaf, c, ic);
    const double ia = (double)(1 << G.levels) / G.a0;
    const int s0 = leaf_start[leaf], s1 = leaf_start[leaf + 1];
    double2* acc = accw + warp * NC;
    for (int j = s0 + warp; j < s1; j += 8) {
        const Src4 s = srt[j];
        const double x = (s.x - c[0]) * ia, y = (s.y - c[1]) * ia, z = (s.z - c[2]) * ia;
        const double r2 = fma(z, z, fma(y, y, x * x));
        if (lane <= p) {
            const int m = lane;
            double rr = 1.0, ri = 0.0;                     // R_m^m = prod_{i<=m} (x + i y) / (2 i)
            for (int i = 1; i <= m; ++i) {
                const double f = 0.5 / (double)i;
                const double t = (rr * x - ri * y) * f;
                ri = (rr * y + ri * x) * f;
                rr = t;
            }
            double p1r = rr, p1i = ri, p2r = 0.0, p2i = 0.0;
            double2* a = acc + cidx(m, m);
            a->x = fma(s.q, rr, a->x); a->y = fma(s.q, ri, a->y);
            for (int n = m + 1; n <= p; ++n) {
                const double f = inv[n * kInvW + m], tz = (double)(2 * n - 1) * z;
                const double cr = (tz * p1r - r2 * p2r) * f, ci = (tz * p1i - r2 * p2i) * f;
                a = acc + cidx(n, m);
                a->x = fma(s.q, cr, a->x); a->y = fma(s.q, ci, a->y);
                p2r = p1r; p2i = p1i; p1r = cr; p1i = ci;
            }
        }
    }
    __syncthreads();
    double2* out = M + (level_offset(G, G.levels) + leaf) * NC;
    for (int t = tid; t < NC; t += 256) {
        double2 v = make_double2(0.0, 0.0);
        for (int w = 0; w < 8; ++w) { v.x += accw[w * NC + t].x; v.y += accw[w * NC + t].y; }
        out[t] = v;
    }
}

// ---- M2L work decomposition (used by m2l_kernel and by l2l_kernel, which adds its partial rows) -----------------------
// Work decomposition as in the pair kernels (sum_kernels.cuh "persistent work decomposition"): the linear sequence of
// units u = group * W + w -- groups of all levels, deepest level first; W = total offset weight of a group -- is dealt
// to a persistent grid in contiguous ranges, so every CTA gets the same weight to within one offset.  A CTA writes
// one partial row per group it touches, row = CTA - first CTA of the group; l2l_kernel adds the rows in that order.
struct M2LLevel { int lev, n_groups, first_group; long long part_off; };   // part_off: this level's rows in Lpart (double2)
struct M2LArgs {
    M2LLevel lv[kMaxLevels];  // deepest level first
    int n_lv;
    int rows;                 // partial rows per group
    long long units;          // n_groups_total * W
    const int* off_list;      // [n_off] dense offset indices (g - t), |d|_inf > kWs, processing order
    const int* off_wprefix;   // [n_off + 1] prefix sums of the offset weights (how many of 8 siblings have it)
    int n_off, W;
};
__host__ __device__ inline int m2l_level_record(const M2LArgs& A, int lev) {
    for (int r = 0; r < A.n_lv; ++r) if (A.lv[r].lev == lev) return r;
    return 0;
}

// ---- plan-time tables ----------------------------------------------------------------------------------------------------
// Rsh[ch][cidx(n,m)] = R_n^m(s_ch), s_ch = ((cx,cy,cz) - 1/2) / 2 for child ch = 4 cx + 2 cy + cz: the shift from the
// parent's centre to the child's, in units of the parent's box side (M2M) -- and the same vector for L2L.
// Stab[off][cidx(N,mu)] = S_N^mu(d), N <= 2p, for the offsets d = (dx,dy,dz) in [-5,5]^3 (off = dense index); entries
// with |d|_inf <= kWs are never read (left zero).  nm[c] = (n << 8) | m.
__global__ void tables_kernel(int p, double2* __restrict__ Rsh, double2* __restrict__ Stab, int* __restrict__ nm,
                              int* __restrict__ pm, int* __restrict__ sfmap) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int NC = nc(p), NS = nc(2 * p);
    if (t < (2 * p + 1) * (2 * p + 1)) {   // expanded S table entry t = fidx(N, mu)
        int N = 0;
        while ((N + 1) * (N + 1) <= t) ++N;
        const int mu = t - N * N - N;
        sfmap[t] = (sp_index(N, mu) << 14) | (cidx(N, mu < 0 ? -mu : mu) << 2) | (mu < 0 ? ((mu & 1) ? 2 : 1) : 0);
    }
    if (t == 0) {   // output pairs (k, l0), l0 even
        int c = 0;
        for (int k = 0; k <= p; ++k)
            for (int l0 = 0; l0 <= k; l0 += 2) pm[c++] = (k << 8) | l0;
    }
    if (t < NC) {
        int n = 0;
        while (cidx(n + 1, 0) <= t) ++n;
        nm[t] = (n << 8) | (t - cidx(n, 0));
    }
    if (t < 8) {
        const double x = ((t >> 2) & 1) ? 0.25 : -0.25, y = ((t >> 1) & 1) ? 0.25 : -0.25, z = (t & 1) ? 0.25 : -0.25;
        const double r2 = x * x + y * y + z * z;
        double2* R = Rsh + t * NC;
        double rr = 1.0, ri = 0.0;
        for (int m = 0; m <= p; ++m) {
            if (m > 0) { const double f = 0.5 / m, u = (rr * x - ri * y) * f; ri = (rr * y + ri * x) * f; rr = u; }
            double p1r = rr, p1i = ri, p2r = 0.0, p2i = 0.0;
            R[cidx(m, m)] = make_double2(rr, ri);
            for (int n = m + 1; n <= p; ++n) {
                const double f = 1.0 / ((double)(n + m) * (double)(n - m)), tz = (2 * n - 1) * z;
                const double cr = (tz * p1r - r2 * p2r) * f, ci = (tz * p1i - r2 * p2i) * f;
                R[cidx(n, m)] = make_double2(cr, ci);
                p2r = p1r; p2i = p1i; p1r = cr; p1i = ci;
            }
        }
    }
    if (t < kOffN) {
        const int dx = t / (kOffW * kOffW) - kOffR, dy = (t / kOffW) % kOffW - kOffR, dz = t % kOffW - kOffR;
        double2* S = Stab + (long long)t * NS;
        const int amax = max(abs(dx), max(abs(dy), abs(dz)));
        if (amax <= kWs) {
            for (int k = 0; k < NS; ++k) S[k] = make_double2(0.0, 0.0);
            return;
        }
        const double x = dx, y = dy, z = dz, r2 = x * x + y * y + z * z, ir2 = 1.0 / r2;
        const int P2 = 2 * p;
        double sr = 1.0 / sqrt(r2), si = 0.0;           // S_m^m = (2m-1) (x + i y) / r^2 S_{m-1}^{m-1}
        for (int m = 0; m <= P2; ++m) {
            if (m > 0) { const double f = (2 * m - 1) * ir2, u = (sr * x - si * y) * f; si = (sr * y + si * x) * f; sr = u; }
            double p1r = sr, p1i = si, p2r = 0.0, p2i = 0.0;
            S[cidx(m, m)] = make_double2(sr, si);
            for (int n = m + 1; n <= P2; ++n) {
                const double tz = (2 * n - 1) * z, g = (double)(n - 1 + m) * (double)(n - 1 - m);
                const double cr = (tz * p1r - g * p2r) * ir2, ci = (tz * p1i - g * p2i) * ir2;
                S[cidx(n, m)] = make_double2(cr, ci);
                p2r = p1r; p2i = p1i; p1r = cr; p1i = ci;
            }
        }
    }
}

// ---- M2M: one CTA per parent box of level lev, one thread per coefficient ---------------------------------------------
// dynamic shared memory: Mc [8][NC], Rs [8][NC] double2
__global__ void __launch_bounds__(256) m2m_kernel(const Geom G, int lev, const double2* __restrict__ Rsh, const int* __restrict__ nm,
                                                  double2* __restrict__ M) {
    extern __shared__ __align__(16) double2 sm2[];
    const int p = G.p, NC = nc(p);
    double2* Mc = sm2;
    double2* Rs = sm2 + 8 * NC;
    const int box = blockIdx.x;
    const int ny = grid_n(G, lev, 1), nz = grid_n(G, lev, 2);
    const int iz = box % nz, iy = (box / nz) % ny, ix = box / (nz * ny);
    const int cy = grid_n(G, lev + 1, 1), cz = grid_n(G, lev + 1, 2);
    const double2* Mchild = M + level_offset(G, lev + 1) * NC;
    for (int t = threadIdx.x; t < 8 * NC; t += 256) {
        const int ch = t / NC, c = t - ch * NC;
        const int jx = 2 * ix + ((ch >> 2) & 1), jy = 2 * iy + ((ch >> 1) & 1), jz = 2 * iz + (ch & 1);
        Mc[t] = Mchild[((long long)(jx * cy + jy) * cz + jz) * NC + c];
        Rs[t] = Rsh[t];
    }
    __syncthreads();
    double2* out = M + (level_offset(G, lev) + box) * NC;
    for (int c = threadIdx.x; c < NC; c += 256) {
        const int n = nm[c] >> 8, m = nm[c] & 255;
        double2 acc = make_double2(0.0, 0.0);
        for (int ch = 0; ch < 8; ++ch) {
            const double2* R = Rs + ch * NC;
            const double2* X = Mc + ch * NC;
            for (int k = 0; k <= n; ++k) {
                const int nn = n - k;
                const double sc = ldexp(1.0, -nn);
                double2 part = make_double2(0.0, 0.0);
                const int l_lo = max(-k, m - nn), l_hi = min(k, m + nn);
                for (int l = l_lo; l <= l_hi; ++l) cfma(part, cget(R, k, l), cget(X, nn, m - l));
                acc.x = fma(sc, part.x, acc.x); acc.y = fma(sc, part.y, acc.y);
            }
        }
        out[c] = acc;
    }
}

// ---- L2L + sum of the M2L partials: one CTA per box of level lev ----------------------------------------------------------
// L[lev][box] = sum_s Lpart[s][box] (+ the parent's local expansion shifted to this box, lev > 0)
// dynamic shared memory: Lp [NC], Rs [NC] double2
__global__ void __launch_bounds__(256) l2l_kernel(const Geom G, int lev, const double2* __restrict__ Rsh, const int* __restrict__ nm,
                                                  const double2* __restrict__ Lpart, const M2LArgs A, int Gm2l,
                                                  double2* __restrict__ L) {
    extern __shared__ __align__(16) double2 sm2[];
    const int p = G.p, NC = nc(p);
    double2* Lp = sm2;
    double2* Rs = sm2 + NC;
    const int box = blockIdx.x;
    const long long nb = boxes_at(G, lev);
    long long parent = box;   // level 0: the box is its own group
    if (lev > 0) {
        const int ny = grid_n(G, lev, 1), nz = grid_n(G, lev, 2);
        const int iz = box % nz, iy = (box / nz) % ny, ix = box / (nz * ny);
        const int py = grid_n(G, lev - 1, 1), pz = grid_n(G, lev - 1, 2);
        parent = ((long long)((ix >> 1) * py + (iy >> 1))) * pz + (iz >> 1);
        const int ch = ((ix & 1) << 2) | ((iy & 1) << 1) | (iz & 1);
        const double2* Lpar = L + (level_offset(G, lev - 1) + parent) * NC;
        for (int t = threadIdx.x; t < NC; t += 256) { Lp[t] = Lpar[t]; Rs[t] = Rsh[ch * NC + t]; }
    }
    __syncthreads();
    // the M2L partial rows of this box's group: the CTAs of m2l_kernel that worked on it, in CTA order
    const M2LLevel lvr = A.lv[m2l_level_record(A, lev)];
    const long long grp = lvr.first_group + parent;
    const int n_rows = cta_of_unit((grp + 1) * A.W - 1, A.units, Gm2l) - cta_of_unit(grp * A.W, A.units, Gm2l) + 1;
    const double2* Lrows = Lpart + lvr.part_off;
    double2* out = L + (level_offset(G, lev) + box) * NC;
    for (int c = threadIdx.x; c < NC; c += 256) {
        const int n = nm[c] >> 8, m = nm[c] & 255;
        double2 acc = make_double2(0.0, 0.0);
        for (int s = 0; s < n_rows; ++s) {
            const double2 v = Lrows[((long long)s * nb + box) * NC + c];
            acc.x += v.x; acc.y += v.y;
        }
        if (lev > 0) {
            double2 sh = make_double2(0.0, 0.0);
            for (int k = n; k <= p; ++k) {
                const int dn = k - n;
                const int l_lo = max(-k, m - dn), l_hi = min(k, m + dn);
                for (int l = l_lo; l <= l_hi; ++l) {
                    const double2 r = cget(Rs, dn, l - m);
                    cfma(sh, make_double2(r.x, -r.y), cget(Lp, k, l));
                }
            }
            const double sc = ldexp(1.0, -(n + 1));
            acc.x = fma(sc, sh.x, acc.x); acc.y = fma(sc, sh.y, acc.y);
        }
        out[c] = acc;
    }
}

// ---- M2L: the translation that dominates the far field -----------------------------------------------------------------
// Unit of work = (sibling group, offset): the <= 8 children of one parent box (level 0: a single box) and one offset;
// a CTA walks a contiguous, weight-balanced range of them.  For an offset d all siblings share S(d) (staged once in shared
// memory, expanded to -N <= mu <= N) and each valid sibling has its own source box t + d (its conj M, expanded to
// -n <= m <= n with the image reflection and the cell weight applied, staged too).  Thread (k, l) keeps the 8 local
// coefficients L_k^l of the siblings in registers: per (n, m) one 128-bit read of S and one broadcast read per sibling
// feed 4 DFMA per sibling.  The CTA's partial sums go to Lpart[row][box]; l2l_kernel adds the rows in CTA order.
// Thread = two neighbouring outputs (k, l0) and (k, l0 + 1), l0 even, of all 8 siblings.  The terms m and -m of a source
// moment M_n^m = a + ib are taken together (M_n^{-m} = (-1)^m conj M_n^m):
//     conj(M_n^m) S^{l+m} + conj(M_n^{-m}) S^{l-m} = a P + b Q,   P = S^{l+m} + (-1)^m S^{l-m},  Q = -i (S^{l+m} - (-1)^m S^{l-m})
// P and Q do not depend on the sibling: 4 real FMA per sibling, output and (m, -m) pair instead of 8, and only the m >= 0
// moments are staged.  S_{n+k}^{l0+1+m} of one step is S_{n+k}^{l0+(m+1)} of the next (and the same downwards), so two
// sliding windows need two new S values per step for both outputs.  Per step and 8 siblings: 2 + 8 shared-memory
// reads, 64 DFMA.
template <int NV>
__device__ __forceinline__ void m2l_step(const double2* __restrict__ Mrow, int mstride, int m, double sgn, double2 up0, double2 up1,
                                         double2 dn0, double2 dn1, double2 (&a0)[NV], double2 (&a1)[NV]) {
    const double2 P0 = make_double2(fma(sgn, dn0.x, up0.x), fma(sgn, dn0.y, up0.y));
    const double2 P1 = make_double2(fma(sgn, dn1.x, up1.x), fma(sgn, dn1.y, up1.y));
    const double2 Q0 = make_double2(fma(-sgn, dn0.y, up0.y), fma(sgn, dn0.x, -up0.x));   // -i (up - sgn dn)
    const double2 Q1 = make_double2(fma(-sgn, dn1.y, up1.y), fma(sgn, dn1.x, -up1.x));
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const double2 mv = Mrow[i * mstride + m];
        a0[i].x = fma(mv.x, P0.x, a0[i].x); a0[i].x = fma(mv.y, Q0.x, a0[i].x);
        a0[i].y = fma(mv.x, P0.y, a0[i].y); a0[i].y = fma(mv.y, Q0.y, a0[i].y);
        a1[i].x = fma(mv.x, P1.x, a1[i].x); a1[i].x = fma(mv.y, Q1.x, a1[i].x);
        a1[i].y = fma(mv.x, P1.y, a1[i].y); a1[i].y = fma(mv.y, Q1.y, a1[i].y);
    }
}
template <int NV>
__device__ __forceinline__ void m2l_inner(const double2* __restrict__ Sfull, const double2* __restrict__ Mf, int mstride,
                                          int p, int k, int l0, double2 (&a0)[NV], double2 (&a1)[NV]) {
    for (int n = 0; n <= p; ++n) {
        const int N = n + k;
        // S_N^{l0 + j}: even j at E[j / 2], odd j at O[(j + 1) / 2]   (parity-split rows, sp_index)
        const double2* E = Sfull + N * (N + 1) + ((l0 + N + (N & 1)) >> 1);
        const double2* O = Sfull + N * (N + 1) + (N + 1) + ((l0 + N + ((N + 1) & 1) - 1) >> 1);
        const double2* Mrow = Mf + cidx(n, 0);
        double2 up0 = E[0], up1 = O[1];                  // (for the half pair l0 = k, up1 / dn1 may leave the row: unused)
        double2 dn0 = up0, dn1 = up1;
#pragma unroll
        for (int i = 0; i < NV; ++i) {                   // m = 0: M_n^0 is real
            const double a = Mrow[i * mstride].x;
            a0[i].x = fma(a, up0.x, a0[i].x); a0[i].y = fma(a, up0.y, a0[i].y);
            a1[i].x = fma(a, up1.x, a1[i].x); a1[i].y = fma(a, up1.y, a1[i].y);
        }
        for (int m = 1; m <= n; m += 2) {
            up0 = up1; up1 = E[(m + 1) >> 1]; dn1 = dn0; dn0 = O[-((m - 1) >> 1)];        // odd m
            m2l_step<NV>(Mrow, mstride, m, -1.0, up0, up1, dn0, dn1, a0, a1);
            if (m + 1 > n) break;
            up0 = up1; up1 = O[(m + 3) >> 1]; dn1 = dn0; dn0 = E[-((m + 1) >> 1)];        // even m + 1
            m2l_step<NV>(Mrow, mstride, m + 1, 1.0, up0, up1, dn0, dn1, a0, a1);
        }
    }
}

constexpr int kM2LThreads = 128;
__host__ __device__ inline int m2l_pairs(int p) {   // sum_k ceil((k+1)/2)
    int s = 0;
    for (int k = 0; k <= p; ++k) s += (k + 2) / 2;
    return s;
}
__host__ __device__ inline int m2l_smem_bytes(int p) {
    return (int)sizeof(double2) * (sp_size(p) + 8 * nc(p));
}

// pm[t] = (k << 8) | l0 of output pair t; sfmap[t] = (cidx(N, |mu|) << 2) | op for the expanded S table entry t =
// fidx(N, mu): op 0 as stored, 1 conj (mu < 0 even), 2 -conj (mu < 0 odd)
template <int NV>
__device__ __forceinline__ void m2l_add(double2 (&acc)[8], const double2 (&tmp)[NV], const int* slot_sib, int done) {
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        const int sid = slot_sib[done + i];
#pragma unroll
        for (int j = 0; j < 8; ++j) if (j == sid) { acc[j].x += tmp[i].x; acc[j].y += tmp[i].y; }
    }
}

__global__ void __launch_bounds__(kM2LThreads) m2l_kernel(const Geom G, const M2LArgs A, const double2* __restrict__ M,
                                                          const double2* __restrict__ Stab, const int* __restrict__ nm,
                                                          const int* __restrict__ pm, const int* __restrict__ sfmap,
                                                          double2* __restrict__ Lpart) {
    extern __shared__ __align__(16) double2 sm2[];
    __shared__ int sib_box[8], sib_flip[8], slot_sib[8];
    __shared__ double sib_w[8];
    __shared__ int s_nv, s_lo, s_hi;
    const int p = G.p, NC = nc(p), NS = nc(2 * p), NSF = (2 * p + 1) * (2 * p + 1), NP = m2l_pairs(p);
    double2* Sfull = sm2;
    double2* Mfull = sm2 + sp_size(p);
    const int tid = threadIdx.x;
    const int Gc = gridDim.x, kc = blockIdx.x;
    const long long u0 = unit_start(kc, A.units, Gc), u1 = unit_start(kc + 1, A.units, Gc);
    if (u1 <= u0) return;
    for (int t = tid; t < sp_size(p); t += kM2LThreads) Sfull[t] = make_double2(0.0, 0.0);   // (pads and unused slots)
    for (long long grp = u0 / A.W; grp <= (u1 - 1) / A.W; ++grp) {
        int r = 0;
        while (r + 1 < A.n_lv && grp >= A.lv[r + 1].first_group) ++r;
        const M2LLevel lv = A.lv[r];
        const int group = (int)(grp - lv.first_group);
        const int row = kc - cta_of_unit(grp * A.W, A.units, Gc);
        const int lev = lv.lev;
        const int nsib = lev == 0 ? 1 : 8;
        int P[3];   // parent coordinates (level 0: the box itself)
        {
            const int gl = lev == 0 ? 0 : lev - 1;
            const int gy = grid_n(G, gl, 1), gz = grid_n(G, gl, 2);
            P[2] = group % gz; P[1] = (group / gz) % gy; P[0] = group / (gz * gy);
        }
        __syncthreads();
        if (tid == 0) {   // this CTA's share of the group's offsets, by weight: offsets whose prefix start lies in [w_lo, w_hi)
            const long long w_lo = max(u0, grp * A.W) - grp * A.W, w_hi = min(u1, (grp + 1) * A.W) - grp * A.W;
            int lo = 0, hi = A.n_off;
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (A.off_wprefix[mid] < w_lo) lo = mid + 1; else hi = mid; }
            s_lo = lo;
            lo = 0; hi = A.n_off;
            while (lo < hi) { const int mid = (lo + hi) >> 1; if (A.off_wprefix[mid] < w_hi) lo = mid + 1; else hi = mid; }
            s_hi = lo;
        }
        __syncthreads();
        const int o_lo = s_lo, o_hi = s_hi;
        const long long nb = boxes_at(G, lev);
        const double2* Mlev = M + level_offset(G, lev) * NC;
        const int ny = grid_n(G, lev, 1), nz = grid_n(G, lev, 2);

        for (int c0 = 0; c0 < NP; c0 += kM2LThreads) {
            const int c = c0 + tid;
            const bool have = c < NP;
            const int k = have ? (pm[c] >> 8) : 0, l0 = have ? (pm[c] & 255) : 0;
            double2 acc0[8], acc1[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) { acc0[i] = make_double2(0.0, 0.0); acc1[i] = make_double2(0.0, 0.0); }
            for (int oi = o_lo; oi < o_hi; ++oi) {
                const int off = A.off_list[oi];
                const int dx = off / (kOffW * kOffW) - kOffR, dy = (off / kOffW) % kOffW - kOffR, dz = off % kOffW - kOffR;
                __syncthreads();   // the previous offset's reads of Sfull / Mfull / sib_* are done
                if (tid < 32) {
                    bool ok = false;
                    ImageBox ib;
                    if (tid < nsib) {
                        const int t[3] = {lev == 0 ? P[0] : 2 * P[0] + ((tid >> 2) & 1), lev == 0 ? P[1] : 2 * P[1] + ((tid >> 1) & 1),
                                          lev == 0 ? P[2] : 2 * P[2] + (tid & 1)};
                        const int g[3] = {t[0] + dx, t[1] + dy, t[2] + dz};
                        ok = true;
                        if (lev > 0)   // the source's parent must be within kWs of the target's parent
                            for (int a = 0; a < 3; ++a) ok = ok && g[a] >= 2 * (P[a] - kWs) && g[a] <= 2 * (P[a] + kWs) + 1;
                        ok = ok && image_box(G, lev, g[0], g[1], g[2], ib);
                    }
                    const unsigned mask = __ballot_sync(0xffffffffu, ok);
                    if (ok) {
                        const int slot = __popc(mask & ((1u << tid) - 1u));
                        sib_box[slot] = ib.box; sib_flip[slot] = ib.fx | (ib.fy << 1) | (ib.fz << 2); sib_w[slot] = ib.w;
                        slot_sib[slot] = tid;
                    }
                    if (tid == 0) s_nv = __popc(mask);
                }
                __syncthreads();
                const int nv = s_nv;
                if (nv == 0) continue;
                // S(t - g) = S(-d), expanded to negative orders
                const double2* S = Stab + (long long)(((kOffR - dx) * kOffW + (kOffR - dy)) * kOffW + (kOffR - dz)) * NS;
                for (int t = tid; t < NSF; t += kM2LThreads) {
                    const int e = sfmap[t];
                    double2 v = S[(e >> 2) & 4095];
                    if (e & 1) v.y = -v.y;
                    if (e & 2) { v.x = -v.x; }
                    Sfull[e >> 14] = v;
                }
                // the (reflected, weighted) source moments of the valid siblings, m >= 0
                for (int t = tid; t < nv * NC; t += kM2LThreads) {
                    const int sl = t / NC, cc = t - sl * NC;
                    const int fl = sib_flip[sl];
                    const double w = sib_w[sl];
                    const int n = nm[cc] >> 8, m = nm[cc] & 255;
                    double2 v = Mlev[(long long)sib_box[sl] * NC + cc];
                    if (fl & 1) v = (m & 1) ? make_double2(-v.x, v.y) : make_double2(v.x, -v.y);   // x: (-1)^m conj
                    if (fl & 2) v.y = -v.y;                                                         // y: conj
                    if ((fl & 4) && ((n + m) & 1)) { v.x = -v.x; v.y = -v.y; }                      // z: (-1)^(n+m)
                    Mfull[t] = make_double2(v.x * w, v.y * w);
                }
                __syncthreads();
                int done = 0;
                while (done < nv) {
                    const int left = nv - done;
                    const double2* Mf = Mfull + done * NC;
                    if (left >= 8) {
                        m2l_inner<8>(Sfull, Mf, NC, p, k, l0, acc0, acc1);   // all eight siblings: slot i is sibling i
                        done += 8;
                    } else if (left >= 4) {
                        double2 t0[4], t1[4];
#pragma unroll
                        for (int i = 0; i < 4; ++i) { t0[i] = make_double2(0.0, 0.0); t1[i] = make_double2(0.0, 0.0); }
                        m2l_inner<4>(Sfull, Mf, NC, p, k, l0, t0, t1);
                        m2l_add<4>(acc0, t0, slot_sib, done); m2l_add<4>(acc1, t1, slot_sib, done);
                        done += 4;
                    } else if (left >= 2) {
                        double2 t0[2], t1[2];
#pragma unroll
                        for (int i = 0; i < 2; ++i) { t0[i] = make_double2(0.0, 0.0); t1[i] = make_double2(0.0, 0.0); }
                        m2l_inner<2>(Sfull, Mf, NC, p, k, l0, t0, t1);
                        m2l_add<2>(acc0, t0, slot_sib, done); m2l_add<2>(acc1, t1, slot_sib, done);
                        done += 2;
                    } else {
                        double2 t0[1], t1[1];
                        t0[0] = make_double2(0.0, 0.0); t1[0] = make_double2(0.0, 0.0);
                        m2l_inner<1>(Sfull, Mf, NC, p, k, l0, t0, t1);
                        m2l_add<1>(acc0, t0, slot_sib, done); m2l_add<1>(acc1, t1, slot_sib, done);
                        done += 1;
                    }
                }
            }
            if (have) {
                const double sg = (k & 1) ? -1.0 : 1.0;
                const int cc = cidx(k, l0);
#pragma unroll
                for (int sI = 0; sI < 8; ++sI) {
                    if (sI < nsib) {
                        const int tx = lev == 0 ? P[0] : 2 * P[0] + ((sI >> 2) & 1), ty = lev == 0 ? P[1] : 2 * P[1] + ((sI >> 1) & 1),
                                  tz = lev == 0 ? P[2] : 2 * P[2] + (sI & 1);
                        const long long box = ((long long)tx * ny + ty) * nz + tz;
                        double2* o = Lpart + lv.part_off + ((long long)row * nb + box) * NC + cc;
                        o[0] = make_double2(sg * acc0[sI].x, sg * acc0[sI].y);
                        if (l0 + 1 <= k) o[1] = make_double2(sg * acc1[sI].x, sg * acc1[sI].y);
                    }
                }
            }
        }
    }   // groups of this CTA
}

// ---- leaves: L2P + P2P --------------------------------------------------------------------------------------------------
// One CTA of 64 threads per chunk of a leaf: up to 4 rows of 64 targets, i.e. a thread owns R <= 4 targets of ONE leaf
// in registers (every smem read of a source feeds R pairs), and the number of rows follows the leaf population, so
// the lanes are full whatever it is (534 targets = 9 rows = chunks of 4 + 4 + 1).  The leaf's
// local expansion is evaluated at the targets (L2P), then the 5^3 neighbour boxes -- images through the near cell table,
// never materialised -- are summed directly (P2P) from 256-source tiles in shared memory with the pair arithmetic of
// near_sum_kernel: the target is moved into the image's frame, sigma o (t - kL); only the bare self term (central
// cell, same particle) is masked.
// dynamic shared memory: Ls [NC] double2, inv [(p+1) * kInvW] double
constexpr int kLeafThreads = 64;
constexpr int kLeafTile = 128;
constexpr int kLeafR = 4;      // rows of kLeafThreads targets per chunk (targets per thread)

// FIELD: also the gradient (forces): out[comp * N + i], comp 0 = phi, 1..3 = grad phi.  The gradient of
// the local expansion uses d/dz R_n^m = R_{n-1}^m, (d/dx + i d/dy) conj R_n^m = conj R_{n-1}^{m-1}:
//   dPsi/dz = sum_k [R_k^0 L_{k+1}^0 + 2 Re sum_{j>=1} conj R_k^j L_{k+1}^j]
//   dPsi/dx + i dPsi/dy = sum_k [sum_{j>=0} conj R_k^j L_{k+1}^{j+1} - sum_{j>=1} R_k^j conj L_{k+1}^{j-1}]
// (checked against finite differences before this was written); the P2P part uses pair_field of sum_kernels.cuh.
template <int REFINE, int R, bool FIELD>
__device__ __forceinline__ void leaf_round(const Geom& G, const int ic[3], const double c[3], const Src4* __restrict__ srt,
                                           const int* __restrict__ idx, const int* __restrict__ leaf_start, int t0, int t1,
                                           Src4* tile, const double2* Ls, const double* inv, long long N, int dx_slab,
                                           double* __restrict__ phi_out /* this slab's [comps][N] */) {
    constexpr int RG = FIELD ? R : 1;
    const int p = G.p, lev = G.levels, tid = threadIdx.x;
    const double ia = (double)(1 << lev) / G.a0;
    const double scale = REFINE == 1 ? 0.5 : 1.0, scale_grad = REFINE == 1 ? -0.125 : -1.0;
    double total[R], totx[RG], toty[RG], totz[RG];
#pragma unroll
    for (int r = 0; r < R; ++r) { total[r] = 0.0; if (FIELD) { totx[r % RG] = 0.0; toty[r % RG] = 0.0; totz[r % RG] = 0.0; } }
    // L2P: (1/a) Re sum conj R_n^m L_n^m, m < 0 folded in (factor 2) -- by the slab dx = 0 only
#pragma unroll 1
    for (int r = 0; r < (dx_slab == 0 ? R : 0); ++r) {
        const Src4 t = srt[min(t0 + r * kLeafThreads + tid, t1 - 1)];
        const double x = (t.x - c[0]) * ia, y = (t.y - c[1]) * ia, z = (t.z - c[2]) * ia;
        const double r2 = fma(z, z, fma(y, y, x * x));
        double rr = 1.0, ri = 0.0, far = 0.0, gpr = 0.0, gpi = 0.0, gz = 0.0;
        for (int m = 0; m <= p; ++m) {
            if (m > 0) { const double f = 0.5 / (double)m, u = (rr * x - ri * y) * f; ri = (rr * y + ri * x) * f; rr = u; }
            double p1r = rr, p1i = ri, p2r = 0.0, p2i = 0.0;
            double s = 0.0, sz = 0.0;
            for (int n = m; n <= p; ++n) {
                double cr, ci;
                if (n == m) { cr = rr; ci = ri; }
                else {
                    const double f = inv[n * kInvW + m], tz = (double)(2 * n - 1) * z;
                    cr = (tz * p1r - r2 * p2r) * f; ci = (tz * p1i - r2 * p2i) * f;
                    p2r = p1r; p2i = p1i; p1r = cr; p1i = ci;
                }
                const double2 lc = Ls[cidx(n, m)];
                s = fma(cr, lc.x, s); s = fma(ci, lc.y, s);
                if (FIELD && n < p) {
                    const double2 lz = Ls[cidx(n + 1, m)], lp = Ls[cidx(n + 1, m + 1)];
                    sz = fma(cr, lz.x, sz); sz = fma(ci, lz.y, sz);
                    gpr = fma(cr, lp.x, gpr); gpr = fma(ci, lp.y, gpr);      // conj(R) L^{m+1}
                    gpi = fma(cr, lp.y, gpi); gpi = fma(-ci, lp.x, gpi);
                    if (m >= 1) {                                            // - R conj(L^{m-1})
                        const double2 lm = Ls[cidx(n + 1, m - 1)];
                        gpr = fma(-cr, lm.x, gpr); gpr = fma(-ci, lm.y, gpr);
                        gpi = fma(-ci, lm.x, gpi); gpi = fma(cr, lm.y, gpi);
                    }
                }
            }
            far += m == 0 ? s : 2.0 * s;
            if (FIELD) gz += m == 0 ? sz : 2.0 * sz;
        }
        // (dynamic index into a register array would spill: select)
#pragma unroll
        for (int k = 0; k < R; ++k) if (k == r) {
            total[k] = far * ia;
            if (FIELD) { totx[k % RG] = gpr * ia * ia; toty[k % RG] = gpi * ia * ia; totz[k % RG] = gz * ia * ia; }
        }
    }
    Src4 me[R];
    int pos[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        pos[r] = min(t0 + r * kLeafThreads + tid, t1 - 1);   // slots past the end repeat the last target and do not store
        me[r] = srt[pos[r]];
    }
    {
        const int dx = dx_slab;
        for (int dy = -kWs; dy <= kWs; ++dy)
            for (int dz = -kWs; dz <= kWs; ++dz) {
                ImageBox ib;
                if (!image_box(G, lev, ic[0] + dx, ic[1] + dy, ic[2] + dz, ib)) continue;
                const int s0 = leaf_start[ib.box], s1 = leaf_start[ib.box + 1];
                if (s0 == s1) continue;
                double tx[R], ty[R], tz[R], acc[R], gx[RG], gy[RG], gz[RG];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    tx[r] = flip(me[r].x - ib.sx, ib.fx); ty[r] = flip(me[r].y - ib.sy, ib.fy); tz[r] = flip(me[r].z - ib.sz, ib.fz);
                    acc[r] = 0.0;
                    if (FIELD) { gx[r % RG] = 0.0; gy[r % RG] = 0.0; gz[r % RG] = 0.0; }
                }
                const bool self_here = ib.central && dx == 0 && dy == 0 && dz == 0;
                for (int base = s0; base < s1; base += kLeafTile) {
                    __syncthreads();
#pragma unroll
                    for (int h = 0; h < kLeafTile / kLeafThreads; ++h) {
                        const int j = base + h * kLeafThreads + tid;
                        tile[h * kLeafThreads + tid] = j < s1 ? srt[j] : Src4{kFar, kFar, kFar, 0.0};
                    }
                    __syncthreads();
                    const int cnt = min(kLeafTile, s1 - base);
                    if (self_here) {
#pragma unroll 1
                        for (int j = 0; j < cnt; ++j) {
                            const double2 xy = *reinterpret_cast<const double2*>(&tile[j].x);
                            const double2 zq = *reinterpret_cast<const double2*>(&tile[j].z);
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                const bool self = base + j == pos[r];
                                if (FIELD)
                                    pair_field<REFINE, 0>(tx[r], ty[r], tz[r], self ? tx[r] + 1.0 : xy.x, self ? ty[r] : xy.y,
                                                          self ? tz[r] : zq.x, self ? 0.0 : zq.y, acc[r], gx[r % RG], gy[r % RG], gz[r % RG]);
                                else
                                    pair<REFINE>(tx[r], ty[r], tz[r], self ? tx[r] + 1.0 : xy.x, self ? ty[r] : xy.y, self ? tz[r] : zq.x,
                                                 self ? 0.0 : zq.y, acc[r]);
                            }
                        }
                    } else {
#pragma unroll 2
                        for (int j = 0; j < cnt; ++j) {
                            const double2 xy = *reinterpret_cast<const double2*>(&tile[j].x);
                            const double2 zq = *reinterpret_cast<const double2*>(&tile[j].z);
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                if (FIELD) pair_field<REFINE, 0>(tx[r], ty[r], tz[r], xy.x, xy.y, zq.x, zq.y, acc[r], gx[r % RG], gy[r % RG], gz[r % RG]);
                                else pair<REFINE>(tx[r], ty[r], tz[r], xy.x, xy.y, zq.x, zq.y, acc[r]);
                            }
                        }
                    }
                }
                const double w = ib.w * scale, wg = ib.w * scale_grad;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    total[r] = fma(w, acc[r], total[r]);
                    if (FIELD) {   // the pair loop ran in the frame of the transformed target: a reflected axis flips back
                        totx[r % RG] = fma(wg, flip(gx[r % RG], ib.fx), totx[r % RG]);
                        toty[r % RG] = fma(wg, flip(gy[r % RG], ib.fy), toty[r % RG]);
                        totz[r % RG] = fma(wg, flip(gz[r % RG], ib.fz), totz[r % RG]);
                    }
                }
            }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int t = t0 + r * kLeafThreads + tid;
        if (t < t1) {
            const long long i = idx[t];
            phi_out[i] = total[r];
            if (FIELD) { phi_out[N + i] = totx[r % RG]; phi_out[2 * N + i] = toty[r % RG]; phi_out[3 * N + i] = totz[r % RG]; }
        }
    }
}

// chunk_start[l] = number of chunks of the leaves before l (a chunk = up to kLeafR rows of kLeafThreads targets of one
// leaf); chunk_start[n_leaves] = total.  Single block.
__global__ void __launch_bounds__(1024) leaf_chunks_kernel(const int* __restrict__ leaf_start, int n_leaves, int* __restrict__ chunk_start) {
    __shared__ int wsum[32];
    __shared__ int carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < n_leaves; base += 1024) {
        const int l = base + threadIdx.x;
        const int n = l < n_leaves ? leaf_start[l + 1] - leaf_start[l] : 0;
        const int v = (n + kLeafThreads * kLeafR - 1) / (kLeafThreads * kLeafR);
        int x = v;
        for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
        if (lane == 31) wsum[warp] = x;
        __syncthreads();
        if (warp == 0) {
            int w = wsum[lane];
            for (int o = 1; o < 32; o <<= 1) { const int y = __shfl_up_sync(0xffffffffu, w, o); if (lane >= o) w += y; }
            wsum[lane] = w;
        }
        __syncthreads();
        if (l < n_leaves) chunk_start[l] = carry + (warp > 0 ? wsum[warp - 1] : 0) + x - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += wsum[31];
        __syncthreads();
    }
    if (threadIdx.x == 0) chunk_start[n_leaves] = carry;
}

// grid: an upper bound of the number of chunks (N / (kLeafThreads * kLeafR) + n_leaves); surplus CTAs return
template <int REFINE, bool FIELD>
__global__ void __launch_bounds__(kLeafThreads) leaf_kernel(const Geom G, const Src4* __restrict__ srt, const int* __restrict__ idx,
                                                            const int* __restrict__ leaf_start, const int* __restrict__ chunk_start,
                                                            int n_leaves, const double2* __restrict__ L, long long N,
                                                            double* __restrict__ slab_out /* [2 kWs + 1][comps][N] */) {
    extern __shared__ __align__(16) double2 sm2[];
    __shared__ __align__(16) Src4 tile[kLeafTile];
    const int p = G.p, NC = nc(p), lev = G.levels;
    double2* Ls = sm2;
    double* inv = reinterpret_cast<double*>(sm2 + NC);
    const int b = blockIdx.x;
    if (b >= chunk_start[n_leaves]) return;
    int lo = 0, hi = n_leaves - 1;   // the leaf with chunk_start[leaf] <= b < chunk_start[leaf + 1]
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (chunk_start[mid] <= b) lo = mid; else hi = mid - 1;
    }
    const int leaf = lo;
    const int s1 = leaf_start[leaf + 1];
    const int t0 = leaf_start[leaf] + (b - chunk_start[leaf]) * (kLeafThreads * kLeafR);
    const int t1 = min(s1, t0 + kLeafThreads * kLeafR);
    fill_inv_table(inv, p);
    const double2* Lleaf = L + (level_offset(G, lev) + leaf) * NC;
    for (int t = threadIdx.x; t < NC; t += kLeafThreads) Ls[t] = Lleaf[t];
    double c[3]; int ic[3];
    box_centre(G, lev, leaf, c, ic);
    __syncthreads();
    // blockIdx.y = the slab dx of the 5 x 5 x 5 neighbour boxes this CTA sums (five times more, five times shorter CTAs:
    // the tail of the launch shrinks accordingly); each slab writes its own partial row, leaf_sum_kernel adds them in order
    const int dx_slab = (int)blockIdx.y - kWs;
    double* phi_out = slab_out + (long long)blockIdx.y * (FIELD ? 4 : 1) * N;
    const int R = (t1 - t0 + kLeafThreads - 1) / kLeafThreads;
    switch (R) {
        case 1: leaf_round<REFINE, 1, FIELD>(G, ic, c, srt, idx, leaf_start, t0, t1, tile, Ls, inv, N, dx_slab, phi_out); break;
        case 2: leaf_round<REFINE, 2, FIELD>(G, ic, c, srt, idx, leaf_start, t0, t1, tile, Ls, inv, N, dx_slab, phi_out); break;
        case 3: leaf_round<REFINE, 3, FIELD>(G, ic, c, srt, idx, leaf_start, t0, t1, tile, Ls, inv, N, dx_slab, phi_out); break;
        default: leaf_round<REFINE, 4, FIELD>(G, ic, c, srt, idx, leaf_start, t0, t1, tile, Ls, inv, N, dx_slab, phi_out); break;
    }
}

// out[c][i] = sum over the slabs, in slab order
__global__ void leaf_sum_kernel(const double* __restrict__ slab, long long n /* comps * N */, double* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double v = 0.0;
#pragma unroll
    for (int sl = 0; sl < 2 * kWs + 1; ++sl) v += slab[(long long)sl * n + i];
    out[i] = v;
}

// ---- step (a) from the same hierarchy: the near sum at arbitrary points (the check targets) --------------------------------
// A check target x may lie outside the central cell (the circumsphere points of PAPER.md:80-82), where no local
// expansion exists; it is served by the MULTIPOLES directly (M2P): with b_l the box of level l that contains x (global
// grid coordinates, any cell), the boxes of b_l's interaction list -- parent within kWs of b_l's parent, more than
// kWs away from b_l; at level 0 every box of the cell table more than kWs away -- are evaluated as
//     phi += (1/a) Re sum_{n,m} conj M_n^m S_n^m((x' - c)/a),      x' = sigma o (x - kL)
// (the target is moved into the frame of the image, as in the pair kernels, so the central box's moments serve
// unreflected), and the leaf boxes within kWs of b_lmax are summed directly.  Same separation and order as M2L, hence
// the same truncation error.  One CTA per target; the threads share the boxes; fixed-order tree reduction.
constexpr int kM2PThreads = 128;

// A target INSIDE the central cell has a leaf with a local expansion: its far field is one L2P (231 terms, the orders m
// shared among the threads) instead of ~2,700 M2P.
// dynamic shared memory: Ls [NC] double2, inv [(p+1) * kInvW] double
__global__ void __launch_bounds__(kM2PThreads) m2p_points_kernel(const Geom G, const double* __restrict__ tgt /* [T,3] centred */,
                                                                 const Src4* __restrict__ srt, const int* __restrict__ leaf_start,
                                                                 const double2* __restrict__ M, const double2* __restrict__ L,
                                                                 double* __restrict__ phi_out) {
    __shared__ double red[kM2PThreads];
    extern __shared__ __align__(16) double2 sm2[];
    const int p = G.p, NC = nc(p), lmax = G.levels, tid = threadIdx.x;
    const double x = tgt[3 * (size_t)blockIdx.x], y = tgt[3 * (size_t)blockIdx.x + 1], z = tgt[3 * (size_t)blockIdx.x + 2];
    const double xc[3] = {x, y, z};
    int gl[3];   // leaf-level box of the target, global coordinates
#pragma unroll
    for (int a = 0; a < 3; ++a) gl[a] = (int)floor((xc[a] + G.half[a]) * (double)(1 << lmax) / G.a0);
    double acc = 0.0;
    bool inside = true;
#pragma unroll
    for (int a = 0; a < 3; ++a) inside = inside && gl[a] >= 0 && gl[a] < grid_n(G, lmax, a);
    if (inside) {   // far field = the leaf's local expansion: thread m takes the order m
        double2* Ls = sm2;
        double* inv = reinterpret_cast<double*>(sm2 + NC);
        const int leaf = (gl[0] * grid_n(G, lmax, 1) + gl[1]) * grid_n(G, lmax, 2) + gl[2];
        const double2* Lleaf = L + (level_offset(G, lmax) + leaf) * NC;
        for (int t = tid; t < NC; t += kM2PThreads) Ls[t] = Lleaf[t];
        fill_inv_table(inv, p);
        __syncthreads();
        if (tid <= p) {
            double c[3]; int ic[3];
            box_centre(G, lmax, leaf, c, ic);
            const double ia = (double)(1 << lmax) / G.a0;
            const double rx = (x - c[0]) * ia, ry = (y - c[1]) * ia, rz = (z - c[2]) * ia;
            const double r2 = fma(rz, rz, fma(ry, ry, rx * rx));
            const int m = tid;
            double rr = 1.0, ri = 0.0;
            for (int i = 1; i <= m; ++i) { const double f = 0.5 / (double)i, u = (rr * rx - ri * ry) * f; ri = (rr * ry + ri * rx) * f; rr = u; }
            double p1r = rr, p1i = ri, p2r = 0.0, p2i = 0.0;
            double2 lc = Ls[cidx(m, m)];
            double s = fma(rr, lc.x, ri * lc.y);
            for (int n = m + 1; n <= p; ++n) {
                const double f = inv[n * kInvW + m], tz = (double)(2 * n - 1) * rz;
                const double cr = (tz * p1r - r2 * p2r) * f, ci = (tz * p1i - r2 * p2i) * f;
                lc = Ls[cidx(n, m)];
                s = fma(cr, lc.x, s); s = fma(ci, lc.y, s);
                p2r = p1r; p2i = p1i; p1r = cr; p1i = ci;
            }
            acc = (m == 0 ? s : 2.0 * s) * ia;
        }
    }
    // far field of a target outside the central cell: multipoles of the interaction lists, all levels
    for (int lev = inside ? -1 : lmax; lev >= 0; --lev) {
        const int sh = lmax - lev;
        const int b[3] = {gl[0] >> sh, gl[1] >> sh, gl[2] >> sh};
        int R[3];   // candidate offsets |d_a| <= R_a
#pragma unroll
        for (int a = 0; a < 3; ++a) R[a] = lev > 0 ? kOffR : (2 * G.shell[a] + 1) * G.base[a] - 1;
        const int wx = 2 * R[0] + 1, wy = 2 * R[1] + 1, wz = 2 * R[2] + 1;
        const double al = G.a0 / (double)(1 << lev), ial = 1.0 / al;
        const double2* Mlev = M + level_offset(G, lev) * NC;
        for (int o = tid; o < wx * wy * wz; o += kM2PThreads) {
            const int dx = o / (wy * wz) - R[0], dy = (o / wz) % wy - R[1], dz = o % wz - R[2];
            if (max(abs(dx), max(abs(dy), abs(dz))) <= kWs) continue;
            const int g[3] = {b[0] + dx, b[1] + dy, b[2] + dz};
            bool ok = true;
            if (lev > 0)
#pragma unroll
                for (int a = 0; a < 3; ++a) { const int P = b[a] >> 1; ok = ok && g[a] >= 2 * (P - kWs) && g[a] <= 2 * (P + kWs) + 1; }
            ImageBox ib;
            if (!ok || !image_box(G, lev, g[0], g[1], g[2], ib)) continue;
            double c[3]; int ic[3];
            box_centre(G, lev, ib.box, c, ic);
            // target in the image's frame, relative to the central box's centre, in box units
            const double rx = (flip(x - ib.sx, ib.fx) - c[0]) * ial, ry = (flip(y - ib.sy, ib.fy) - c[1]) * ial,
                         rz = (flip(z - ib.sz, ib.fz) - c[2]) * ial;
            const double r2 = fma(rz, rz, fma(ry, ry, rx * rx)), ir2 = 1.0 / r2;
            const double2* Mb = Mlev + (long long)ib.box * NC;
            double sr = rsqrt_cubic(r2), si = 0.0, sum = 0.0;      // S_0^0 = 1/r
            for (int m = 0; m <= p; ++m) {
                if (m > 0) { const double f = (double)(2 * m - 1) * ir2, u = (sr * rx - si * ry) * f; si = (sr * ry + si * rx) * f; sr = u; }
                double p1r = sr, p1i = si, p2r = 0.0, p2i = 0.0;
                double2 mc = Mb[cidx(m, m)];
                double s = fma(mc.x, sr, mc.y * si);
                for (int n = m + 1; n <= p; ++n) {
                    const double tz = (double)(2 * n - 1) * rz, gg = (double)(n - 1 + m) * (double)(n - 1 - m);
                    const double cr = (tz * p1r - gg * p2r) * ir2, ci = (tz * p1i - gg * p2i) * ir2;
                    mc = Mb[cidx(n, m)];
                    s = fma(mc.x, cr, s); s = fma(mc.y, ci, s);
                    p2r = p1r; p2i = p1i; p1r = cr; p1i = ci;
                }
                sum += m == 0 ? s : 2.0 * s;
            }
            acc = fma(ib.w * ial, sum, acc);
        }
    }
    // near field: the leaf boxes within kWs, pair by pair (cubic refinement: step (a) feeds the fit)
    for (int o = 0; o < (2 * kWs + 1) * (2 * kWs + 1) * (2 * kWs + 1); ++o) {
        const int dx = o / 25 - kWs, dy = (o / 5) % 5 - kWs, dz = o % 5 - kWs;
        ImageBox ib;
        if (!image_box(G, lmax, gl[0] + dx, gl[1] + dy, gl[2] + dz, ib)) continue;
        const int s0 = leaf_start[ib.box], s1 = leaf_start[ib.box + 1];
        const double tx = flip(x - ib.sx, ib.fx), ty = flip(y - ib.sy, ib.fy), tz = flip(z - ib.sz, ib.fz);
        double a2 = 0.0;
        for (int j = s0 + tid; j < s1; j += kM2PThreads) {
            const Src4 s = srt[j];
            pair<2>(tx, ty, tz, s.x, s.y, s.z, s.q, a2);
        }
        acc = fma(ib.w, a2, acc);
    }
    red[tid] = acc;
    __syncthreads();
    for (int o = kM2PThreads / 2; o > 0; o >>= 1) {
        if (tid < o) red[tid] += red[tid + o];
        __syncthreads();
    }
    if (tid == 0) phi_out[blockIdx.x] = red[0];
}

}  // namespace fmm
}  // namespace hsma
