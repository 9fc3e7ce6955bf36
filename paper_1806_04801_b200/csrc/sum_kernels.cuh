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

// ---- persistent work decomposition ------------------------------------------
// The work of one launch is the linear sequence of units u = (target block b, source tile t, cell c),
// cell fastest: u = (b * n_tiles + t) * C + c, U units in all.  The grid is persistent: G CTAs (one
// wave: resident CTAs per SM x SMs), CTA k owns the contiguous range [unit_start(k), unit_start(k+1)),
// so every CTA gets U/G units to within one unit and there is no tail wave.  A target block is covered by
// a few consecutive CTAs; each writes its partial sums to row (k - first CTA of the block) of `part`,
// and finish_phi_kernel adds the rows in that fixed order (no atomics: bit-reproducible).
__host__ __device__ inline long long unit_start(long long k, long long U, int G) { return (k * U) / G; }
__host__ __device__ inline int cta_of_unit(long long u, long long U, int G) {
    long long k = (u * G) / U;
    while (k + 1 < G && unit_start(k + 1, U, G) <= u) ++k;
    while (k > 0 && unit_start(k, U, G) > u) --k;
    return (int)k;
}
// rows of `part` that are enough for any block: CTAs overlapping an interval of Ub units
__host__ __device__ inline int part_rows(long long U, long long Ub, int G) {
    const long long per = U / G > 0 ? U / G : 1;
    return (int)(Ub / per + 2);
}

struct PartLayout {      // how finish_phi_kernel finds the partial rows of one pair kernel
    const double* part;  // [rows][T], or nullptr
    long long U, Ub;     // units in all / per target block
    int G;               // CTAs of the launch
    int block_targets;   // targets per block (kThreads * R)
    // sphere-culled near set: the source count lives on the device (dyn[1] = source tiles), Ub = dyn[1] * cells
    const long long* dyn = nullptr;
    int cells = 1;
};
// units per block / in all of a layout whose source count is device-resident
__device__ __forceinline__ void layout_units(const PartLayout& L, long long T, long long& U, long long& Ub) {
    U = L.U; Ub = L.Ub;
    if (L.dyn) {
        Ub = L.dyn[1] * L.cells;
        U = ((T + L.block_targets - 1) / L.block_targets) * Ub;
    }
}

struct QInfo { double qmag; int uniform; int pad; };  // all |q| equal to qmag (charge_stats_kernel)

struct NearArgs {
    const double* tgt;   // targets, `tstride` doubles apart (3 = xyz rows, 4 = packed Src4 rows)
    int tstride;
    long long T;         // number of targets
    long long t_first;   // target t is row tgt_index[t_first + t] of tgt (row t_first + t if tgt_index is null)
    const int* tgt_index;
    const Src4* src;     // packed by pack_sources_kernel: tiles of kTile records, sign-sorted, padded with q = 0 at kFar
    long long n_src;     // valid sources
    long long n_tiles;   // padded source count / kTile
    const int* tile_np;  // [n_tiles] sources with q >= 0 at the front of each tile
    const int* slot_of;  // [n_src] packed index of source i (needed only for the self exclusion)
    const QInfo* qinfo;  // null: always multiply by q
    const Cell* cells;   // [C]
    int C;
    long long units;     // U = ntb * n_tiles * C
    // sphere-culled near set: the image list is built on the device and its length never visits the host.  dyn[0] =
    // sources, dyn[1] = source tiles replace n_src / n_tiles, and units = ntb * dyn[1] * C (null: the values above)
    const long long* dyn;
    long long ntb;
    long long self_offset;  // >= 0: target t is source (self_offset + t); its bare term is skipped
    double scale;        // applied to the cell weights (0.5 for the Newton form, see below)
    double scale_grad;   // FIELD: weight of the gradient sums (-1/8 Newton, -1 cubic)
    double* part;        // [part_rows][T] partial sums ([part_rows][4][T] in the FIELD form)
};

// One pair: acc += q / |d|.
//  REFINE 1: y0 = seed; q*y = (q*y0) * (kNewton3 - r2*y0^2) / 2  (one Newton step; the 1/2 lives in `scale`)
//            -> 3 DADD + DMUL + 2 DFMA (r2) + MUFU + DMUL + DMUL + DFMA + DFMA = 10 FP64-pipe instructions
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

// The same pair with the charge factored out (all |q| equal, tiles sign-sorted): acc += y or acc -= y.
//  REFINE 1: 3 DADD + DMUL + 2 DFMA + MUFU + DMUL + DFMA + DFMA = 9 FP64-pipe instructions (the negation is
//  an operand modifier); REFINE 2: 11.
template <int REFINE, bool NEG>
__device__ __forceinline__ void pair_unit(double tx, double ty, double tz, double sx, double sy, double sz, double& acc) {
    const double dx = tx - sx, dy = ty - sy, dz = tz - sz;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double y0 = rsqrt_seed(r2);
    const double t = y0 * y0;
    if (REFINE == 1) {
        const double g = fma(-r2, t, kNewton3);
        acc = NEG ? fma(-y0, g, acc) : fma(y0, g, acc);
    } else {
        const double e = fma(-r2, t, 1.0);
        const double h = fma(e, 0.375, 0.5);
        const double k = fma(e, h, 1.0);
        acc = NEG ? fma(-y0, k, acc) : fma(y0, k, acc);
    }
}

// Potential AND gradient (forces, Eq.(9)): with a = 2y (Newton) or y (cubic),
//   phi += s q a,   G += s q a^3 d   (d = t - source; grad_t q/|d| = -q d/|d|^3: the sign and the powers of 2
//   live in the cell weights).  SIGN 0: multiply by q (generic), +1/-1: all |q| equal, sign from the tile half.
//   FP64-pipe instructions per pair: generic 16 (Newton) / 18 (cubic); uniform 15 / 17.
template <int REFINE, int SIGN>
__device__ __forceinline__ void pair_field(double tx, double ty, double tz, double sx, double sy, double sz, double sq,
                                           double& acc, double& gx, double& gy, double& gz) {
    const double dx = tx - sx, dy = ty - sy, dz = tz - sz;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double y0 = rsqrt_seed(r2);
    const double t = y0 * y0;
    double k;
    if (REFINE == 1) {
        k = fma(-r2, t, kNewton3);
    } else {
        const double e = fma(-r2, t, 1.0);
        const double h = fma(e, 0.375, 0.5);
        k = fma(e, h, 1.0);
    }
    const double a = y0 * k;
    const double u = SIGN == 0 ? sq * a : a;
    const double v = u * (a * a);
    if (SIGN >= 0) {
        acc += u;
        gx = fma(v, dx, gx); gy = fma(v, dy, gy); gz = fma(v, dz, gz);
    } else {
        acc -= u;
        gx = fma(-v, dx, gx); gy = fma(-v, dy, gy); gz = fma(-v, dz, gz);
    }
}

constexpr int near_min_ctas(int R) { return R >= 8 ? 1 : (R == 4 ? 2 : (R == 2 ? 3 : 4)); }

// UNIFORM selects the loop form at compile time; the host launches both instantiations and the one that does
// not match the device-side flag QInfo.uniform returns at once (no host synchronisation to pick a kernel,
// and each instantiation keeps only its own loops: fewer live registers, better schedules).
// FIELD: also accumulate the gradient; partial rows then hold 4 components per target, part[(row*4 + comp)*T + t],
// comp 0 = phi, 1..3 = grad phi (in the frame of the ORIGINAL target: a reflected axis flips its component back).
template <int R, int REFINE, bool UNIFORM, bool FIELD>
__device__ __forceinline__ void near_sum_body(const NearArgs& a) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    __shared__ Cell cells[kMaxCells];

    constexpr int kUnroll = R >= 4 ? 2 : 4;  // sources per unrolled body (measured best on B200)
    if ((a.qinfo != nullptr && a.qinfo->uniform != 0) != UNIFORM) return;
    const int tid = threadIdx.x;
    const int G = gridDim.x, k = blockIdx.x;
    const long long u0 = unit_start(k, a.units, G), u1 = unit_start(k + 1, a.units, G);
    if (u1 <= u0) return;  // (never: the host launches G <= U CTAs)
    const long long Ub = a.n_tiles * a.C;
    const long long V0 = u0 / a.C, V1 = (u1 - 1) / a.C;  // visits v = b * n_tiles + t of this CTA

    for (int c = tid; c < a.C; c += kThreads) cells[c] = a.cells[c];
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&full[0], kTile * sizeof(Src4));
        bulk_g2s(tile[0], a.src + (V0 % a.n_tiles) * kTile, kTile * sizeof(Src4), &full[0]);
    }
    const double qmag = UNIFORM ? a.qinfo->qmag : 1.0;

    constexpr int RG = FIELD ? R : 1;  // gradient accumulators exist only in the FIELD form
    double ox[R], oy[R], oz[R], tot[R];
    double totx[RG], toty[RG], totz[RG];
    // visits are walked with 32-bit state: block b, tile tl inside the block
    const int nvis = (int)(V1 - V0) + 1;
    const int nt = (int)a.n_tiles;
    int b = (int)(V0 / a.n_tiles), tl = (int)(V0 - (long long)b * a.n_tiles);
    const int c_first = (int)(u0 - V0 * a.C), c_last = (int)(u1 - 1 - V1 * a.C) + 1;
    bool fresh = true;  // targets of block b not loaded yet
    // partial sums of block b go to row (k - first CTA that works on b)
    auto store_block = [&](int blk) {
        const int row = k - cta_of_unit(blk * Ub, a.units, G);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long t = (long long)blk * (kThreads * R) + r * kThreads + tid;
            if (t < a.T) {
                if (FIELD) {
                    double* o = a.part + (long long)row * 4 * a.T + t;
                    o[0] = tot[r]; o[a.T] = totx[r % RG]; o[2 * a.T] = toty[r % RG]; o[3 * a.T] = totz[r % RG];
                } else {
                    a.part[(long long)row * a.T + t] = tot[r];
                }
            }
        }
    };

    for (int it = 0; it < nvis; ++it) {
        const int st = it & 1;
        if (tid == 0 && it + 1 < nvis) {  // buffer st^1 was released by the barrier that ended the previous visit
            const int tn = tl + 1 == nt ? 0 : tl + 1;
            mbar_expect_tx(&full[st ^ 1], kTile * sizeof(Src4));
            bulk_g2s(tile[st ^ 1], a.src + (long long)tn * kTile, kTile * sizeof(Src4), &full[st ^ 1]);
        }
        const long long tb = (long long)b * (kThreads * R);
        if (fresh) {
            fresh = false;
            // targets owned by this thread (tail threads recompute target T-1 and do not store)
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
        const int np = a.tile_np[tl];
        const int nv = (int)min((long long)kTile, a.n_src - (long long)tl * kTile);
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        // self: target t is source self_offset + t (same tile after the in-tile sort).  Block-uniform test
        // whether this tile holds any of the block's own sources.
        const long long j0 = (long long)tl * kTile;
        const long long self_lo = a.self_offset + tb, self_hi = a.self_offset + min(a.T, tb + (long long)kThreads * R);
        const bool tile_has_self = a.self_offset >= 0 && j0 < self_hi && j0 + kTile > self_lo;
        const int c_lo = it == 0 ? c_first : 0;
        const int c_hi = it == nvis - 1 ? c_last : a.C;

        for (int c = c_lo; c < c_hi; ++c) {
            const Cell cell = cells[c];
            double tx[R], ty[R], tz[R], acc[R];
            double gx[RG], gy[RG], gz[RG];
#pragma unroll
            for (int r = 0; r < R; ++r) {
                tx[r] = flip(ox[r] - cell.sx, cell.fx);
                ty[r] = flip(oy[r] - cell.sy, cell.fy);
                tz[r] = flip(oz[r] - cell.sz, cell.fz);
                acc[r] = 0.0;
                if (FIELD) { gx[r % RG] = 0.0; gy[r % RG] = 0.0; gz[r % RG] = 0.0; }
            }
            double w = cell.w * a.scale;
            double wg = cell.w * a.scale_grad;
            if (cell.central && tile_has_self) {
                // masked path: the pair (t, j = slot of source self_offset + t) has r2 = 0; give it r2 = 1, q = 0
                int sj[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const long long i = a.self_offset + min(tb + r * kThreads + tid, a.T - 1);
                    const long long slot = a.slot_of ? (long long)a.slot_of[i] : i;
                    sj[r] = (int)max(-1LL, min((long long)kTile, slot - j0));
                }
#pragma unroll 1
                for (int j = 0; j < kTile; ++j) {
                    const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                    const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const bool self = j == sj[r];
                        if (FIELD)
                            pair_field<REFINE, 0>(tx[r], ty[r], tz[r], self ? tx[r] + 1.0 : xy.x, self ? ty[r] : xy.y,
                                                  self ? tz[r] : zq.x, self ? 0.0 : zq.y, acc[r], gx[r % RG], gy[r % RG], gz[r % RG]);
                        else
                            pair<REFINE>(tx[r], ty[r], tz[r], self ? tx[r] + 1.0 : xy.x, self ? ty[r] : xy.y,
                                         self ? tz[r] : zq.x, self ? 0.0 : zq.y, acc[r]);
                    }
                }
            } else if (UNIFORM) {
                w *= qmag;
                wg *= qmag;
#pragma unroll kUnroll
                for (int j = 0; j < np; ++j) {
                    const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                    const double sz = s[j].z;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (FIELD) pair_field<REFINE, 1>(tx[r], ty[r], tz[r], xy.x, xy.y, sz, 1.0, acc[r], gx[r % RG], gy[r % RG], gz[r % RG]);
                        else pair_unit<REFINE, false>(tx[r], ty[r], tz[r], xy.x, xy.y, sz, acc[r]);
                    }
                }
#pragma unroll kUnroll
                for (int j = np; j < nv; ++j) {
                    const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                    const double sz = s[j].z;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (FIELD) pair_field<REFINE, -1>(tx[r], ty[r], tz[r], xy.x, xy.y, sz, 1.0, acc[r], gx[r % RG], gy[r % RG], gz[r % RG]);
                        else pair_unit<REFINE, true>(tx[r], ty[r], tz[r], xy.x, xy.y, sz, acc[r]);
                    }
                }
            } else {
#pragma unroll kUnroll
                for (int j = 0; j < kTile; ++j) {
                    const double2 xy = *reinterpret_cast<const double2*>(&s[j].x);
                    const double2 zq = *reinterpret_cast<const double2*>(&s[j].z);
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (FIELD) pair_field<REFINE, 0>(tx[r], ty[r], tz[r], xy.x, xy.y, zq.x, zq.y, acc[r], gx[r % RG], gy[r % RG], gz[r % RG]);
                        else pair<REFINE>(tx[r], ty[r], tz[r], xy.x, xy.y, zq.x, zq.y, acc[r]);
                    }
                }
            }
#pragma unroll
            for (int r = 0; r < R; ++r) {
                tot[r] = fma(w, acc[r], tot[r]);
                if (FIELD) {
                    totx[r % RG] = fma(wg, flip(gx[r % RG], cell.fx), totx[r % RG]);
                    toty[r % RG] = fma(wg, flip(gy[r % RG], cell.fy), toty[r % RG]);
                    totz[r % RG] = fma(wg, flip(gz[r % RG], cell.fz), totz[r % RG]);
                }
            }
        }
        __syncthreads();  // everyone is done with tile[st] before it is refilled
        if (++tl == nt) {   // next visit starts the next target block
            store_block(b);
            tl = 0; ++b; fresh = true;
        }
    }
    if (!fresh) store_block(b);
}

template <int R, int REFINE, bool UNIFORM, bool FIELD = false>
__global__ void __launch_bounds__(kThreads, near_min_ctas(FIELD ? 2 * R : R)) near_sum_kernel(const NearArgs a) {
    near_sum_body<R, REFINE, UNIFORM, FIELD>(a);
}
// The same with the source count read from device memory (sphere-culled near set: the image list is built on the device
// and its length never visits the host): dyn[0] = sources, dyn[1] = source tiles replace n_src / n_tiles, and
// units = ntb * dyn[1] * C.  A separate instantiation, so that the kernel above keeps exactly its register allocation
// (folding the choice into it cost the R = 8 loop 2.7 % at 244 registers).
template <int R, int REFINE, bool UNIFORM, bool FIELD = false>
__global__ void __launch_bounds__(kThreads, near_min_ctas(FIELD ? 2 * R : R)) near_sum_dyn_kernel(const NearArgs a) {
    NearArgs b = a;
    b.n_src = a.dyn[0];
    b.n_tiles = a.dyn[1];
    b.units = a.ntb * b.n_tiles * a.C;
    near_sum_body<R, REFINE, UNIFORM, FIELD>(b);
}

// ---- step (b), symmetric form (Newton's third law) ---------------------------------------------
// When the targets ARE the sources (step (b) over all N, Eq.(5) with the self term left out), the
// image sum is symmetric: the image of source j in cell (k, sigma) lies as far from target i as the image of
// source i in the partner cell (-sigma o k, sigma), which has the same weight gamma^|k| (the cell
// table is closed under that map).  So one evaluation y = w / |r_i - img_c(r_j)| serves two sums:
//     phi_i += q_j y      (row sum, in the registers of the thread that owns target i)
//     phi_j += q_i y      (column sum: reduced over the 8 targets of a thread, over the cells, then over the lanes)
// and only the unordered pairs are walked: target block I (kSymBlock packed sources = kSymR tiles) meets source
// tiles J >= I * kSymR.  The block's own tiles ("diagonal" visits) are done as ordered pairs (row sums only,
// self term masked in the central cell); every later tile gives both.  Per unordered pair (Newton form):
// 3 DADD + DMUL + 2 DFMA (r2) + MUFU + DMUL (t) + DFMA (g) + DMUL (y) + 2 DFMA = 11 FP64-pipe instructions, i.e.
// 5.5 per pair interaction against 9 in near_sum_kernel (5.8 with the per-source work below).  Images are made
// by moving the SOURCE here (p = g o s + shift with g = +-1: one DFMA per coordinate, per source and cell, shared
// by the 8 targets of the thread), so nothing per-cell lives in registers on the target side and the
// column sums of a chunk of kSymS sources stay in registers across all cells: one warp reduction per source
// and tile visit, not per cell.
// Work decomposition: visits v = (I, J) in block-major order, each cut into kSymChunks chunks of kSymS sources;
// the fine units f = v * kSymChunks + chunk are dealt to the persistent grid in contiguous ranges exactly as in
// near_sum_kernel (balance to within one chunk).  Row sums go to part[row][packed index] (row = CTA - first CTA
// of the block), column sums to col[v][j]; sym_gather_kernel adds both in a fixed order (deterministic).
constexpr int kSymR = 8;                        // targets per thread
constexpr int kSymS = 4;                        // sources per chunk
constexpr int kSymChunks = kTile / kSymS;       // chunks per tile visit
constexpr int kSymBlock = kThreads * kSymR;     // targets per block
constexpr int kSymMaxCells = 128;               // cell table entries of this form (static shared memory <= 48 KB)
// first visit of block I (block I visits tiles I*kSymR .. n_tiles-1)
__host__ __device__ inline long long sym_visit0(long long I, long long n_tiles) {
    return I * n_tiles - (long long)kSymR * (I * (I - 1) / 2);
}

struct SymArgs {
    const Src4* src;     // packed sources (pack_sources_kernel); targets are the same records
    long long n_src, n_tiles;
    int n_blocks;        // ceil(n_tiles / kSymR)
    const Cell* cells;
    int C;
    long long f_begin;   // this launch walks the fine units [f_begin, f_begin + fine) of the F = sym_visit0(n_blocks) *
    long long fine;      // kSymChunks in all (one rank: everything; R ranks: a contiguous 1/R each)
    double scale;        // 0.5 for the Newton form (y is twice the reciprocal distance)
    double scale_grad;   // gradient form only: -1/4 (Newton), -1 (cubic)
    // One launch ("wave") walks a bounded range of fine units, so its scratch is bounded too: the
    // row sums of the blocks blk_base .. blk_base + part_blocks - 1 and one column line per visit from v_base on.
    int blk_base, part_blocks;
    long long v_base;
    double* part;        // [rows][part_blocks * kSymBlock]           (gradient form: [rows][4][...])
    double* col;         // [visits of the wave][kTile]               (gradient form: [visits][4][kTile])
};

template <int REFINE>
__device__ __forceinline__ double sym_recip(double dx, double dy, double dz) {
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double y0 = rsqrt_seed(r2);
    const double t = y0 * y0;
    if (REFINE == 1) {
        const double g = fma(-r2, t, kNewton3);
        return y0 * g;
    } else {
        const double e = fma(-r2, t, 1.0);
        const double h = fma(e, 0.375, 0.5);
        const double k = fma(e, h, 1.0);
        return y0 * k;
    }
}

template <int REFINE>
__global__ void __launch_bounds__(kThreads, 1) near_sym_kernel(const SymArgs a) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    struct SymCell { double sx, sy, sz, w, gx, gy, gz; int central, pad; };  // g = -1 on a reflected axis, else +1
    __shared__ SymCell cells[kSymMaxCells];
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

    for (int c = tid; c < a.C; c += kThreads) {
        const Cell g = a.cells[c];
        cells[c] = SymCell{g.sx, g.sy, g.sz, g.w * a.scale, g.fx ? -1.0 : 1.0, g.fy ? -1.0 : 1.0, g.fz ? -1.0 : 1.0, g.central, 0};
    }
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
        const int ch_lo = it == 0 ? ch_first : 0;
        const int ch_hi = it == nvis - 1 ? ch_last : kSymChunks;

        for (int ch = ch_lo; ch < ch_hi; ++ch) {
            const int j0 = ch * S;
            double sx[S], sy[S], sz[S], sq[S], colp[S];
#pragma unroll
            for (int i = 0; i < S; ++i) {
                const double2 xy = *reinterpret_cast<const double2*>(&s[j0 + i].x);
                const double2 zq = *reinterpret_cast<const double2*>(&s[j0 + i].z);
                sx[i] = xy.x; sy[i] = xy.y; sz[i] = zq.x; sq[i] = zq.y;
                colp[i] = 0.0;
            }
#pragma unroll 1
            for (int c = 0; c < a.C; ++c) {
                const SymCell cell = cells[c];
                const double wc = cell.w;
                if (diag && cell.central) {
                    // the block's own tile, bare terms: target (r = rd, tid) IS source j = tid; skip that pair
#pragma unroll 1
                    for (int i = 0; i < S; ++i) {   // (read from the tile again: no dynamic indexing of registers)
                        const double2 xy = *reinterpret_cast<const double2*>(&s[j0 + i].x);
                        const double2 zq = *reinterpret_cast<const double2*>(&s[j0 + i].z);
                        const double wq = zq.y * wc;
                        const bool mine = j0 + i == tid;
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const bool self = mine && r == rd;
                            const double y = sym_recip<REFINE>(ox[r] - (self ? ox[r] + 1.0 : xy.x), oy[r] - xy.y, oz[r] - zq.x);
                            tot[r] = fma(self ? 0.0 : wq, y, tot[r]);
                        }
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < S; ++i) {
                        const double px = fma(cell.gx, sx[i], cell.sx);   // image = sign o r + shift (exact: g = +-1)
                        const double py = fma(cell.gy, sy[i], cell.sy);
                        const double pz = fma(cell.gz, sz[i], cell.sz);
                        const double wq = sq[i] * wc;
                        double cj = 0.0;
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const double y = sym_recip<REFINE>(ox[r] - px, oy[r] - py, oz[r] - pz);
                            tot[r] = fma(wq, y, tot[r]);
                            cj = fma(oq[r], y, cj);
                        }
                        colp[i] = fma(wc, cj, colp[i]);
                    }
                }
            }
            if (!diag) {
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    double v = colp[i];
#pragma unroll
                    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    if (lane == 0) colw[warp][j0 + i] = v;
                }
            }
        }
        __syncthreads();  // tile[st] may be refilled; colw is complete
        if (!diag) {
            const int j = tid;  // kTile == kThreads
            if (j >= ch_lo * S && j < ch_hi * S) {
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

// ---- step (b), symmetric form with the gradient (forces, Eq.(9)) ------------------------------
// One evaluation now feeds phi_i, grad phi_i, phi_j and grad phi_j.  With d = r_i - img_c(r_j) and v = w / |d|^3:
//   grad_i (q_j w / |d|)           = -q_j v d                      (the source is moved, so d is in the original frame)
//   grad_j (q_i w / |r_j - img'|)  = +q_i v (sigma_c o d)          (partner cell: d' = -sigma_c o d, same |d|)
// Per evaluation (Newton): 3 DADD + DMUL + 2 DFMA (r2) + MUFU + 3 DMUL (y0^2, y, y^2) + DFMA (g) + DMUL (v)
// + row: DFMA + DMUL + 3 DFMA + column: DFMA + DMUL + 3 DFMA = 21 FP64-pipe instructions, i.e. 10.5 per pair
// interaction against 15 in near_sum_kernel<.., FIELD>.  The reflection signs, the cell weight and the powers of
// two of the Newton form (y = 2/|d|, v = 8/|d|^3) are applied once per (source, cell) and at the stores.
// Layouts: part[(row * 4 + comp) * Tp + packed index], col[(visit * 4 + comp) * kTile + j], comp 0 = phi,
// 1..3 = grad phi.  Work decomposition, diagonal visits and determinism as in near_sym_kernel.
constexpr int kSymFS = 2;                       // sources per chunk of the gradient form (register budget)
constexpr int kSymFChunks = kTile / kSymFS;
constexpr int kSymFieldDynSmem = ((kThreads / 32) * 4 * kTile + 2 * kSymR * kThreads) * (int)sizeof(double);

template <int REFINE>
__global__ void __launch_bounds__(kThreads, 1) near_sym_field_kernel(const SymArgs a) {
    __shared__ __align__(128) Src4 tile[kStages][kTile];
    __shared__ __align__(8) uint64_t full[kStages];
    struct SymCell { double sx, sy, sz, w, gx, gy, gz; int central, pad; };
    __shared__ SymCell cells[kSymMaxCells];
    // dynamic shared memory (kSymFieldDynSmem): colw [kThreads / 32][4][kTile] (64 KB), then x, y of the block's
    // targets, txy [R][kThreads] double2 (32 KB; slot [r][tid] is written and read by thread tid only).  With phi and
    // grad phi accumulators for 8 targets the register file is full, and this kernel is bound by dependent-issue
    // latency (ncu: stall_wait 2.1 per issue with everything in registers): half of the target coordinates and the
    // chunk's sources are therefore re-read from shared memory (one conflict-free 128-bit load per evaluation), which
    // frees ~48 registers for independent pair chains: 99.9 -> 85.0 ms at N = 65,536 (FP64 issue 71 % -> 84 %; all
    // four target words in shared memory: 86.0 ms).
    extern __shared__ __align__(16) double colw[];
    double2* txy = reinterpret_cast<double2*>(colw + (kThreads / 32) * 4 * kTile);

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

    for (int c = tid; c < a.C; c += kThreads) {
        const Cell g = a.cells[c];
        cells[c] = SymCell{g.sx, g.sy, g.sz, g.w * a.scale, g.fx ? -1.0 : 1.0, g.fy ? -1.0 : 1.0, g.fz ? -1.0 : 1.0, g.central, 0};
    }
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&full[0], kTile * sizeof(Src4));
        bulk_g2s(tile[0], a.src + (long long)J * kTile, kTile * sizeof(Src4), &full[0]);
    }

    double oz[R], oq[R], tot[R], tgx[R], tgy[R], tgz[R];
    const int nvis = (int)(V1 - V0) + 1;
    const int ch_first = (int)(f0 - V0 * kSymFChunks), ch_last = (int)(f1 - 1 - V1 * kSymFChunks) + 1;
    const long long Tp = (long long)a.part_blocks * kSymBlock;
    const double sg = a.scale_grad;   // gradient sums -> grad phi: -1/4 (Newton: v = 8/|d|^3 against the 1/2 in w), -1 (cubic)
    bool fresh = true;
    auto store_block = [&](int blk) {
        const int row = k - cta_of_unit(max(sym_visit0(blk, nt) * kSymFChunks, a.f_begin) - a.f_begin, a.fine, G);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            double* o = a.part + (long long)row * 4 * Tp + (long long)(blk - a.blk_base) * kSymBlock + r * kThreads + tid;
            o[0] = tot[r]; o[Tp] = sg * tgx[r]; o[2 * Tp] = sg * tgy[r]; o[3 * Tp] = sg * tgz[r];
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
#pragma unroll
            for (int r = 0; r < R; ++r) {
                const int tt = I * R + r;
                const Src4 t = a.src[(long long)min(tt, nt - 1) * kTile + tid];
                txy[r * kThreads + tid] = make_double2(t.x, t.y);   // read back by this thread only
                oz[r] = t.z; oq[r] = tt < nt ? t.q : 0.0;
                tot[r] = 0.0; tgx[r] = 0.0; tgy[r] = 0.0; tgz[r] = 0.0;
            }
        }
        const int rd = J - I * R;
        const bool diag = rd < R;
        mbar_wait(&full[st], (it >> 1) & 1);
        const Src4* __restrict__ s = tile[st];
        const int ch_lo = it == 0 ? ch_first : 0;
        const int ch_hi = it == nvis - 1 ? ch_last : kSymFChunks;
        double* colv = a.col + (V0 + it - a.v_base) * 4 * kTile;

        for (int ch = ch_lo; ch < ch_hi; ++ch) {
            const int j0 = ch * S;
            double cp[S], cx[S], cy[S], cz[S];
#pragma unroll
            for (int i = 0; i < S; ++i) { cp[i] = 0.0; cx[i] = 0.0; cy[i] = 0.0; cz[i] = 0.0; }
#pragma unroll 1
            for (int c = 0; c < a.C; ++c) {
                const SymCell cell = cells[c];
                const double wc = cell.w;
                if (diag && cell.central) {
#pragma unroll 1
                    for (int i = 0; i < S; ++i) {
                        const double2 xy = *reinterpret_cast<const double2*>(&s[j0 + i].x);
                        const double2 zq = *reinterpret_cast<const double2*>(&s[j0 + i].z);
                        const double wq = zq.y * wc;
                        const bool mine = j0 + i == tid;
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const bool self = mine && r == rd;
                            const double2 oxy = txy[r * kThreads + tid];
                            const double dx = oxy.x - (self ? oxy.x + 1.0 : xy.x), dy = oxy.y - xy.y, dz = oz[r] - zq.x;
                            const double y = sym_recip<REFINE>(dx, dy, dz);
                            const double wm = self ? 0.0 : wq;
                            const double wv = wm * (y * (y * y));
                            tot[r] = fma(wm, y, tot[r]);
                            tgx[r] = fma(wv, dx, tgx[r]); tgy[r] = fma(wv, dy, tgy[r]); tgz[r] = fma(wv, dz, tgz[r]);
                        }
                    }
                } else {
#pragma unroll
                    for (int i = 0; i < S; ++i) {
                        const double2 xy = *reinterpret_cast<const double2*>(&s[j0 + i].x);
                        const double2 zq = *reinterpret_cast<const double2*>(&s[j0 + i].z);
                        const double px = fma(cell.gx, xy.x, cell.sx);
                        const double py = fma(cell.gy, xy.y, cell.sy);
                        const double pz = fma(cell.gz, zq.x, cell.sz);
                        const double wq = zq.y * wc;
                        double cj = 0.0, gx = 0.0, gy = 0.0, gz = 0.0;
#pragma unroll
                        for (int r = 0; r < R; ++r) {
                            const double2 oxy = txy[r * kThreads + tid];
                            const double dx = oxy.x - px, dy = oxy.y - py, dz = oz[r] - pz;
                            const double y = sym_recip<REFINE>(dx, dy, dz);
                            const double v = y * (y * y);
                            const double oqr = oq[r];
                            const double wv = wq * v, ov = oqr * v;
                            tot[r] = fma(wq, y, tot[r]);
                            tgx[r] = fma(wv, dx, tgx[r]); tgy[r] = fma(wv, dy, tgy[r]); tgz[r] = fma(wv, dz, tgz[r]);
                            cj = fma(oqr, y, cj);
                            gx = fma(ov, dx, gx); gy = fma(ov, dy, gy); gz = fma(ov, dz, gz);
                        }
                        cp[i] = fma(wc, cj, cp[i]);
                        cx[i] = fma(wc * cell.gx, gx, cx[i]); cy[i] = fma(wc * cell.gy, gy, cy[i]); cz[i] = fma(wc * cell.gz, gz, cz[i]);
                    }
                }
            }
            if (!diag) {
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    double v0 = cp[i], v1 = cx[i], v2 = cy[i], v3 = cz[i];
#pragma unroll
                    for (int o = 16; o; o >>= 1) {
                        v0 += __shfl_xor_sync(0xffffffffu, v0, o); v1 += __shfl_xor_sync(0xffffffffu, v1, o);
                        v2 += __shfl_xor_sync(0xffffffffu, v2, o); v3 += __shfl_xor_sync(0xffffffffu, v3, o);
                    }
                    if (lane == 0) {
                        double* o = colw + (warp * 4) * kTile + j0 + i;
                        o[0] = v0; o[kTile] = v1; o[2 * kTile] = v2; o[3 * kTile] = v3;
                    }
                }
            }
        }
        __syncthreads();  // tile[st] may be refilled; colw is complete
        if (!diag) {
            // grad_j = +q_i v sigma o d: the factor sg of the row side carries a minus sign, hence -sg here
            const int j = tid;  // kTile == kThreads
            if (j >= ch_lo * S && j < ch_hi * S) {
#pragma unroll
                for (int comp = 0; comp < 4; ++comp) {
                    double v = 0.0;
#pragma unroll
                    for (int w = 0; w < kThreads / 32; ++w) v += colw[(w * 4 + comp) * kTile + j];
                    colv[comp * kTile + j] = comp == 0 ? v : -sg * v;
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

// What one wave (launch) of the symmetric kernels left behind, for the gathers below.
struct SymWave {
    long long f_begin, fine;   // fine units of the wave
    long long v_base;          // first visit of the wave (column line 0)
    int blk_lo, blk_hi;        // blocks the wave's visits belong to (row sums: part_blocks = blk_hi - blk_lo + 1)
    int G;                     // CTAs of the wave
    int first;                 // 1: the first wave of the evaluate (out is written, not added to)
};

// FIELD form of sym_gather_kernel: out[comp * N + t], comp 0 = phi, 1..3 = grad phi, original source order.
__global__ void sym_gather_field_kernel(const double* __restrict__ part, const double* __restrict__ col,
                                        const int* __restrict__ slot_of, long long N, long long n_tiles, const SymWave w,
                                        double* __restrict__ out) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= N) return;
    const long long p = slot_of[t];
    const int I = (int)(p / kSymBlock), J = (int)(p / kTile), j = (int)(p % kTile);
    const long long Tp = (long long)(w.blk_hi - w.blk_lo + 1) * kSymBlock;
    const long long f_end = w.f_begin + w.fine;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    if (!w.first) {
#pragma unroll
        for (int c = 0; c < 4; ++c) v[c] = out[c * N + t];
    }
    const long long lo = max(sym_visit0(I, n_tiles) * kSymFChunks, w.f_begin), hi = min(sym_visit0(I + 1, n_tiles) * kSymFChunks, f_end);
    if (lo < hi) {
        const int first = cta_of_unit(lo - w.f_begin, w.fine, w.G), last = cta_of_unit(hi - 1 - w.f_begin, w.fine, w.G);
        const long long pw = p - (long long)w.blk_lo * kSymBlock;
        for (int r = 0; r <= last - first; ++r)
#pragma unroll
            for (int c = 0; c < 4; ++c) v[c] += part[((long long)r * 4 + c) * Tp + pw];
    }
    for (int b = w.blk_lo; b <= min(w.blk_hi, I - 1); ++b) {
        const long long vis = sym_visit0(b, n_tiles) + (J - b * kSymR);
        const long long f = vis * kSymFChunks + j / kSymFS;
        if (f >= w.f_begin && f < f_end)
#pragma unroll
            for (int c = 0; c < 4; ++c) v[c] += col[((vis - w.v_base) * 4 + c) * kTile + j];
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) out[c * N + t] = v[c];
}

// phi of step (b) in the ORIGINAL source order: for each wave in turn, row sums (fixed CTA order) + column sums (blocks
// in order) of the fine units the wave walked; over the waves of one rank this adds up to its share of the near sum.
__global__ void sym_gather_kernel(const double* __restrict__ part, const double* __restrict__ col,
                                  const int* __restrict__ slot_of, long long N, long long n_tiles, const SymWave w,
                                  double* __restrict__ out) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= N) return;
    const long long p = slot_of[t];
    const int I = (int)(p / kSymBlock), J = (int)(p / kTile), j = (int)(p % kTile);
    const long long Tp = (long long)(w.blk_hi - w.blk_lo + 1) * kSymBlock;
    const long long f_end = w.f_begin + w.fine;
    double v = w.first ? 0.0 : out[t];
    const long long lo = max(sym_visit0(I, n_tiles) * kSymChunks, w.f_begin), hi = min(sym_visit0(I + 1, n_tiles) * kSymChunks, f_end);
    if (lo < hi) {
        const int first = cta_of_unit(lo - w.f_begin, w.fine, w.G), last = cta_of_unit(hi - 1 - w.f_begin, w.fine, w.G);
        const long long pw = p - (long long)w.blk_lo * kSymBlock;
        for (int r = 0; r <= last - first; ++r) v += part[(long long)r * Tp + pw];
    }
    for (int b = w.blk_lo; b <= min(w.blk_hi, I - 1); ++b) {
        const long long vis = sym_visit0(b, n_tiles) + (J - b * kSymR);
        const long long f = vis * kSymChunks + j / kSymS;
        if (f >= w.f_begin && f < f_end) v += col[(vis - w.v_base) * kTile + j];
    }
    out[t] = v;
}

struct NodeArgs {
    const double* tgt;
    int tstride;
    long long T;
    long long t_first;   // target t is row tgt_index[t_first + t] of tgt (row t_first + t if tgt_index is null)
    const int* tgt_index;
    const Node8* nodes;  // padded to a multiple of kTile/2 with zero-strength records at kFar
    long long n_tiles;   // tiles of kTile/2 nodes (same 8 KB stage size)
    long long units;     // U = ntb * n_tiles (the decomposition above with C = 1)
    double* part;        // [part_rows][T] ([part_rows][4][T] in the FIELD form)
};

// phi(t) = sum_j Q_j/rho - P_j.(t - R_j)/rho^3  = sum_j y (Q_j - (P_j.d) y^2),  y = 1/rho,
// with the exact normal dipole P_j = D_j n_j (reading S9).  y by the cubic step (relative ~1e-19
// before rounding).  3 DADD + 3 (r2) + 5 (rsqrt) + 3 (P.d) + DMUL (y^2) + DFMA + DFMA = 17 FP64 instructions.
// FIELD: also grad phi = y^3 [ (3 (P.d) y^2 - Q) d - P ]  (+ DMUL y^3, DMUL 3 y^2, DFMA, 3 DFMA, 3 DFMA = 26).
template <int R, bool FIELD = false>
__global__ void __launch_bounds__(kThreads, near_min_ctas(FIELD ? 2 * R : R)) node_sum_kernel(const NodeArgs a) {
    constexpr int kNT = kTile / 2;
    __shared__ __align__(128) Node8 tile[kStages][kNT];
    __shared__ __align__(8) uint64_t full[kStages];
    const int tid = threadIdx.x;
    const int G = gridDim.x, k = blockIdx.x;
    const long long V0 = unit_start(k, a.units, G), V1 = unit_start(k + 1, a.units, G) - 1;  // inclusive
    if (V1 < V0) return;
    if (tid == 0) {
        for (int s = 0; s < kStages; ++s) mbar_init(&full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
        mbar_expect_tx(&full[0], kNT * sizeof(Node8));
        bulk_g2s(tile[0], a.nodes + (V0 % a.n_tiles) * kNT, kNT * sizeof(Node8), &full[0]);
    }
    constexpr int RG = FIELD ? R : 1;
    double tx[R], ty[R], tz[R], acc[R];
    double gx[RG], gy[RG], gz[RG];
    long long cur_b = -1;
    auto store_block = [&](long long b) {
        const int row = k - cta_of_unit(b * a.n_tiles, a.units, G);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const long long t = b * (kThreads * R) + r * kThreads + tid;
            if (t < a.T) {
                if (FIELD) {
                    double* o = a.part + (long long)row * 4 * a.T + t;
                    o[0] = acc[r]; o[a.T] = gx[r % RG]; o[2 * a.T] = gy[r % RG]; o[3 * a.T] = gz[r % RG];
                } else {
                    a.part[(long long)row * a.T + t] = acc[r];
                }
            }
        }
    };
    for (long long v = V0; v <= V1; ++v) {
        const int it = (int)(v - V0), st = it & 1;
        const long long b = v / a.n_tiles;
        if (tid == 0 && v < V1) {
            mbar_expect_tx(&full[st ^ 1], kNT * sizeof(Node8));
            bulk_g2s(tile[st ^ 1], a.nodes + ((v + 1) % a.n_tiles) * kNT, kNT * sizeof(Node8), &full[st ^ 1]);
        }
        if (b != cur_b) {
            if (cur_b >= 0) store_block(cur_b);
            cur_b = b;
#pragma unroll
            for (int r = 0; r < R; ++r) {
                long long t = b * (kThreads * R) + r * kThreads + tid;
                t = a.t_first + (t < a.T ? t : a.T - 1);
                if (a.tgt_index) t = a.tgt_index[t];
                const double* p = a.tgt + t * a.tstride;
                tx[r] = p[0]; ty[r] = p[1]; tz[r] = p[2];
                acc[r] = 0.0;
                if (FIELD) { gx[r % RG] = 0.0; gy[r % RG] = 0.0; gz[r % RG] = 0.0; }
            }
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
                const double y2 = y * y;
                const double u = fma(-pd, y2, zq.y);
                acc[r] = fma(y, u, acc[r]);
                if (FIELD) {
                    const double y3 = y2 * y;
                    const double c = fma(3.0 * y2, pd, -zq.y);       // 3 (P.d) y^2 - Q
                    gx[r % RG] = fma(y3, fma(c, dx, -pxy.x), gx[r % RG]);
                    gy[r % RG] = fma(y3, fma(c, dy, -pxy.y), gy[r % RG]);
                    gz[r % RG] = fma(y3, fma(c, dz, -pz), gz[r % RG]);
                }
            }
        }
        __syncthreads();
    }
    store_block(cur_b);
}

// ---- H1 pre-pass: centre the coordinates, pack (x,y,z,q) and sort each tile by the sign of q ----
// One block = one tile of kTile sources.  Inside a tile the records are stably partitioned: the n_pos
// sources with q >= 0 first, then the negative ones (tile_np[tile] = n_pos); pads (q = 0 at kFar) stay
// behind the valid records.  slot_of[i] = index of source i in the packed array (same tile, so the
// "does this tile hold my own sources" test of the self exclusion is unchanged).  With all |q| equal
// (QInfo.uniform, found by charge_stats_kernel) the sum kernels then never multiply by q: they add
// over the positive part, subtract over the negative part and scale the cell weight by |q|.
// Also writes per block [sum q, sum |q|, min |q|, max |q|] for charge_stats_kernel.
__global__ void __launch_bounds__(kTile) pack_sources_kernel(const double* __restrict__ xyz, const double* __restrict__ q,
                                                           long long N, double hx, double hy, double hz,
                                                           Src4* __restrict__ out, int* __restrict__ slot_of,
                                                           int* __restrict__ tile_np, double* __restrict__ stats /* [gridDim.x][4] */,
                                                           const long long* __restrict__ dynN = nullptr /* device-resident N */) {
    if (dynN) { N = dynN[0]; if ((long long)blockIdx.x * kTile >= N) return; }
    __shared__ int wpos[kTile / 32], wneg[kTile / 32];
    __shared__ double sh[4][kTile / 32];
    const int tid = threadIdx.x, w = tid >> 5, l = tid & 31;
    const long long i = (long long)blockIdx.x * kTile + tid;
    const bool valid = i < N;
    Src4 s;
    if (valid) { s.x = xyz[3 * i] - hx; s.y = xyz[3 * i + 1] - hy; s.z = xyz[3 * i + 2] - hz; s.q = q[i]; }
    else { s.x = kFar; s.y = kFar; s.z = kFar; s.q = 0.0; }
    const bool pos = valid && !(s.q < 0.0), neg = valid && s.q < 0.0;
    const unsigned bp = __ballot_sync(0xffffffffu, pos), bn = __ballot_sync(0xffffffffu, neg);
    if (l == 0) { wpos[w] = __popc(bp); wneg[w] = __popc(bn); }
    // block statistics of q
    double a = valid ? s.q : 0.0, b = fabs(a), mn = valid ? b : 1e300, mx = valid ? b : 0.0;
    for (int o = 16; o; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o);
        mn = fmin(mn, __shfl_down_sync(0xffffffffu, mn, o)); mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    }
    if (l == 0) { sh[0][w] = a; sh[1][w] = b; sh[2][w] = mn; sh[3][w] = mx; }
    __syncthreads();
    int before_pos = 0, before_neg = 0, npos = 0, nneg = 0;
#pragma unroll
    for (int k = 0; k < kTile / 32; ++k) {
        if (k < w) { before_pos += wpos[k]; before_neg += wneg[k]; }
        npos += wpos[k]; nneg += wneg[k];
    }
    const unsigned lower = (1u << l) - 1u;
    int slot;
    if (pos) slot = before_pos + __popc(bp & lower);
    else if (neg) slot = npos + before_neg + __popc(bn & lower);
    else slot = tid;  // pads: the valid sources of a tile are its first threads, so pads keep their place
    out[(long long)blockIdx.x * kTile + slot] = s;
    if (valid) slot_of[i] = (int)(blockIdx.x * kTile + slot);
    if (tid == 0) {
        tile_np[blockIdx.x] = npos;
        double A = 0.0, B = 0.0, MN = 1e300, MX = 0.0;
        for (int k = 0; k < kTile / 32; ++k) { A += sh[0][k]; B += sh[1][k]; MN = fmin(MN, sh[2][k]); MX = fmax(MX, sh[3][k]); }
        stats[4 * blockIdx.x] = A; stats[4 * blockIdx.x + 1] = B; stats[4 * blockIdx.x + 2] = MN; stats[4 * blockIdx.x + 3] = MX;
    }
}

// ---- paper-literal near set: the images inside the auxiliary sphere ----
// Entry e = c * N + j of the (cell, source) table, cells in the order `order[c]` (central cell first, so that
// image i < N is source i).  inside(e): |sign o r_j + shift|^2 <= R^2.  Pass 1 counts per block of kTile entries,
// scan_counts_kernel turns the counts into offsets (single block), pass 2 writes the compacted list in order:
// xyz_img [N_s,3], q_img [N_s] = w_c q_j.  The list is then packed like any source array and summed with the
// identity cell.
__device__ __forceinline__ bool image_of(const double* __restrict__ xyz, const double* __restrict__ q, long long N,
                                         double hx, double hy, double hz, const Cell* __restrict__ cells,
                                         const int* __restrict__ order, long long e, long long total, double R2,
                                         double out[4]) {
    if (e >= total) return false;
    const int c = order[e / N];
    const long long j = e - (e / N) * N;
    const Cell cell = cells[c];
    // image = sign o r + shift  (the pair kernels use the equivalent transform of the target instead)
    const double x = flip(xyz[3 * j] - hx, cell.fx) + cell.sx;
    const double y = flip(xyz[3 * j + 1] - hy, cell.fy) + cell.sy;
    const double z = flip(xyz[3 * j + 2] - hz, cell.fz) + cell.sz;
    out[0] = x; out[1] = y; out[2] = z; out[3] = cell.w * q[j];
    return x * x + y * y + z * z <= R2;
}
__global__ void __launch_bounds__(kTile) image_count_kernel(const double* __restrict__ xyz, const double* __restrict__ q,
                                                          long long N, double hx, double hy, double hz,
                                                          const Cell* __restrict__ cells, const int* __restrict__ order,
                                                          int C, double R2, long long* __restrict__ block_count) {
    __shared__ int wc[kTile / 32];
    const long long e = (long long)blockIdx.x * kTile + threadIdx.x;
    double r[4];
    const bool in = image_of(xyz, q, N, hx, hy, hz, cells, order, e, (long long)C * N, R2, r);
    const unsigned b = __ballot_sync(0xffffffffu, in);
    if ((threadIdx.x & 31) == 0) wc[threadIdx.x >> 5] = __popc(b);
    __syncthreads();
    if (threadIdx.x == 0) {
        int n = 0;
        for (int k = 0; k < kTile / 32; ++k) n += wc[k];
        block_count[blockIdx.x] = n;
    }
}
// in place: counts -> exclusive offsets; total -> counts[n].  Single block of 1024 threads, chunked.
__global__ void __launch_bounds__(1024) scan_counts_kernel(long long* __restrict__ counts, long long n) {
    __shared__ long long sh[1024];
    __shared__ long long carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (long long base = 0; base < n; base += 1024) {
        const long long i = base + threadIdx.x;
        const long long v = i < n ? counts[i] : 0;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const long long t = threadIdx.x >= o ? sh[threadIdx.x - o] : 0;
            __syncthreads();
            sh[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < n) counts[i] = carry + sh[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 0) carry += sh[1023];
        __syncthreads();
    }
    if (threadIdx.x == 0) counts[n] = carry;
}
// dyn[0] = images inside the sphere, dyn[1] = their tiles; flags[2] = 1 if a source itself lies outside the sphere
// (fewer images than sources) or the list would overflow the 32-bit packed indices
__global__ void image_finalize_kernel(const long long* __restrict__ counts_total, long long N, long long* __restrict__ dyn,
                                      int* __restrict__ flags) {
    const long long Ns = counts_total[0];
    dyn[0] = Ns;
    dyn[1] = (Ns + kTile - 1) / kTile;
    if (Ns < N || Ns > 2000000000LL) flags[2] = 1;
}
__global__ void __launch_bounds__(kTile) image_scatter_kernel(const double* __restrict__ xyz, const double* __restrict__ q,
                                                            long long N, double hx, double hy, double hz,
                                                            const Cell* __restrict__ cells, const int* __restrict__ order,
                                                            int C, double R2, const long long* __restrict__ block_offset,
                                                            double* __restrict__ xyz_img, double* __restrict__ q_img) {
    __shared__ int wc[kTile / 32];
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    const long long e = (long long)blockIdx.x * kTile + threadIdx.x;
    double r[4];
    const bool in = image_of(xyz, q, N, hx, hy, hz, cells, order, e, (long long)C * N, R2, r);
    const unsigned b = __ballot_sync(0xffffffffu, in);
    if (l == 0) wc[w] = __popc(b);
    __syncthreads();
    if (in) {
        int before = 0;
        for (int k = 0; k < w; ++k) before += wc[k];
        const long long o = block_offset[blockIdx.x] + before + __popc(b & ((1u << l) - 1u));
        xyz_img[3 * o] = r[0]; xyz_img[3 * o + 1] = r[1]; xyz_img[3 * o + 2] = r[2];
        q_img[o] = r[3];
    }
}

// Single block: sum q, sum |q| -> scal[0..1]; neutrality flag (reading S17); QInfo (all |q| equal, bit for bit).
__global__ void __launch_bounds__(1024) charge_stats_kernel(const double* __restrict__ stats, long long nblocks,
                                                            int need_neutral, double* __restrict__ scal,
                                                            QInfo* __restrict__ qi, int* __restrict__ flags,
                                                            const long long* __restrict__ dyn = nullptr /* dyn[1] = blocks */) {
    if (dyn) nblocks = dyn[1];
    __shared__ double sh[4][32];
    double a = 0.0, b = 0.0, mn = 1e300, mx = 0.0;
    for (long long i = threadIdx.x; i < nblocks; i += blockDim.x) {
        a += stats[4 * i]; b += stats[4 * i + 1]; mn = fmin(mn, stats[4 * i + 2]); mx = fmax(mx, stats[4 * i + 3]);
    }
    for (int o = 16; o; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o);
        mn = fmin(mn, __shfl_down_sync(0xffffffffu, mn, o)); mx = fmax(mx, __shfl_down_sync(0xffffffffu, mx, o));
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) { sh[0][w] = a; sh[1][w] = b; sh[2][w] = mn; sh[3][w] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        a = 0.0; b = 0.0; mn = 1e300; mx = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { a += sh[0][k]; b += sh[1][k]; mn = fmin(mn, sh[2][k]); mx = fmax(mx, sh[3][k]); }
        scal[0] = a; scal[1] = b;
        qi->uniform = (mn == mx) ? 1 : 0;
        qi->qmag = mx;
        qi->pad = 0;
        if (need_neutral && fabs(a) > 1e-12 * b) flags[1] = 1;
    }
}

// ---- H7: phi = sum over partial rows (fixed order), U block partials --------------------------
// The rows of a target block are those of the CTAs that worked on it, in CTA order (PartLayout).
__device__ __forceinline__ double sum_part_rows(const PartLayout& L, long long t, long long T) {
    if (!L.part) return 0.0;
    const long long b = t / L.block_targets;
    long long U, Ub;
    layout_units(L, T, U, Ub);
    const int first = cta_of_unit(b * Ub, U, L.G), last = cta_of_unit((b + 1) * Ub - 1, U, L.G);
    double s = 0.0;
    for (int k = 0; k <= last - first; ++k) s += L.part[(long long)k * T + t];
    return s;
}
// FIELD form of the finish: phi, force F_i = -q_i grad phi(r_i) or, without charges, grad phi itself.
__device__ __forceinline__ void sum_part_rows4(const PartLayout& L, long long t, long long T, double out[4]) {
    if (!L.part) return;
    const long long b = t / L.block_targets;
    long long U, Ub;
    layout_units(L, T, U, Ub);
    const int first = cta_of_unit(b * Ub, U, L.G), last = cta_of_unit((b + 1) * Ub - 1, U, L.G);
    for (int k = 0; k <= last - first; ++k)
#pragma unroll
        for (int c = 0; c < 4; ++c) out[c] += L.part[((long long)k * 4 + c) * T + t];
}
__global__ void finish_field_kernel(const PartLayout Lb, const PartLayout Lc, long long T,
                                    const Src4* __restrict__ src, const int* __restrict__ slot_of, long long t_first,
                                    double* __restrict__ phi, double* __restrict__ vec /* [T,3] */,
                                    double* __restrict__ u_part /* [gridDim.x] or null */) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (t < T) {
        double sb[4] = {0.0, 0.0, 0.0, 0.0}, sc[4] = {0.0, 0.0, 0.0, 0.0};
        sum_part_rows4(Lb, t, T, sb);
        sum_part_rows4(Lc, t, T, sc);
        const double v = sb[0] + sc[0];
        if (phi) phi[t] = v;
        const double qi = src ? src[slot_of[t_first + t]].q : -1.0;   // no charges: write +grad
        vec[3 * t] = -qi * (sb[1] + sc[1]); vec[3 * t + 1] = -qi * (sb[2] + sc[2]); vec[3 * t + 2] = -qi * (sb[3] + sc[3]);
        if (src) e = qi * v;
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

__global__ void finish_phi_kernel(const PartLayout Lb, const PartLayout Lc, long long T,
                                  const Src4* __restrict__ src, const int* __restrict__ slot_of, long long t_first,
                                  double* __restrict__ phi, double* __restrict__ u_part /* [gridDim.x] or null */) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (t < T) {
        const double v = sum_part_rows(Lb, t, T) + sum_part_rows(Lc, t, T);
        phi[t] = v;
        if (src) e = src[slot_of[t_first + t]].q * v;
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

// H7 for a part of the pair work (multi-GPU): phi_part[t] over ALL N targets = this part's share of the
// near sum + the node sum for the targets t0 <= t < t1 only; U_part = 1/2 sum q phi_part.  Both add up over the parts.
__global__ void finish_part_kernel(const double* __restrict__ near, const PartLayout Lc, long long N, long long t0,
                                   long long t1, const Src4* __restrict__ src, const int* __restrict__ slot_of,
                                   double* __restrict__ phi, double* __restrict__ u_part) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (t < N) {
        double v = near[t];
        if (t >= t0 && t < t1) v += sum_part_rows(Lc, t - t0, t1 - t0);
        phi[t] = v;
        e = src[slot_of[t]].q * v;
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

// The same with forces: near [4][N] (phi, grad phi of this part's share), node sum rows in the FIELD layout for the
// targets t0..t1-1; phi (may be null) and F = -q grad phi [N,3] are partial sums over the parts.
__global__ void finish_part_field_kernel(const double* __restrict__ near, const PartLayout Lc, long long N, long long t0,
                                         long long t1, const Src4* __restrict__ src, const int* __restrict__ slot_of,
                                         double* __restrict__ phi, double* __restrict__ vec, double* __restrict__ u_part) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (t < N) {
        double v[4] = {near[t], near[N + t], near[2 * N + t], near[3 * N + t]};
        if (t >= t0 && t < t1) sum_part_rows4(Lc, t - t0, t1 - t0, v);
        const double qi = src[slot_of[t]].q;
        if (phi) phi[t] = v[0];
        vec[3 * t] = -qi * v[1]; vec[3 * t + 1] = -qi * v[2]; vec[3 * t + 2] = -qi * v[3];
        e = qi * v[0];
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
