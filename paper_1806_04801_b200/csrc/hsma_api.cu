// C-ABI of include/hsma.h: plan (preparation step) and evaluate (update step,
// PAPER.md:142).  Host orchestration only; every arithmetic step of the path is a kernel in
// sum_kernels.cuh / fit_kernels.cuh.  No CPU fallback exists.
#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"
#include "fit_kernels.cuh"
#include "fmm_host.cuh"
#include "geometry.h"
#include "hsma.h"
#include "peak.cuh"
#include "sum_kernels.cuh"
#include "lattice_kernels.cuh"

namespace hsma {
std::atomic<long long> g_launches{0};

#define CU(x)                                     \
    do {                                          \
        if ((x) != cudaSuccess) return HSMA_ERR_CUDA; \
    } while (0)

// bumped whenever any plan buffer is (re)allocated: captured graphs hold raw pointers.  Process-wide and atomic: a bump by
// another plan (another host thread) only drops this plan's graph, it can never be missed.
static std::atomic<size_t> g_alloc_epoch{0};

template <class T>
struct DevBuf {  // growable device buffer owned by the plan
    T* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t n) {
        if (n <= cap) return cudaSuccess;
        ++g_alloc_epoch;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        cudaError_t e = cudaMalloc(&p, n * sizeof(T));
        if (e == cudaSuccess) cap = n;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

static int g_num_sm = 0;
static int num_sm() {
    if (!g_num_sm) {
        int dev = 0;
        cudaGetDevice(&dev);
        if (cudaDeviceGetAttribute(&g_num_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || g_num_sm <= 0)
            g_num_sm = 148;
    }
    return g_num_sm;
}

// Persistent launch shape of one pair kernel (sum_kernels.cuh "work decomposition").
struct Launch {
    int R;            // targets per thread
    int ntb;          // target blocks of kThreads * R
    long long Ub, U;  // units per block / in all
    int G;            // CTAs = min(resident CTAs, U)
    int rows;         // rows of the partial-sum buffer
    PartLayout layout(const double* part, const long long* dyn = nullptr, int cells = 1) const {
        PartLayout L{part, U, Ub, G, kThreads * R};
        L.dyn = dyn; L.cells = cells;
        return L;
    }
};

template <class K>
static int resident_ctas(K kernel) {
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kThreads, 0) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    return per_sm * num_sm();
}
// resident CTAs of near_sum_kernel<R, REFINE, *, FIELD>: the smaller of the two loop forms (one launch shape)
template <int R, int REFINE, bool FIELD>
static int near_resident_of() {
    return std::min(resident_ctas(near_sum_kernel<R, REFINE, false, FIELD>), resident_ctas(near_sum_kernel<R, REFINE, true, FIELD>));
}
static int near_resident(int R, int refine, bool field) {
    static int cache[4][2][2] = {};
    const int i = R == 8 ? 3 : (R == 4 ? 2 : (R == 2 ? 1 : 0)), j = refine == 1 ? 0 : 1, f = field ? 1 : 0;
    int& c = cache[i][j][f];
    if (!c) {
        if (!field) {
            if (refine == 1) c = R == 8 ? near_resident_of<8, 1, false>() : R == 4 ? near_resident_of<4, 1, false>() : R == 2 ? near_resident_of<2, 1, false>() : near_resident_of<1, 1, false>();
            else c = R == 8 ? near_resident_of<8, 2, false>() : R == 4 ? near_resident_of<4, 2, false>() : R == 2 ? near_resident_of<2, 2, false>() : near_resident_of<1, 2, false>();
        } else {  // FIELD: R <= 4
            if (refine == 1) c = R == 4 ? near_resident_of<4, 1, true>() : R == 2 ? near_resident_of<2, 1, true>() : near_resident_of<1, 1, true>();
            else c = R == 4 ? near_resident_of<4, 2, true>() : R == 2 ? near_resident_of<2, 2, true>() : near_resident_of<1, 2, true>();
        }
    }
    return c;
}
static int node_resident(int R, bool field) {
    static int cache[4][2] = {};
    int& c = cache[R == 8 ? 3 : R == 4 ? 2 : (R == 2 ? 1 : 0)][field ? 1 : 0];
    if (!c) {
        if (!field) c = R == 8 ? resident_ctas(node_sum_kernel<8, false>) : R == 4 ? resident_ctas(node_sum_kernel<4, false>) : R == 2 ? resident_ctas(node_sum_kernel<2, false>) : resident_ctas(node_sum_kernel<1, false>);
        else c = R == 4 ? resident_ctas(node_sum_kernel<4, true>) : R == 2 ? resident_ctas(node_sum_kernel<2, true>) : resident_ctas(node_sum_kernel<1, true>);
    }
    return c;
}

// Targets per thread: the largest R in {Rmax, .., 2, 1} that (i) leaves every resident CTA at least 4 units
// and (ii) wastes at most 6 % of its target slots on the padding of the last block; if none qualifies, the
// R with the least padding among those that satisfy (i), else R = 1.
template <class Resident>
static Launch choose_launch(long long T, long long units_per_block, int Rmax, Resident resident) {
    auto shape = [&](int R) {
        Launch L;
        L.R = R;
        L.ntb = (int)((T + (long long)kThreads * R - 1) / ((long long)kThreads * R));
        L.Ub = units_per_block;
        L.U = L.ntb * L.Ub;
        L.G = (int)std::min<long long>(resident(R), L.U);
        L.rows = part_rows(L.U, L.Ub, L.G);
        return L;
    };
    int best = 1;
    double best_fill = 0.0;
    for (int R = Rmax; R >= 1; R /= 2) {
        const Launch L = shape(R);
        if (R > 1 && L.U < 4LL * resident(R)) continue;
        const double fill = (double)T / ((double)L.ntb * kThreads * R);
        if (fill >= 0.94) { best = R; break; }
        if (fill > best_fill + 1e-9) { best_fill = fill; best = R; }
    }
    return shape(best);
}

// The packed sources of one evaluate (pack_sources_kernel) as the pair kernels need them.
struct Packed {
    const Src4* src; long long n_src, n_tiles; const int* tile_np; const int* slot_of; const QInfo* qinfo;
    const long long* dyn = nullptr;   // sphere-culled near set: device-resident {n_src, n_tiles} (n_src, n_tiles above are estimates)
};

template <bool UNIFORM, bool FIELD>
static void launch_near_form(const Launch& L, int refine, const NearArgs& a, cudaStream_t st) {
#define NEAR_LAUNCH(K)                                                                                   \
    do {                                                                                                 \
        if (refine == 1) {                                                                               \
            if (L.R == 8) { if (!FIELD) K<8, 1, UNIFORM, false><<<L.G, kThreads, 0, st>>>(a); }          \
            else if (L.R == 4) K<4, 1, UNIFORM, FIELD><<<L.G, kThreads, 0, st>>>(a);                     \
            else if (L.R == 2) K<2, 1, UNIFORM, FIELD><<<L.G, kThreads, 0, st>>>(a);                     \
            else K<1, 1, UNIFORM, FIELD><<<L.G, kThreads, 0, st>>>(a);                                   \
        } else {                                                                                         \
            if (L.R == 8) { if (!FIELD) K<8, 2, UNIFORM, false><<<L.G, kThreads, 0, st>>>(a); }          \
            else if (L.R == 4) K<4, 2, UNIFORM, FIELD><<<L.G, kThreads, 0, st>>>(a);                     \
            else if (L.R == 2) K<2, 2, UNIFORM, FIELD><<<L.G, kThreads, 0, st>>>(a);                     \
            else K<1, 2, UNIFORM, FIELD><<<L.G, kThreads, 0, st>>>(a);                                   \
        }                                                                                                \
    } while (0)
    if (a.dyn) NEAR_LAUNCH(near_sum_dyn_kernel);   // sphere-culled near set: device-resident source count
    else NEAR_LAUNCH(near_sum_kernel);
#undef NEAR_LAUNCH
    HSMA_COUNT_LAUNCH();
}

// part must hold L.rows * T doubles (x 4 with field).  tgt_index: null, or the row of each target inside tgt.
static void launch_near(const Launch& L, bool field, const double* tgt, int tstride, const int* tgt_index, long long T,
                        long long t_first, const Packed& P, const Cell* cells, int C, long long self_offset, int refine,
                        double* part, cudaStream_t st) {
    NearArgs a;
    a.tgt = tgt; a.tstride = tstride; a.tgt_index = tgt_index; a.T = T; a.t_first = t_first;
    a.src = P.src; a.n_src = P.n_src; a.n_tiles = P.n_tiles; a.tile_np = P.tile_np; a.slot_of = P.slot_of; a.qinfo = P.qinfo;
    a.cells = cells; a.C = C; a.units = L.U; a.self_offset = self_offset; a.dyn = P.dyn; a.ntb = L.ntb;
    a.scale = refine == 1 ? 0.5 : 1.0; a.scale_grad = refine == 1 ? -0.125 : -1.0; a.part = part;
    // generic form always; the uniform-|q| form too when the charge statistics are available (each returns at
    // once unless QInfo.uniform selects it)
    if (field) {
        launch_near_form<false, true>(L, refine, a, st);
        if (a.qinfo) launch_near_form<true, true>(L, refine, a, st);
    } else {
        launch_near_form<false, false>(L, refine, a, st);
        if (a.qinfo) launch_near_form<true, false>(L, refine, a, st);
    }
}
// Ordered pairs, lattice-factored (lattice_kernels.cuh near_lat_sum_kernel): R in {2, 1} -- the 27+ image chains of one
// pair already fill the FP64 pipe, so more targets per thread buy nothing -- and units of kLatChunk sources.
using LatNearFn = void (*)(const NearArgs, const LatGeom);
static LatNearFn lat_near_fn(int R, int refine, bool field, int shape) {
#define HSMA_LAT_SHAPE(RR, RF, FD)                                                          \
    (shape == 1 ? (LatNearFn)near_lat_sum_kernel<RR, RF, FD, 1, 1, 1, 0>                    \
                : shape == 2 ? (LatNearFn)near_lat_sum_kernel<RR, RF, FD, 1, 1, 1, 7>       \
                : shape == 4 ? (LatNearFn)near_lat_sum_kernel<RR, RF, FD, 1, 1, 1, 4>       \
                             : (LatNearFn)near_lat_sum_kernel<RR, RF, FD, 1, 1, 2, 4>)
    if (R == 2) {
        if (refine == 1) return field ? HSMA_LAT_SHAPE(2, 1, true) : HSMA_LAT_SHAPE(2, 1, false);
        return field ? HSMA_LAT_SHAPE(2, 2, true) : HSMA_LAT_SHAPE(2, 2, false);
    }
    if (refine == 1) return field ? HSMA_LAT_SHAPE(1, 1, true) : HSMA_LAT_SHAPE(1, 1, false);
    return field ? HSMA_LAT_SHAPE(1, 2, true) : HSMA_LAT_SHAPE(1, 2, false);
#undef HSMA_LAT_SHAPE
}
static int lat_near_resident(int R, int refine, bool field, int shape) {
    static int cache[2][2][2][5] = {};
    int& c = cache[R == 2 ? 1 : 0][refine == 1 ? 0 : 1][field ? 1 : 0][shape];
    if (!c) c = resident_ctas(lat_near_fn(R, refine, field, shape));
    return c;
}
static Launch choose_near_lat(long long T, long long n_tiles, int refine, bool field, int shape) {
    return choose_launch(T, n_tiles * kLatChunks, 2, [=](int R) { return lat_near_resident(R, refine, field, shape); });
}
static void launch_near_lat(const Launch& L, bool field, const double* tgt, int tstride, const int* tgt_index, long long T,
                            long long t_first, const Packed& P, long long self_offset, int refine, int shape, LatGeom g,
                            double* part, cudaStream_t st) {
    NearArgs a;
    a.tgt = tgt; a.tstride = tstride; a.tgt_index = tgt_index; a.T = T; a.t_first = t_first;
    a.src = P.src; a.n_src = P.n_src; a.n_tiles = P.n_tiles; a.tile_np = P.tile_np; a.slot_of = P.slot_of; a.qinfo = nullptr;
    a.cells = nullptr; a.C = kLatChunks; a.units = L.U; a.self_offset = self_offset; a.dyn = nullptr; a.ntb = L.ntb;
    a.scale = refine == 1 ? 0.5 : 1.0; a.scale_grad = 0.0; a.part = part;
    for (int m = 0; m < 8; ++m) g.wpow[m] *= a.scale;
    g.cgrad = refine == 1 ? 0.125 : 1.0;
    lat_near_fn(L.R, refine, field, shape)<<<L.G, kThreads, 0, st>>>(a, g);
    HSMA_COUNT_LAUNCH();
}
static Launch choose_near(long long T, long long n_tiles, int C, int refine, bool field = false) {
    return choose_launch(T, n_tiles * C, field ? 4 : 8, [refine, field](int R) { return near_resident(R, refine, field); });
}

// Symmetric form of step (b) (sum_kernels.cuh near_sym_kernel): launch shape and buffers.  The fine units of one rank
// are walked in `waves` (launches) of at most wave_fine units each, so that the column-sum scratch (one 2 KB line per
// visit of a wave; 8 KB with the gradient) stays below the plan's cap whatever N is: O(N) memory, DESIGN.md 6.12.
struct SymLaunch {
    int n_blocks, rows, chunks;
    long long visits, f_begin, fine;
    int n_waves, resident;
    long long wave_fine;       // fine units per wave (the last one takes what is left)
    long long wave_visits;     // column lines to reserve: max over waves of (last visit - first visit + 1)
    int wave_blocks;           // row-sum blocks to reserve: max over waves of the blocks a wave touches
};
constexpr size_t kSymColCapDefault = 64u << 20;   // bytes of column scratch per wave (fits L2 beside the sources)
static int sym_resident(int refine) {
    static int cache[2] = {0, 0};
    int& c = cache[refine == 1 ? 0 : 1];
    if (!c) c = refine == 1 ? resident_ctas(near_sym_kernel<1>) : resident_ctas(near_sym_kernel<2>);
    return c;
}
// Kernels with more than 48 KB of shared memory: raise the limit once per kernel AND per device (a function attribute
// belongs to the device that was current when it was set; one mask per call site, bit = device ordinal mod 64).
template <class K>
static void ensure_dyn_smem(K kernel, int bytes, std::atomic<unsigned long long>& done) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); dev = 0; }
    const unsigned long long bit = 1ull << (dev & 63);
    if (done.load(std::memory_order_relaxed) & bit) return;
    if (cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) != cudaSuccess) cudaGetLastError();
    done.fetch_or(bit, std::memory_order_relaxed);
}
template <int REFINE>
static void ensure_sym_field_smem() {
    static std::atomic<unsigned long long> done{0};
    ensure_dyn_smem(near_sym_field_kernel<REFINE>, kSymFieldDynSmem, done);
}
// the gradient form needs 64 KB of dynamic shared memory
template <int REFINE>
static int sym_field_resident_of() {
    ensure_sym_field_smem<REFINE>();
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, near_sym_field_kernel<REFINE>, kThreads, kSymFieldDynSmem) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    return per_sm * num_sm();
}
static int sym_field_resident(int refine) {
    static int cache[2] = {0, 0};
    int& c = cache[refine == 1 ? 0 : 1];
    if (!c) c = refine == 1 ? sym_field_resident_of<1>() : sym_field_resident_of<2>();
    return c;
}
static int sym_block_of_visit(long long v, long long n_tiles, int n_blocks) {
    int lo = 0, hi = n_blocks - 1;   // largest I with sym_visit0(I) <= v
    while (lo < hi) {
        const int mid = (lo + hi + 1) / 2;
        if (sym_visit0(mid, n_tiles) <= v) lo = mid; else hi = mid - 1;
    }
    return lo;
}
// wave w of a launch shape
static SymWave sym_wave(const SymLaunch& L, long long n_tiles, int w) {
    SymWave W;
    W.f_begin = L.f_begin + (long long)w * L.wave_fine;
    W.fine = std::min(L.wave_fine, L.f_begin + L.fine - W.f_begin);
    W.v_base = W.f_begin / L.chunks;
    const long long v_last = (W.f_begin + W.fine - 1) / L.chunks;
    W.blk_lo = sym_block_of_visit(W.v_base, n_tiles, L.n_blocks);
    W.blk_hi = sym_block_of_visit(v_last, n_tiles, L.n_blocks);
    W.G = (int)std::max<long long>(1, std::min<long long>(L.resident, W.fine));
    W.first = w == 0;
    return W;
}
// part / n_parts: the contiguous share [F * part / n_parts, F * (part + 1) / n_parts) of the F fine units (multi-GPU)
static SymLaunch choose_sym(long long n_tiles, int refine, size_t col_cap_bytes, int part = 0, int n_parts = 1, bool field = false) {
    SymLaunch L;
    L.chunks = field ? kSymFChunks : kSymChunks;
    L.n_blocks = (int)((n_tiles + kSymR - 1) / kSymR);
    L.visits = sym_visit0(L.n_blocks, n_tiles);
    const long long F = L.visits * L.chunks;
    L.f_begin = F * part / n_parts;
    L.fine = F * (part + 1) / n_parts - L.f_begin;
    L.resident = field ? sym_field_resident(refine) : sym_resident(refine);
    // waves: equal shares of the fine units, each spanning at most cap / line bytes visits (and at least 2 visits)
    const long long line = (long long)kTile * sizeof(double) * (field ? 4 : 1);
    const long long cap_visits = std::max<long long>(2, (long long)(col_cap_bytes / (size_t)line));
    const long long my_visits = L.fine > 0 ? (L.f_begin + L.fine - 1) / L.chunks - L.f_begin / L.chunks + 1 : 0;
    L.n_waves = (int)std::max<long long>(1, (my_visits + cap_visits - 2) / (cap_visits - 1));
    L.wave_fine = std::max<long long>(1, (L.fine + L.n_waves - 1) / L.n_waves);
    L.n_waves = L.fine > 0 ? (int)((L.fine + L.wave_fine - 1) / L.wave_fine) : 0;
    L.rows = 1; L.wave_visits = 1; L.wave_blocks = 1;
    for (int w = 0; w < L.n_waves; ++w) {
        const SymWave W = sym_wave(L, n_tiles, w);
        L.wave_visits = std::max(L.wave_visits, (W.f_begin + W.fine - 1) / L.chunks - W.v_base + 1);
        L.wave_blocks = std::max(L.wave_blocks, W.blk_hi - W.blk_lo + 1);
        for (int I = W.blk_lo; I <= W.blk_hi; ++I) {
            const long long lo = std::max(sym_visit0(I, n_tiles) * L.chunks, W.f_begin);
            const long long hi = std::min(sym_visit0(I + 1, n_tiles) * L.chunks, W.f_begin + W.fine);
            if (lo >= hi) continue;
            const int first = cta_of_unit(lo - W.f_begin, W.fine, W.G), last = cta_of_unit(hi - 1 - W.f_begin, W.fine, W.G);
            L.rows = std::max(L.rows, last - first + 1);
        }
    }
    return L;
}
// The symmetric form pays when most visits are off the diagonal (a diagonal visit costs 11 instructions per ORDERED
// pair): from 32 source tiles on, and while the cell table fits its shared-memory copy.
// (the gradient form breaks even at 32 tiles too: 1.01x at N = 8192, 1.13x at 16,384, 1.26x at 262,144)
static bool sym_applies(long long n_tiles, int C) { return n_tiles >= 32 && C <= kSymMaxCells; }

static Launch choose_node(long long T, long long n_tiles, bool field = false) {
    return choose_launch(T, n_tiles, field ? 4 : 8, [field](int R) { return node_resident(R, field); });
}
static void launch_node(const Launch& L, bool field, const double* tgt, int tstride, const int* tgt_index, long long T,
                        long long t_first, const Node8* nodes, long long n_tiles, double* part, cudaStream_t st) {
    NodeArgs a;
    a.tgt = tgt; a.tstride = tstride; a.tgt_index = tgt_index; a.T = T; a.t_first = t_first; a.nodes = nodes; a.n_tiles = n_tiles;
    a.units = L.U; a.part = part;
    if (field) {
        if (L.R == 4) node_sum_kernel<4, true><<<L.G, kThreads, 0, st>>>(a);
        else if (L.R == 2) node_sum_kernel<2, true><<<L.G, kThreads, 0, st>>>(a);
        else node_sum_kernel<1, true><<<L.G, kThreads, 0, st>>>(a);
    } else {
        if (L.R == 8) node_sum_kernel<8, false><<<L.G, kThreads, 0, st>>>(a);
        else if (L.R == 4) node_sum_kernel<4, false><<<L.G, kThreads, 0, st>>>(a);
        else if (L.R == 2) node_sum_kernel<2, false><<<L.G, kThreads, 0, st>>>(a);
        else node_sum_kernel<1, false><<<L.G, kThreads, 0, st>>>(a);
    }
    HSMA_COUNT_LAUNCH();
}

}  // namespace hsma

using namespace hsma;

// Lattice-factored kernels (lattice_kernels.cuh): the shapes instantiated, by (near_shell, reflecting axes).
static int lat_shape_of(const int shell[3], const bool refl[3]) {
    const int mask = (refl[0] ? 1 : 0) | (refl[1] ? 2 : 0) | (refl[2] ? 4 : 0);
    if (shell[0] == 1 && shell[1] == 1 && shell[2] == 1 && mask == 0) return 1;
    if (shell[0] == 1 && shell[1] == 1 && shell[2] == 1 && mask == 7) return 2;
    if (shell[0] == 1 && shell[1] == 1 && shell[2] == 2 && mask == 4) return 3;
    if (shell[0] == 1 && shell[1] == 1 && shell[2] == 1 && mask == 4) return 4;
    return 0;
}

struct hsma_plan {
    hsma_plan_desc d;
    cudaStream_t stream = nullptr;
    double R0 = 0.0, half[3] = {0, 0, 0};
    bool pairs = false;       // fully periodic: all rows are differences x_i / x~_i, constant column dropped
    bool slab_bc = false;     // grounded slab: pair rows wrapped in x,y + Dirichlet rows on the plates
    int drop = 0;             // 1: the constant column is dropped, A_00 = 0
    bool neumann = false;     // gamma = +1 walls: derivative rows
    bool face_pairs = false;  // periodic kind closed by value + normal-derivative pairs on opposite faces
    bool need_grad = false;   // some row is a derivative row: step (a) runs its FIELD form
    RowDesc* row_desc = nullptr;  // [rows]
    double* pcg = nullptr;    // [Kt,3] grad Phi_in at the check targets (need_grad)
    bool need_neutral = false;
    int rows = 0, ncol = 0, Kt = 0, C_near = 0, C_rhs = 0, refine = 1;
    long long node_tiles = 0;
    double rhs_sign = -1.0;
    // plan-owned device data
    Cell* cells_near = nullptr;
    Cell* cell_identity = nullptr;   // one cell: no shift, weight 1, central (sphere-culled near set)
    int* cell_order = nullptr;       // central cell first (sphere-culled near set)
    bool sphere = false;
    double fd_dr = 0.0;              // > 0: three-sphere dipole
    long long n_node_records = 0, last_images = 0;
    // image list of the sphere-culled near set (grown as needed)
    DevBuf<long long> img_counts;
    DevBuf<double> img_xyz, img_q, img_stats;
    DevBuf<Src4> img_src;
    DevBuf<int> img_slot_of, img_tile_np;
    QInfo* img_qinfo = nullptr;
    long long* img_dyn = nullptr;    // device {images inside the sphere, their tiles} of the last evaluate
    Cell* cells_rhs = nullptr;   // == cells_near for the boundary closure
    double* chk = nullptr;       // [Kt,3]
    double* nrm = nullptr;       // [M,3]
    double* wq = nullptr;        // [M]
    Node8* nodes = nullptr;      // packed, padded
    double *Fm = nullptr, *tau = nullptr, *Qm = nullptr, *Rm = nullptr, *Pinv = nullptr;
    double *pc = nullptr, *rhs = nullptr, *cvec = nullptr, *A_full = nullptr, *scalars = nullptr;  // scalars[8]
    int* flags = nullptr;        // [0] rank deficient, [1] not neutral
    // scratch grown to the largest N seen
    DevBuf<Src4> src;
    DevBuf<int> slot_of, tile_np;
    QInfo* qinfo = nullptr;
    DevBuf<double> part_a, part_b, part_c, red, xyz_in, q_in, phi_dev, force_dev;
    DevBuf<double> sym_col, sym_phi;   // symmetric form of step (b): column sums per visit of one wave, phi_near in source order
    int lat_shape = 0;           // lattice-factored kernels (lattice_kernels.cuh): 0 none, else index into the instantiated shapes
    bool lat_on = true;          // hsma_plan_set_image_factoring
    LatGeom lat;                 // shifts k L_a and gamma^m (unscaled)
    size_t sym_col_cap = kSymColCapDefault;   // hsma_plan_set_sym_scratch_cap: bytes of column scratch per wave
    hsma::fmm::State fmm;              // near_algorithm = FMM: tables and scratch of the sub-quadratic form of step (b)
    long long fmm_min_N = 0;           // near_algorithm = AUTO: the FMM from this N on
    int pair_form = 0;                 // hsma_plan_set_pair_form: 0 = automatic, 1 = ordered pairs only, 2 = symmetric wherever possible
    int last_pair_form = 1;            // what the last evaluate used for step (b): 1 ordered, 2 symmetric
    long long last_launches = 0;
    hsma_status sticky = HSMA_OK;
    // CUDA graph of the whole evaluate: captured on the second call with identical arguments,
    // replayed while the arguments and every plan buffer stay the same
    struct GraphKey {
        const void *xyz = nullptr, *q = nullptr, *phi = nullptr, *U = nullptr, *F = nullptr;
        long long N = -1, t0 = 0, t1 = 0;
        bool operator==(const GraphKey& o) const {
            return xyz == o.xyz && q == o.q && phi == o.phi && U == o.U && F == o.F && N == o.N && t0 == o.t0 && t1 == o.t1;
        }
    };
    GraphKey gkey_seen, gkey;
    size_t gepoch_seen = 0, gepoch = 0;
    cudaGraphExec_t gexec = nullptr;
    long long glaunches = 0, greplays = 0;
    // stage timing (hsma_plan_set_timing): events ev[0..7] bracket the stages of one evaluate
    bool timing = false;
    cudaEvent_t ev[10] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    bool last_far_timed = false;       // ev[7], ev[8] bracket the FMM far field of the last evaluate
    bool ev_valid = false;
};

// ------------------------------------------------------------------------------------------------
// plan
// ------------------------------------------------------------------------------------------------
static void plan_free(hsma_plan* p) {
    if (!p) return;
    if (p->cells_rhs && p->cells_rhs != p->cells_near) cudaFree(p->cells_rhs);
    void* ptrs[] = {p->cells_near, p->chk, p->nrm, p->wq, p->nodes, p->Fm, p->tau, p->Qm, p->Rm, p->Pinv,
                    p->pc, p->rhs, p->cvec, p->A_full, p->scalars, p->flags};
    for (void* q : ptrs) if (q) cudaFree(q);
    p->src.release(); p->slot_of.release(); p->tile_np.release(); if (p->qinfo) cudaFree(p->qinfo);
    if (p->cell_identity) cudaFree(p->cell_identity);
    if (p->row_desc) cudaFree(p->row_desc);
    if (p->pcg) cudaFree(p->pcg);
    if (p->cell_order) cudaFree(p->cell_order);
    if (p->img_qinfo) cudaFree(p->img_qinfo);
    if (p->img_dyn) cudaFree(p->img_dyn);
    p->img_counts.release(); p->img_xyz.release(); p->img_q.release(); p->img_stats.release(); p->img_src.release();
    p->img_slot_of.release(); p->img_tile_np.release();
    p->part_a.release(); p->part_b.release(); p->part_c.release(); p->red.release(); p->sym_col.release(); p->sym_phi.release();
    p->xyz_in.release(); p->q_in.release(); p->phi_dev.release(); p->force_dev.release();
    p->fmm.release();
    for (cudaEvent_t e : p->ev) if (e) cudaEventDestroy(e);
    if (p->gexec) cudaGraphExecDestroy(p->gexec);
    delete p;
}

template <class T>
static cudaError_t upload(T** dst, const std::vector<T>& v, cudaStream_t st) {
    cudaError_t e = cudaMalloc(dst, std::max<size_t>(1, v.size()) * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpyAsync(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice, st);
}

extern "C" hsma_status hsma_plan_create_ex(const hsma_plan_desc* desc, void* cuda_stream, hsma_plan** plan_out) {
    if (!desc || !plan_out || desc->struct_size != sizeof(hsma_plan_desc)) return HSMA_ERR_INVALID_ARG;
    const hsma_plan_desc& d = *desc;
    if (d.kind < 0 || d.kind > 2 || d.p < 1 || d.p > kMaxP || d.M < 8 || d.K < 1) return HSMA_ERR_INVALID_ARG;
    if (d.closure != HSMA_CLOSURE_BOUNDARY && d.closure != HSMA_CLOSURE_FAR_DATA && d.closure != HSMA_CLOSURE_FACE_PAIRS)
        return HSMA_ERR_INVALID_ARG;
    if (d.closure == HSMA_CLOSURE_FACE_PAIRS && d.kind != HSMA_BC_PERIODIC) return HSMA_ERR_INVALID_ARG;
    if (d.rsqrt_refine < 0 || d.rsqrt_refine > 2) return HSMA_ERR_INVALID_ARG;
    if (d.near_mode != HSMA_NEAR_WHOLE_CELLS && d.near_mode != HSMA_NEAR_SPHERE) return HSMA_ERR_INVALID_ARG;
    if (d.dipole_mode != HSMA_DIPOLE_EXACT && d.dipole_mode != HSMA_DIPOLE_FD3) return HSMA_ERR_INVALID_ARG;
    if (d.near_mode == HSMA_NEAR_SPHERE && d.closure == HSMA_CLOSURE_FAR_DATA) return HSMA_ERR_INVALID_ARG;
    if (d.fd_dr_rel < 0.0 || d.fd_dr_rel > 0.1) return HSMA_ERR_INVALID_ARG;
    if (d.near_algorithm != HSMA_NEAR_ALG_DIRECT && d.near_algorithm != HSMA_NEAR_ALG_FMM && d.near_algorithm != HSMA_NEAR_ALG_AUTO)
        return HSMA_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a)
        if (!(d.L[a] > 0.0) || d.near_shell[a] < 0 || d.near_shell[a] > 8) return HSMA_ERR_INVALID_ARG;
    if (d.kind == HSMA_BC_PERIODIC && d.closure == HSMA_CLOSURE_FAR_DATA) return HSMA_ERR_INVALID_ARG;
    if (d.kind != HSMA_BC_PERIODIC && d.closure == HSMA_CLOSURE_BOUNDARY && d.gamma != -1.0 && d.gamma != 1.0)
        return HSMA_ERR_INVALID_ARG;  // reading S16: a dielectric wall has no boundary closure (far-data closure only);
                                      // gamma = -1 closes by Dirichlet rows, gamma = +1 by Neumann rows
    // reading S7: whole-cell near set is valid iff R0 < R_aux <= min_a (s_a + 1/2) L_a
    const double R0 = 0.5 * std::sqrt(d.L[0] * d.L[0] + d.L[1] * d.L[1] + d.L[2] * d.L[2]);
    double bound = 1e300;
    for (int a = 0; a < 3; ++a) bound = std::min(bound, (d.near_shell[a] + 0.5) * d.L[a]);
    if (!(d.R_aux > R0 && d.R_aux <= bound * (1 + 1e-14))) return HSMA_ERR_GEOMETRY;

    hsma_plan* p = new (std::nothrow) hsma_plan;
    if (!p) return HSMA_ERR_ALLOC;
    p->d = d; p->d.check_xyz = nullptr;
    p->stream = (cudaStream_t)cuda_stream;
    p->R0 = R0;
    for (int a = 0; a < 3; ++a) p->half[a] = 0.5 * d.L[a];
    p->pairs = d.kind == HSMA_BC_PERIODIC && d.closure == HSMA_CLOSURE_BOUNDARY;
    p->face_pairs = d.kind == HSMA_BC_PERIODIC && d.closure == HSMA_CLOSURE_FACE_PAIRS;
    p->slab_bc = d.kind == HSMA_BC_SLAB_XY_PERIODIC_Z_MIRROR && d.closure == HSMA_CLOSURE_BOUNDARY;
    p->neumann = d.kind != HSMA_BC_PERIODIC && d.closure == HSMA_CLOSURE_BOUNDARY && d.gamma == 1.0;
    p->need_neutral = (d.kind != HSMA_BC_MIRROR_CAVITY && !p->slab_bc) || p->neumann;   // grounded walls screen a net charge
    p->refine = d.rsqrt_refine;  // 0 = by size, see evaluate_impl
    p->rhs_sign = d.closure == HSMA_CLOSURE_FAR_DATA ? 1.0 : -1.0;
    p->sphere = d.near_mode == HSMA_NEAR_SPHERE;
    p->fd_dr = d.dipole_mode == HSMA_DIPOLE_FD3 ? (d.fd_dr_rel > 0.0 ? d.fd_dr_rel : 1e-5) * d.R_aux : 0.0;
    cudaStream_t st = p->stream;
#define PCU(x) do { if ((x) != cudaSuccess) { plan_free(p); return HSMA_ERR_CUDA; } } while (0)

    // cell tables
    std::vector<Cell> near = make_cells(d.kind, d.L, d.near_shell, d.gamma, nullptr);
    std::vector<Cell> rhsc;
    if (d.closure == HSMA_CLOSURE_FAR_DATA) {
        for (int a = 0; a < 3; ++a) if (d.far_shell[a] < d.near_shell[a] || d.far_shell[a] > 16) { plan_free(p); return HSMA_ERR_INVALID_ARG; }
        rhsc = make_cells(d.kind, d.L, d.far_shell, d.gamma, d.near_shell);
        if (rhsc.empty()) { plan_free(p); return HSMA_ERR_INVALID_ARG; }
    }
    if ((int)near.size() > kMaxCells || (int)rhsc.size() > kMaxCells) { plan_free(p); return HSMA_ERR_INVALID_ARG; }
    p->C_near = (int)near.size();
    PCU(upload(&p->cells_near, near, st));
    {
        bool refl[3];
        reflecting_axes(d.kind, refl);
        p->lat_shape = p->sphere ? 0 : lat_shape_of(d.near_shell, refl);
        for (int a = 0; a < 3; ++a)
            for (int k = -2; k <= 2; ++k) p->lat.sh[a][k + 2] = k * d.L[a];
        for (int m = 0; m < 8; ++m) p->lat.wpow[m] = m == 0 ? 1.0 : std::pow(d.gamma, (double)m);
        for (int a = 0; a < 3; ++a)
            for (int k = -2; k <= 2; ++k) p->lat.wa[a][k + 2] = (refl[a] && k != 0) ? std::pow(d.gamma, (double)std::abs(k)) : 1.0;
        for (int i = 0; i < 5; ++i)
            for (int j = 0; j < 5; ++j) p->lat.wxy[i][j] = p->lat.wa[0][i] * p->lat.wa[1][j];
        p->lat.cgrad = 1.0;
    }
    if (p->sphere) {
        Cell id;
        id.sx = id.sy = id.sz = 0.0; id.w = 1.0; id.fx = id.fy = id.fz = 0; id.central = 1;
        PCU(upload(&p->cell_identity, std::vector<Cell>(1, id), st));
        std::vector<int> order;
        for (int c = 0; c < (int)near.size(); ++c) if (near[c].central) order.push_back(c);
        for (int c = 0; c < (int)near.size(); ++c) if (!near[c].central) order.push_back(c);
        PCU(upload(&p->cell_order, order, st));
        PCU(cudaMalloc(&p->img_qinfo, sizeof(QInfo)));
        PCU(cudaMalloc(&p->img_dyn, 2 * sizeof(long long)));
        PCU(cudaMemsetAsync(p->img_dyn, 0, 2 * sizeof(long long), st));
    }
    if (d.near_algorithm == HSMA_NEAR_ALG_FMM || d.near_algorithm == HSMA_NEAR_ALG_AUTO) {
        bool refl[3];
        reflecting_axes(d.kind, refl);
        const hsma_status fs = fmm::setup(p->fmm, d, refl, st);
        if (fs != HSMA_OK && d.near_algorithm == HSMA_NEAR_ALG_FMM) { plan_free(p); return fs; }
        if (fs != HSMA_OK) { p->fmm.release(); p->fmm.enabled = false; cudaGetLastError(); }   // AUTO: the direct sum serves this geometry
        p->fmm_min_N = d.near_algorithm == HSMA_NEAR_ALG_AUTO ? 36864 : 0;
    }
    if (rhsc.empty()) { p->cells_rhs = p->cells_near; p->C_rhs = p->C_near; }
    else { p->C_rhs = (int)rhsc.size(); PCU(upload(&p->cells_rhs, rhsc, st)); }

    // monitoring points and the rows of the least-squares problem, PAPER.md:74-82 (RowDesc in fit_kernels.cuh)
    const double tol_wall = 1e-12 * std::max({d.L[0], d.L[1], d.L[2]});
    std::vector<double> chk;
    std::vector<RowDesc> rowd;
    if (p->face_pairs) {
        // K points on the lower faces x_a = -L_a/2 and their partners x + L_a e_a on the opposite
        // faces; one value row and one normal-derivative row per pair (value rows alone are rank deficient, S15)
        std::vector<double> x;
        if (d.check_xyz) x.assign(d.check_xyz, d.check_xyz + 3 * (size_t)d.K);
        else { bool use[3] = {true, true, true}; x = default_face_points(d.K, d.L, use, /*lower_only=*/true); }
        std::vector<double> xp = x;
        std::vector<int> axis(d.K, -1);
        for (int i = 0; i < d.K; ++i) {
            for (int a = 0; a < 3 && axis[i] < 0; ++a)
                if (std::fabs(x[3 * (size_t)i + a] + 0.5 * d.L[a]) <= tol_wall) axis[i] = a;
            if (axis[i] < 0) { plan_free(p); return HSMA_ERR_INVALID_ARG; }   // not on a lower face
            xp[3 * (size_t)i + axis[i]] += d.L[axis[i]];
        }
        chk = x; chk.insert(chk.end(), xp.begin(), xp.end());
        for (int i = 0; i < d.K; ++i) rowd.push_back(RowDesc{i, d.K + i, -1, 0});
        for (int i = 0; i < d.K; ++i) rowd.push_back(RowDesc{i, d.K + i, axis[i], 0});
        p->drop = 1;
        p->need_grad = true;
    } else {
        std::vector<double> x;   // the user's / default points: circumsphere points (periodic) or wall points
        if (d.check_xyz) x.assign(d.check_xyz, d.check_xyz + 3 * (size_t)d.K);
        else if (p->pairs) x = fibonacci_checkpoints(d.K, R0);
        else {
            bool use[3] = {!p->slab_bc, !p->slab_bc, true};   // slab: points on the two plates only
            x = default_face_points(d.K, d.L, use);
        }
        int n_pair = 0;
        if (p->pairs || p->slab_bc) {
            // x~ = x - L round(x/L) on the periodic axes; rows with x~ = x carry no information
            const std::vector<double> sph = p->pairs ? x : fibonacci_checkpoints(d.K, R0);
            const int wrap_axes = p->pairs ? 3 : 2;
            std::vector<double> a, b;
            for (int i = 0; i < d.K; ++i) {
                double w[3]; bool moved = false;
                for (int c = 0; c < 3; ++c) {
                    const double v = sph[3 * (size_t)i + c];
                    w[c] = c < wrap_axes ? v - d.L[c] * std::nearbyint(v / d.L[c]) : v;
                    moved = moved || std::fabs(v - w[c]) > 0.0;
                }
                if (!moved) continue;
                for (int c = 0; c < 3; ++c) { a.push_back(sph[3 * (size_t)i + c]); b.push_back(w[c]); }
            }
            n_pair = (int)(a.size() / 3);
            chk = a; chk.insert(chk.end(), b.begin(), b.end());
            for (int i = 0; i < n_pair; ++i) rowd.push_back(RowDesc{i, n_pair + i, -1, 0});
        }
        if (!p->pairs) {   // wall rows (cavity, slab) or data rows (far-data closure)
            const int first_axis = d.kind == HSMA_BC_MIRROR_CAVITY ? 0 : 2;
            for (int i = 0; i < d.K; ++i) {
                int axis = -1;
                if (p->neumann) {   // the wall the point lies on: the reflecting axis with |x_a| = L_a/2
                    for (int a = first_axis; a < 3 && axis < 0; ++a)
                        if (std::fabs(std::fabs(x[3 * (size_t)i + a]) - 0.5 * d.L[a]) <= tol_wall) axis = a;
                    if (axis < 0) { plan_free(p); return HSMA_ERR_INVALID_ARG; }   // a wall point that is on no wall
                }
                rowd.push_back(RowDesc{2 * n_pair + i, -1, axis, 0});
            }
            chk.insert(chk.end(), x.begin(), x.end());
        }
        p->drop = (p->pairs || p->neumann) ? 1 : 0;   // no row sees the constant harmonic
        p->need_grad = p->neumann;
    }
    p->rows = (int)rowd.size();
    p->Kt = (int)(chk.size() / 3);
    p->ncol = d.p * d.p - p->drop;
    if (p->rows < p->ncol || p->ncol < 1) { plan_free(p); return HSMA_ERR_RANK_DEFICIENT; }
    PCU(upload(&p->chk, chk, st));
    PCU(upload(&p->row_desc, rowd, st));

    // integration nodes
    std::vector<double> nrm, wq;
    if (!make_nodes(d.M, d.R_aux, d.quad_rule, nrm, wq)) { plan_free(p); return HSMA_ERR_INVALID_ARG; }
    PCU(upload(&p->nrm, nrm, st));
    PCU(upload(&p->wq, wq, st));
    constexpr int kNT = kTile / 2;
    p->n_node_records = p->fd_dr > 0.0 ? 3LL * d.M : d.M;
    p->node_tiles = (p->n_node_records + kNT - 1) / kNT;
    {
        std::vector<Node8> pad((size_t)p->node_tiles * kNT);
        for (auto& n : pad) { n.x = n.y = n.z = kFar; n.q = n.px = n.py = n.pz = n.pad = 0.0; }
        PCU(upload(&p->nodes, pad, st));
    }

    // fitting matrix and its QR (device)
    const size_t mn = (size_t)p->rows * p->ncol;
    PCU(cudaMalloc(&p->Fm, mn * sizeof(double)));
    PCU(cudaMalloc(&p->Qm, mn * sizeof(double)));
    PCU(cudaMalloc(&p->Rm, (size_t)p->ncol * p->ncol * sizeof(double)));
    PCU(cudaMalloc(&p->Pinv, mn * sizeof(double)));
    PCU(cudaMalloc(&p->tau, p->ncol * sizeof(double)));
    PCU(cudaMalloc(&p->pc, p->Kt * sizeof(double)));
    if (p->need_grad) PCU(cudaMalloc(&p->pcg, 3 * (size_t)p->Kt * sizeof(double)));
    PCU(cudaMalloc(&p->rhs, p->rows * sizeof(double)));
    PCU(cudaMalloc(&p->cvec, p->ncol * sizeof(double)));
    PCU(cudaMalloc(&p->A_full, d.p * d.p * sizeof(double)));
    PCU(cudaMalloc(&p->scalars, 8 * sizeof(double)));
    PCU(cudaMalloc(&p->flags, 4 * sizeof(int)));
    PCU(cudaMalloc(&p->qinfo, sizeof(QInfo)));
    PCU(cudaMemsetAsync(p->flags, 0, 4 * sizeof(int), st));
    PCU(cudaMemsetAsync(p->A_full, 0, d.p * d.p * sizeof(double), st));
    build_fit_matrix_kernel<<<(p->rows + 127) / 128, 128, 0, st>>>(p->chk, p->row_desc, p->rows, p->drop, d.p, 1.0 / R0, p->Fm);
    HSMA_COUNT_LAUNCH();
    householder_qr_kernel<<<1, 1024, 0, st>>>(p->Fm, p->rows, p->ncol, p->tau, p->Qm, p->Rm, p->flags);
    HSMA_COUNT_LAUNCH();
    pinv_kernel<<<(p->rows + 63) / 64, 64, 0, st>>>(p->Qm, p->Rm, p->rows, p->ncol, p->Pinv);
    HSMA_COUNT_LAUNCH();
    int hflags[4] = {0, 0, 0, 0};
    PCU(cudaMemcpyAsync(hflags, p->flags, sizeof(hflags), cudaMemcpyDeviceToHost, st));
    PCU(cudaStreamSynchronize(st));
    PCU(cudaGetLastError());
    if (hflags[0]) { plan_free(p); return HSMA_ERR_RANK_DEFICIENT; }
#undef PCU
    *plan_out = p;
    return HSMA_OK;
}

extern "C" hsma_status hsma_plan_create(double L, int boundary_kind, int near_shell, double R_aux, int p, int M_fib,
                                        void* cuda_stream, hsma_plan** plan_out) {
    hsma_plan_desc d;
    std::memset(&d, 0, sizeof(d));
    d.struct_size = sizeof(d);
    d.kind = boundary_kind;
    for (int a = 0; a < 3; ++a) { d.L[a] = L; d.near_shell[a] = near_shell; }
    d.gamma = boundary_kind == HSMA_BC_PERIODIC ? 1.0 : -1.0;
    d.R_aux = R_aux; d.p = p; d.M = M_fib;
    d.K = 2 * p * p;  // PAPER.md:163 N_m = 2 P^2
    d.closure = HSMA_CLOSURE_BOUNDARY;
    d.quad_rule = HSMA_QUAD_SPIRAL;
    if (boundary_kind == HSMA_BC_SLAB_XY_PERIODIC_Z_MIRROR) return HSMA_ERR_INVALID_ARG;  // needs far_shell: use _ex
    return hsma_plan_create_ex(&d, cuda_stream, plan_out);
}

extern "C" hsma_status hsma_plan_destroy(hsma_plan* plan) {
    if (!plan) return HSMA_ERR_INVALID_ARG;
    cudaStreamSynchronize(plan->stream);
    plan_free(plan);
    return HSMA_OK;
}

// ------------------------------------------------------------------------------------------------
// evaluate (update step; Table I)
// ------------------------------------------------------------------------------------------------
namespace hsma {
__global__ void unpack_nodes_kernel(const Node8* __restrict__ n, int M, double* __restrict__ Q, double* __restrict__ P) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= M) return;
    if (Q) Q[j] = n[j].q;
    if (P) { P[3 * j] = n[j].px; P[3 * j + 1] = n[j].py; P[3 * j + 2] = n[j].pz; }
}
__global__ void node_positions_kernel(const double* __restrict__ nrm, double R, int M, double* __restrict__ xyz) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < 3 * M) xyz[j] = R * nrm[j];
}
}  // namespace hsma

// force_out non-null: the FIELD kernels also produce F_i = -q_i grad Phi(r_i)
// Phases of the update step (multi-GPU): the check-point sums of step (a) can be sharded over ranks too.
//   kPhaseAll     the whole evaluate
//   kPhaseCheck   H1 + step (a) for the check targets c0 <= i < c1 only, into the plan's pc (pcg); nothing else
//   kPhaseRest    H1 + fit + mapping + (b) + (c) + finish with the plan's pc (pcg) AS THEY ARE (hsma_set_check_sums)
enum { kPhaseAll = 0, kPhaseCheck = 1, kPhaseRest = 2 };
static bool lat_applies(const hsma_plan* p, const Cell* cells) { return p->lat_on && p->lat_shape != 0 && cells == p->cells_near; }
template <int REFINE, int SX, int SY, int SZ, int MASK>
static void launch_lat_sym_of(int G, const SymArgs& a, const LatGeom& g, cudaStream_t st) {
    static std::atomic<unsigned long long> done{0};
    ensure_dyn_smem(near_lat_sym_kernel<REFINE, SX, SY, SZ, MASK>, kSymWideDynSmem, done);
    near_lat_sym_kernel<REFINE, SX, SY, SZ, MASK><<<G, kSymWideThreads, kSymWideDynSmem, st>>>(a, g);
}
static void launch_lat_sym(int shape, int refine, int G, const SymArgs& a, const LatGeom& g, cudaStream_t st) {
#define HSMA_LAT_SYM(SX, SY, SZ, MASK)                                              \
    do {                                                                            \
        if (refine == 1) launch_lat_sym_of<1, SX, SY, SZ, MASK>(G, a, g, st);       \
        else launch_lat_sym_of<2, SX, SY, SZ, MASK>(G, a, g, st);                   \
    } while (0)
    if (shape == 1) HSMA_LAT_SYM(1, 1, 1, 0);
    else if (shape == 2) HSMA_LAT_SYM(1, 1, 1, 7);
    else if (shape == 4) HSMA_LAT_SYM(1, 1, 1, 4);
    else HSMA_LAT_SYM(1, 1, 2, 4);
#undef HSMA_LAT_SYM
}
template <int REFINE, int SX, int SY, int SZ, int MASK>
static void launch_lat_sym_field_of(int G, const SymArgs& a, const LatGeom& g, cudaStream_t st) {
    static std::atomic<unsigned long long> done{0};
    ensure_dyn_smem(near_lat_sym_field_kernel<REFINE, SX, SY, SZ, MASK>, kLatFieldDynSmem, done);
    near_lat_sym_field_kernel<REFINE, SX, SY, SZ, MASK><<<G, kThreads, kLatFieldDynSmem, st>>>(a, g);
}
static void launch_lat_sym_field(int shape, int refine, int G, const SymArgs& a, const LatGeom& g, cudaStream_t st) {
#define HSMA_LAT_SYMF(SX, SY, SZ, MASK)                                                 \
    do {                                                                                \
        if (refine == 1) launch_lat_sym_field_of<1, SX, SY, SZ, MASK>(G, a, g, st);     \
        else launch_lat_sym_field_of<2, SX, SY, SZ, MASK>(G, a, g, st);                 \
    } while (0)
    if (shape == 1) HSMA_LAT_SYMF(1, 1, 1, 0);
    else if (shape == 2) HSMA_LAT_SYMF(1, 1, 1, 7);
    else if (shape == 4) HSMA_LAT_SYMF(1, 1, 1, 4);
    else HSMA_LAT_SYMF(1, 1, 2, 4);
#undef HSMA_LAT_SYMF
}

// Buffers of the symmetric form (row partials and column sums of ONE wave, near sum in source order); comps = 4 with
// the gradient.  Bounded by the plan's cap on the column scratch: O(N) in all.
static cudaError_t reserve_sym(hsma_plan* p, const SymLaunch& ss, long long N, size_t comps) {
    cudaError_t e = p->part_b.reserve((size_t)ss.rows * ss.wave_blocks * kSymBlock * comps);
    if (e == cudaSuccess) e = p->sym_col.reserve((size_t)ss.wave_visits * kTile * comps);
    if (e == cudaSuccess) e = p->sym_phi.reserve((size_t)N * comps);
    return e;
}
// near_sym(_field)_kernel over the fine units of `ss`, wave by wave, each followed by its gather into p->sym_phi ([N], or
// [4][N] with the gradient): the first wave writes, the others add, in wave order (deterministic).
static void launch_sym(hsma_plan* p, const SymLaunch& ss, bool field, int refine, const Cell* cells, int C, long long N,
                       long long n_tiles, cudaStream_t st) {
    SymArgs a;
    a.src = p->src.p; a.n_src = N; a.n_tiles = n_tiles; a.n_blocks = ss.n_blocks; a.cells = cells; a.C = C;
    a.scale = refine == 1 ? 0.5 : 1.0; a.scale_grad = refine == 1 ? -0.25 : -1.0;
    a.part = p->part_b.p; a.col = p->sym_col.p;
    const unsigned gb = (unsigned)((N + 255) / 256);
    const bool lat = lat_applies(p, cells);
    LatGeom lg = p->lat;
    for (int m = 0; m < 8; ++m) lg.wpow[m] *= a.scale;
    lg.cgrad = refine == 1 ? 0.125 : 1.0;
    if (ss.n_waves == 0) {   // a part with no fine units: its share of the near sum is zero
        cudaMemsetAsync(p->sym_phi.p, 0, (size_t)N * (field ? 4 : 1) * sizeof(double), st);
        return;
    }
    for (int w = 0; w < ss.n_waves; ++w) {
        const SymWave W = sym_wave(ss, n_tiles, w);
        a.f_begin = W.f_begin; a.fine = W.fine; a.v_base = W.v_base; a.blk_base = W.blk_lo; a.part_blocks = W.blk_hi - W.blk_lo + 1;
        if (field) {
            if (lat) launch_lat_sym_field(p->lat_shape, refine, W.G, a, lg, st);
            else if (refine == 1) { ensure_sym_field_smem<1>(); near_sym_field_kernel<1><<<W.G, kThreads, kSymFieldDynSmem, st>>>(a); }
            else { ensure_sym_field_smem<2>(); near_sym_field_kernel<2><<<W.G, kThreads, kSymFieldDynSmem, st>>>(a); }
            HSMA_COUNT_LAUNCH();
            sym_gather_field_kernel<<<gb, 256, 0, st>>>(p->part_b.p, p->sym_col.p, p->slot_of.p, N, n_tiles, W, p->sym_phi.p);
        } else {
            if (lat) launch_lat_sym(p->lat_shape, refine, W.G, a, lg, st);
            else if (refine == 1) near_sym_kernel<1><<<W.G, kThreads, 0, st>>>(a);
            else near_sym_kernel<2><<<W.G, kThreads, 0, st>>>(a);
            HSMA_COUNT_LAUNCH();
            sym_gather_kernel<<<gb, 256, 0, st>>>(p->part_b.p, p->sym_col.p, p->slot_of.p, N, n_tiles, W, p->sym_phi.p);
        }
        HSMA_COUNT_LAUNCH();
    }
}

// part / n_parts (kPhaseRest only, n_parts >= 1 given): the PART form of the multi-GPU path, DESIGN.md 8 -- step (b)
// in symmetric form over this part's share of the fine units, phi_out [N] = that share + step (c) for t0 <= t < t1.
static hsma_status evaluate_impl(hsma_plan* p, const double* xyz, const double* q, long long N, long long t0,
                                 long long t1, double* phi_out, double* energy_out, double* force_out = nullptr,
                                 int phase = kPhaseAll, long long c0 = 0, long long c1 = -1, int part = 0, int n_parts = 0) {
    if (!p || !xyz || !q || N < 1 || t0 < 0 || t1 > N || t0 > t1 ||
        (phase != kPhaseCheck && !phi_out && !force_out && t1 > t0))
        return HSMA_ERR_INVALID_ARG;
    if (phase == kPhaseAll) { c0 = 0; c1 = p->Kt; }
    if (phase == kPhaseCheck && (c0 < 0 || c1 > p->Kt || c0 > c1)) return HSMA_ERR_INVALID_ARG;
    const bool field = force_out != nullptr;
    cudaStream_t st = p->stream;
    const long long before = g_launches;
    const long long n_tiles = (N + kTile - 1) / kTile, Npad = n_tiles * kTile;
    const hsma_plan_desc& d = p->d;

#define MARK(i) do { if (p->timing) cudaEventRecord(p->ev[i], st); } while (0)
    p->ev_valid = false;
    MARK(0);
    // H1 pre-pass: centre + pack + in-tile sign sort; charge statistics (neutrality flag, uniform |q|)
    if (N > 2000000000LL) return HSMA_ERR_INVALID_ARG;  // packed indices are 32-bit
    if (p->src.reserve((size_t)Npad) != cudaSuccess || p->slot_of.reserve((size_t)N) != cudaSuccess ||
        p->tile_np.reserve((size_t)n_tiles) != cudaSuccess)
        return HSMA_ERR_ALLOC;
    if (p->red.reserve((size_t)std::max(4 * n_tiles, (N + 255) / 256 + 1)) != cudaSuccess) return HSMA_ERR_ALLOC;
    pack_sources_kernel<<<(unsigned)n_tiles, kTile, 0, st>>>(xyz, q, N, p->half[0], p->half[1], p->half[2], p->src.p,
                                                           p->slot_of.p, p->tile_np.p, p->red.p);
    charge_stats_kernel<<<1, 1024, 0, st>>>(p->red.p, n_tiles, p->need_neutral ? 1 : 0, p->scalars + 2, p->qinfo, p->flags);
    HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH();
    Packed P{p->src.p, N, n_tiles, p->tile_np.p, p->slot_of.p, p->qinfo};   // what the near sums read
    const Cell *cells_a = p->cells_rhs, *cells_b = p->cells_near;
    int C_a = p->C_rhs, C_b = p->C_near;
    long long n_tiles_near = n_tiles;
    p->last_images = N * (long long)p->C_near;
    const long long* dyn = nullptr;   // sphere-culled near set: device-resident source count of the pair kernels
    long long nt_lo = n_tiles, nt_hi = n_tiles;   // bounds of the source tiles (partial-row allocation)
    if (p->sphere) {
        // paper-literal near set: explicit list of the images inside the sphere, central cell first
        // (image i < N is source i), packed like a source array and summed with the identity cell.  The length of the
        // list stays on the device (img_dyn): buffers are sized for the whole cell table, grids for the worst case
        // (surplus CTAs return), the persistent pair kernels and the finish read the count themselves -- no host
        // synchronisation, so the evaluate can be captured and replayed as a CUDA graph like the other modes.
        const long long entries = (long long)p->C_near * N, blocks = (entries + kTile - 1) / kTile;
        const double R2 = d.R_aux * d.R_aux;
        if (entries > 2000000000LL) return HSMA_ERR_INVALID_ARG;
        const long long nt_max = blocks;
        if (p->img_counts.reserve((size_t)blocks + 1) != cudaSuccess || p->img_xyz.reserve(3 * (size_t)entries) != cudaSuccess ||
            p->img_q.reserve((size_t)entries) != cudaSuccess || p->img_src.reserve((size_t)nt_max * kTile) != cudaSuccess ||
            p->img_slot_of.reserve((size_t)entries) != cudaSuccess || p->img_tile_np.reserve((size_t)nt_max) != cudaSuccess ||
            p->img_stats.reserve(4 * (size_t)nt_max + 2) != cudaSuccess)
            return HSMA_ERR_ALLOC;
        image_count_kernel<<<(unsigned)blocks, kTile, 0, st>>>(xyz, q, N, p->half[0], p->half[1], p->half[2], p->cells_near,
                                                              p->cell_order, p->C_near, R2, p->img_counts.p);
        scan_counts_kernel<<<1, 1024, 0, st>>>(p->img_counts.p, blocks);
        image_finalize_kernel<<<1, 1, 0, st>>>(p->img_counts.p + blocks, N, p->img_dyn, p->flags);
        image_scatter_kernel<<<(unsigned)blocks, kTile, 0, st>>>(xyz, q, N, p->half[0], p->half[1], p->half[2], p->cells_near,
                                                                p->cell_order, p->C_near, R2, p->img_counts.p, p->img_xyz.p,
                                                                p->img_q.p);
        pack_sources_kernel<<<(unsigned)nt_max, kTile, 0, st>>>(p->img_xyz.p, p->img_q.p, entries, 0.0, 0.0, 0.0, p->img_src.p,
                                                               p->img_slot_of.p, p->img_tile_np.p, p->img_stats.p, p->img_dyn);
        charge_stats_kernel<<<1, 1024, 0, st>>>(p->img_stats.p, nt_max, 0, p->img_stats.p + 4 * nt_max, p->img_qinfo, p->flags,
                                                p->img_dyn);
        for (int i = 0; i < 6; ++i) HSMA_COUNT_LAUNCH();
        // host-side ESTIMATE of the list (launch shapes only): the sphere's share of the cell block
        const double vol = 4.18879020478639098 * d.R_aux * d.R_aux * d.R_aux / (d.L[0] * d.L[1] * d.L[2]);
        const long long Ns_est = std::max<long long>(N, std::min<long long>(entries, (long long)(vol * (double)N)));
        const long long nt_img = (Ns_est + kTile - 1) / kTile;
        P = Packed{p->img_src.p, Ns_est, nt_img, p->img_tile_np.p, p->img_slot_of.p, p->img_qinfo, p->img_dyn};
        cells_a = cells_b = p->cell_identity;
        C_a = C_b = 1;
        n_tiles_near = nt_img;
        p->last_images = Ns_est;
        dyn = p->img_dyn;
        nt_lo = n_tiles; nt_hi = nt_max;
    }
    // rows of a partial-sum buffer when the source tiles are only known to lie in [nt_lo, nt_hi] (sphere-culled set)
    auto rows_for = [&](const Launch& L, int C) {
        int r = L.rows;
        if (dyn)
            for (long long nt : {nt_lo, nt_hi, n_tiles_near}) {
                const long long Ub = nt * C, U = (long long)L.ntb * Ub;
                r = std::max(r, part_rows(U, Ub, L.G) + 1);
            }
        return r;
    };

    // near_algorithm = FMM: step (b) over all N targets (potentials) by the fast multipole method; its
    // upward pass (leaf sort, P2M, M2M) comes first because step (a) can use the multipoles too
    const bool use_fmm = p->fmm.enabled && N >= p->fmm_min_N && phase == kPhaseAll && n_parts == 0 && t0 == 0 && t1 == N && p->pair_form == 0;
    if (use_fmm) {
        hsma_status fs = fmm::upward(p->fmm, xyz, q, N, p->half, g_alloc_epoch, st);
        if (fs != HSMA_OK) return fs;
        // the far field of (b) (M2L, L2L) does not depend on the fit either; it comes before step (a) because check
        // targets inside the central cell read their leaf's local expansion.  Timed on its own (ms_out[7]).
        if (p->timing) cudaEventRecord(p->ev[7], st);
        fs = fmm::far_field(p->fmm, N, p->half, g_alloc_epoch, st);
        if (fs != HSMA_OK) return fs;
        if (p->timing) cudaEventRecord(p->ev[8], st);
    }
    p->last_far_timed = use_fmm && p->timing;
    // H2 (a): Phi_in (or the far-cell data) at the monitoring points c0..c1-1 -> pc [Kt]
    if (use_fmm && p->cells_rhs == p->cells_near && !p->need_grad && c1 > c0) {
        // the check targets from the same hierarchy: multipoles of the interaction lists + direct sum over the near leaves
        MARK(1);
        const hsma_status fs = fmm::points(p->fmm, p->chk + 3 * c0, c1 - c0, N, p->half, p->pc + c0, st);
        if (fs != HSMA_OK) return fs;
        MARK(2);
    } else if (phase != kPhaseRest && c1 > c0) {
        const long long Tc = c1 - c0;
        const bool fa = p->need_grad;   // derivative rows need grad Phi_in at the check targets: the FIELD form of (a)
        const bool lat_a = lat_applies(p, cells_a);
        const Launch s = lat_a ? choose_near_lat(Tc, n_tiles_near, 2, fa, p->lat_shape) : choose_near(Tc, n_tiles_near, C_a, 2, fa);
        if (p->part_a.reserve((size_t)rows_for(s, C_a) * Tc * (fa ? 4 : 1)) != cudaSuccess) return HSMA_ERR_ALLOC;
        MARK(1);
        // (a) always cubic: it feeds the fit
        if (lat_a) launch_near_lat(s, fa, p->chk, 3, nullptr, Tc, c0, P, -1, 2, p->lat_shape, p->lat, p->part_a.p, st);
        else launch_near(s, fa, p->chk, 3, nullptr, Tc, c0, P, cells_a, C_a, -1, 2, p->part_a.p, st);
        MARK(2);
        if (fa)
            finish_field_kernel<<<(unsigned)((Tc + 255) / 256), 256, 0, st>>>(s.layout(p->part_a.p, dyn, C_a), PartLayout{nullptr, 1, 1, 1, 1}, Tc, nullptr, nullptr, 0, p->pc + c0, p->pcg + 3 * c0, nullptr);
        else
            finish_phi_kernel<<<(unsigned)((Tc + 255) / 256), 256, 0, st>>>(s.layout(p->part_a.p, dyn, C_a), PartLayout{nullptr, 1, 1, 1, 1}, Tc, nullptr, nullptr, 0, p->pc + c0, nullptr);
        HSMA_COUNT_LAUNCH();
    } else {
        MARK(1); MARK(2);
    }
    if (phase == kPhaseCheck) {
        MARK(3); MARK(4); MARK(5); MARK(6);
        p->ev_valid = p->timing;
        p->last_launches = g_launches - before;
        if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); p->sticky = HSMA_ERR_CUDA; return HSMA_ERR_CUDA; }
        return HSMA_OK;
    }
    // H3: least squares, Eq.(7)
    ls_apply_kernel<<<(p->ncol + 7) / 8, 256, 0, st>>>(p->pc, p->pcg, p->row_desc, p->rows, p->ncol, p->drop, p->rhs_sign,
                                                       p->Pinv, p->rhs, p->A_full);
    HSMA_COUNT_LAUNCH();
    // H4: harmonic surface mapping, Eq.(10),(11) PAPER.md:99-105
    surface_mapping_kernel<<<(d.M + 127) / 128, 128, 0, st>>>(p->A_full, d.p, d.R_aux / p->R0, d.R_aux, p->nrm, p->wq,
                                                              d.M, p->fd_dr, p->nodes);
    HSMA_COUNT_LAUNCH();

    const long long T = t1 - t0;
    if (n_parts > 0) {
        // PART form (multi-GPU): this part's share of the unordered pairs of (b) for ALL targets, (c) for
        // the targets t0..t1-1; phi_out [N] and U add up over the parts
        if (p->sphere || !sym_applies(n_tiles, C_b) || part < 0 || part >= n_parts || (!phi_out && !field)) return HSMA_ERR_INVALID_ARG;
        const int refine = p->refine ? p->refine : ((double)N * (double)p->last_images < 4294967296.0 ? 2 : 1);
        const size_t comps = field ? 4 : 1;
        const SymLaunch ss = choose_sym(n_tiles, refine, p->sym_col_cap, part, n_parts, field);
        if (reserve_sym(p, ss, N, comps) != cudaSuccess) return HSMA_ERR_ALLOC;
        Launch sc{};
        if (T > 0) {
            sc = choose_node(T, p->node_tiles, field);
            if (p->part_c.reserve((size_t)sc.rows * T * comps) != cudaSuccess) return HSMA_ERR_ALLOC;
        }
        p->last_pair_form = 2;
        MARK(3);
        launch_sym(p, ss, field, refine, cells_b, C_b, N, n_tiles, st);
        MARK(4);
        if (T > 0)
            launch_node(sc, field, reinterpret_cast<const double*>(p->src.p), 4, p->slot_of.p, T, t0, p->nodes, p->node_tiles, p->part_c.p, st);
        MARK(5);
        const long long fb = (N + 255) / 256;
        const PartLayout layout_c = T > 0 ? sc.layout(p->part_c.p) : PartLayout{nullptr, 1, 1, 1, 1};
        if (field)
            finish_part_field_kernel<<<(unsigned)fb, 256, 0, st>>>(p->sym_phi.p, layout_c, N, t0, t1, p->src.p, p->slot_of.p, phi_out,
                                                                   force_out, energy_out ? p->red.p : nullptr);
        else
            finish_part_kernel<<<(unsigned)fb, 256, 0, st>>>(p->sym_phi.p, layout_c, N, t0, t1, p->src.p, p->slot_of.p, phi_out,
                                                             energy_out ? p->red.p : nullptr);
        HSMA_COUNT_LAUNCH();
        if (energy_out) {
            reduce_rows_kernel<<<1, 1024, 0, st>>>(p->red.p, fb, 1, 1, 0.5, energy_out);
            HSMA_COUNT_LAUNCH();
        }
    } else if (T > 0) {
        // H5 (b): near images at the sources, self excluded
        const int refine = p->refine ? p->refine : ((double)N * (double)p->last_images < 4294967296.0 ? 2 : 1);
        // rsqrt_refine = 0: the cubic step while (b) is latency-bound anyway (< 2^32 pairs), Newton above
        const size_t comps = field ? 4 : 1;
        bool sym = !use_fmm && !p->sphere && p->pair_form != 1 && t0 == 0 && t1 == N && sym_applies(n_tiles, C_b);
        const bool lat_b = lat_applies(p, cells_b);
        Launch sb = lat_b ? choose_near_lat(T, n_tiles_near, refine, field, p->lat_shape) : choose_near(T, n_tiles_near, C_b, refine, field);
        if (use_fmm && p->sym_phi.reserve((size_t)N * comps) != cudaSuccess) return HSMA_ERR_ALLOC;
        SymLaunch ss{};
        if (sym) {
            ss = choose_sym(n_tiles, refine, p->sym_col_cap, 0, 1, field);
            if (reserve_sym(p, ss, N, comps) != cudaSuccess) {
                // never fail where the ordered kernel would succeed: in automatic mode fall back to it
                cudaGetLastError();
                if (p->pair_form == 2) return HSMA_ERR_ALLOC;
                sym = false;
            }
        }
        if (!sym && !use_fmm && p->part_b.reserve((size_t)rows_for(sb, C_b) * T * comps) != cudaSuccess) return HSMA_ERR_ALLOC;
        p->last_pair_form = use_fmm ? 3 : (sym ? 2 : 1);
        const Launch sc = choose_node(T, p->node_tiles, field);
        if (p->part_c.reserve((size_t)sc.rows * T * comps) != cudaSuccess) return HSMA_ERR_ALLOC;
        MARK(3);
        PartLayout layout_b = sb.layout(p->part_b.p, dyn, C_b);
        if (use_fmm) {
            const hsma_status fs = fmm::leaves(p->fmm, N, p->half, refine, field, p->sym_phi.p, g_alloc_epoch, st);
            if (fs != HSMA_OK) return fs;
            layout_b = PartLayout{p->sym_phi.p, 1, 1, 1, (int)std::min<long long>(T, 2147483647LL)};
        } else if (sym) {
            // every unordered (source, source) pair once: row sums + column sums, then phi_near in source order
            launch_sym(p, ss, field, refine, cells_b, C_b, N, n_tiles, st);
            layout_b = PartLayout{p->sym_phi.p, 1, 1, 1, (int)std::min<long long>(T, 2147483647LL)};
        } else if (lat_b) {
            launch_near_lat(sb, field, reinterpret_cast<const double*>(p->src.p), 4, p->slot_of.p, T, t0, P, t0, refine,
                            p->lat_shape, p->lat, p->part_b.p, st);
        } else {
            launch_near(sb, field, reinterpret_cast<const double*>(p->src.p), 4, p->slot_of.p, T, t0, P, cells_b, C_b,
                        t0, refine, p->part_b.p, st);
        }
        MARK(4);
        // H6 (c): sphere nodes, charge + dipole
        launch_node(sc, field, reinterpret_cast<const double*>(p->src.p), 4, p->slot_of.p, T, t0, p->nodes, p->node_tiles, p->part_c.p, st);
        MARK(5);
        // H7: phi (forces) and U
        const long long fb = (T + 255) / 256;
        if (field)
            finish_field_kernel<<<(unsigned)fb, 256, 0, st>>>(layout_b, sc.layout(p->part_c.p), T, p->src.p, p->slot_of.p, t0,
                                                              phi_out, force_out, energy_out ? p->red.p : nullptr);
        else
            finish_phi_kernel<<<(unsigned)fb, 256, 0, st>>>(layout_b, sc.layout(p->part_c.p), T, p->src.p, p->slot_of.p, t0, phi_out,
                                                            energy_out ? p->red.p : nullptr);
        HSMA_COUNT_LAUNCH();
        if (energy_out) {
            reduce_rows_kernel<<<1, 1024, 0, st>>>(p->red.p, fb, 1, 1, 0.5, energy_out);
            HSMA_COUNT_LAUNCH();
        }
    } else {
        MARK(3); MARK(4); MARK(5);
        if (energy_out && cudaMemsetAsync(energy_out, 0, sizeof(double), st) != cudaSuccess) return HSMA_ERR_CUDA;
    }
    MARK(6);
#undef MARK
    p->ev_valid = p->timing;
    p->last_launches = g_launches - before;
    if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); p->sticky = HSMA_ERR_CUDA; return HSMA_ERR_CUDA; }
    return HSMA_OK;
}

// Whole-evaluate CUDA graph (SURVEY.md 8(d) trap (v): configs 1-3 are launch-latency bound).  The launch sequence
// of an evaluate depends only on (N, t0, t1, force or not) and on pointers; every data-dependent decision (uniform
// |q|, neutrality) is taken on the device.  So: the first call with a given argument set runs normally (and sizes the
// buffers), the second one is captured into a graph, later ones replay it with one cudaGraphLaunch.  Not used on the
// legacy default stream (it cannot be captured), with stage timing on, or with the sphere-culled near set (which
// reads the image count back).  Any reallocation of a plan buffer invalidates the graph.
static hsma_status evaluate_graphed(hsma_plan* p, const double* xyz, const double* q, long long N, long long t0,
                                    long long t1, double* phi_out, double* energy_out, double* force_out) {
    if (!p) return HSMA_ERR_INVALID_ARG;
    cudaStream_t st = p->stream;
    if (st == nullptr || p->timing) return evaluate_impl(p, xyz, q, N, t0, t1, phi_out, energy_out, force_out);
    hsma_plan::GraphKey key;
    key.xyz = xyz; key.q = q; key.phi = phi_out; key.U = energy_out; key.F = force_out; key.N = N; key.t0 = t0; key.t1 = t1;
    if (p->gexec && key == p->gkey && p->gepoch == g_alloc_epoch) {
        if (cudaGraphLaunch(p->gexec, st) != cudaSuccess) { cudaGetLastError(); p->sticky = HSMA_ERR_CUDA; return HSMA_ERR_CUDA; }
        g_launches += p->glaunches;
        p->last_launches = p->glaunches;
        ++p->greplays;
        return HSMA_OK;
    }
    if (key == p->gkey_seen && p->gepoch_seen == g_alloc_epoch) {   // second identical call: capture it
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
            const long long before = g_launches;
            const hsma_status s = evaluate_impl(p, xyz, q, N, t0, t1, phi_out, energy_out, force_out);
            const cudaError_t e = cudaStreamEndCapture(st, &graph);
            const long long captured = g_launches - before;
            g_launches = before;   // nothing has run yet
            if (s == HSMA_OK && e == cudaSuccess && graph && p->gepoch_seen == g_alloc_epoch) {
                if (p->gexec) { cudaGraphExecDestroy(p->gexec); p->gexec = nullptr; }
                if (cudaGraphInstantiate(&p->gexec, graph, 0) == cudaSuccess) {
                    cudaGraphDestroy(graph);
                    p->gkey = key; p->gepoch = g_alloc_epoch; p->glaunches = captured;
                    if (cudaGraphLaunch(p->gexec, st) != cudaSuccess) { cudaGetLastError(); p->sticky = HSMA_ERR_CUDA; return HSMA_ERR_CUDA; }
                    g_launches += captured;
                    p->last_launches = captured;
                    ++p->greplays;
                    return HSMA_OK;
                }
                p->gexec = nullptr;
            }
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            if (s != HSMA_OK) return s;   // argument / allocation error reported as usual, nothing was enqueued
        } else {
            cudaGetLastError();
        }
        p->gkey_seen = hsma_plan::GraphKey();   // capture not possible here: stop trying for this argument set
        return evaluate_impl(p, xyz, q, N, t0, t1, phi_out, energy_out, force_out);
    }
    const hsma_status s = evaluate_impl(p, xyz, q, N, t0, t1, phi_out, energy_out, force_out);
    p->gkey_seen = key;
    p->gepoch_seen = g_alloc_epoch;   // after the call: its own buffer growth is included
    return s;
}

extern "C" hsma_status hsma_evaluate(hsma_plan* plan, const double* xyz, const double* q, long long N, double* phi_out,
                                     double* energy_out) {
    return evaluate_graphed(plan, xyz, q, N, 0, N, phi_out, energy_out, nullptr);
}

extern "C" hsma_status hsma_evaluate_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                           long long t0, long long t1, double* phi_out, double* energy_out) {
    return evaluate_graphed(plan, xyz, q, N, t0, t1, phi_out, energy_out, nullptr);
}

extern "C" hsma_status hsma_evaluate_forces(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                            double* phi_out, double* force_out, double* energy_out) {
    if (!force_out) return HSMA_ERR_INVALID_ARG;
    return evaluate_graphed(plan, xyz, q, N, 0, N, phi_out, energy_out, force_out);
}

extern "C" hsma_status hsma_evaluate_forces_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                                  long long t0, long long t1, double* phi_out, double* force_out,
                                                  double* energy_out) {
    if (!force_out && t1 > t0) return HSMA_ERR_INVALID_ARG;
    if (t1 == t0) return evaluate_impl(plan, xyz, q, N, t0, t1, phi_out, energy_out);
    return evaluate_graphed(plan, xyz, q, N, t0, t1, phi_out, energy_out, force_out);
}

// ---- multi-GPU: step (a) sharded over the check targets --------------------------------------------
extern "C" hsma_status hsma_check_sums_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                             long long c0, long long c1) {
    return evaluate_impl(plan, xyz, q, N, 0, 0, nullptr, nullptr, nullptr, kPhaseCheck, c0, c1);
}
extern "C" hsma_status hsma_get_check_sums(hsma_plan* p, long long c0, long long c1, double* pc_out, double* pcg_out) {
    if (!p || c0 < 0 || c1 > p->Kt || c0 > c1 || !pc_out || (p->need_grad && !pcg_out)) return HSMA_ERR_INVALID_ARG;
    if (c1 == c0) return HSMA_OK;
    CU(cudaMemcpyAsync(pc_out, p->pc + c0, (size_t)(c1 - c0) * sizeof(double), cudaMemcpyDeviceToDevice, p->stream));
    if (p->need_grad) CU(cudaMemcpyAsync(pcg_out, p->pcg + 3 * c0, 3 * (size_t)(c1 - c0) * sizeof(double), cudaMemcpyDeviceToDevice, p->stream));
    return HSMA_OK;
}
extern "C" hsma_status hsma_set_check_sums(hsma_plan* p, long long c0, long long c1, const double* pc_in, const double* pcg_in) {
    if (!p || c0 < 0 || c1 > p->Kt || c0 > c1 || !pc_in || (p->need_grad && !pcg_in)) return HSMA_ERR_INVALID_ARG;
    if (c1 == c0) return HSMA_OK;
    CU(cudaMemcpyAsync(p->pc + c0, pc_in, (size_t)(c1 - c0) * sizeof(double), cudaMemcpyDeviceToDevice, p->stream));
    if (p->need_grad) CU(cudaMemcpyAsync(p->pcg + 3 * c0, pcg_in, 3 * (size_t)(c1 - c0) * sizeof(double), cudaMemcpyDeviceToDevice, p->stream));
    return HSMA_OK;
}
extern "C" hsma_status hsma_evaluate_rest_shard(hsma_plan* plan, const double* xyz, const double* q, long long N,
                                                long long t0, long long t1, double* phi_out, double* force_out,
                                                double* energy_out) {
    return evaluate_impl(plan, xyz, q, N, t0, t1, phi_out, energy_out, force_out, kPhaseRest);
}

extern "C" hsma_status hsma_evaluate_rest_part(hsma_plan* plan, const double* xyz, const double* q, long long N, int part,
                                               int n_parts, long long t0, long long t1, double* phi_part_out,
                                               double* force_part_out, double* energy_part_out) {
    if (n_parts < 1) return HSMA_ERR_INVALID_ARG;
    return evaluate_impl(plan, xyz, q, N, t0, t1, phi_part_out, energy_part_out, force_part_out, kPhaseRest, 0, -1, part, n_parts);
}
extern "C" int hsma_plan_part_form_applies(const hsma_plan* p, long long N) {
    if (!p || N < 1) return 0;
    return !p->sphere && p->pair_form != 1 && sym_applies((N + kTile - 1) / kTile, p->C_near) ? 1 : 0;
}

extern "C" hsma_status hsma_plan_sync(hsma_plan* plan) {
    if (!plan) return HSMA_ERR_INVALID_ARG;
    int hf[4] = {0, 0, 0, 0};
    cudaError_t e = cudaMemcpyAsync(hf, plan->flags, sizeof(hf), cudaMemcpyDeviceToHost, plan->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(plan->stream);
    hsma_status s = plan->sticky;
    plan->sticky = HSMA_OK;
    if (e != cudaSuccess) { cudaGetLastError(); return HSMA_ERR_CUDA; }
    if (hf[1]) {
        cudaMemsetAsync(plan->flags + 1, 0, sizeof(int), plan->stream);
        if (s == HSMA_OK) s = HSMA_ERR_NOT_NEUTRAL;
    }
    if (hf[2]) {   // sphere-culled near set: a source outside the auxiliary sphere (found on the device)
        cudaMemsetAsync(plan->flags + 2, 0, sizeof(int), plan->stream);
        if (s == HSMA_OK) s = HSMA_ERR_GEOMETRY;
    }
    return s;
}

static hsma_status host_impl(hsma_plan* p, const double* xyz_host, const double* q_host, long long N, long long t0,
                             long long t1, double* phi_host, double* force_host, double* energy_host) {
    if (!p || !xyz_host || !q_host || N < 1 || t0 < 0 || t1 > N || t0 > t1) return HSMA_ERR_INVALID_ARG;
    const long long T = t1 - t0;
    const bool field = force_host != nullptr && T > 0;
    if (p->xyz_in.reserve(3 * (size_t)N) != cudaSuccess || p->q_in.reserve((size_t)N) != cudaSuccess ||
        p->phi_dev.reserve((size_t)std::max(1LL, T)) != cudaSuccess ||
        (field && p->force_dev.reserve(3 * (size_t)T) != cudaSuccess))
        return HSMA_ERR_ALLOC;
    cudaStream_t st = p->stream;
    CU(cudaMemcpyAsync(p->xyz_in.p, xyz_host, 3 * (size_t)N * sizeof(double), cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(p->q_in.p, q_host, (size_t)N * sizeof(double), cudaMemcpyHostToDevice, st));
    hsma_status s = evaluate_graphed(p, p->xyz_in.p, p->q_in.p, N, t0, t1, p->phi_dev.p, p->scalars, field ? p->force_dev.p : nullptr);
    if (s != HSMA_OK) return s;
    if (phi_host && T > 0)
        CU(cudaMemcpyAsync(phi_host, p->phi_dev.p, (size_t)T * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (field) CU(cudaMemcpyAsync(force_host, p->force_dev.p, 3 * (size_t)T * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (energy_host) CU(cudaMemcpyAsync(energy_host, p->scalars, sizeof(double), cudaMemcpyDeviceToHost, st));
    return hsma_plan_sync(p);
}

extern "C" hsma_status hsma_evaluate_shard_host(hsma_plan* p, const double* xyz_host, const double* q_host,
                                                long long N, long long t0, long long t1, double* phi_host,
                                                double* energy_host) {
    return host_impl(p, xyz_host, q_host, N, t0, t1, phi_host, nullptr, energy_host);
}

extern "C" hsma_status hsma_evaluate_forces_host(hsma_plan* p, const double* xyz_host, const double* q_host, long long N,
                                                 double* phi_host, double* force_host, double* energy_host) {
    if (!force_host) return HSMA_ERR_INVALID_ARG;
    return host_impl(p, xyz_host, q_host, N, 0, N, phi_host, force_host, energy_host);
}

extern "C" hsma_status hsma_evaluate_host(hsma_plan* p, const double* xyz_host, const double* q_host, long long N,
                                          double* phi_host, double* energy_host) {
    return hsma_evaluate_shard_host(p, xyz_host, q_host, N, 0, N, phi_host, energy_host);
}

// ------------------------------------------------------------------------------------------------
// introspection, raw kernels, microbenchmark
// ------------------------------------------------------------------------------------------------
extern "C" const char* hsma_status_string(int s) {
    switch (s) {
        case HSMA_OK: return "HSMA_OK";
        case HSMA_ERR_INVALID_ARG: return "HSMA_ERR_INVALID_ARG";
        case HSMA_ERR_GEOMETRY: return "HSMA_ERR_GEOMETRY: R_aux must lie in (R0, min_a (shell_a + 1/2) L_a]";
        case HSMA_ERR_NOT_NEUTRAL: return "HSMA_ERR_NOT_NEUTRAL: periodic axes need sum q = 0";
        case HSMA_ERR_CUDA: return "HSMA_ERR_CUDA";
        case HSMA_ERR_ALLOC: return "HSMA_ERR_ALLOC";
        case HSMA_ERR_RANK_DEFICIENT: return "HSMA_ERR_RANK_DEFICIENT";
        case HSMA_ERR_TOO_LARGE: return "HSMA_ERR_TOO_LARGE: sizes beyond the fixed scratch of hsma_direct_sum_static (N, T <= 65,536, C <= 32, 16 MiB in all)";
        default: return "HSMA_ERR_UNKNOWN";
    }
}

extern "C" hsma_status hsma_plan_info(hsma_plan* p, long long* w) {
    if (!p || !w) return HSMA_ERR_INVALID_ARG;
    if (p->sphere && p->img_dyn) {   // the image count lives on the device: fetch it for the caller (synchronises)
        long long h[2] = {0, 0};
        if (cudaMemcpyAsync(h, p->img_dyn, sizeof(h), cudaMemcpyDeviceToHost, p->stream) == cudaSuccess &&
            cudaStreamSynchronize(p->stream) == cudaSuccess && h[0] > 0)
            p->last_images = h[0];
    }
    w[0] = p->rows; w[1] = p->ncol; w[2] = p->Kt; w[3] = p->C_near; w[4] = p->C_rhs; w[5] = p->d.M; w[6] = p->d.p;
    w[7] = p->last_launches; w[8] = p->last_images; w[9] = p->n_node_records; w[10] = p->need_grad ? 1 : 0; w[11] = p->greplays;
    return HSMA_OK;
}

static hsma_status d2d(hsma_plan* p, void* dst, const void* src, size_t bytes) {
    if (!p || !dst) return HSMA_ERR_INVALID_ARG;
    CU(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToDevice, p->stream));
    return HSMA_OK;
}
extern "C" hsma_status hsma_get_coeffs(hsma_plan* p, double* A_out) {
    return p ? d2d(p, A_out, p->A_full, (size_t)p->d.p * p->d.p * sizeof(double)) : HSMA_ERR_INVALID_ARG;
}
extern "C" hsma_status hsma_get_rhs(hsma_plan* p, double* rhs_out) {
    return p ? d2d(p, rhs_out, p->rhs, (size_t)p->rows * sizeof(double)) : HSMA_ERR_INVALID_ARG;
}
extern "C" hsma_status hsma_get_check_targets(hsma_plan* p, double* xyz_out) {
    return p ? d2d(p, xyz_out, p->chk, 3 * (size_t)p->Kt * sizeof(double)) : HSMA_ERR_INVALID_ARG;
}
extern "C" hsma_status hsma_get_nodes(hsma_plan* p, double* xyz_out, double* w_out) {
    if (!p) return HSMA_ERR_INVALID_ARG;
    if (xyz_out) {
        node_positions_kernel<<<(3 * p->d.M + 255) / 256, 256, 0, p->stream>>>(p->nrm, p->d.R_aux, p->d.M, xyz_out);
        HSMA_COUNT_LAUNCH();
    }
    if (w_out) return d2d(p, w_out, p->wq, (size_t)p->d.M * sizeof(double));
    return HSMA_OK;
}
extern "C" hsma_status hsma_get_surface(hsma_plan* p, double* Q_out, double* P_out) {
    if (!p) return HSMA_ERR_INVALID_ARG;
    unpack_nodes_kernel<<<(p->d.M + 255) / 256, 256, 0, p->stream>>>(p->nodes, p->d.M, Q_out, P_out);
    HSMA_COUNT_LAUNCH();
    return HSMA_OK;
}
extern "C" hsma_status hsma_get_fit_residual(hsma_plan* p, double* rms_out) {
    if (!p || !rms_out) return HSMA_ERR_INVALID_ARG;
    r_times_a_kernel<<<1, 256, 0, p->stream>>>(p->Rm, p->A_full, p->ncol, p->drop, p->cvec);
    fit_residual_kernel<<<1, 1024, 0, p->stream>>>(p->rhs, p->rows, p->ncol, p->Qm, p->cvec, p->scalars + 4);
    HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH();
    CU(cudaMemcpyAsync(rms_out, p->scalars + 4, sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    CU(cudaStreamSynchronize(p->stream));
    return HSMA_OK;
}

namespace hsma {
__global__ void pack_nodes_kernel(const double* __restrict__ R, const double* __restrict__ Q, const double* __restrict__ P,
                                  long long M, long long Mpad, Node8* __restrict__ out) {
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Mpad) return;
    Node8 n;
    if (j < M) { n.x = R[3 * j]; n.y = R[3 * j + 1]; n.z = R[3 * j + 2]; n.q = Q[j]; n.px = P[3 * j]; n.py = P[3 * j + 1]; n.pz = P[3 * j + 2]; }
    else { n.x = n.y = n.z = kFar; n.q = n.px = n.py = n.pz = 0.0; }
    n.pad = 0.0;
    out[j] = n;
}
}  // namespace hsma

static hsma_status direct_impl(const double* tgt, long long T, const double* src, const double* q, long long N,
                               const double* shift_host, const double* sign_host, const double* w_host, int C,
                               int central_cell, long long self_offset, int refine, double* phi_out, double* grad_out,
                               void* cuda_stream) {
    const bool field = grad_out != nullptr;
    if (!tgt || !src || !q || !shift_host || !sign_host || !w_host || (!phi_out && !grad_out)) return HSMA_ERR_INVALID_ARG;
    if (T < 1 || N < 1 || C < 1 || C > kMaxCells || (refine != 1 && refine != 2)) return HSMA_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    std::vector<Cell> cells(C);
    for (int c = 0; c < C; ++c) {
        cells[c].sx = shift_host[3 * c]; cells[c].sy = shift_host[3 * c + 1]; cells[c].sz = shift_host[3 * c + 2];
        cells[c].w = w_host[c];
        cells[c].fx = sign_host[3 * c] < 0; cells[c].fy = sign_host[3 * c + 1] < 0; cells[c].fz = sign_host[3 * c + 2] < 0;
        cells[c].central = (c == central_cell);
    }
    const long long n_tiles = (N + kTile - 1) / kTile, Npad = n_tiles * kTile;
    const Launch s = choose_near(T, n_tiles, C, refine, field);
    if (N > 2000000000LL) return HSMA_ERR_INVALID_ARG;
    Cell* dc = nullptr; Src4* ds = nullptr; double* part = nullptr; double* stats = nullptr; int* idx = nullptr;
    QInfo* qi = nullptr; int* flags = nullptr;
    hsma_status rc = HSMA_OK;
    // idx: slot_of [N] then tile_np [n_tiles]; stats: per tile [4] then scal [2]
    if (cudaMalloc(&dc, C * sizeof(Cell)) != cudaSuccess || cudaMalloc(&ds, Npad * sizeof(Src4)) != cudaSuccess ||
        cudaMalloc(&part, (size_t)s.rows * T * (field ? 4 : 1) * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&stats, (size_t)(4 * n_tiles + 2) * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&idx, (size_t)(N + n_tiles) * sizeof(int)) != cudaSuccess || cudaMalloc(&qi, sizeof(QInfo)) != cudaSuccess ||
        cudaMalloc(&flags, 4 * sizeof(int)) != cudaSuccess) {
        rc = HSMA_ERR_ALLOC;
    } else {
        cudaMemcpyAsync(dc, cells.data(), C * sizeof(Cell), cudaMemcpyHostToDevice, st);
        pack_sources_kernel<<<(unsigned)n_tiles, kTile, 0, st>>>(src, q, N, 0.0, 0.0, 0.0, ds, idx, idx + N, stats);
        charge_stats_kernel<<<1, 1024, 0, st>>>(stats, n_tiles, 0, stats + 4 * n_tiles, qi, flags);
        HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH();
        const Packed P{ds, N, n_tiles, idx + N, idx, qi};
        launch_near(s, field, tgt, 3, nullptr, T, 0, P, dc, C, central_cell >= 0 ? self_offset : -1, refine, part, st);
        if (field)
            finish_field_kernel<<<(unsigned)((T + 255) / 256), 256, 0, st>>>(s.layout(part), PartLayout{nullptr, 1, 1, 1, 1}, T, nullptr, nullptr, 0, phi_out, grad_out, nullptr);
        else
            finish_phi_kernel<<<(unsigned)((T + 255) / 256), 256, 0, st>>>(s.layout(part), PartLayout{nullptr, 1, 1, 1, 1}, T, nullptr, nullptr, 0, phi_out, nullptr);
        HSMA_COUNT_LAUNCH();
        if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = HSMA_ERR_CUDA;
    }
    for (void* ptr : {(void*)dc, (void*)ds, (void*)part, (void*)stats, (void*)idx, (void*)qi, (void*)flags})
        if (ptr) cudaFree(ptr);
    return rc;
}

extern "C" hsma_status hsma_direct_sum(const double* tgt, long long T, const double* src, const double* q, long long N,
                                       const double* shift_host, const double* sign_host, const double* w_host, int C,
                                       int central_cell, long long self_offset, int refine, double* phi_out,
                                       void* cuda_stream) {
    if (!phi_out) return HSMA_ERR_INVALID_ARG;
    return direct_impl(tgt, T, src, q, N, shift_host, sign_host, w_host, C, central_cell, self_offset, refine, phi_out,
                       nullptr, cuda_stream);
}
extern "C" hsma_status hsma_direct_field(const double* tgt, long long T, const double* src, const double* q, long long N,
                                         const double* shift_host, const double* sign_host, const double* w_host, int C,
                                         int central_cell, long long self_offset, int refine, double* phi_out,
                                         double* grad_out, void* cuda_stream) {
    if (!grad_out) return HSMA_ERR_INVALID_ARG;
    return direct_impl(tgt, T, src, q, N, shift_host, sign_host, w_host, C, central_cell, self_offset, refine, phi_out,
                       grad_out, cuda_stream);
}

static hsma_status node_impl(const double* tgt, long long T, const double* R, const double* Q, const double* P,
                             long long M, double* phi_out, double* grad_out, void* cuda_stream) {
    const bool field = grad_out != nullptr;
    if (!tgt || !R || !Q || !P || (!phi_out && !grad_out) || T < 1 || M < 1) return HSMA_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    constexpr int kNT = kTile / 2;
    const long long n_tiles = (M + kNT - 1) / kNT, Mpad = n_tiles * kNT;
    const Launch s = choose_node(T, n_tiles, field);
    Node8* dn = nullptr; double* part = nullptr;
    hsma_status rc = HSMA_OK;
    if (cudaMalloc(&dn, Mpad * sizeof(Node8)) != cudaSuccess || cudaMalloc(&part, (size_t)s.rows * T * (field ? 4 : 1) * sizeof(double)) != cudaSuccess) {
        rc = HSMA_ERR_ALLOC;
    } else {
        pack_nodes_kernel<<<(unsigned)((Mpad + 255) / 256), 256, 0, st>>>(R, Q, P, M, Mpad, dn);
        HSMA_COUNT_LAUNCH();
        launch_node(s, field, tgt, 3, nullptr, T, 0, dn, n_tiles, part, st);
        if (field)
            finish_field_kernel<<<(unsigned)((T + 255) / 256), 256, 0, st>>>(PartLayout{nullptr, 1, 1, 1, 1}, s.layout(part), T, nullptr, nullptr, 0, phi_out, grad_out, nullptr);
        else
            finish_phi_kernel<<<(unsigned)((T + 255) / 256), 256, 0, st>>>(PartLayout{nullptr, 1, 1, 1, 1}, s.layout(part), T, nullptr, nullptr, 0, phi_out, nullptr);
        HSMA_COUNT_LAUNCH();
        if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) rc = HSMA_ERR_CUDA;
    }
    if (dn) cudaFree(dn);
    if (part) cudaFree(part);
    return rc;
}

extern "C" hsma_status hsma_node_sum(const double* tgt, long long T, const double* R, const double* Q, const double* P,
                                     long long M, double* phi_out, void* cuda_stream) {
    if (!phi_out) return HSMA_ERR_INVALID_ARG;
    return node_impl(tgt, T, R, Q, P, M, phi_out, nullptr, cuda_stream);
}
extern "C" hsma_status hsma_node_field(const double* tgt, long long T, const double* R, const double* Q, const double* P,
                                       long long M, double* phi_out, double* grad_out, void* cuda_stream) {
    if (!grad_out) return HSMA_ERR_INVALID_ARG;
    return node_impl(tgt, T, R, Q, P, M, phi_out, grad_out, cuda_stream);
}

extern "C" hsma_status hsma_fp64_peak(double seconds, double* tflops_out, double* sm_clock_mhz_out) {
    if (!tflops_out || !(seconds > 0.0) || seconds > 30.0) return HSMA_ERR_INVALID_ARG;
    int dev = 0, khz = 0;
    CU(cudaGetDevice(&dev));
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    double* out = nullptr;
    CU(cudaMalloc(&out, sizeof(double)));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = num_sm() * 8;
    int iters = 2000;
    float ms = 0.f;
    hsma_status rc = HSMA_OK;
    for (int pass = 0; pass < 3 && rc == HSMA_OK; ++pass) {  // calibrate, then one long timed launch
        cudaEventRecord(e0);
        dfma_peak_kernel<<<blocks, 256>>>(out, iters, 0.999999, 1e-9);
        HSMA_COUNT_LAUNCH();
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { rc = HSMA_ERR_CUDA; break; }
        cudaEventElapsedTime(&ms, e0, e1);
        if (pass < 2) {
            const double scale = seconds * 1e3 / std::max(1e-3, (double)ms) * (pass == 0 ? 0.1 : 1.0);
            iters = (int)std::max(100.0, std::min(2.0e8, iters * scale * (pass == 0 ? 1.0 : 1.0)));
            if (pass == 1) iters = (int)std::max(100.0, std::min(2.0e8, (double)iters));
        }
    }
    if (rc == HSMA_OK) {
        const double fma = (double)blocks * 256.0 * (double)iters * (double)kPeakFmaPerThreadIter;
        *tflops_out = 2.0 * fma / (ms * 1e-3) * 1e-12;
        if (sm_clock_mhz_out) *sm_clock_mhz_out = khz * 1e-3;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    return rc;
}

extern "C" hsma_status hsma_plan_set_timing(hsma_plan* p, int enable) {
    if (!p) return HSMA_ERR_INVALID_ARG;
    if (enable)
        for (cudaEvent_t& e : p->ev)
            if (!e) CU(cudaEventCreate(&e));
    p->timing = enable != 0;
    p->ev_valid = false;
    return HSMA_OK;
}

extern "C" hsma_status hsma_plan_set_pair_form(hsma_plan* p, int form) {
    if (!p || form < 0 || form > 2) return HSMA_ERR_INVALID_ARG;
    p->pair_form = form;
    ++g_alloc_epoch;   // a captured evaluate graph holds the other form's launches
    return HSMA_OK;
}

extern "C" int hsma_plan_last_pair_form(const hsma_plan* p) { return p ? p->last_pair_form : 0; }

extern "C" hsma_status hsma_plan_fmm_info(hsma_plan* p, long long* w) {
    if (!p || !w || !p->fmm.enabled) return HSMA_ERR_INVALID_ARG;
    w[0] = p->fmm.p; w[1] = p->fmm.last_levels;
    w[2] = p->fmm.last_levels > 0 ? ((long long)p->fmm.base[0] * p->fmm.base[1] * p->fmm.base[2]) << (3 * p->fmm.last_levels) : 0;
    w[3] = (p->cells_rhs == p->cells_near && !p->need_grad) ? 1 : 0;
    return HSMA_OK;
}

extern "C" hsma_status hsma_plan_set_sym_scratch_cap(hsma_plan* p, long long bytes) {
    if (!p || bytes < 0) return HSMA_ERR_INVALID_ARG;
    p->sym_col_cap = bytes == 0 ? kSymColCapDefault : (size_t)bytes;
    ++g_alloc_epoch;   // a captured evaluate graph holds the old wave structure
    return HSMA_OK;
}
extern "C" hsma_status hsma_plan_set_image_factoring(hsma_plan* p, int on) {
    if (!p || on < 0 || on > 1) return HSMA_ERR_INVALID_ARG;
    p->lat_on = on != 0;
    ++g_alloc_epoch;   // a captured evaluate graph holds the other kernels
    return HSMA_OK;
}
extern "C" int hsma_plan_image_factoring(const hsma_plan* p) { return p && p->lat_on && p->lat_shape != 0 ? 1 : 0; }
extern "C" long long hsma_plan_scratch_bytes(const hsma_plan* p) {
    if (!p) return 0;
    size_t b = p->src.cap * sizeof(Src4) + (p->slot_of.cap + p->tile_np.cap) * sizeof(int) +
               (p->part_a.cap + p->part_b.cap + p->part_c.cap + p->red.cap + p->sym_col.cap + p->sym_phi.cap) * sizeof(double) +
               p->img_counts.cap * sizeof(long long) + (p->img_xyz.cap + p->img_q.cap + p->img_stats.cap) * sizeof(double) +
               p->img_src.cap * sizeof(Src4) + (p->img_slot_of.cap + p->img_tile_np.cap) * sizeof(int) + p->fmm.scratch_bytes();
    return (long long)b;
}

extern "C" hsma_status hsma_plan_get_timing(hsma_plan* p, double* ms_out) {
    if (!p || !ms_out || !p->timing || !p->ev_valid) return HSMA_ERR_INVALID_ARG;
    CU(cudaEventSynchronize(p->ev[6]));
    double ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = 0; i < 6; ++i) {
        float f = 0.f;
        CU(cudaEventElapsedTime(&f, p->ev[i], p->ev[i + 1]));
        ms[i] = f;
    }
    float tot = 0.f;
    CU(cudaEventElapsedTime(&tot, p->ev[0], p->ev[6]));
    ms[6] = tot;
    if (p->last_far_timed) {   // the FMM far field ran inside the pre-pass interval: report it on its own
        float far = 0.f;
        CU(cudaEventElapsedTime(&far, p->ev[7], p->ev[8]));
        ms[7] = far;
        ms[0] -= far;
    }
    for (int i = 0; i < 8; ++i) ms_out[i] = ms[i];
    return HSMA_OK;
}

extern "C" long long hsma_launch_count(void) { return g_launches; }

// ---- allocation-free raw direct sum: hsma_direct_sum_static (include/hsma.h) ---------------------------------------
// The same launches as hsma_direct_sum (pack_sources_kernel, charge_stats_kernel, near_sum_kernel, finish_phi_kernel)
// with every scratch buffer -- cell table, packed sources, slots, tile statistics, partial rows -- carved out of ONE
// file-scope device array of fixed size, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops).
// Every GPU that loads the library holds the array until the process exits.  In host code `g_static_scratch` is a
// host-side stand-in for the symbol, NOT a device address: the address comes from cudaGetSymbolAddress, once per device,
// with that device current.
namespace hsma {
constexpr size_t kStaticScratchBytes = 16u << 20;      // 16 MiB
constexpr long long kStaticMaxN = 65536, kStaticMaxT = 65536;
constexpr int kStaticMaxC = 32;
constexpr int kStaticMaxDevices = 64;
struct StaticCells { Cell c[kStaticMaxC]; };           // 1536 B: travels as a kernel argument, no host-to-device copy
__global__ void static_cells_kernel(const StaticCells t, int C, Cell* __restrict__ out, int* __restrict__ flags) {
    const int i = threadIdx.x;
    if (i < C) out[i] = t.c[i];
    if (i < 4) flags[i] = 0;                           // what must start at zero (the array keeps the last call's contents)
}
}  // namespace hsma

static __device__ __align__(256) unsigned char g_static_scratch[hsma::kStaticScratchBytes];

static std::mutex g_static_mu;
static unsigned char* g_static_ptr[hsma::kStaticMaxDevices] = {};

// device address of the scratch array on the CURRENT device (looked up once per device)
static hsma_status static_scratch_address(unsigned char** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kStaticMaxDevices) { cudaGetLastError(); return HSMA_ERR_CUDA; }
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) { cudaGetLastError(); return HSMA_ERR_CUDA; }
        g_static_ptr[dev] = static_cast<unsigned char*>(ptr);
    }
    *out = g_static_ptr[dev];
    return HSMA_OK;
}

extern "C" hsma_status hsma_static_scratch_setup(void) {
    unsigned char* p = nullptr;
    return static_scratch_address(&p);
}
extern "C" long long hsma_static_scratch_bytes(void) { return (long long)kStaticScratchBytes; }
// test hook: overwrite the whole array with `byte` (0xFF: every double a NaN) on `cuda_stream`, so that a test can show
// that a call reads nothing a previous call (or nobody) left behind
extern "C" hsma_status hsma_static_scratch_fill(int byte, void* cuda_stream) {
    unsigned char* p = nullptr;
    const hsma_status rs = static_scratch_address(&p);
    if (rs != HSMA_OK) return rs;
    if (cudaMemsetAsync(p, byte, kStaticScratchBytes, (cudaStream_t)cuda_stream) != cudaSuccess) { cudaGetLastError(); return HSMA_ERR_CUDA; }
    return HSMA_OK;
}

extern "C" hsma_status hsma_direct_sum_static(const double* tgt, long long T, const double* src, const double* q, long long N,
                                              const double* shift_host, const double* sign_host, const double* w_host, int C,
                                              int central_cell, long long self_offset, int refine, double* phi_out,
                                              void* cuda_stream) {
    if (!tgt || !src || !q || !shift_host || !sign_host || !w_host || !phi_out) return HSMA_ERR_INVALID_ARG;
    if (T < 1 || N < 1 || C < 1 || (refine != 1 && refine != 2)) return HSMA_ERR_INVALID_ARG;
    if (T > kStaticMaxT || N > kStaticMaxN || C > kStaticMaxC) return HSMA_ERR_TOO_LARGE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    StaticCells cells;
    for (int c = 0; c < kStaticMaxC; ++c) {
        Cell& k = cells.c[c];
        k.sx = k.sy = k.sz = 0.0; k.w = 0.0; k.fx = k.fy = k.fz = 0; k.central = 0;
        if (c >= C) continue;
        k.sx = shift_host[3 * c]; k.sy = shift_host[3 * c + 1]; k.sz = shift_host[3 * c + 2];
        k.w = w_host[c];
        k.fx = sign_host[3 * c] < 0; k.fy = sign_host[3 * c + 1] < 0; k.fz = sign_host[3 * c + 2] < 0;
        k.central = (c == central_cell);
    }
    const long long n_tiles = (N + kTile - 1) / kTile, Npad = n_tiles * kTile;
    const Launch s = choose_near(T, n_tiles, C, refine, false);
    // carve the array: every piece 256-byte aligned
    auto up = [](size_t b) { return (b + 255) & ~(size_t)255; };
    size_t off = 0;
    const size_t o_cells = off; off += up(kStaticMaxC * sizeof(Cell));
    const size_t o_qi = off;    off += up(sizeof(QInfo));
    const size_t o_flags = off; off += up(4 * sizeof(int));
    const size_t o_src = off;   off += up((size_t)Npad * sizeof(Src4));
    const size_t o_idx = off;   off += up((size_t)(N + n_tiles) * sizeof(int));       // slot_of [N] then tile_np [n_tiles]
    const size_t o_stats = off; off += up((size_t)(4 * n_tiles + 2) * sizeof(double)); // per tile [4] then scalars [2]
    const size_t o_part = off;  off += up((size_t)s.rows * T * sizeof(double));
    if (off > kStaticScratchBytes) return HSMA_ERR_TOO_LARGE;
    unsigned char* base = nullptr;
    const hsma_status rs = static_scratch_address(&base);
    if (rs != HSMA_OK) return rs;
    Cell* dc = reinterpret_cast<Cell*>(base + o_cells);
    QInfo* qi = reinterpret_cast<QInfo*>(base + o_qi);
    int* flags = reinterpret_cast<int*>(base + o_flags);
    Src4* ds = reinterpret_cast<Src4*>(base + o_src);
    int* idx = reinterpret_cast<int*>(base + o_idx);
    double* stats = reinterpret_cast<double*>(base + o_stats);
    double* part = reinterpret_cast<double*>(base + o_part);
    static_cells_kernel<<<1, 32, 0, st>>>(cells, C, dc, flags);
    pack_sources_kernel<<<(unsigned)n_tiles, kTile, 0, st>>>(src, q, N, 0.0, 0.0, 0.0, ds, idx, idx + N, stats);
    charge_stats_kernel<<<1, 1024, 0, st>>>(stats, n_tiles, 0, stats + 4 * n_tiles, qi, flags);
    HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH();
    const Packed P{ds, N, n_tiles, idx + N, idx, qi};
    launch_near(s, false, tgt, 3, nullptr, T, 0, P, dc, C, central_cell >= 0 ? self_offset : -1, refine, part, st);
    finish_phi_kernel<<<(unsigned)((T + 255) / 256), 256, 0, st>>>(s.layout(part), PartLayout{nullptr, 1, 1, 1, 1}, T, nullptr, nullptr, 0, phi_out, nullptr);
    HSMA_COUNT_LAUNCH();
    if (cudaPeekAtLastError() != cudaSuccess) { cudaGetLastError(); return HSMA_ERR_CUDA; }
    return HSMA_OK;
}
