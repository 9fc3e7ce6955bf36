// Host orchestration of the FMM form of step (b) (fmm_kernels.cuh).  Plan time: geometry checks and
// the translation tables.  Evaluate time: sort by leaf -> P2M -> M2M up -> M2L (all levels, one launch) -> L2L down
// (+ sum of the M2L partial rows) -> leaves (L2P + P2P; with forces also their gradients).  No host synchronisation, no atomics in floating point: a given
// (N, plan) is bit-reproducible.
#pragma once
#include <algorithm>
#include <cmath>
#include <vector>

#include "fmm_kernels.cuh"
#include "hsma.h"

namespace hsma {
namespace fmm {

template <class T>
struct Buf {   // growable device buffer (same contract as DevBuf in hsma_api.cu; `epoch` is bumped on reallocation)
    T* p = nullptr;
    size_t cap = 0;
    cudaError_t reserve(size_t n, std::atomic<size_t>& epoch) {
        if (n <= cap) return cudaSuccess;
        ++epoch;
        if (p) cudaFree(p);
        p = nullptr; cap = 0;
        const cudaError_t e = cudaMalloc(&p, n * sizeof(T));
        if (e == cudaSuccess) cap = n;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
};

struct State {
    bool enabled = false;
    int p = 20, levels_req = 0, last_levels = 0;
    int base[3] = {1, 1, 1}, refl[3] = {0, 0, 0}, shell[3] = {0, 0, 0};
    double a0 = 0.0, L[3] = {0, 0, 0};
    double* w_lut = nullptr;
    double2 *Rsh = nullptr, *Stab = nullptr;
    int *nm = nullptr, *pm = nullptr, *sfmap = nullptr, *off_list = nullptr, *off_wprefix = nullptr;
    int n_off = 0, W = 0;      // offsets of the M2L list and their total weight
    Buf<int> key_a, key_b, idx_a, idx_b, leaf_start, chunk_start;
    Buf<long long> counts;
    Buf<Src4> srt;
    Buf<double> slab;             // leaf kernel: one partial row per slab of neighbour boxes
    Buf<double2> Mx, Lx, Lpart;   // multipole / local expansions of all levels, M2L partial sums
    void release() {
        for (void* q : {(void*)w_lut, (void*)Rsh, (void*)Stab, (void*)nm, (void*)pm, (void*)sfmap, (void*)off_list, (void*)off_wprefix}) if (q) cudaFree(q);
        w_lut = nullptr; Rsh = Stab = nullptr; nm = pm = sfmap = off_list = off_wprefix = nullptr;
        key_a.release(); key_b.release(); idx_a.release(); idx_b.release(); leaf_start.release(); chunk_start.release(); counts.release();
        srt.release(); Mx.release(); Lx.release(); Lpart.release(); slab.release();
    }
    size_t scratch_bytes() const {
        return (key_a.cap + key_b.cap + idx_a.cap + idx_b.cap + leaf_start.cap + chunk_start.cap) * sizeof(int) + counts.cap * sizeof(long long) +
               srt.cap * sizeof(Src4) + (Mx.cap + Lx.cap + Lpart.cap) * sizeof(double2) + slab.cap * sizeof(double);
    }
};

// Geometry the FMM form supports: whole-cell near set, cubic boxes (every L_a an integer multiple of the smallest
// side), level-0 offsets inside the M2L table.  Returns HSMA_ERR_INVALID_ARG otherwise.
inline hsma_status setup(State& S, const hsma_plan_desc& d, const bool refl[3], cudaStream_t st) {
    if (d.near_mode != HSMA_NEAR_WHOLE_CELLS) return HSMA_ERR_INVALID_ARG;
    S.p = d.fmm_order > 0 ? d.fmm_order : 20;
    if (S.p < 2 || S.p > kMaxOrder) return HSMA_ERR_INVALID_ARG;
    if (d.fmm_levels < 0 || d.fmm_levels >= kMaxLevels) return HSMA_ERR_INVALID_ARG;
    S.levels_req = d.fmm_levels;
    const double Lmin = std::min({d.L[0], d.L[1], d.L[2]});
    for (int a = 0; a < 3; ++a) {
        const double r = d.L[a] / Lmin;
        S.base[a] = (int)std::llround(r);
        if (S.base[a] < 1 || S.base[a] > 4 || std::fabs(r - S.base[a]) > 1e-12) return HSMA_ERR_INVALID_ARG;
        S.refl[a] = refl[a] ? 1 : 0;
        S.shell[a] = d.near_shell[a];
        S.L[a] = d.L[a];
        if ((d.near_shell[a] + 1) * S.base[a] - 1 > kOffR) return HSMA_ERR_INVALID_ARG;   // level-0 offsets beyond the table
    }
    S.a0 = Lmin;
    // cell weights gamma^|k| over the reflecting axes (the same expression as make_cells)
    const int wx = 2 * S.shell[0] + 1, wy = 2 * S.shell[1] + 1, wz = 2 * S.shell[2] + 1;
    std::vector<double> lut((size_t)wx * wy * wz);
    for (int kx = -S.shell[0]; kx <= S.shell[0]; ++kx)
        for (int ky = -S.shell[1]; ky <= S.shell[1]; ++ky)
            for (int kz = -S.shell[2]; kz <= S.shell[2]; ++kz) {
                const int k[3] = {kx, ky, kz};
                int order = 0;
                for (int a = 0; a < 3; ++a) if (refl[a]) order += std::abs(k[a]);
                lut[((size_t)(kx + S.shell[0]) * wy + (ky + S.shell[1])) * wz + (kz + S.shell[2])] =
                    order > 0 ? std::pow(d.gamma, (double)order) : 1.0;
            }
    // offsets |d|_inf > kWs in lexicographic order; weight = how many of the 8 siblings can have the offset
    std::vector<int> off, wpre(1, 0);
    for (int dx = -kOffR; dx <= kOffR; ++dx)
        for (int dy = -kOffR; dy <= kOffR; ++dy)
            for (int dz = -kOffR; dz <= kOffR; ++dz) {
                if (std::max({std::abs(dx), std::abs(dy), std::abs(dz)}) <= kWs) continue;
                off.push_back(((dx + kOffR) * kOffW + (dy + kOffR)) * kOffW + (dz + kOffR));
                const int w = (std::abs(dx) == kOffR ? 1 : 2) * (std::abs(dy) == kOffR ? 1 : 2) * (std::abs(dz) == kOffR ? 1 : 2);
                wpre.push_back(wpre.back() + w);
            }
    S.n_off = (int)off.size();
    S.W = wpre.back();
    const int NC = nc(S.p), NS = nc(2 * S.p);
#define FCU(x) do { if ((x) != cudaSuccess) return HSMA_ERR_CUDA; } while (0)
    FCU(cudaMalloc(&S.w_lut, lut.size() * sizeof(double)));
    FCU(cudaMemcpyAsync(S.w_lut, lut.data(), lut.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    FCU(cudaMalloc(&S.off_list, off.size() * sizeof(int)));
    FCU(cudaMemcpyAsync(S.off_list, off.data(), off.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    FCU(cudaMalloc(&S.off_wprefix, wpre.size() * sizeof(int)));
    FCU(cudaMemcpyAsync(S.off_wprefix, wpre.data(), wpre.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    FCU(cudaMalloc(&S.Rsh, 8 * (size_t)NC * sizeof(double2)));
    FCU(cudaMalloc(&S.Stab, (size_t)kOffN * NS * sizeof(double2)));
    FCU(cudaMalloc(&S.nm, NC * sizeof(int)));
    FCU(cudaMalloc(&S.pm, m2l_pairs(S.p) * sizeof(int)));
    const int NSF = (2 * S.p + 1) * (2 * S.p + 1);
    FCU(cudaMalloc(&S.sfmap, NSF * sizeof(int)));
    tables_kernel<<<(std::max({kOffN, NC, NSF}) + 127) / 128, 128, 0, st>>>(S.p, S.Rsh, S.Stab, S.nm, S.pm, S.sfmap);
    HSMA_COUNT_LAUNCH();
    FCU(cudaStreamSynchronize(st));   // the host vectors above go out of scope
    FCU(cudaFuncSetAttribute(m2l_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, m2l_smem_bytes(S.p)));
    FCU(cudaFuncSetAttribute(m2m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 16 * NC * (int)sizeof(double2)));
    FCU(cudaFuncSetAttribute(p2m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             8 * NC * (int)sizeof(double2) + (S.p + 1) * kInvW * (int)sizeof(double)));
#undef FCU
    S.enabled = true;
    return HSMA_OK;
}

// leaf level: about 500 particles per leaf balances P2P (125 neighbour boxes) against M2L (875 translations of
// O(p^4) each) at p = 20; at least level 1
inline int choose_levels(const State& S, long long N) {
    if (S.levels_req > 0) return S.levels_req;
    const double base_boxes = (double)S.base[0] * S.base[1] * S.base[2];
    const double want = (double)N / (500.0 * base_boxes);
    int lev = (int)std::lround(std::log(std::max(want, 1.0)) / std::log(8.0));
    return std::max(1, std::min(kMaxLevels - 1, lev));
}

inline int resident_m2l(int p) {
    int per_sm = 0, dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, m2l_kernel, kM2LThreads, m2l_smem_bytes(p)) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    return per_sm * sms;
}

inline Geom make_geom(const State& S, long long N, const double half[3]) {
    Geom G;
    for (int a = 0; a < 3; ++a) { G.base[a] = S.base[a]; G.shell[a] = S.shell[a]; G.refl[a] = S.refl[a]; G.half[a] = half[a]; G.L[a] = S.L[a]; }
    G.levels = choose_levels(S, N);
    G.p = S.p; G.a0 = S.a0; G.w_lut = S.w_lut;
    return G;
}

// Upward pass of one evaluate: leaf sort, sorted source records, P2M, M2M.  Afterwards the multipoles of all levels
// are in S.Mx (used by step (a) through `points` and by step (b) through `downward`).
inline hsma_status upward(State& S, const double* xyz, const double* q, long long N, const double half[3],
                          std::atomic<size_t>& epoch, cudaStream_t st) {
    if (N > 2000000000LL) return HSMA_ERR_INVALID_ARG;
    const Geom G = make_geom(S, N, half);
    S.last_levels = G.levels;
    const int NC = nc(S.p);
    const long long n_leaves = boxes_at(G, G.levels), n_boxes = level_offset(G, G.levels + 1);
    if (n_leaves >= 65536) return HSMA_ERR_INVALID_ARG;
    const long long n_blk = (N + 255) / 256;
#define FR(x) do { if ((x) != cudaSuccess) return HSMA_ERR_ALLOC; } while (0)
    FR(S.key_a.reserve((size_t)N, epoch)); FR(S.key_b.reserve((size_t)N, epoch));
    FR(S.idx_a.reserve((size_t)N, epoch)); FR(S.idx_b.reserve((size_t)N, epoch));
    FR(S.leaf_start.reserve((size_t)n_leaves + 1, epoch)); FR(S.chunk_start.reserve((size_t)n_leaves + 1, epoch));
    FR(S.counts.reserve((size_t)(256 * n_blk + 256), epoch));
    FR(S.srt.reserve((size_t)N, epoch));
    FR(S.Mx.reserve((size_t)n_boxes * NC, epoch)); FR(S.Lx.reserve((size_t)n_boxes * NC, epoch));
#undef FR
    const unsigned gN = (unsigned)n_blk;
    key_kernel<<<gN, 256, 0, st>>>(xyz, N, G, S.key_a.p, S.idx_a.p);
    HSMA_COUNT_LAUNCH();
    // two stable 8-bit passes: a -> b -> a
    for (int pass = 0; pass < 2; ++pass) {
        const int* kin = pass == 0 ? S.key_a.p : S.key_b.p;
        const int* iin = pass == 0 ? S.idx_a.p : S.idx_b.p;
        int* kout = pass == 0 ? S.key_b.p : S.key_a.p;
        int* iout = pass == 0 ? S.idx_b.p : S.idx_a.p;
        radix_hist_kernel<<<gN, 256, 0, st>>>(kin, N, 8 * pass, n_blk, S.counts.p);
        radix_rowscan_kernel<<<256, 1024, 0, st>>>(S.counts.p, n_blk, S.counts.p + 256 * n_blk);
        radix_base_kernel<<<1, 256, 0, st>>>(S.counts.p + 256 * n_blk);
        radix_scatter_kernel<<<gN, 256, 0, st>>>(kin, iin, N, 8 * pass, n_blk, S.counts.p, S.counts.p + 256 * n_blk, kout, iout);
        HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH();
    }
    leaf_start_kernel<<<(unsigned)((n_leaves + 1 + 255) / 256), 256, 0, st>>>(S.key_a.p, N, (int)n_leaves, S.leaf_start.p);
    gather_sorted_kernel<<<gN, 256, 0, st>>>(xyz, q, S.idx_a.p, N, half[0], half[1], half[2], S.srt.p);
    HSMA_COUNT_LAUNCH(); HSMA_COUNT_LAUNCH();
    const int inv_bytes = (S.p + 1) * kInvW * (int)sizeof(double);
    p2m_kernel<<<(unsigned)n_leaves, 256, 8 * NC * sizeof(double2) + inv_bytes, st>>>(G, S.srt.p, S.leaf_start.p, S.Mx.p);
    HSMA_COUNT_LAUNCH();
    for (int lev = G.levels - 1; lev >= 0; --lev) {
        m2m_kernel<<<(unsigned)boxes_at(G, lev), 256, 16 * NC * sizeof(double2), st>>>(G, lev, S.Rsh, S.nm, S.Mx.p);
        HSMA_COUNT_LAUNCH();
    }
    return HSMA_OK;
}

// Step (a) from the hierarchy built by `upward` and `far_field`: the near sum at T arbitrary points (centred coordinates, device).
inline hsma_status points(State& S, const double* tgt, long long T, long long N, const double half[3], double* phi_out,
                          cudaStream_t st) {
    if (T < 1) return HSMA_OK;
    const Geom G = make_geom(S, N, half);
    const size_t smem = nc(S.p) * sizeof(double2) + (S.p + 1) * kInvW * sizeof(double);
    m2p_points_kernel<<<(unsigned)T, kM2PThreads, smem, st>>>(G, tgt, S.srt.p, S.leaf_start.p, S.Mx.p, S.Lx.p, phi_out);
    HSMA_COUNT_LAUNCH();
    return HSMA_OK;
}

// Far field of step (b): M2L at every level, L2L down.  Afterwards the local expansions of all boxes are in S.Lx (used by
// step (a) for check targets inside the central cell, and by `leaves`).
inline hsma_status far_field(State& S, long long N, const double half[3], std::atomic<size_t>& epoch, cudaStream_t st) {
    const Geom G = make_geom(S, N, half);
    const int NC = nc(S.p);
    // M2L launch shape: one persistent wave over the units (group, offset weight), deepest level first
    M2LArgs A;
    A.n_lv = 0;
    A.W = S.W;
    int n_groups_total = 0;
    for (int lev = G.levels; lev >= 0; --lev) {
        M2LLevel& r = A.lv[A.n_lv++];
        r.lev = lev;
        r.n_groups = (int)(lev == 0 ? boxes_at(G, 0) : boxes_at(G, lev - 1));
        r.first_group = n_groups_total;
        n_groups_total += r.n_groups;
    }
    A.units = (long long)n_groups_total * A.W;
    const int Gm2l = (int)std::min<long long>(resident_m2l(S.p), A.units);
    A.rows = part_rows(A.units, A.W, Gm2l);
    long long part_elems = 0;
    for (int r = 0; r < A.n_lv; ++r) {
        A.lv[r].part_off = part_elems;
        part_elems += (long long)A.rows * boxes_at(G, A.lv[r].lev) * NC;
    }
    A.off_list = S.off_list; A.off_wprefix = S.off_wprefix; A.n_off = S.n_off;
    if (S.Lpart.reserve((size_t)part_elems, epoch) != cudaSuccess) return HSMA_ERR_ALLOC;
    m2l_kernel<<<(unsigned)Gm2l, kM2LThreads, m2l_smem_bytes(S.p), st>>>(G, A, S.Mx.p, S.Stab, S.nm, S.pm, S.sfmap, S.Lpart.p);
    HSMA_COUNT_LAUNCH();
    for (int lev = 0; lev <= G.levels; ++lev) {
        l2l_kernel<<<(unsigned)boxes_at(G, lev), 256, 2 * NC * sizeof(double2), st>>>(G, lev, S.Rsh, S.nm, S.Lpart.p, A, Gm2l, S.Lx.p);
        HSMA_COUNT_LAUNCH();
    }
    return HSMA_OK;
}

// Step (b) at all N sources, original order, into phi_out [N] ([4][N] with forces): the leaves (L2P + P2P) after
// `far_field`.  refine as in the direct kernels (1 Newton, 2 cubic) for the P2P part.
inline hsma_status leaves(State& S, long long N, const double half[3], int refine, bool field, double* phi_out,
                          std::atomic<size_t>& epoch, cudaStream_t st) {
    const Geom G = make_geom(S, N, half);
    const int NC = nc(S.p);
    const long long n_leaves = boxes_at(G, G.levels);
    const int inv_bytes = (S.p + 1) * kInvW * (int)sizeof(double);
    const size_t leaf_smem = NC * sizeof(double2) + inv_bytes;
    leaf_chunks_kernel<<<1, 1024, 0, st>>>(S.leaf_start.p, (int)n_leaves, S.chunk_start.p);
    HSMA_COUNT_LAUNCH();
    const unsigned gl = (unsigned)(N / (kLeafThreads * kLeafR) + n_leaves);
    // field: phi_out is [4][N]: phi, grad phi (forces)
    const long long comps_n = (field ? 4 : 1) * N;
    if (S.slab.reserve((size_t)(2 * kWs + 1) * comps_n, epoch) != cudaSuccess) return HSMA_ERR_ALLOC;
    const dim3 gl3(gl, 2 * kWs + 1);
#define LEAF(RF, FL) leaf_kernel<RF, FL><<<gl3, kLeafThreads, leaf_smem, st>>>(G, S.srt.p, S.idx_a.p, S.leaf_start.p, S.chunk_start.p, (int)n_leaves, S.Lx.p, N, S.slab.p)
    if (field) { if (refine == 1) LEAF(1, true); else LEAF(2, true); }
    else { if (refine == 1) LEAF(1, false); else LEAF(2, false); }
#undef LEAF
    HSMA_COUNT_LAUNCH();
    leaf_sum_kernel<<<(unsigned)((comps_n + 255) / 256), 256, 0, st>>>(S.slab.p, comps_n, phi_out);
    HSMA_COUNT_LAUNCH();
    return HSMA_OK;
}

}  // namespace fmm
}  // namespace hsma
