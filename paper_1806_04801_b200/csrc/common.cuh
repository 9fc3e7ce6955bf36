// Shared device/host helpers of the CUDA path (sm_100a).  Nothing here is used by oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <atomic>

namespace hsma {

// ---- launch accounting (hsma_launch_count) --------------------------------------------------
extern std::atomic<long long> g_launches;
#define HSMA_COUNT_LAUNCH() (++::hsma::g_launches)

// ---- geometry of the all-pairs kernels ------------------------------------------------------
constexpr int kThreads = 256;     // threads per CTA of the pair kernels
constexpr int kTile = 256;        // sources per shared-memory tile (one 8 KB bulk copy)
constexpr int kStages = 2;        // double buffering
constexpr int kMaxCells = 448;    // cell table entries kept in shared memory (441 = 7x7x9 fits)
constexpr double kFar = 1.0e6;    // coordinate of the q=0 padding sources

// packed source record: 32 B, one 128-bit pair of loads per source (x,y | z,q)
struct __align__(16) Src4 { double x, y, z, q; };
// packed node record: 64 B (Rx,Ry,Rz,Qh | Px,Py,Pz,0) with Qh, P pre-scaled (see node_sum_kernel)
struct __align__(16) Node8 { double x, y, z, q, px, py, pz, pad; };

// one near (or far) image cell: image = sign o r + shift, weight w
struct Cell { double sx, sy, sz, w; int fx, fy, fz, central; };  // f = 1 if that axis is reflected

// ---- PTX: mbarrier + 1-D bulk async copy (TMA engine, SASS UBLKCP) --------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy, completion signalled on `bar` (bytes: multiple of 16, 16-B aligned)
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---- reciprocal square root ----------------------------------------------------------------
// fp64-input hardware seed (SASS MUFU.RSQ64H): ~22 significant bits, low word zero.
__device__ __forceinline__ double rsqrt_seed(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}
// seed + one cubic (Halley) step: y = y0 (1 + e/2 + 3e^2/8), e = 1 - x y0^2; relative error ~ e^3
__device__ __forceinline__ double rsqrt_cubic(double x) {
    const double y0 = rsqrt_seed(x);
    const double e = fma(-x, y0 * y0, 1.0);
    const double h = fma(e, 0.375, 0.5);
    return fma(y0 * e, h, y0);
}

__device__ __forceinline__ double flip(double v, int f) { return f ? -v : v; }

}  // namespace hsma
