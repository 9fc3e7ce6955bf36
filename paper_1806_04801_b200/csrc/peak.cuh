// DFMA-only microbenchmark: the measured FP64 roofline denominator.
// 8 independent FMA chains per thread, 8 CTAs x 256 threads per SM, no memory traffic in the loop.
// The chain is c = fma(c, c, b): with fma(c, a, b) and a, b shared by all chains the two loop-invariant
// operands collide in one register bank and the pipe issues at only 92 % (measured on B200); with two
// distinct source registers per instruction it reaches 99.5 % of 64 lanes x clock.
#pragma once
#include "common.cuh"

namespace hsma {

__global__ void __launch_bounds__(256) dfma_peak_kernel(double* out, int iters, double a, double b) {
    double c0 = threadIdx.x * 1e-3 * a, c1 = c0 * 0.5, c2 = c0 * 0.25, c3 = c0 * 0.125, c4 = c0 * 0.7, c5 = c0 * 0.3,
           c6 = c0 * 0.9, c7 = c0 * 0.1;   // all in [0, 0.26): c <- c*c + b stays bounded
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            c0 = fma(c0, c0, b); c1 = fma(c1, c1, b); c2 = fma(c2, c2, b); c3 = fma(c3, c3, b);
            c4 = fma(c4, c4, b); c5 = fma(c5, c5, b); c6 = fma(c6, c6, b); c7 = fma(c7, c7, b);
        }
    }
    const double s = ((c0 + c1) + (c2 + c3)) + ((c4 + c5) + (c6 + c7));
    if (s == 123.456) out[0] = s;  // never true; keeps the chains alive
}
constexpr long long kPeakFmaPerThreadIter = 16 * 8;

}  // namespace hsma
