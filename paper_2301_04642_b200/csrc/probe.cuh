// Issue-rate ceiling of the FP64 tensor pipe (rfoe_probe_fp64_peak): the squaring kernel's inner loop -- 8 warps per
// SM, 32 independent mma.m8n8k4.f64 accumulator pairs per warp (SASS DMMA.8x8x4) -- with its shared-memory operand
// loads removed, so nothing but the tensor pipe limits it.  The number it yields is the denominator of the squaring's
// roofline fraction: MEASURED_PEAKS.json carries no FP64 figure and the profiling guide lists no FP64 nominal.
#pragma once
#include "ptx_sm100.cuh"

namespace rfoe {

constexpr int PROBE_THREADS = 256;
constexpr double PROBE_FLOPS_PER_WARP_ITER = 4.0 * 32.0 * 512.0;   // 4 k4-steps x 32 DMMAs x (8*8*4 FMA = 512 flops)

__global__ void __launch_bounds__(PROBE_THREADS, 1)
fp64_peak_probe_kernel(long long iters, const double* __restrict__ seed, double* __restrict__ sink)
{
    // operands come from memory so the loop cannot be folded; values are small enough to stay finite for any iters
    const double a_seed = seed[0], b_seed = seed[1];
    double a[8], b[4], acc[8][4][2];
#pragma unroll
    for (int mi = 0; mi < 8; ++mi) a[mi] = a_seed * (double)(mi + 1 + (threadIdx.x & 3));
#pragma unroll
    for (int ni = 0; ni < 4; ++ni) b[ni] = b_seed * (double)(ni + 1 + (threadIdx.x >> 5));
#pragma unroll
    for (int mi = 0; mi < 8; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
#pragma unroll
            for (int mi = 0; mi < 8; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], a[mi], b[ni]);
    }
    double v = 0.0;
#pragma unroll
    for (int mi = 0; mi < 8; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) v += acc[mi][ni][0] + acc[mi][ni][1];
    if (v == 123.456) sink[0] = v;   // never true for the seeds used; keeps the accumulators live
}

}  // namespace rfoe
