// Tail of a squaring launch (rows A4 + A5).  All tiles cost the same, so a launch of n_t tiles on 148 SMs runs in
// ceil(n_t / 148) waves and the last one may be nearly empty (k = 8192: 2080 tiles = 14.05 waves -> 15; k = 1024: 36
// tiles on 148 SMs).  The host
// (plan_tail in rfoe.cu) therefore hands the last T tiles to sym_square_kernel<2>, which cuts their contraction
// into S slices (T x S CTAs fill whole waves of 1/S the length) and stores raw accumulators tile-contiguously;
// tail_fixup_kernel below adds the slices in ascending order and applies exactly the fused epilogue of the main
// kernel: Out = c2 C + c1 E + c0 I to (I,J) and mirrored to (J,I), and the five partial sums of the tile
// (PAPER.md:39, 72), to every destination of `dst` (one for a single-GPU run, all ranks for a sharded P2P run).
// Which tiles are tail tiles depends only on (n_t, K extent, SM count), so a sharded run
// computes every tile with the same arithmetic as the single-GPU run.
#pragma once
#include "sym_square.cuh"

namespace rfoe {

constexpr int TAIL_THREADS = 1024;   // 32 x 32: one element of every 32 x 32 sub-block per thread

__global__ void __launch_bounds__(TAIL_THREADS)
tail_fixup_kernel(const double* __restrict__ ws, int n_slices, int n_tail, const int2* __restrict__ tile_map,
                  const double* __restrict__ E, int ld, int kvalid,
                  const StepCoef* __restrict__ coef, const __grid_constant__ PeerSet dst)
{
    __shared__ double sm[32][33];
    __shared__ double red[5][32];
    const int2 tile = tile_map[blockIdx.x];
    const int I = tile.x, J = tile.y;
    const bool diag = (I == J);
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 32
    const double* T = ws + (size_t)blockIdx.x * (SQ_BM * SQ_BM);
    const size_t slice_stride = (size_t)n_tail * (SQ_BM * SQ_BM);
    const double c2 = coef->c2, c1 = coef->c1, c0 = coef->c0;
    double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
    for (int bi = 0; bi < 4; ++bi)
        for (int bj = diag ? bi : 0; bj < 4; ++bj) {
            __syncthreads();
            {
                const int r = bi * 32 + ty, c = bj * 32 + tx;
                const int row = I * SQ_BM + r, col = J * SQ_BM + c;
                const double* src = T + r * SQ_BM + c;
                const double ev = E[(size_t)row * ld + col];
                double cv = 0.0;
                int s = 0;
                for (; s + 4 <= n_slices; s += 4) {       // four loads in flight, added in ascending slice order
                    const double x0 = src[(size_t)s * slice_stride], x1 = src[(size_t)(s + 1) * slice_stride];
                    const double x2 = src[(size_t)(s + 2) * slice_stride], x3 = src[(size_t)(s + 3) * slice_stride];
                    cv += x0; cv += x1; cv += x2; cv += x3;
                }
                for (; s < n_slices; ++s) cv += src[(size_t)s * slice_stride];
                double v = fma(c2, cv, c1 * ev);
                const double d = cv - ev;
                double w = 1.0;
                if (diag) {
                    w = (col > row) ? 2.0 : ((col == row) ? 1.0 : 0.0);
                    if (col == row) {
                        if (row < kvalid) v += c0;
                        p_tr += v;
                        p_trc += cv;
                    }
                }
                sm[ty][tx] = v;
                if (!diag || col >= row)
                    for (int q = 0; q < dst.n; ++q) dst.out[q][(size_t)row * ld + col] = v;
                p_ss = fma(w * v, v, p_ss);
                p_err = fma(w * d, d, p_err);
                p_ce = fma(w * cv, ev, p_ce);
            }
            __syncthreads();
            {
                // mirrored element (col, row): col = J*128 + bj*32 + ty, row = I*128 + bi*32 + tx
                const int col = J * SQ_BM + bj * 32 + ty, row = I * SQ_BM + bi * 32 + tx;
                if (!diag || col > row)
                    for (int q = 0; q < dst.n; ++q) dst.out[q][(size_t)col * ld + row] = sm[tx][ty];
            }
        }
    if (!diag) { p_ss *= 2.0; p_err *= 2.0; p_ce *= 2.0; }
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        p_tr += __shfl_xor_sync(0xffffffffu, p_tr, m);
        p_ss += __shfl_xor_sync(0xffffffffu, p_ss, m);
        p_err += __shfl_xor_sync(0xffffffffu, p_err, m);
        p_trc += __shfl_xor_sync(0xffffffffu, p_trc, m);
        p_ce += __shfl_xor_sync(0xffffffffu, p_ce, m);
    }
    if (tx == 0) { red[0][ty] = p_tr; red[1][ty] = p_ss; red[2][ty] = p_err; red[3][ty] = p_trc; red[4][ty] = p_ce; }
    __syncthreads();
    if (threadIdx.x < SQ_NPART) {
        double v = 0.0;
        if (threadIdx.x < 5)
            for (int w = 0; w < 32; ++w) v += red[threadIdx.x][w];
        for (int q = 0; q < dst.n; ++q) dst.rec[q][(size_t)(dst.rec_offset + (int)blockIdx.x) * SQ_NPART + threadIdx.x] = v;
    }
}

}  // namespace rfoe
