// Steps either side of the expansion (reading R-RR).
//
// The paper's setting: the M x M Kohn-Sham matrix H "is orthogonally projected onto a carefully
// constructed subspace ... (Rayleigh-Ritz step)", the k x k projected H^p goes through RFOE, which "approximate[s]
// the density matrix in the subspace".  With the basis stored one state per row (Psi: k x M, M >> k):
//   before:  H^p = Psi HPsi^T           sym_square_kernel<2> (sym_square.cuh) + project_reduce_kernel (here)
//   after :  Y = P Psi                  apply_kernel (here): FP64 DMMA, P row panels and Psi blocks by TMA
//            rho_m = sum_i Psi_im Y_im  density_partial_kernel + density_reduce_kernel (HBM-bound)
#pragma once
#include "ptx_sm100.cuh"
#include "sym_square.cuh"

namespace rfoe {

// ------------------------------------------------------------------------------------------------------------
// Sum the K-slices of one projected tile in ascending slice order, write it to H^p (k x k, ld = k) and mirror it
// (the upper triangle is the definition; H^p must be bitwise symmetric for rfoe_expand).  One CTA per upper tile,
// 32 x 32 sub-blocks through shared memory so both the direct and the mirrored rows are written as 256-byte runs.
// rec[tile] = {Tr, sum of squares (off-diagonal entries counted twice), 0...}.
__global__ void __launch_bounds__(256)
project_reduce_kernel(const double* __restrict__ ws, int n_slices, int n_tiles, const int2* __restrict__ tile_map,
                      int k, double* __restrict__ Hp, double* __restrict__ rec)
{
    __shared__ double sm[32][33];
    __shared__ double red[2][8];
    const int2 tile = tile_map[blockIdx.x];
    const int I = tile.x, J = tile.y;
    const bool diag = (I == J);
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8
    const double* T = ws + (size_t)blockIdx.x * (SQ_BM * SQ_BM);
    const size_t slice_stride = (size_t)n_tiles * (SQ_BM * SQ_BM);
    double p_tr = 0.0, p_ss = 0.0;
    for (int bi = 0; bi < 4; ++bi)
        for (int bj = diag ? bi : 0; bj < 4; ++bj) {
            __syncthreads();
#pragma unroll
            for (int y = ty; y < 32; y += 8) {
                const int r = bi * 32 + y, c = bj * 32 + tx;
                double v = 0.0;
                for (int s = 0; s < n_slices; ++s) v += T[(size_t)s * slice_stride + r * SQ_BM + c];
                sm[y][tx] = v;
                const int gi = I * SQ_BM + r, gj = J * SQ_BM + c;
                if (gi < k && gj < k && gj >= gi) {
                    Hp[(size_t)gi * k + gj] = v;
                    if (gi == gj) { p_tr += v; p_ss = fma(v, v, p_ss); }
                    else p_ss = fma(2.0 * v, v, p_ss);
                }
            }
            __syncthreads();
#pragma unroll
            for (int y = ty; y < 32; y += 8) {
                // mirrored element: H^p(gj, gi) with gj = J*128 + bj*32 + y (row), gi = I*128 + bi*32 + tx
                const int gj = J * SQ_BM + bj * 32 + y, gi = I * SQ_BM + bi * 32 + tx;
                if (gi < k && gj < k && gj > gi) Hp[(size_t)gj * k + gi] = sm[tx][y];
            }
        }
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        p_tr += __shfl_xor_sync(0xffffffffu, p_tr, m);
        p_ss += __shfl_xor_sync(0xffffffffu, p_ss, m);
    }
    if (tx == 0) { red[0][ty] = p_tr; red[1][ty] = p_ss; }
    __syncthreads();
    if (threadIdx.x < SQ_NPART) {
        double v = 0.0;
        if (threadIdx.x < 2)
            for (int w = 0; w < 8; ++w) v += red[threadIdx.x][w];
        rec[(size_t)blockIdx.x * SQ_NPART + threadIdx.x] = v;
    }
}

// ------------------------------------------------------------------------------------------------------------
// Y = P Psi  (k x k times k x M): C(i, m) = sum_j P(i, j) Psi(j, m).
// Tile 128 (i) x 128 (m), K chunks of 16 (j).  Operand A = P row panel, K-contiguous, exactly the squaring
// kernel's panel (128 rows x 128 bytes, 128B swizzle).  Operand B = Psi, whose contraction index j is the SLOW
// index: eight TMA boxes of 16 (j) x 16 (m) per chunk, each a 2 KiB swizzled sub-panel [j][16 m].
// Bank-conflict-free fragment loads need a permuted contraction order inside a 16-chunk -- k4-step q, lane k index
// kk reads j = 8 (q >> 1) + 2 kk + ((kk ^ q) & 1), i.e. {0,3,4,7}, {1,2,5,6}, {8,11,12,15}, {9,10,13,14} -- used for A
// and B alike (a contraction may be summed in any order), and fragment row r of A maps to panel row
// {0,1,4,5,2,3,6,7}[r] inside each 8-row group: every 16-lane half of a 64-bit load then hits 16 distinct 8-byte
// bank pairs for both operands (derivation in DESIGN.md section 12).
constexpr int AP_BN = 128;
constexpr int AP_BBOX_BYTES = SQ_BK * 16 * 8;                           // 2 KiB: 16 j-rows x 16 m
constexpr int AP_STAGE_BYTES = SQ_PANEL_BYTES + 8 * AP_BBOX_BYTES;       // 32 KiB
constexpr int AP_SMEM_BYTES = SQ_STAGES * AP_STAGE_BYTES + 1024;

__global__ void __launch_bounds__(SQ_THREADS, 1)
apply_kernel(const __grid_constant__ CUtensorMap tmP, const __grid_constant__ CUtensorMap tmPsi,
             double* __restrict__ Y, int k, long long M, long long ldy, int kt_total, int vec_ok)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[SQ_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[SQ_STAGES];

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int I = blockIdx.x;                 // i tile (fastest: the resident CTAs share a few Psi blocks in L2)
    const int Mt = blockIdx.y;                // m tile
    const int KT = kt_total;

    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full0 = smem_u32(&full_bar[0]);
    const uint32_t empty0 = smem_u32(&empty_bar[0]);

    if (threadIdx.x == 0) {
        for (int s = 0; s < SQ_STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, SQ_CONSUMER_WARPS);
        }
        mbar_fence_init();
        tma_prefetch_desc(&tmP);
        tma_prefetch_desc(&tmPsi);
    }
    __syncthreads();

    int ld_kt = 0, ld_s = 0;
    uint32_t ld_ph = 0;
    auto issue_loads = [&](int upto) {
        while (ld_kt < upto) {
            if (ld_kt >= SQ_STAGES && !mbar_test(empty0 + 8 * ld_s, ld_ph ^ 1u)) break;
            const uint32_t fb = full0 + 8 * ld_s;
            const uint32_t dstA = smem_base + ld_s * AP_STAGE_BYTES;
            if (elect_one()) {
                mbar_expect_tx(fb, AP_STAGE_BYTES);
                tma_load_2d(dstA, &tmP, ld_kt * SQ_BK, I * SQ_BM, fb);
#pragma unroll
                for (int cb = 0; cb < 8; ++cb)
                    tma_load_2d(dstA + SQ_PANEL_BYTES + cb * AP_BBOX_BYTES, &tmPsi, Mt * AP_BN + cb * 16, ld_kt * SQ_BK, fb);
            }
            __syncwarp();
            ++ld_kt;
            if (++ld_s == SQ_STAGES) { ld_s = 0; ld_ph ^= 1u; }
        }
    };
    if (warp == 0) issue_loads(min(KT, SQ_STAGES));

    const int warp_m = warp >> 2;      // 0..1 -> 64 tile rows
    const int warp_n = warp & 3;       // 0..3 -> 32 tile cols
    const int r = lane >> 2;           // fragment row of A / column of B
    const int kk = lane & 3;           // k index inside a k4-step; C column pair
    const int rmap = (r & 1) | ((r & 2) << 1) | ((r & 4) >> 1);   // 0,1,4,5,2,3,6,7
    // A: element (row R, j) at R*128 + (((j>>1) ^ (R&7)) << 4) + (j&1)*8;   R & 7 = rmap for every 8-row group
    // B: element (j, mm) of box cb at cb*2048 + j*128 + (((mm>>1) ^ (j&7)) << 4) + (mm&1)*8
    uint32_t offA[4], offB[4][2];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int j = 8 * (q >> 1) + 2 * kk + ((kk ^ q) & 1);
        offA[q] = (uint32_t)((((j >> 1) ^ rmap) << 4) + (j & 1) * 8);
#pragma unroll
        for (int odd = 0; odd < 2; ++odd) {
            const int mm = odd * 8 + r;
            offB[q][odd] = (uint32_t)(j * 128 + ((((mm >> 1) ^ (j & 7)) << 4)) + (mm & 1) * 8);
        }
    }
    const uint32_t rowA = (uint32_t)(warp_m * 64 + rmap) * 128u;
    const uint32_t baseB = (uint32_t)SQ_PANEL_BYTES + (uint32_t)(warp_n * 2) * AP_BBOX_BYTES;

    double acc[8][4][2];
#pragma unroll
    for (int mi = 0; mi < 8; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;

    auto load_frag = [&](double (&a)[8], double (&b)[4], uint32_t st, int q) {
#pragma unroll
        for (int mi = 0; mi < 8; ++mi) a[mi] = lds_f64(st + rowA + (uint32_t)(mi * 1024) + offA[q]);
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) b[ni] = lds_f64(st + baseB + (uint32_t)((ni >> 1) * AP_BBOX_BYTES) + offB[q][ni & 1]);
    };
    auto mma_step = [&](const double (&a)[8], const double (&b)[4]) {
#pragma unroll
        for (int mi = 0; mi < 8; ++mi)
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], a[mi], b[ni]);
    };

    // same software pipeline as the squaring kernel: fragments one k4-step ahead, across stage boundaries
    int s = 0;
    uint32_t ph = 0;
    double a0[8], b0[4], a1[8], b1[4];
    mbar_wait(full0, 0);
    uint32_t st = smem_base;
    load_frag(a0, b0, st, 0);
    for (int kt = 0; kt < KT; ++kt) {
        if (warp == 0) {
            issue_loads(min(KT, kt + SQ_STAGES));
            // Warp 0 is the only producer AND a consumer, and it blocks on chunk kt+1 further down: that chunk must have been
            // issued by then, or nobody ever would.  It normally was, five iterations ago; if another warp still holds its stage
            // (a 5-chunk skew, which the 6-stage ring permits), wait HERE, where waiting cannot deadlock (that warp has its data).
            while (ld_kt < min(KT, kt + 2)) issue_loads(min(KT, kt + SQ_STAGES));
        }
        int s1 = s + 1;
        uint32_t ph1 = ph;
        if (s1 == SQ_STAGES) { s1 = 0; ph1 ^= 1u; }
        const uint32_t stn = smem_base + s1 * AP_STAGE_BYTES;
        load_frag(a1, b1, st, 1);
        mma_step(a0, b0);
        load_frag(a0, b0, st, 2);
        mma_step(a1, b1);
        load_frag(a1, b1, st, 3);
        if (kt + 1 < KT) mbar_wait(full0 + 8 * s1, ph1);
        mma_step(a0, b0);
        load_frag(a0, b0, stn, 0);      // after the last stage this reads stale smem; unused
        mma_step(a1, b1);
        __syncwarp();
        if (lane == 0) mbar_arrive(empty0 + 8 * s);
        s = s1; ph = ph1; st = stn;
    }

    // epilogue: C fragment (mi, ni): row = rmap-permuted, cols 2 kk + {0, 1} of the 8-column block
#pragma unroll
    for (int mi = 0; mi < 8; ++mi) {
        const int row = I * SQ_BM + warp_m * 64 + mi * 8 + rmap;
        if (row >= k) continue;
        double* yrow = Y + (size_t)row * (size_t)ldy;
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) {
            const long long col = (long long)Mt * AP_BN + warp_n * 32 + ni * 8 + 2 * kk;
            if (vec_ok && col + 1 < M) {
                *reinterpret_cast<double2*>(yrow + col) = make_double2(acc[mi][ni][0], acc[mi][ni][1]);
            } else {
                if (col < M) yrow[col] = acc[mi][ni][0];
                if (col + 1 < M) yrow[col + 1] = acc[mi][ni][1];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------------
// rho_m = sum_i Psi_im Y_im = diag(Psi^T P Psi): column sums over the k states, HBM-bound (16 k M bytes).
// The k rows are cut into gridDim.y slices; part[slice][m] is summed in ascending slice order by the second kernel.
__global__ void __launch_bounds__(256)
density_partial_kernel(const double* __restrict__ Psi, long long ld, const double* __restrict__ Y, long long ldy,
                       int k, long long M, int rows_per_slice, double* __restrict__ part)
{
    const long long m = (long long)blockIdx.x * 256 + threadIdx.x;
    if (m >= M) return;
    const int i0 = blockIdx.y * rows_per_slice;
    const int i1 = min(k, i0 + rows_per_slice);
    double acc = 0.0;
    int i = i0;
    for (; i + 4 <= i1; i += 4) {
        double p[4], y[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            p[u] = Psi[(size_t)(i + u) * ld + m];
            y[u] = Y[(size_t)(i + u) * ldy + m];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) acc = fma(p[u], y[u], acc);
    }
    for (; i < i1; ++i) acc = fma(Psi[(size_t)i * ld + m], Y[(size_t)i * ldy + m], acc);
    part[(size_t)blockIdx.y * M + m] = acc;
}

__global__ void __launch_bounds__(256)
density_reduce_kernel(const double* __restrict__ part, int n_slices, long long M, double* __restrict__ rho)
{
    const long long m = (long long)blockIdx.x * 256 + threadIdx.x;
    if (m >= M) return;
    double acc = 0.0;
    for (int s = 0; s < n_slices; ++s) acc += part[(size_t)s * M + m];
    rho[m] = acc;
}

}  // namespace rfoe
