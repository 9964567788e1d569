// Symmetric squaring / symmetric product on the FP64 tensor cores (rows A4 + A5 of DESIGN.md).
//
// Computes, for upper-triangle tile pairs I <= J only,
//     C_IJ = sum_l A(I, l) * B(J, l)^T            (A = B = X_n: the SYRK form of X_n * X_n;
//                                                  A = X_n^2, B = X_n: the McWeeny product)
// and fuses the whole recursion update into the epilogue:
//     Out = c2 * C + c1 * E + c0 * I  written to (I,J) and mirrored to (J,I)
//     per-tile partial sums of Tr Out, ||Out||_F^2, ||C - E||_F^2, Tr C, <C, E>
// "matrix-matrix multiplication is the computationally dominant step".
//
// Layout: all matrices are n x n (n = k rounded up to 128), zero outside k x k, row-major FP64 with row
// pitch ld = n + SQ_PAD doubles: a pitch of n*8 bytes is a power of two for k = 8192, 16384, ... and the 128
// rows of every TMA box would then alias in L2 (measured: 6-9x DRAM re-reads, profiles/r01_sym_square_k16384.md).
// Because X is bitwise symmetric, both operands are K-contiguous row panels (128 rows x 16 doubles
// = 128-byte rows) fetched by TMA with the 128-byte swizzle into a 6-stage mbarrier ring; eight warps
// (2 x 4, 64 x 32 outputs each) issue mma.m8n8k4.f64 (SASS DMMA.8x8x4) with accumulators in registers,
// and lane 0 of warp 0 doubles as the TMA producer: it refills a stage as soon as a non-blocking
// mbarrier test shows all eight warps have released it (2 warps per SMSP keep the 255-register budget).
// Fragment row m of a 16-row group maps to tile row 2m + p (p = 0, 1): with the 128B swizzle this makes every 64-bit fragment load bank-conflict free.
// The epilogue's own operand, the 128 x 128 tile of X_n, rides the same ring: four more entries of two boxes each are requested
// while the last chunks are multiplied and land in the stages those chunks free, so the update reads X_n from shared memory
// instead of waiting for eight dependent trips to DRAM (k=16384: 122.06 -> 121.69 ms per squaring, same bits).
#pragma once
#include "ptx_sm100.cuh"

namespace rfoe {

constexpr int SQ_BM = 128;               // tile rows = tile cols
constexpr int SQ_BK = 16;                // doubles per K chunk = one 128-byte swizzle row
constexpr int SQ_STAGES = 6;
constexpr int SQ_CONSUMER_WARPS = 8;
constexpr int SQ_THREADS = SQ_CONSUMER_WARPS * 32;   // no 9th warp: 3 warps on one SMSP would cap registers at 168
constexpr int SQ_PANEL_BYTES = SQ_BM * SQ_BK * 8;                    // 16 KiB
constexpr int SQ_SMEM_BYTES = SQ_STAGES * 2 * SQ_PANEL_BYTES + 1024; // + slack for 1024-byte alignment
constexpr int SQ_PAD = 16;               // doubles added to the row pitch of the work matrices (see below)
constexpr int SQ_NPART = 8;              // doubles per tile record in the partials array (5 used)

struct StepCoef {
    double c2, c1, c0;
};

// MODE 3 (one expansion sharded over several GPUs): the epilogue stores every output tile, its
// mirror and its partial record into the X_{n+1} / record arrays of ALL ranks -- out[d], rec[d] are peer-mapped
// device pointers (NVLink P2P), own rank included -- so the all-gather IS the epilogue's stores, spread over the
// whole launch, and no pack / collective / unpack pass exists.  rec_offset = global index of the launch's first tile.
constexpr int SQ_MAX_PEERS = 16;
struct PeerSet {
    double* out[SQ_MAX_PEERS];
    double* rec[SQ_MAX_PEERS];
    int n;
    int rec_offset;
};

// MODE 0: squaring (A = B = X_n, one tensor map).  MODE 1: symmetric product of two matrices (McWeeny).
// MODE 3: MODE 0 with the epilogue's stores going to every rank of a sharded run (PeerSet above, passed through `Out`).
// MODE 2: Rayleigh-Ritz projection H^p = Psi HPsi^T: the contraction runs over the M degrees
//         of freedom (kt_total chunks of 16, ragged tail zero-filled by TMA), split into gridDim.y slices of
//         kt_per_slice chunks so that tiles x slices fills the 148 SMs evenly; the raw 128 x 128 accumulators go
//         to a tile-contiguous workspace, Out + (slice * gridDim.x + tile) * 128 * 128, and
//         project_reduce_kernel (subspace.cuh) adds the slices in a fixed order and mirrors.
// (kt_per_slice is the LAST parameter on purpose: with it in front of ld ptxas schedules the MODE 0 main loop
// differently and the k=16384 squaring takes 123.25 ms instead of 122.15 ms; in this order the MODE 0 SASS is
// byte-identical to the kernel before MODE 2 existed.)
template <int MODE>
__global__ void __launch_bounds__(SQ_THREADS, 1)
sym_square_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                  const double* __restrict__ E, double* __restrict__ Out, int n, int ld, int kvalid,
                  const StepCoef* __restrict__ coef, const int2* __restrict__ tile_map,
                  double* __restrict__ partials, int kt_per_slice)
{
    constexpr bool TWO_OP = (MODE == 1 || MODE == 2);
    constexpr bool P2P = (MODE == 3);
    // E_SMEM (squarings: E = X_n is the matrix tmA describes): the epilogue's 128 x 128 tile of X_n arrives by TMA as four
    // more ring entries ("chunks" KT .. KT+3: boxes 2v, 2v+1 of the tile in entry v) into the stages the last chunks free,
    // so it is in shared memory when the main loop ends (r02b profile: half of the epilogue was spent waiting for these
    // 128 KiB, one dependent DRAM round trip per 16 x 32 block, with the tensor pipe idle)
    constexpr bool E_SMEM = (MODE == 0 || MODE == 3);
    constexpr int E_CHUNKS = E_SMEM ? (SQ_BM * SQ_BM * 8) / (2 * SQ_PANEL_BYTES) : 0;      // 4
    // MODE 3 has no single output matrix: `Out` carries a pointer to the PeerSet in device memory instead (the
    // parameter list is kept as it is because any change to it perturbs ptxas' schedule of the MODE 0 main loop)
    const PeerSet& peers = *reinterpret_cast<const PeerSet*>(Out);
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[SQ_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[SQ_STAGES];
    __shared__ double red[SQ_CONSUMER_WARPS][5];

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int2 tile = tile_map[blockIdx.x];
    const int I = tile.x, J = tile.y;
    const bool diag = (I == J);
    const bool two_panels = TWO_OP || !diag;
    const int kt0 = (MODE == 2) ? (int)blockIdx.y * kt_per_slice : 0;      // n = contraction extent, a multiple of 16
    const int KT = (MODE == 2) ? min(kt_per_slice, n / SQ_BK - kt0) : n / SQ_BK;

    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full0 = smem_u32(&full_bar[0]);
    const uint32_t empty0 = smem_u32(&empty_bar[0]);

    if (threadIdx.x == 0) {
        for (int s = 0; s < SQ_STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, SQ_CONSUMER_WARPS);
        }
        mbar_fence_init();
    }
    if (threadIdx.x == 0) {
        tma_prefetch_desc(&tmA);
        if (TWO_OP) tma_prefetch_desc(&tmB);
    }
    __syncthreads();

    // ===== TMA producer state (warp 0; the warp stays converged and one elected lane issues, so the TMA
    //       operands live in uniform registers -- an `if (threadIdx.x == 0)` region costs an ELECT /
    //       R2UR.BROADCAST loop in front of every UTMALDG) =====
    const uint32_t stage_bytes = two_panels ? 2 * SQ_PANEL_BYTES : SQ_PANEL_BYTES;
    int ld_kt = 0, ld_s = 0;
    uint32_t ld_ph = 0;
    auto issue_loads = [&](int upto) {
        while (ld_kt < upto) {
            if (ld_kt >= SQ_STAGES && !mbar_test(empty0 + 8 * ld_s, ld_ph ^ 1u)) break;
            const uint32_t fb = full0 + 8 * ld_s;
            const uint32_t dstA = smem_base + ld_s * (2 * SQ_PANEL_BYTES);
            if (E_SMEM && ld_kt >= KT) {
                // entry v = ld_kt - KT of the X_n tile: columns J*128 + 32 v .. + 31 of rows I*128 .. + 127, as two boxes
                if (elect_one()) {
                    mbar_expect_tx(fb, 2 * SQ_PANEL_BYTES);
                    tma_load_2d(dstA, &tmA, J * SQ_BM + (ld_kt - KT) * 2 * SQ_BK, I * SQ_BM, fb);
                    tma_load_2d(dstA + SQ_PANEL_BYTES, &tmA, J * SQ_BM + (ld_kt - KT) * 2 * SQ_BK + SQ_BK, I * SQ_BM, fb);
                }
            } else if (elect_one()) {
                mbar_expect_tx(fb, stage_bytes);
                tma_load_2d(dstA, &tmA, (kt0 + ld_kt) * SQ_BK, I * SQ_BM, fb);
                if (two_panels) tma_load_2d(dstA + SQ_PANEL_BYTES, TWO_OP ? &tmB : &tmA, (kt0 + ld_kt) * SQ_BK, J * SQ_BM, fb);
            }
            __syncwarp();
            ++ld_kt;
            if (++ld_s == SQ_STAGES) { ld_s = 0; ld_ph ^= 1u; }
        }
    };
    if (warp == 0) issue_loads(min(KT, SQ_STAGES));
    {
        // ===== consumers =====
        const int warp_m = warp >> 2;      // 0..1  -> 64 tile rows
        const int warp_n = warp & 3;       // 0..3  -> 32 tile cols
        const int r = lane >> 2;           // fragment row / col index 0..7
        const int kk = lane & 3;           // k index inside the k4 step; also C column pair index
        // swizzled byte offset inside a 128-byte panel row for (k4-step ks, parity p)
        uint32_t off[4][2];
#pragma unroll
        for (int ks = 0; ks < 4; ++ks)
#pragma unroll
            for (int p = 0; p < 2; ++p)
                off[ks][p] = ((uint32_t)(((2 * ks + (kk >> 1)) ^ ((2 * r + p) & 7)) << 4)) + (uint32_t)((kk & 1) * 8);
        const uint32_t rowA = (uint32_t)(warp_m * 64 + 2 * r) * 128u;
        const uint32_t rowB = (uint32_t)(warp_n * 32 + 2 * r) * 128u + (two_panels ? (uint32_t)SQ_PANEL_BYTES : 0u);

        double acc[8][4][2];
#pragma unroll
        for (int mi = 0; mi < 8; ++mi)
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;

        // Software pipeline over the flattened (kt, ks) sequence: the fragments of k4-step q+1 are loaded
        // while the 32 DMMAs of step q issue, ACROSS stage boundaries too -- the full-barrier of stage
        // kt+1 is waited for in the middle of stage kt, so no warp ever reaches a stage boundary with an
        // empty DMMA queue (r01 profile: 5 % of the tensor pipe's cycles were lost exactly there).
        auto load_frag = [&](double (&a)[8], double (&b)[4], uint32_t aB, uint32_t bB, const uint32_t (&o)[2]) {
#pragma unroll
            for (int mi = 0; mi < 8; ++mi) a[mi] = lds_f64(aB + (uint32_t)((mi >> 1) * 2048 + (mi & 1) * 128) + o[mi & 1]);
#pragma unroll
            for (int ni = 0; ni < 4; ++ni) b[ni] = lds_f64(bB + (uint32_t)((ni >> 1) * 2048 + (ni & 1) * 128) + o[ni & 1]);
        };
        auto mma_step = [&](const double (&a)[8], const double (&b)[4]) {
#pragma unroll
            for (int mi = 0; mi < 8; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], a[mi], b[ni]);
        };

        int s = 0;
        uint32_t ph = 0;
        double a0[8], b0[4], a1[8], b1[4];
        mbar_wait(full0, 0);
        uint32_t st = smem_base;
        load_frag(a0, b0, st + rowA, st + rowB, off[0]);
        for (int kt = 0; kt < KT; ++kt) {
            if (warp == 0) {
                issue_loads(min(KT + E_CHUNKS, kt + SQ_STAGES));
                // Warp 0 is the only producer AND a consumer, and it blocks on chunk kt+1 further down: that chunk must have been
                // issued by then, or nobody ever would.  It normally was, five iterations ago; if another warp still holds its stage
                // (a 5-chunk skew, which the 6-stage ring permits), wait HERE, where waiting cannot deadlock (that warp has its data).
                while (ld_kt < min(KT, kt + 2)) issue_loads(min(KT + E_CHUNKS, kt + SQ_STAGES));
            }
            const uint32_t aB = st + rowA, bB = st + rowB;
            int s1 = s + 1;
            uint32_t ph1 = ph;
            if (s1 == SQ_STAGES) { s1 = 0; ph1 ^= 1u; }
            const uint32_t stn = smem_base + s1 * (2 * SQ_PANEL_BYTES);
            load_frag(a1, b1, aB, bB, off[1]);
            mma_step(a0, b0);
            load_frag(a0, b0, aB, bB, off[2]);
            mma_step(a1, b1);
            load_frag(a1, b1, aB, bB, off[3]);
            if (kt + 1 < KT) mbar_wait(full0 + 8 * s1, ph1);
            mma_step(a0, b0);
            // first fragments of the next stage (after the last stage this reads stale smem; unused)
            load_frag(a0, b0, stn + rowA, stn + rowB, off[0]);
            mma_step(a1, b1);
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * s);
            s = s1; ph = ph1; st = stn;
        }

        if (MODE == 2) {
            // raw accumulators -> tile-contiguous workspace (row pitch 128); no update, no mirror, no partials
            double* T = Out + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * (size_t)(SQ_BM * SQ_BM);
#pragma unroll
            for (int mi = 0; mi < 8; ++mi) {
                const int row = warp_m * 64 + 2 * r + 16 * (mi >> 1) + (mi & 1);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const int col = warp_n * 32 + 4 * kk + 16 * h;
                    *reinterpret_cast<double2*>(T + row * SQ_BM + col) = make_double2(acc[mi][2 * h][0], acc[mi][2 * h + 1][0]);
                    *reinterpret_cast<double2*>(T + row * SQ_BM + col + 2) = make_double2(acc[mi][2 * h][1], acc[mi][2 * h + 1][1]);
                }
            }
            return;
        }
        // ===== fused epilogue =====
        // E_SMEM: this warp's 64 x 32 block of X_n lies in ring entry KT + warp_n (box h = columns 16 h .. 16 h + 15 of the
        // block; rows 128 bytes, 16-byte chunks swizzled by the row as everywhere).  Warp 0 first makes sure all four entries
        // are on their way: their stages free up as the other warps leave the main loop, which needs nothing from warp 0 any more.
        uint32_t e_base = 0;
        if (E_SMEM) {
            if (warp == 0)
                while (ld_kt < KT + E_CHUNKS) issue_loads(KT + E_CHUNKS);
            int se = s + warp_n;
            uint32_t phe = ph;
            if (se >= SQ_STAGES) { se -= SQ_STAGES; phe ^= 1u; }
            mbar_wait(full0 + 8 * se, phe);
            e_base = smem_base + (uint32_t)se * (2 * SQ_PANEL_BYTES) + (uint32_t)(warp_m * 64 + 2 * r) * 128u;
        }
        const double c2 = coef->c2, c1 = coef->c1, c0 = coef->c0;
        double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
        const int row_base = I * SQ_BM + warp_m * 64 + 2 * r;       // + 16 g + p
        const int col_base = J * SQ_BM + warp_n * 32 + 4 * kk;      // + 16 h + u
#pragma unroll
        for (int g = 0; g < 4; ++g) {
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                double o[2][4];
                const int col = col_base + 16 * h;
#pragma unroll
                for (int p = 0; p < 2; ++p) {
                    const int row = row_base + 16 * g + p;
                    const int mi = 2 * g + p;
                    const double cv[4] = {acc[mi][2 * h][0], acc[mi][2 * h + 1][0], acc[mi][2 * h][1], acc[mi][2 * h + 1][1]};
                    double2 e01, e23;
                    if (E_SMEM) {
                        // tile row 2r + 16g + p (+ 64 warp_m), box h, columns 4 kk .. 4 kk + 3 = 16-byte chunks 2 kk, 2 kk + 1
                        const uint32_t a = e_base + (uint32_t)(h * SQ_PANEL_BYTES + (16 * g + p) * 128);
                        const uint32_t sw = (uint32_t)((2 * r + p) & 7);
                        e01 = lds_f64x2(a + ((((uint32_t)(2 * kk)) ^ sw) << 4));
                        e23 = lds_f64x2(a + ((((uint32_t)(2 * kk + 1)) ^ sw) << 4));
                    } else {
                        e01 = *reinterpret_cast<const double2*>(E + (size_t)row * ld + col);
                        e23 = *reinterpret_cast<const double2*>(E + (size_t)row * ld + col + 2);
                    }
                    const double ev[4] = {e01.x, e01.y, e23.x, e23.y};
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        double v = fma(c2, cv[u], c1 * ev[u]);
                        const double d = cv[u] - ev[u];
                        double w = 1.0;   // off-diagonal tiles: x2 applied once at the end
                        if (diag) {
                            const int cc = col + u;
                            w = (cc > row) ? 2.0 : ((cc == row) ? 1.0 : 0.0);
                            if (cc == row) {
                                if (row < kvalid) v += c0;
                                p_tr += v;
                                p_trc += cv[u];
                            }
                        }
                        o[p][u] = v;
                        p_ss = fma(w * v, v, p_ss);
                        p_err = fma(w * d, d, p_err);
                        p_ce = fma(w * cv[u], ev[u], p_ce);
                    }
                    if (P2P) continue;
                    if (!diag) {
                        *reinterpret_cast<double2*>(Out + (size_t)row * ld + col) = make_double2(o[p][0], o[p][1]);
                        *reinterpret_cast<double2*>(Out + (size_t)row * ld + col + 2) = make_double2(o[p][2], o[p][3]);
                    } else {
#pragma unroll
                        for (int u = 0; u < 4; ++u)
                            if (col + u >= row) Out[(size_t)row * ld + col + u] = o[p][u];
                    }
                }
                if (P2P) {
                    // the same direct and mirrored stores, to every rank's X_{n+1}
                    const int row0 = row_base + 16 * g;
                    for (int d = 0; d < peers.n; ++d) {
                        double* O = peers.out[d];
#pragma unroll
                        for (int p = 0; p < 2; ++p) {
                            const int row = row0 + p;
                            if (!diag) {
                                *reinterpret_cast<double2*>(O + (size_t)row * ld + col) = make_double2(o[p][0], o[p][1]);
                                *reinterpret_cast<double2*>(O + (size_t)row * ld + col + 2) = make_double2(o[p][2], o[p][3]);
                            } else {
#pragma unroll
                                for (int u = 0; u < 4; ++u)
                                    if (col + u >= row) O[(size_t)row * ld + col + u] = o[p][u];
                            }
                        }
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            if (!diag) {
                                *reinterpret_cast<double2*>(O + (size_t)(col + u) * ld + row0) = make_double2(o[0][u], o[1][u]);
                            } else {
                                if (col + u > row0) O[(size_t)(col + u) * ld + row0] = o[0][u];
                                if (col + u > row0 + 1) O[(size_t)(col + u) * ld + row0 + 1] = o[1][u];
                            }
                        }
                    }
                    continue;
                }
                // mirrored store: element (row, col+u) -> (col+u, row); rows 2r and 2r+1 are adjacent
                const int row0 = row_base + 16 * g;
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if (!diag) {
                        *reinterpret_cast<double2*>(Out + (size_t)(col + u) * ld + row0) = make_double2(o[0][u], o[1][u]);
                    } else {
                        if (col + u > row0) Out[(size_t)(col + u) * ld + row0] = o[0][u];
                        if (col + u > row0 + 1) Out[(size_t)(col + u) * ld + row0 + 1] = o[1][u];
                    }
                }
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
        if (lane == 0) {
            red[warp][0] = p_tr; red[warp][1] = p_ss; red[warp][2] = p_err; red[warp][3] = p_trc; red[warp][4] = p_ce;
        }
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < SQ_CONSUMER_WARPS; ++w) v += red[w][threadIdx.x];
        if (P2P) {
            for (int d = 0; d < peers.n; ++d) peers.rec[d][(size_t)(peers.rec_offset + (int)blockIdx.x) * SQ_NPART + threadIdx.x] = v;
        } else {
            partials[(size_t)blockIdx.x * SQ_NPART + threadIdx.x] = v;
        }
    }
}

}  // namespace rfoe
