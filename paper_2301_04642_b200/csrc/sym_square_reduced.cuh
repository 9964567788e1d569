// Reduced-precision symmetric squaring on the 5th-generation tensor cores (row A8 of DESIGN.md):
// the paper's mixed-precision RFOE runs the squarings far from convergence in FP32.
// Here an "FP32 step" is a three-product split: X = Xh + Xl with two 11-significant-bit parts (FP16, scaled; see
// "Operand format" below), and
//     C = Xh Xh^T  +  (Xh Xl^T + Xl Xh^T)          (Xl Xl^T, 2^-22 relative, is dropped)
// computed by tcgen05.mma (kind::f16) with TWO FP32 accumulators in tensor memory (the exact-product
// head term and the small cross terms are accumulated separately and added in FP64 in the epilogue).
// Two measures keep the tensor cores' FP32 accumulation (which TRUNCATES: measured, a systematic bias of
// ~(k/8) 2^-24 on coherent sums such as the diagonal of X^2, enough to push eigenvalues past 1 and make SP2
// diverge) at plain-FP32 accuracy:
//   * shift: with d = Tr X / k the product is taken of Z = X - d I (zero-mean diagonal, small entries) and
//     X^2 = Z^2 + 2 d X - d^2 I is completed exactly in FP64 in the epilogue;
//   * chunking: the head term is accumulated in tensor memory over 256 k values only, then drained by the
//     (otherwise idle) epilogue warps into FP32 register sums with round-to-nearest adds, double-buffered.
// The master copy of X stays FP64: the epilogue is the same as the FP64 kernel's -- Out = c2 C + c1 X
// + c0 I written to (I,J) and mirrored, five FP64 partial sums per tile -- so the recursion, its
// scalars and its control flow are unchanged; only the product is reduced precision.
//
// Roles (320 threads): warp 0 = TMA producer, warp 1 = TMEM allocator + MMA issuer (both warps stay converged
// and one elected lane issues, so the TMA / tcgen05 operands live in uniform registers), warps 2..9 = epilogue: warp w reads
// the 32 TMEM lanes (tile rows) of quarter w % 4 and owns 64 of the tile's 128 columns (two warps per quarter: 64 FP32 head
// sums per thread instead of 128 -- no spills -- and twice the threads behind the FP64 epilogue's memory latency; round 1's
// four warps spent 38 % of the kernel there at k=8192).
// Clusters of two CTAs own the tiles (I, J0) and (I, J0+1): they share the row panels Zh(I), Zl(I), each
// CTA fetches half of them and TMA-multicasts it to both (25 % fewer L2 requests per CTA; measured: no
// change in time -- the kernel runs into the 1 kW power cap).
// A stage is refilled only after BOTH CTAs' MMAs have
// read it (multicast tcgen05.commit on both empty barriers).  A row with an odd number of tiles ends in a
// phantom tile (J0+1 = m): that CTA loads zeros (TMA out-of-bounds fill), serves its half of the shared
// panels and writes nothing but a zero partial record.
//
// Operand format (RFOE_REDUCED_F16, default 1).  The two parts only carry 11 significant bits each, which is what
// FP16 holds, and |Z_ij| <= ||Z||_2 <= 1 bounds their range: with Zh = fp16(2^15 z) 2^-15 and Zl = fp16(2^26 (z - Zh))
// 2^-26 every product Zh Zh, Zh Zl is exact in FP32 exactly as with tf32 parts, entries down to 2^-29 keep full
// precision, and the three products run as tcgen05.mma.kind::f16 (K = 16 per instruction, twice the tf32 rate, half
// the operand bytes through TMA and shared memory).  The scalings 2^-30 / 2^-41 are undone in the FP64 epilogue.
// RFOE_REDUCED_F16 = 0 keeps the original tf32 parts (kind::tf32, K = 8).
//
// This file holds the split pass, the constants and the ONE-CTA-PER-TILE form of the kernel (RFOE_OPT_REDUCED_PAIR = 0); the
// default form issues the same products as CTA-pair MMAs (tcgen05.mma.cta_group::2): sym_square_reduced_pair.cuh.
#pragma once
#include <cuda_fp16.h>

#include "ptx_sm100.cuh"
#include "sym_square.cuh"

#ifndef RFOE_REDUCED_F16
#define RFOE_REDUCED_F16 1
#endif

namespace rfoe {

#if RFOE_REDUCED_F16
typedef __half tq_elem_t;
constexpr int TQ_UK = 16;                  // K of one tcgen05.mma.kind::f16
constexpr double TQ_SCALE_HI = 32768.0;    // 2^15
constexpr double TQ_SCALE_LO = 67108864.0; // 2^26
#else
typedef float tq_elem_t;
constexpr int TQ_UK = 8;                   // K of one tcgen05.mma.kind::tf32
constexpr double TQ_SCALE_HI = 1.0;
constexpr double TQ_SCALE_LO = 1.0;
#endif
constexpr double TQ_UNSCALE_HEAD = 1.0 / (TQ_SCALE_HI * TQ_SCALE_HI);
constexpr double TQ_UNSCALE_CROSS = 1.0 / (TQ_SCALE_HI * TQ_SCALE_LO);
constexpr int TQ_BM = 128;                 // tile rows = cols (UMMA M = N = 128, cta_group::1)
constexpr int TQ_BK = 128 / (int)sizeof(tq_elem_t);   // elements per K chunk = one 128-byte swizzle row (32 tf32 / 64 f16)
constexpr int TQ_STAGES = 3;
#ifndef TQ_EPI_WARPS_N
#define TQ_EPI_WARPS_N 8
#endif
constexpr int TQ_EPI_WARPS = TQ_EPI_WARPS_N;             // 4 TMEM lane quarters x (TQ_EPI_WARPS / 4) column ranges
constexpr int TQ_THREADS = 64 + 32 * TQ_EPI_WARPS;
constexpr int TQ_EPI_COLS = TQ_BM / (TQ_EPI_WARPS / 4);  // columns per epilogue warp
constexpr int TQ_PANEL_BYTES = TQ_BM * 128;                       // 16 KiB
constexpr int TQ_STAGE_BYTES = 4 * TQ_PANEL_BYTES;               // A_hi, A_lo, B_hi, B_lo
constexpr int TQ_SMEM_BYTES = TQ_STAGES * TQ_STAGE_BYTES + 1024; // + slack for 1024-byte alignment
constexpr int TQ_CHUNK_KT = 256 / TQ_BK;   // K chunks per tensor-memory accumulation run: 256 k values
constexpr int TQ_TMEM_COLS = 512;          // head accumulator x 2 (double-buffered) + cross-term accumulator
constexpr int TQ_HALF_BYTES = TQ_PANEL_BYTES / 2;                // 64 rows of a panel
constexpr int TQ_PAD = 128 / (int)sizeof(tq_elem_t);   // elements added to the row pitch of the hi / lo matrices

// HBM-bound: split the FP64 work matrix (n x n, pitch ld) into the hi and lo part matrices (n x n, pitch ld32
// elements) of Z = X - d I, d = *trace / kvalid (rows >= kvalid stay zero).
// FP16 parts: hi = fp16(2^15 z), lo = fp16(2^26 (z - 2^-15 hi)), the residual exact in FP64 (|z| <= 1: no overflow).
// tf32 parts (RFOE_REDUCED_F16 = 0): hi = tf32(fl32(z)), lo = tf32(fl32(z - hi)).
__global__ void __launch_bounds__(256)
split_parts_kernel(const double* __restrict__ X, int n, int ld, int kvalid, const double* __restrict__ trace,
                  tq_elem_t* __restrict__ Hi, tq_elem_t* __restrict__ Lo, int ld32)
{
    const double d = *trace / (double)kvalid;
    const int lane = threadIdx.x & 31;
    const int wglobal = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int wtotal = gridDim.x * 8;
    for (int i = wglobal; i < n; i += wtotal) {
        const double2* row = reinterpret_cast<const double2*>(X + (size_t)i * ld);
#if RFOE_REDUCED_F16
        __half2* hrow = reinterpret_cast<__half2*>(Hi + (size_t)i * ld32);
        __half2* lrow = reinterpret_cast<__half2*>(Lo + (size_t)i * ld32);
#else
        float2* hrow = reinterpret_cast<float2*>(Hi + (size_t)i * ld32);
        float2* lrow = reinterpret_cast<float2*>(Lo + (size_t)i * ld32);
#endif
#pragma unroll 4
        for (int j = lane; j < n / 2; j += 32) {
            double2 x = row[j];
            if (2 * j == i && i < kvalid) x.x -= d;
            if (2 * j + 1 == i && i < kvalid) x.y -= d;
#if RFOE_REDUCED_F16
            // |z| <= ||Z||_2 <= 1 inside an expansion (spectrum of X in [0,1]); the clamp only keeps a caller's
            // out-of-contract matrix (|z| >= 2) from producing infinities
            x.x = fmin(fmax(x.x, -1.99), 1.99);
            x.y = fmin(fmax(x.y, -1.99), 1.99);
            const __half hx = __double2half(x.x * TQ_SCALE_HI), hy = __double2half(x.y * TQ_SCALE_HI);
            const double rx = x.x - (double)__half2float(hx) * (1.0 / TQ_SCALE_HI);      // exact in FP64
            const double ry = x.y - (double)__half2float(hy) * (1.0 / TQ_SCALE_HI);
            hrow[j] = __halves2half2(hx, hy);
            lrow[j] = __halves2half2(__double2half(rx * TQ_SCALE_LO), __double2half(ry * TQ_SCALE_LO));
#else
            float2 h, l;
            h.x = to_tf32((float)x.x);
            h.y = to_tf32((float)x.y);
            l.x = to_tf32((float)(x.x - (double)h.x));
            l.y = to_tf32((float)(x.y - (double)h.y));
            hrow[j] = h;
            lrow[j] = l;
#endif
        }
    }
}

__global__ void __launch_bounds__(TQ_THREADS, 1)
sym_square_reduced_kernel(const __grid_constant__ CUtensorMap tmHi, const __grid_constant__ CUtensorMap tmLo,
                       const double* __restrict__ E, double* __restrict__ Out, int n, int ld, int kvalid,
                       const double* __restrict__ trace, const StepCoef* __restrict__ coef,
                       const int2* __restrict__ pair_map, int m_tiles, double* __restrict__ partials)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[TQ_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[TQ_STAGES];
    __shared__ __align__(8) uint64_t hfull_bar[2];    // head accumulator b holds a finished chunk
    __shared__ __align__(8) uint64_t hempty_bar[2];   // head accumulator b has been drained
    __shared__ uint32_t tmem_base_sh;
    __shared__ double red[TQ_EPI_WARPS][5];

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t crank = cluster_ctarank();               // 0 or 1
    const int2 pair = pair_map[blockIdx.x >> 1];
    const int I = pair.x, J = pair.y + (int)crank;
    const bool phantom = (J >= m_tiles);
    const bool diag = (I == J);
    const int KT = n / TQ_BK;

    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full0 = smem_u32(&full_bar[0]);
    const uint32_t empty0 = smem_u32(&empty_bar[0]);
    const uint32_t hfull0 = smem_u32(&hfull_bar[0]);
    const uint32_t hempty0 = smem_u32(&hempty_bar[0]);

    if (threadIdx.x == 0) {
        for (int s = 0; s < TQ_STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, 2);      // this CTA's MMA commit + the peer's
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(hfull0 + 8 * b, 1);
            mbar_init(hempty0 + 8 * b, TQ_EPI_WARPS);     // lane 0 of each epilogue warp
        }
        mbar_fence_init();
        tma_prefetch_desc(&tmHi);
        tma_prefetch_desc(&tmLo);
    }
    if (warp == 1) tmem_alloc<TQ_TMEM_COLS>(smem_u32(&tmem_base_sh));
    tc_fence_before();
    cluster_sync_all();                         // barriers of both CTAs initialised before any multicast lands
    tc_fence_after();
    const uint32_t tmem = tmem_base_sh;

    if (warp == 0) {
        // ===== TMA producer (the warp stays converged; one elected lane issues) =====
        {
            int s = 0;
            uint32_t ph = 0;
            for (int kt = 0; kt < KT; ++kt) {
                mbar_wait_bounded(empty0 + 8 * s, ph ^ 1u);              // both CTAs have consumed this stage
                const uint32_t fb = full0 + 8 * s;
                const uint32_t dst = smem_base + s * TQ_STAGE_BYTES;
                if (elect_one()) {
                mbar_expect_tx(fb, TQ_STAGE_BYTES);                     // 2 x 8 KiB from me + 2 x 8 KiB from the peer + 32 KiB own
                const int c0 = kt * TQ_BK;
                // my half of the shared row panels, to both CTAs
                tma_load_2d_mc(dst + crank * TQ_HALF_BYTES, &tmHi, c0, I * TQ_BM + (int)crank * 64, fb, (uint16_t)3);
                tma_load_2d_mc(dst + TQ_PANEL_BYTES + crank * TQ_HALF_BYTES, &tmLo, c0, I * TQ_BM + (int)crank * 64, fb, (uint16_t)3);
                // my own column panels (rows of tile column J; beyond the matrix for a phantom tile -> zeros)
                tma_load_2d(dst + 2 * TQ_PANEL_BYTES, &tmHi, c0, J * TQ_BM, fb);
                tma_load_2d(dst + 2 * TQ_PANEL_BYTES + TQ_HALF_BYTES, &tmHi, c0, J * TQ_BM + 64, fb);
                tma_load_2d(dst + 3 * TQ_PANEL_BYTES, &tmLo, c0, J * TQ_BM, fb);
                tma_load_2d(dst + 3 * TQ_PANEL_BYTES + TQ_HALF_BYTES, &tmLo, c0, J * TQ_BM + 64, fb);
                }
                __syncwarp();
                if (++s == TQ_STAGES) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer (converged warp, one elected lane): 3 tcgen05.mma per 8-wide k step =====
        {
#if RFOE_REDUCED_F16
            constexpr uint32_t idesc = umma_idesc_f16(TQ_BM, TQ_BM);
#define RFOE_UMMA umma_f16
#else
            constexpr uint32_t idesc = umma_idesc_tf32(TQ_BM, TQ_BM);
#define RFOE_UMMA umma_tf32
#endif
            int s = 0;
            uint32_t ph = 0;
            for (int kt = 0; kt < KT; ++kt) {
                const int kc = kt % TQ_CHUNK_KT;             // position inside the chunk
                const int hb = (kt / TQ_CHUNK_KT) & 1;       // head accumulator of this chunk
                if (kc == 0 && kt >= 2 * TQ_CHUNK_KT) {      // buffer reused: wait until its previous chunk is drained
                    mbar_wait_bounded(hempty0 + 8 * hb, (uint32_t)((kt / (2 * TQ_CHUNK_KT)) - 1) & 1u);
                    tc_fence_after();
                }
                mbar_wait_bounded(full0 + 8 * s, ph);
                tc_fence_after();
                const uint32_t a_hi = smem_base + s * TQ_STAGE_BYTES;
                const uint32_t a_lo = a_hi + TQ_PANEL_BYTES;
                const uint64_t dAh = umma_desc_k128(a_hi), dAl = umma_desc_k128(a_lo);
                const uint64_t dBh = umma_desc_k128(a_hi + 2 * TQ_PANEL_BYTES);
                const uint64_t dBl = umma_desc_k128(a_hi + 3 * TQ_PANEL_BYTES);
                const uint32_t t_head = tmem + hb * TQ_BM, t_cross = tmem + 2 * TQ_BM;
                if (elect_one()) {
#pragma unroll
                for (int ks = 0; ks < TQ_BK / TQ_UK; ++ks) {
                    const uint64_t o = (uint64_t)(ks * TQ_UK * (int)sizeof(tq_elem_t) >> 4);   // 32 bytes per k step, in 16-byte units
                    RFOE_UMMA(t_head, dAh + o, dBh + o, idesc, (kc | ks) != 0);   // head: Zh Zh^T (products exact in FP32)
                    RFOE_UMMA(t_cross, dAh + o, dBl + o, idesc, (kt | ks) != 0);  // cross terms: tiny, one long accumulation
                    RFOE_UMMA(t_cross, dAl + o, dBh + o, idesc, 1u);
                }
                umma_commit_mc(empty0 + 8 * s, (uint16_t)3);   // frees the stage in BOTH CTAs' producers' view
                if (kc == TQ_CHUNK_KT - 1 || kt == KT - 1) umma_commit(hfull0 + 8 * hb);   // chunk complete
                }
                __syncwarp();
                if (++s == TQ_STAGES) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ===== epilogue warps: TMEM -> registers -> fused FP64 update, mirror, partial sums =====
        const int q = warp & 3;                   // TMEM lane quarter this warp may access
        const int ew = warp - 2;                  // 0..7
        const int c_lo = (ew >> 2) * TQ_EPI_COLS; // this warp's 64 columns of the tile
        const int row = I * TQ_BM + q * 32 + lane;
        const uint32_t trow = tmem + ((uint32_t)(q * 32) << 16);
        // ---- drain the head accumulator chunk by chunk into FP32 register sums (round-to-nearest adds)
        float hsum[TQ_EPI_COLS];
        const int NC = (KT + TQ_CHUNK_KT - 1) / TQ_CHUNK_KT;
#pragma unroll 1
        for (int ch = 0; ch < NC; ++ch) {
            const int hb = ch & 1;
            mbar_wait_bounded(hfull0 + 8 * hb, (uint32_t)(ch >> 1) & 1u);
            tc_fence_after();
#pragma unroll
            for (int cb = 0; cb < TQ_EPI_COLS; cb += 16) {
                float v[16];
                tmem_ld16(trow + hb * TQ_BM + c_lo + cb, v);
#pragma unroll
                for (int u = 0; u < 16; ++u) hsum[cb + u] = (ch == 0) ? v[u] : __fadd_rn(hsum[cb + u], v[u]);
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(hempty0 + 8 * hb);
        }
        // ---- the last chunk's commit also covers every cross-term MMA: finish in FP64
        if (phantom) {
            if (lane == 0) { red[ew][0] = red[ew][1] = red[ew][2] = red[ew][3] = red[ew][4] = 0.0; }
        } else {
        const double d = *trace / (double)kvalid;
        const double c2 = coef->c2, c1 = coef->c1, c0 = coef->c0;
        double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
        const double* erow = E + (size_t)row * ld + (size_t)J * TQ_BM + c_lo;
        double* orow = Out + (size_t)row * ld + (size_t)J * TQ_BM + c_lo;
        // Global accesses of the 32 x 16 block a warp handles per step go through a staging patch in the operand ring (free
        // by now: the last commit covers every MMA of this CTA, and the peer's multicasts into this CTA were needed by them):
        // with lane = row (the TMEM layout) a 16-byte load or store touches 32 rows -- 32 sectors for 512 bytes; staged, 8
        // lanes cover one row's 128 bytes and an instruction covers 4 whole rows.  Patch layout: element (r, c) at
        // r * 16 + 2 * ((c / 2) ^ (r & 7)) + (c & 1): conflict-free 16-byte accesses both by row (lane = r) and by quarter
        // warp (8 lanes = one row).
        double* const stg_e = reinterpret_cast<double*>(smem_raw + (smem_base - smem_u32(smem_raw))) + ew * 1024;
        double* const stg_o = stg_e + 512;
        const int srow = lane >> 3, sch = lane & 7;            // coalesced side: row inside a group of 4, 16-byte chunk of the row
        const double* eblk = E + (size_t)(I * TQ_BM + q * 32) * ld + (size_t)J * TQ_BM + c_lo;
        double* oblk = Out + (size_t)(I * TQ_BM + q * 32) * ld + (size_t)J * TQ_BM + c_lo;
#pragma unroll
        for (int cb = 0; cb < TQ_EPI_COLS; cb += 16) {
            float xx[16];
            tmem_ld16(trow + 2 * TQ_BM + c_lo + cb, xx);
            double ev[16], o[16];
            if (!diag) {
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int rr = 4 * i + srow;
                    const double2 v = *reinterpret_cast<const double2*>(eblk + (size_t)rr * ld + cb + 2 * sch);
                    *reinterpret_cast<double2*>(stg_e + rr * 16 + 2 * (sch ^ (rr & 7))) = v;
                }
                __syncwarp();
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const double2 e2 = *reinterpret_cast<const double2*>(stg_e + lane * 16 + 2 * (j ^ (lane & 7)));
                    ev[2 * j] = e2.x; ev[2 * j + 1] = e2.y;
                }
            } else {
#pragma unroll
                for (int u = 0; u < 16; u += 2) {
                    const double2 e2 = *reinterpret_cast<const double2*>(erow + cb + u);
                    ev[u] = e2.x; ev[u + 1] = e2.y;
                }
            }
            const int col = J * TQ_BM + c_lo + cb;
#pragma unroll
            for (int u = 0; u < 16; ++u) {
                // X^2 = Z^2 + 2 d X - d^2 I   (Z = X - d I on rows < kvalid)
                double cv = fma(2.0 * d, ev[u], (double)hsum[cb + u] * TQ_UNSCALE_HEAD + (double)xx[u] * TQ_UNSCALE_CROSS);
                double v;
                const double d0 = cv - ev[u];
                double w = 1.0;                   // off-diagonal tiles: x2 applied once at the end
                if (diag) {
                    const int cc = col + u;
                    w = (cc > row) ? 2.0 : ((cc == row) ? 1.0 : 0.0);
                    if (cc == row && row < kvalid) cv -= d * d;
                    v = fma(c2, cv, c1 * ev[u]);
                    if (cc == row) {
                        if (row < kvalid) v += c0;
                        p_tr += v;
                        p_trc += cv;
                    }
                } else {
                    v = fma(c2, cv, c1 * ev[u]);
                }
                const double dd = diag ? (cv - ev[u]) : d0;
                o[u] = v;
                p_ss = fma(w * v, v, p_ss);
                p_err = fma(w * dd, dd, p_err);
                p_ce = fma(w * cv, ev[u], p_ce);
            }
            if (!diag) {
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    *reinterpret_cast<double2*>(stg_o + lane * 16 + 2 * (j ^ (lane & 7))) = make_double2(o[2 * j], o[2 * j + 1]);
#pragma unroll
                for (int u = 0; u < 16; ++u) Out[(size_t)(col + u) * ld + row] = o[u];   // mirror: lanes = consecutive rows
                __syncwarp();
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int rr = 4 * i + srow;
                    const double2 v = *reinterpret_cast<const double2*>(stg_o + rr * 16 + 2 * (sch ^ (rr & 7)));
                    *reinterpret_cast<double2*>(oblk + (size_t)rr * ld + cb + 2 * sch) = v;
                }
                __syncwarp();
            } else {
#pragma unroll
                for (int u = 0; u < 16; ++u) {
                    if (col + u >= row) orow[cb + u] = o[u];
                    if (col + u > row) Out[(size_t)(col + u) * ld + row] = o[u];
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
            red[ew][0] = p_tr; red[ew][1] = p_ss; red[ew][2] = p_err; red[ew][3] = p_trc; red[ew][4] = p_ce;
        }
        }
    }
    __syncwarp();
    tc_fence_before();
    cluster_sync_all();                         // the peer's commits / multicasts into this CTA are over
    if (warp == 1) tmem_dealloc<TQ_TMEM_COLS>(tmem);
    if (threadIdx.x < 5)
    {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < TQ_EPI_WARPS; ++w) v += red[w][threadIdx.x];      // fixed order
        partials[(size_t)blockIdx.x * SQ_NPART + threadIdx.x] = v;
    }
}

}  // namespace rfoe
