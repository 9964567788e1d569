// Reduced-precision symmetric squaring (row A8), CTA-PAIR form: sym_square_reduced.cuh's three-product split
//     C = Zh Zh^T + (Zh Zl^T + Zl Zh^T),   Z = X - (Tr X / k) I = Zh + Zl  (scaled FP16 parts),
// its chunked head accumulation and its FP64 epilogue, with the products issued as tcgen05.mma.cta_group::2.
//
// Why.  With one CTA per tile every 128 x 128 x 16 MMA reads 4 KiB of A and 4 KiB of B from shared memory in the 64 cycles
// it runs: 128 B/clk, all a Blackwell SM's shared memory delivers -- and the TMA writes of the next stage (16 KiB per k16
// step for the four panels) come on top: 40 KiB per 192 cycles of tensor work, i.e. the loop is shared-memory bound at
// ~61 % of the pipe (measured: 52 % active at the capped clock).  A CTA pair splits B between the two SMs of a TPC:
//   CTA r of the pair (tiles (I, J0) and (I, J0 + 1)) holds ITS OWN column panels Zh(J0 + r), Zl(J0 + r) as "A" (128
//   rows) and rows 64 r .. 64 r + 63 of the shared row panels Zh(I), Zl(I) as its half of "B" (N = 128), and gets
//       D_r = Z(J0 + r) Z(I)^T = C(I, J0 + r)^T        (128 x 128, FP32, in its own tensor memory)
//   from ONE instruction issued by the leader (cluster rank 0) with M = 256.
// Per k16 step and SM: 3 x (4 + 2) KiB of operand reads + 12 KiB of TMA writes = 30 KiB (was 40), 48 KiB per stage (was 64:
// four stages fit instead of three), and no multicast: each CTA loads exactly what lives in its own shared memory.
// The tile arrives TRANSPOSED (lanes = rows of block J, columns = rows of block I).  X is bitwise symmetric and the
// epilogue writes every element to (I,J) and (J,I) anyway, so the epilogue is the single-CTA one with I and J exchanged:
// it reads X_n's block (J, I), stores block (J, I) directly and block (I, J) as the mirror.  Operand order of the two cross
// products is chosen so that every FP32 sum adds the same products in the same order as the single-CTA kernel (measured: the
// two kernels agree to ~3e-12 absolute on entries of size 1, not to the bit -- the M = 256 instruction rounds differently).
//
// Protocol (per CTA: warp 0 = TMA producer, warp 1 = tensor-memory allocator and, in the leader only, MMA issuer, warps
// 2..9 = epilogue):
//   full[s]   lives in the LEADER: its producer expects the bytes of both CTAs' stage (96 KiB); both CTAs' TMA loads
//             (cp.async.bulk.tensor ... cta_group::2) complete on it.
//   empty[s]  in each CTA: one arrival, the leader's multicast tcgen05.commit after the MMAs that read the stage.
//   hfull[b]  in each CTA: multicast commit when head accumulator b holds a finished 256-k chunk (the last one also covers
//             all cross-term MMAs).
//   hempty[b] in the LEADER: lane 0 of every epilogue warp of BOTH CTAs arrives after draining buffer b (remote arrive).
// Every wait is bounded (trap after ~2 s), as in the single-CTA kernel.
#pragma once
#include "sym_square_reduced.cuh"

namespace rfoe {

constexpr int TP_STAGES = 4;
constexpr int TP_STAGE_BYTES = 2 * TQ_PANEL_BYTES + 2 * TQ_HALF_BYTES;     // Zh(J), Zl(J) + my 64 rows of Zh(I), Zl(I): 48 KiB
constexpr int TP_SMEM_BYTES = TP_STAGES * TP_STAGE_BYTES + 1024;           // + slack for 1024-byte alignment

#if RFOE_REDUCED_F16
__global__ void __launch_bounds__(TQ_THREADS, 1)
sym_square_reduced_pair_kernel(const __grid_constant__ CUtensorMap tmHi, const __grid_constant__ CUtensorMap tmLo,
                               const double* __restrict__ E, double* __restrict__ Out, int n, int ld, int kvalid,
                               const double* __restrict__ trace, const StepCoef* __restrict__ coef,
                               const int2* __restrict__ pair_map, int m_tiles, double* __restrict__ partials)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[TP_STAGES];    // used in the leader
    __shared__ __align__(8) uint64_t empty_bar[TP_STAGES];
    __shared__ __align__(8) uint64_t hfull_bar[2];
    __shared__ __align__(8) uint64_t hempty_bar[2];          // used in the leader
    __shared__ uint32_t tmem_base_sh;
    __shared__ double red[TQ_EPI_WARPS][5];

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const uint32_t crank = cluster_ctarank();                // 0 = leader
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
        for (int s = 0; s < TP_STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);       // the leader's producer (arrive + expect_tx of both CTAs' bytes)
            mbar_init(empty0 + 8 * s, 1);      // the leader's multicast commit
        }
        for (int b = 0; b < 2; ++b) {
            mbar_init(hfull0 + 8 * b, 1);
            mbar_init(hempty0 + 8 * b, 2 * TQ_EPI_WARPS);     // lane 0 of each epilogue warp of both CTAs
        }
        mbar_fence_init();
        tma_prefetch_desc(&tmHi);
        tma_prefetch_desc(&tmLo);
    }
    if (warp == 1) tmem_alloc_pair<TQ_TMEM_COLS>(smem_u32(&tmem_base_sh));
    tc_fence_before();
    cluster_sync_all();                         // both CTAs' barriers exist before anything remote arrives on them
    tc_fence_after();
    const uint32_t tmem = tmem_base_sh;

    if (warp == 0) {
        // ===== TMA producer, both CTAs (the warp stays converged; one elected lane issues) =====
        int s = 0;
        uint32_t ph = 0;
        for (int kt = 0; kt < KT; ++kt) {
            mbar_wait_bounded(empty0 + 8 * s, ph ^ 1u);                  // the pair's MMAs have read this stage (in both CTAs)
            const uint32_t fb_leader = map_to_cta(full0 + 8 * s, 0);
            const uint32_t dst = smem_base + s * TP_STAGE_BYTES;
            if (elect_one()) {
                if (crank == 0) mbar_expect_tx(full0 + 8 * s, 2 * TP_STAGE_BYTES);
                const int c0 = kt * TQ_BK;
                // my own column panels (rows of tile column J; beyond the matrix for a phantom tile -> zeros)
                tma_load_2d_pair(dst, &tmHi, c0, J * TQ_BM, fb_leader);
                tma_load_2d_pair(dst + TQ_HALF_BYTES, &tmHi, c0, J * TQ_BM + 64, fb_leader);
                tma_load_2d_pair(dst + TQ_PANEL_BYTES, &tmLo, c0, J * TQ_BM, fb_leader);
                tma_load_2d_pair(dst + TQ_PANEL_BYTES + TQ_HALF_BYTES, &tmLo, c0, J * TQ_BM + 64, fb_leader);
                // my 64 rows of the shared row panels
                tma_load_2d_pair(dst + 2 * TQ_PANEL_BYTES, &tmHi, c0, I * TQ_BM + (int)crank * 64, fb_leader);
                tma_load_2d_pair(dst + 2 * TQ_PANEL_BYTES + TQ_HALF_BYTES, &tmLo, c0, I * TQ_BM + (int)crank * 64, fb_leader);
            }
            __syncwarp();
            if (++s == TP_STAGES) { s = 0; ph ^= 1u; }
        }
    } else if (warp == 1) {
        if (crank == 0) {
            // ===== MMA issuer, leader only (converged warp, one elected lane): 3 pair MMAs per k16 step =====
            constexpr uint32_t idesc = umma_idesc_f16(2 * TQ_BM, TQ_BM);   // M = 256 over the pair, N = 128
            int s = 0;
            uint32_t ph = 0;
            for (int kt = 0; kt < KT; ++kt) {
                const int kc = kt % TQ_CHUNK_KT;             // position inside the chunk
                const int hb = (kt / TQ_CHUNK_KT) & 1;       // head accumulator of this chunk
                if (kc == 0 && kt >= 2 * TQ_CHUNK_KT) {      // buffer reused: both CTAs must have drained its previous chunk
                    mbar_wait_bounded(hempty0 + 8 * hb, (uint32_t)((kt / (2 * TQ_CHUNK_KT)) - 1) & 1u);
                    tc_fence_after();
                }
                mbar_wait_bounded(full0 + 8 * s, ph);
                tc_fence_after();
                const uint32_t a_hi = smem_base + s * TP_STAGE_BYTES;
                const uint64_t dAh = umma_desc_k128(a_hi), dAl = umma_desc_k128(a_hi + TQ_PANEL_BYTES);
                const uint64_t dBh = umma_desc_k128(a_hi + 2 * TQ_PANEL_BYTES);
                const uint64_t dBl = umma_desc_k128(a_hi + 2 * TQ_PANEL_BYTES + TQ_HALF_BYTES);
                const uint32_t t_head = tmem + hb * TQ_BM, t_cross = tmem + 2 * TQ_BM;
                if (elect_one()) {
#pragma unroll
                    for (int ks = 0; ks < TQ_BK / TQ_UK; ++ks) {
                        const uint64_t o = (uint64_t)(ks * TQ_UK * (int)sizeof(tq_elem_t) >> 4);   // 32 bytes per k step, in 16-byte units
                        umma_f16_pair(t_head, dAh + o, dBh + o, idesc, (kc | ks) != 0);    // head: Zh(J) Zh(I)^T
                        umma_f16_pair(t_cross, dAl + o, dBh + o, idesc, (kt | ks) != 0);   // Zl(J) Zh(I)^T (= Zh(I) Zl(J)^T transposed: first, as there)
                        umma_f16_pair(t_cross, dAh + o, dBl + o, idesc, 1u);               // Zh(J) Zl(I)^T
                    }
                    umma_commit_pair_mc(empty0 + 8 * s, (uint16_t)3);      // frees the stage in both CTAs
                    if (kc == TQ_CHUNK_KT - 1 || kt == KT - 1) umma_commit_pair_mc(hfull0 + 8 * hb, (uint16_t)3);   // chunk complete
                }
                __syncwarp();
                if (++s == TP_STAGES) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ===== epilogue warps, both CTAs: TMEM -> registers -> fused FP64 update, mirror, partial sums.  The tile is
        //       C(I,J)^T: lanes = rows of block J, columns = rows of block I; sym_square_reduced.cuh's epilogue with I <-> J =====
        const uint32_t hempty_leader = map_to_cta(hempty0, 0);
        const int q = warp & 3;                   // TMEM lane quarter this warp may access
        const int ew = warp - 2;                  // 0..7
        const int c_lo = (ew >> 2) * TQ_EPI_COLS; // this warp's 64 columns of the tile
        const int row = J * TQ_BM + q * 32 + lane;
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
            if (lane == 0) mbar_arrive_cluster(hempty_leader + 8 * hb);
        }
        // ---- the last chunk's commit also covers every cross-term MMA: finish in FP64
        if (phantom) {
            if (lane == 0) { red[ew][0] = red[ew][1] = red[ew][2] = red[ew][3] = red[ew][4] = 0.0; }
        } else {
        const double d = *trace / (double)kvalid;
        const double c2 = coef->c2, c1 = coef->c1, c0 = coef->c0;
        double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
        const double* erow = E + (size_t)row * ld + (size_t)I * TQ_BM + c_lo;
        double* orow = Out + (size_t)row * ld + (size_t)I * TQ_BM + c_lo;
        // Global accesses of the 32 x 16 block a warp handles per step go through a staging patch in the operand ring (free
        // by now: the last commit covers every MMA of this CTA, and the peer's multicasts into this CTA were needed by them):
        // with lane = row (the TMEM layout) a 16-byte load or store touches 32 rows -- 32 sectors for 512 bytes; staged, 8
        // lanes cover one row's 128 bytes and an instruction covers 4 whole rows.  Patch layout: element (r, c) at
        // r * 16 + 2 * ((c / 2) ^ (r & 7)) + (c & 1): conflict-free 16-byte accesses both by row (lane = r) and by quarter
        // warp (8 lanes = one row).
        double* const stg_e = reinterpret_cast<double*>(smem_raw + (smem_base - smem_u32(smem_raw))) + ew * 1024;
        double* const stg_o = stg_e + 512;
        const int srow = lane >> 3, sch = lane & 7;            // coalesced side: row inside a group of 4, 16-byte chunk of the row
        const double* eblk = E + (size_t)(J * TQ_BM + q * 32) * ld + (size_t)I * TQ_BM + c_lo;
        double* oblk = Out + (size_t)(J * TQ_BM + q * 32) * ld + (size_t)I * TQ_BM + c_lo;
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
            const int col = I * TQ_BM + c_lo + cb;
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
    cluster_sync_all();                         // the pair's MMAs (which read both CTAs' shared memory) and remote arrivals are over
    if (warp == 1) tmem_dealloc_pair<TQ_TMEM_COLS>(tmem);
    if (threadIdx.x < 5)
    {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < TQ_EPI_WARPS; ++w) v += red[w][threadIdx.x];      // fixed order
        partials[(size_t)blockIdx.x * SQ_NPART + threadIdx.x] = v;
    }
}

#endif  // RFOE_REDUCED_F16

}  // namespace rfoe
