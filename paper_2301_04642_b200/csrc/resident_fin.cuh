// The whole recursion in ONE persistent launch, FINISHER form (resident.cuh's kernel with one grid barrier per step instead of
// two; used where a CTA's range of the chunk-unit stream is 0.7 ... 2.0 tiles long: k = 1792 ... 2816 on 148 SMs).
//
// Same stream-K partition (rs_boundary), same ring, same redundant decision.  What differs is who completes a tile that is cut
// between CTAs.  In resident.cuh every holder stores its raw partial tile, everybody meets at a grid barrier, and the split
// tiles are finished in 16-row bands spread over all warps of the grid (then a second barrier).  Here the FIRST holder of a tile
// finishes it: a CTA's range is [tail of tile a | whole tiles | head of tile b], processed in that order, so
//   the tail of tile a (a segment that continues somebody else's tile) is the first thing the CTA computes: it is DONATED
//     at once -- raw accumulators to workspace slot b, one flag per warp -- more than 100 us before anybody needs it;
//   the head of tile b (a segment that starts a tile) is the last thing it computes: its accumulators stay in registers,
//     the parts of the following holders are added in ascending order of the contraction index (the same order, hence the
//     same bits, as resident.cuh's bands), and the ordinary fused epilogue runs from registers.  Both the donated parts and
//     the tile of X_n the epilogue needs arrive THROUGH THE OPERAND RING, behind the last chunks: the workspace is described
//     by a third tensor map (tmW: 128-column tiles one below the other, the operands' box shape), so a part is four more ring
//     entries and is added with the same swizzled shared-memory reads the epilogue uses for X_n -- 128 accumulator registers
//     leave no room for global loads in flight (a version with 32 ld.global per thread took twice as long to finish a tile).
// Only a CTA whose whole range lies inside one tile (k=2048: 12 of 148) donates at the END of its range; its finisher waits
// for that one flag -- a store, a fence and an L2 round trip after everybody has finished multiplying anyway.
// No block-level synchronisation in donating or finishing: finisher warp w needs exactly the 64 x 32 block donor warp w wrote.
#pragma once
#include "resident.cuh"

namespace rfoe {

constexpr int RF_E_ENTRIES = (SQ_BM * SQ_BM * 8) / (2 * SQ_PANEL_BYTES);      // ring entries that hold a 128 x 128 tile of X_n: 4

__global__ void __launch_bounds__(SQ_THREADS, 1)
resident_finisher_kernel(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1,
                         const __grid_constant__ CUtensorMap tmW, const __grid_constant__ ResidentPlan p)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[SQ_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[SQ_STAGES];
    __shared__ double red[SQ_CONSUMER_WARPS][5];
    __shared__ double sh3[SQ_CONSUMER_WARPS][3];
    __shared__ __align__(16) Ctrl cs;      // this CTA's copy of the control block

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int b = blockIdx.x, G = gridDim.x;
    const int KT = p.KT;

    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    double* const tsm = reinterpret_cast<double*>(smem_raw + (smem_base - smem_u32(smem_raw)));
    const uint32_t full0 = smem_u32(&full_bar[0]);
    const uint32_t empty0 = smem_u32(&empty_bar[0]);
    constexpr uint32_t STAGE_BYTES = 2 * SQ_PANEL_BYTES;

    if (threadIdx.x == 0) {
        for (int s = 0; s < SQ_STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, SQ_CONSUMER_WARPS);
        }
        mbar_fence_init();
        tma_prefetch_desc(&tm0);
        tma_prefetch_desc(&tm1);
        tma_prefetch_desc(&tmW);
    }
    {
        const int* src = reinterpret_cast<const int*>(p.ctrl);
        int* dst = reinterpret_cast<int*>(&cs);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctrl) / sizeof(int)); i += SQ_THREADS) dst[i] = __ldcg(src + i);
    }
    __syncthreads();

    const int u_begin = rs_boundary(p, b), u_end = rs_boundary(p, b + 1);
    const int n_units = u_end - u_begin;
    // This CTA's last segment: if it STARTS a tile without completing it, this CTA finishes that tile (it is the tile's first
    // holder; the fin_nseg - 1 CTAs after it hold the rest and donate their parts).  Static over the steps.
    const int t_last = (u_end - 1) / KT;
    const int last_u0 = max(u_begin, t_last * KT);
    const bool has_fin = (last_u0 == t_last * KT) && (u_end < (t_last + 1) * KT);
    int fin_nseg = 1;
    if (has_fin)
        while (b + fin_nseg < G && rs_boundary(p, b + fin_nseg) < (t_last + 1) * KT) ++fin_nseg;
    const int2 fin_ij = p.tile_map[t_last];
    // ring entries per step: the chunk units, then (finisher only) the donated parts of the tile, RF_E_ENTRIES entries each, in
    // ascending order of the contraction index, then the tile of X_n the epilogue needs -- all in the operand ring's box layout
    const int n_entries = n_units + (has_fin ? RF_E_ENTRIES * fin_nseg : 0);

    // ring state: lives across segments AND steps (the mbarrier phases simply keep alternating)
    int ld_s = 0;
    uint32_t ld_ph = 0;
    long long ld_total = 0;          // producer (warp 0): loads issued since the kernel began
    int s = 0;
    uint32_t ph = 0;                 // consumers
    unsigned epoch = 0;
    unsigned long long step_ns = 0, ph_ns[5] = {0, 0, 0, 0, 0};
    const bool timer = (b == 0 && threadIdx.x == 0);

    // consumer geometry, as in sym_square_kernel: 2 x 4 warps of 64 x 32 outputs, fragment row m <-> tile row 2m + p
    const int warp_m = warp >> 2, warp_n = warp & 3;
    const int r = lane >> 2, kk = lane & 3;
    uint32_t off[4][2];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks)
#pragma unroll
        for (int q = 0; q < 2; ++q)
            off[ks][q] = ((uint32_t)(((2 * ks + (kk >> 1)) ^ ((2 * r + q) & 7)) << 4)) + (uint32_t)((kk & 1) * 8);
    const uint32_t rowA = (uint32_t)(warp_m * 64 + 2 * r) * 128u;
    const uint32_t rowB = (uint32_t)(warp_n * 32 + 2 * r) * 128u + (uint32_t)SQ_PANEL_BYTES;   // always two panels here

    while (cs.action == ACT_SP2) {
        const int cur = cs.step & 1;
        const CUtensorMap* tm = cur ? &tm1 : &tm0;
        const double* __restrict__ E = cur ? p.W1 : p.W0;
        double* __restrict__ Out = cur ? p.W0 : p.W1;
        double* __restrict__ rec = cur ? p.rec1 : p.rec0;
        unsigned long long t_start = 0, t_a = 0, t_b = 0;
        if (timer) t_start = t_a = globaltimer_ns();

        // ================= MM: this CTA's range of chunk units =================
        const unsigned step_epoch = (unsigned)cs.step + 1u;
        int ld_r = 0;                                   // ring entries of this step already requested
        int p_tile = u_begin / KT, p_kt = u_begin - p_tile * KT;
        int2 p_ij = p.tile_map[n_units > 0 ? p_tile : 0];
        auto issue_loads = [&](int upto) {
            while (ld_r < upto) {
                if (ld_total >= SQ_STAGES && !mbar_test(empty0 + 8 * ld_s, ld_ph ^ 1u)) break;
                const uint32_t fb = full0 + 8 * ld_s;
                const uint32_t dstA = smem_base + ld_s * STAGE_BYTES;
                const bool chunk = ld_r < n_units;
                if (chunk) {
                    if (elect_one()) {
                        mbar_expect_tx(fb, STAGE_BYTES);
                        tma_load_2d(dstA, tm, p_kt * SQ_BK, p_ij.x * SQ_BM, fb);
                        tma_load_2d(dstA + SQ_PANEL_BYTES, tm, p_kt * SQ_BK, p_ij.y * SQ_BM, fb);
                    }
                } else {
                    // columns 32 v .. 32 v + 31 (two boxes) of a 128 x 128 tile: part `part` of the tile being finished (raw
                    // accumulators in workspace slot b + part + 1, once all eight warps of that CTA have flagged them), or, last, X_n's block (I, J)
                    const int part = (ld_r - n_units) / RF_E_ENTRIES, v = (ld_r - n_units) % RF_E_ENTRIES;
                    if (part < fin_nseg - 1) {
                        const unsigned f = ld_volatile_u32(p.dflags + (b + part + 1) * SQ_CONSUMER_WARPS + (lane & 7));
                        if (!__all_sync(0xffffffffu, (int)(f - step_epoch) >= 0)) break;
                        __threadfence();
                        fence_proxy_async_all();          // the donor's ordinary stores, now read by TMA
                        if (elect_one()) {
                            mbar_expect_tx(fb, STAGE_BYTES);
                            tma_load_2d(dstA, &tmW, v * 2 * SQ_BK, (b + part + 1) * SQ_BM, fb);
                            tma_load_2d(dstA + SQ_PANEL_BYTES, &tmW, v * 2 * SQ_BK + SQ_BK, (b + part + 1) * SQ_BM, fb);
                        }
                    } else if (elect_one()) {
                        mbar_expect_tx(fb, STAGE_BYTES);
                        tma_load_2d(dstA, tm, fin_ij.y * SQ_BM + v * 2 * SQ_BK, fin_ij.x * SQ_BM, fb);
                        tma_load_2d(dstA + SQ_PANEL_BYTES, tm, fin_ij.y * SQ_BM + v * 2 * SQ_BK + SQ_BK, fin_ij.x * SQ_BM, fb);
                    }
                }
                __syncwarp();
                ++ld_r;
                ++ld_total;
                if (++ld_s == SQ_STAGES) { ld_s = 0; ld_ph ^= 1u; }
                if (chunk && ++p_kt == KT) {
                    p_kt = 0;
                    ++p_tile;
                    if (ld_r < n_units) p_ij = p.tile_map[p_tile];
                }
            }
        };
        int done = 0;                                   // ring entries of this step already consumed
        // warp 0 is producer and consumer: before it blocks on a stage, the load into that stage must have been issued
        auto ensure_issued = [&](int upto) {
            issue_loads(min(n_entries, done + SQ_STAGES));
            while (ld_r < min(n_entries, upto)) issue_loads(min(n_entries, done + SQ_STAGES));
        };


        int u = u_begin;
        while (u < u_end) {
            const int tile = u / KT;
            const int kt0 = u - tile * KT;
            const int len = min(KT - kt0, u_end - u);
            const int2 ij = p.tile_map[tile];
            const int I = ij.x, J = ij.y;
            const bool diag = (I == J);

            double acc[8][4][2];
#pragma unroll
            for (int mi = 0; mi < 8; ++mi)
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) acc[mi][ni][0] = acc[mi][ni][1] = 0.0;
            auto load_frag = [&](double (&a)[8], double (&bf)[4], uint32_t aB, uint32_t bB, const uint32_t (&o)[2]) {
#pragma unroll
                for (int mi = 0; mi < 8; ++mi) a[mi] = lds_f64(aB + (uint32_t)((mi >> 1) * 2048 + (mi & 1) * 128) + o[mi & 1]);
#pragma unroll
                for (int ni = 0; ni < 4; ++ni) bf[ni] = lds_f64(bB + (uint32_t)((ni >> 1) * 2048 + (ni & 1) * 128) + o[ni & 1]);
            };
            auto mma_step = [&](const double (&a)[8], const double (&bf)[4]) {
#pragma unroll
                for (int mi = 0; mi < 8; ++mi)
#pragma unroll
                    for (int ni = 0; ni < 4; ++ni) dmma_8x8x4(acc[mi][ni][0], acc[mi][ni][1], a[mi], bf[ni]);
            };

            double a0[8], b0[4], a1[8], b1[4];
            if (warp == 0) ensure_issued(done + 1);
            mbar_wait_safe(full0 + 8 * s, ph);
            uint32_t st = smem_base + s * STAGE_BYTES;
            load_frag(a0, b0, st + rowA, st + rowB, off[0]);
            for (int i = 0; i < len; ++i) {
                if (warp == 0) ensure_issued(done + 2);
                const uint32_t aB = st + rowA, bB = st + rowB;
                int s1 = s + 1;
                uint32_t ph1 = ph;
                if (s1 == SQ_STAGES) { s1 = 0; ph1 ^= 1u; }
                const uint32_t stn = smem_base + s1 * STAGE_BYTES;
                load_frag(a1, b1, aB, bB, off[1]);
                mma_step(a0, b0);
                load_frag(a0, b0, aB, bB, off[2]);
                mma_step(a1, b1);
                load_frag(a1, b1, aB, bB, off[3]);
                if (i + 1 < len) mbar_wait_safe(full0 + 8 * s1, ph1);
                mma_step(a0, b0);
                load_frag(a0, b0, stn + rowA, stn + rowB, off[0]);      // last chunk of a segment: stale, reloaded below
                mma_step(a1, b1);
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * s);
                s = s1; ph = ph1; st = stn;
                ++done;
            }

            if (kt0 != 0) {
                // a segment that CONTINUES a tile another CTA started: donate it.  Raw accumulators -> workspace slot b (each
                // warp its own 64 x 32 block), then this warp's flag: the finisher's warp of the same index needs nothing else.
                // It is the first thing this CTA does in a step (or all it does), so the finisher rarely waits.
                double* T = p.ws + (size_t)b * RS_TILE_ELEMS;
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
                __syncwarp();
                if (lane == 0) {
                    fence_proxy_async_all();              // these ordinary stores will be read by the finisher's TMA
                    __threadfence();
                    st_volatile_u32(p.dflags + b * SQ_CONSUMER_WARPS + warp, step_epoch);
                }
            } else {
                // a tile this CTA started: whole (len == KT), or to be finished here with the parts of the CTAs after it, added in
                // ascending order of the contraction index; then the fused epilogue of sym_square_kernel (update, mirror, sums)
                const bool fin = (len != KT);
                uint32_t e_base = 0;
                if (fin) {
                    // the other holders' parts, in ascending order, from the ring (each warp reads entry warp_n: its 32 columns;
                    // it waits for and releases all RF_E_ENTRIES entries of a part -- a stage may only be released by a warp that
                    // has seen its load complete, or the release would count for the stage's previous occupant)
                    for (int part = 0; part < fin_nseg; ++part) {
                        if (warp == 0) ensure_issued(done + RF_E_ENTRIES);       // spins on the donor's flags / free stages if it must
                        int sv = s;
                        uint32_t phv = ph;
                        uint32_t base = 0;
#pragma unroll
                        for (int v = 0; v < RF_E_ENTRIES; ++v) {
                            mbar_wait_safe(full0 + 8 * sv, phv);
                            if (v == warp_n) base = smem_base + (uint32_t)sv * STAGE_BYTES + (uint32_t)(warp_m * 64 + 2 * r) * 128u;
                            if (++sv == SQ_STAGES) { sv = 0; phv ^= 1u; }
                        }
                        if (part == fin_nseg - 1) { e_base = base; break; }       // X_n's tile: read by the epilogue, released after it
#pragma unroll
                        for (int g = 0; g < 4; ++g)
#pragma unroll
                            for (int h = 0; h < 2; ++h)
#pragma unroll
                                for (int q = 0; q < 2; ++q) {
                                    const int mi = 2 * g + q;
                                    const uint32_t a = base + (uint32_t)(h * SQ_PANEL_BYTES + (16 * g + q) * 128);
                                    const uint32_t sw = (uint32_t)((2 * r + q) & 7);
                                    const double2 x = lds_f64x2(a + ((((uint32_t)(2 * kk)) ^ sw) << 4));
                                    const double2 y = lds_f64x2(a + ((((uint32_t)(2 * kk + 1)) ^ sw) << 4));
                                    acc[mi][2 * h][0] += x.x; acc[mi][2 * h + 1][0] += x.y;
                                    acc[mi][2 * h][1] += y.x; acc[mi][2 * h + 1][1] += y.y;
                                }
                        __syncwarp();
#pragma unroll
                        for (int v = 0; v < RF_E_ENTRIES; ++v) {
                            if (lane == 0) mbar_arrive(empty0 + 8 * s);
                            if (++s == SQ_STAGES) { s = 0; ph ^= 1u; }
                        }
                        done += RF_E_ENTRIES;
                    }
                }
                const double c2 = cs.coef.c2, c1 = cs.coef.c1, c0 = cs.coef.c0;
                const int ld = p.ld;
                double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
                const int row_base = I * SQ_BM + warp_m * 64 + 2 * r;
                const int col_base = J * SQ_BM + warp_n * 32 + 4 * kk;
#pragma unroll
                for (int g = 0; g < 4; ++g) {
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        double o[2][4];
                        const int col = col_base + 16 * h;
#pragma unroll
                        for (int q = 0; q < 2; ++q) {
                            const int row = row_base + 16 * g + q;
                            const int mi = 2 * g + q;
                            const double cv[4] = {acc[mi][2 * h][0], acc[mi][2 * h + 1][0], acc[mi][2 * h][1], acc[mi][2 * h + 1][1]};
                            double2 e01, e23;
                            if (fin) {
                                const uint32_t a = e_base + (uint32_t)(h * SQ_PANEL_BYTES + (16 * g + q) * 128);
                                const uint32_t sw = (uint32_t)((2 * r + q) & 7);
                                e01 = lds_f64x2(a + ((((uint32_t)(2 * kk)) ^ sw) << 4));
                                e23 = lds_f64x2(a + ((((uint32_t)(2 * kk + 1)) ^ sw) << 4));
                            } else {
                                e01 = __ldcg(reinterpret_cast<const double2*>(E + (size_t)row * ld + col));
                                e23 = __ldcg(reinterpret_cast<const double2*>(E + (size_t)row * ld + col + 2));
                            }
                            const double ev[4] = {e01.x, e01.y, e23.x, e23.y};
#pragma unroll
                            for (int u2 = 0; u2 < 4; ++u2) {
                                double v = fma(c2, cv[u2], c1 * ev[u2]);
                                const double d = cv[u2] - ev[u2];
                                double w = 1.0;
                                if (diag) {
                                    const int cc = col + u2;
                                    w = (cc > row) ? 2.0 : ((cc == row) ? 1.0 : 0.0);
                                    if (cc == row) {
                                        if (row < p.kvalid) v += c0;
                                        p_tr += v;
                                        p_trc += cv[u2];
                                    }
                                }
                                o[q][u2] = v;
                                p_ss = fma(w * v, v, p_ss);
                                p_err = fma(w * d, d, p_err);
                                p_ce = fma(w * cv[u2], ev[u2], p_ce);
                            }
                            if (!diag) {
                                *reinterpret_cast<double2*>(Out + (size_t)row * ld + col) = make_double2(o[q][0], o[q][1]);
                                *reinterpret_cast<double2*>(Out + (size_t)row * ld + col + 2) = make_double2(o[q][2], o[q][3]);
                            } else {
#pragma unroll
                                for (int u2 = 0; u2 < 4; ++u2)
                                    if (col + u2 >= row) Out[(size_t)row * ld + col + u2] = o[q][u2];
                            }
                        }
                        const int row0 = row_base + 16 * g;
#pragma unroll
                        for (int u2 = 0; u2 < 4; ++u2) {
                            if (!diag) {
                                *reinterpret_cast<double2*>(Out + (size_t)(col + u2) * ld + row0) = make_double2(o[0][u2], o[1][u2]);
                            } else {
                                if (col + u2 > row0) Out[(size_t)(col + u2) * ld + row0] = o[0][u2];
                                if (col + u2 > row0 + 1) Out[(size_t)(col + u2) * ld + row0 + 1] = o[1][u2];
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
                if (lane == 0) { red[warp][0] = p_tr; red[warp][1] = p_ss; red[warp][2] = p_err; red[warp][3] = p_trc; red[warp][4] = p_ce; }
                if (fin) {
                    // release the four entries of the X_n tile
                    __syncwarp();
#pragma unroll
                    for (int v = 0; v < RF_E_ENTRIES; ++v) {
                        if (lane == 0) mbar_arrive(empty0 + 8 * s);
                        if (++s == SQ_STAGES) { s = 0; ph ^= 1u; }
                    }
                    done += RF_E_ENTRIES;
                }
                __syncthreads();
                if (threadIdx.x < 5) {
                    double v = 0.0;
#pragma unroll
                    for (int w = 0; w < SQ_CONSUMER_WARPS; ++w) v += red[w][threadIdx.x];
                    rec[(size_t)tile * SQ_NPART + threadIdx.x] = v;
                }
                __syncthreads();
            }
            u += len;
        }
        if (timer) { t_b = globaltimer_ns(); ph_ns[0] += t_b - t_a; t_a = t_b; }
        grid_barrier(p.flags, G, epoch);                  // the ONE barrier of a step: X_{n+1} and every tile record are complete
        if (timer) { t_b = globaltimer_ns(); ph_ns[1] += t_b - t_a; t_a = t_b; }

        // ================= CTL: the same sums, the same decision, in every CTA =================
        {
            double t1, s1, e2;
            record_sums_cg(rec, p.n_tiles, sh3, t1, s1, e2);
            if (threadIdx.x == 0) control_update(&cs, t1, s1, e2);
            __syncthreads();
        }
        if (timer) { t_b = globaltimer_ns(); ph_ns[4] += t_b - t_a; step_ns += t_b - t_start; }
    }

    if (b == 0) {
        const int* src = reinterpret_cast<const int*>(&cs);
        int* dst = reinterpret_cast<int*>(p.ctrl);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctrl) / sizeof(int)); i += SQ_THREADS) dst[i] = src[i];
        if (threadIdx.x == 0) {
            p.timing[0] = step_ns;
            for (int i = 0; i < 5; ++i) p.timing[1 + i] = ph_ns[i];
        }
    }
}

}  // namespace rfoe
