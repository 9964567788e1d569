// The whole recursion in ONE persistent launch (rows A3-A6 of DESIGN.md for H^p small enough to stay on chip).
//
// A recursion step of a small problem is short -- k=256: 2.5e7 flops, a microsecond of tensor work; k=2048: 250 us --
// so the launch-per-step path spends its time elsewhere: a host round trip per step (the one scalar of A3), two kernel
// boundaries, and, for k=2048, 136 tiles on 148 SMs.  Here a cooperative grid of G <= 148 CTAs (one per SM) stays
// resident for the whole expansion and runs, per step:
//   MM   the step's work is the stream of U = n_tiles x KT "chunk units" (tile, 16-wide slice of the contraction) in
//        tile order; CTA b takes the contiguous range [b U / G, (b+1) U / G) -- every SM gets the same number of DMMAs
//        (stream-K).  Units arrive by TMA through the same 6-stage mbarrier ring as sym_square_kernel, which keeps
//        running across tile boundaries, so there is no pipeline refill between segments.  A tile that lies wholly in
//        one range gets the fused epilogue of sym_square.cuh straight from registers; the two (at most) partial
//        segments at the ends of a range go to a workspace as raw accumulators.
//   --   grid barrier (one flag per CTA, release / acquire, no atomics)
//   FIX  every split tile is finished in 8 bands of 16 rows spread over all CTAs: its segments are added in ascending
//        order of the contraction index (fixed order: reproducible bits), then exactly the fused epilogue -- update
//        c2 C + c1 X + c0 I, mirror (through shared memory, 128-byte runs), the five partial sums.
//   --   grid barrier
//   CTL  EVERY CTA sums all records in the same fixed order and takes the step's decision (control_update) on its own
//        shared-memory copy of the control block: identical inputs, identical code, identical decisions, so there is
//        no broadcast and no third barrier.  CTA 0 writes the history back at the end.
// The host is not in the loop at all: it enqueues bounds, affine map, first decision, this kernel and the output pass
// and synchronises once.  Cross-CTA data (X_n written by other SMs, raw segments, records) is read through L2
// (ld.global.cg / TMA), never through L1, and both sides of every barrier carry a fence.proxy.async because TMA reads
// what ordinary stores wrote.
#pragma once
#include "control.cuh"
#include "sym_square.cuh"

namespace rfoe {

constexpr int RS_MAX_N = 4096;                       // padded size up to which rfoe_expand takes this path
constexpr int RS_BANDS = 8;                          // fix-up bands per split tile
constexpr int RS_BAND_ROWS = SQ_BM / RS_BANDS;       // 16
constexpr int RS_TILE_ELEMS = SQ_BM * SQ_BM;
constexpr int RS_MAX_SPLIT = 1024;
constexpr int RS_SMEM_BYTES = SQ_SMEM_BYTES;

struct ResidentPlan {
    int n, ld, kvalid, KT;        // padded size, row pitch, true size, chunks per tile (n / 16)
    int n_tiles, n_split, G, pad_;
    long long U;                  // n_tiles * KT chunk units per step
    const int2* tile_map;         // (I, J) of every upper-triangle tile, the usual order
    const int2* split;            // per split tile: (tile, first CTA that holds a segment of it)
    double* W0;                   // the two work matrices (ping-pong by step parity)
    double* W1;
    double* ws;                   // 2 G slots of 128 x 128 raw accumulators (slot 2b: segment that continues a tile, 2b+1: that starts one)
    double* rec0;                 // records of even / odd steps: n_tiles tile records (split tiles' stay zero) + 8 per split tile
    double* rec1;
    unsigned* flags;              // G grid-barrier flags, zero at launch
    Ctrl* ctrl;
    unsigned long long* timing;   // [0]: ns CTA 0 spent in the steps (MM + FIX + CTL), for rfoe_stats_t.square_ms
};

__device__ __forceinline__ unsigned ld_acquire_gpu_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu_u32(unsigned* p, unsigned v)
{
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// All CTAs of the (cooperative, co-resident) grid: everything written before is visible to everybody after.
__device__ __forceinline__ void grid_barrier(unsigned* flags, int G, unsigned& epoch)
{
    ++epoch;
    fence_proxy_async_all();      // ordinary stores before later TMA (async proxy) reads of the same data
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) st_release_gpu_u32(flags + blockIdx.x, epoch);
    if ((int)threadIdx.x < G) {
        const long long t0 = clock64();
        while ((int)(ld_acquire_gpu_u32(flags + threadIdx.x) - epoch) < 0)
            if (clock64() - t0 > 4000000000LL) __trap();      // a lost CTA must not hang the GPU
    }
    __syncthreads();
    fence_proxy_async_all();
}

// block_sum_strided (control.cuh) reading through L2: the records were written by other SMs during this launch
__device__ inline double block_sum_strided_cg(const double* __restrict__ p, int n, int stride, double* sh)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v += __ldcg(p + (size_t)i * stride);
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int m = blockDim.x >> 1; m >= 1; m >>= 1) {
        if ((int)threadIdx.x < m) sh[threadIdx.x] += sh[threadIdx.x + m];
        __syncthreads();
    }
    const double r = sh[0];
    __syncthreads();
    return r;
}

// FIX phase, one band (16 rows) of one split tile: segments added in ascending order, then the fused epilogue.
// tsm: 16 x 129 doubles of shared memory (the idle operand ring); red: 8 x 5 doubles.
__device__ __forceinline__ void resident_fixup_band(const ResidentPlan& p, int q, int G, const double* __restrict__ E,
                                                    double* __restrict__ Out, double* __restrict__ rec, double c2, double c1,
                                                    double c0, double* tsm, double (*red)[5])
{
    const int j = q / RS_BANDS, band = q % RS_BANDS;
    const int2 sp = p.split[j];
    const int tile = sp.x;
    const int2 ij = p.tile_map[tile];
    const int I = ij.x, J = ij.y;
    const bool diag = (I == J);
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31;
    const int rl = t >> 4;                     // row inside the band
    const int r = band * RS_BAND_ROWS + rl;    // row inside the tile
    const int cl = (t & 15) * 8;               // first of this thread's 8 columns
    const int row = I * SQ_BM + r, col = J * SQ_BM + cl;
    const int ld = p.ld;

    double cv[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) cv[u] = 0.0;
    const long long t0u = (long long)tile * p.KT, t1u = t0u + p.KT;
    for (int bb = sp.y;; ++bb) {
        const long long rb = (long long)bb * p.U / G, rb1 = (long long)(bb + 1) * p.U / G;
        const int slot = (rb > t0u) ? 2 * bb : 2 * bb + 1;
        const double2* src = reinterpret_cast<const double2*>(p.ws + (size_t)slot * RS_TILE_ELEMS + r * SQ_BM + cl);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double2 x = __ldcg(src + i);
            cv[2 * i] += x.x;
            cv[2 * i + 1] += x.y;
        }
        if (rb1 >= t1u) break;
    }
    double ev[8];
    {
        const double2* e2p = reinterpret_cast<const double2*>(E + (size_t)row * ld + col);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const double2 x = __ldcg(e2p + i);
            ev[2 * i] = x.x;
            ev[2 * i + 1] = x.y;
        }
    }
    double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
    double o[8];
#pragma unroll
    for (int u = 0; u < 8; ++u) {
        double v = fma(c2, cv[u], c1 * ev[u]);
        const double d = cv[u] - ev[u];
        double w = 1.0;
        if (diag) {
            const int cc = col + u;
            w = (cc > row) ? 2.0 : ((cc == row) ? 1.0 : 0.0);
            if (cc == row) {
                if (row < p.kvalid) v += c0;
                p_tr += v;
                p_trc += cv[u];
            }
        }
        o[u] = v;
        p_ss = fma(w * v, v, p_ss);
        p_err = fma(w * d, d, p_err);
        p_ce = fma(w * cv[u], ev[u], p_ce);
    }
    if (!diag) {
        double2* dst = reinterpret_cast<double2*>(Out + (size_t)row * ld + col);
#pragma unroll
        for (int i = 0; i < 4; ++i) dst[i] = make_double2(o[2 * i], o[2 * i + 1]);
    } else {
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (col + u >= row) Out[(size_t)row * ld + col + u] = o[u];
    }
#pragma unroll
    for (int u = 0; u < 8; ++u) tsm[rl * 129 + cl + u] = o[u];
    __syncthreads();
    {
        // mirror: element (row, col) -> (col, row); thread = (column cc of the tile, 8 of the band's 16 rows): 64-byte runs
        const int cc = t >> 1, half = t & 1;
        const int mrow = J * SQ_BM + cc;                                   // row of the mirrored element
        const int mcol = I * SQ_BM + band * RS_BAND_ROWS + half * 8;       // its first column
        double m[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) m[i] = tsm[(half * 8 + i) * 129 + cc];
        if (!diag) {
            double2* dst = reinterpret_cast<double2*>(Out + (size_t)mrow * ld + mcol);
#pragma unroll
            for (int i = 0; i < 4; ++i) dst[i] = make_double2(m[2 * i], m[2 * i + 1]);
        } else {
#pragma unroll
            for (int i = 0; i < 8; ++i)
                if (mrow > mcol + i) Out[(size_t)mrow * ld + mcol + i] = m[i];
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
    __syncthreads();
    if (t < 5) {
        double v = 0.0;
#pragma unroll
        for (int w = 0; w < SQ_CONSUMER_WARPS; ++w) v += red[w][t];
        rec[(size_t)(p.n_tiles + j * RS_BANDS + band) * SQ_NPART + t] = v;
    }
    __syncthreads();      // tsm and red are reused by the next band
}

__global__ void __launch_bounds__(SQ_THREADS, 1)
resident_recursion_kernel(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1,
                          const __grid_constant__ ResidentPlan p)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[SQ_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[SQ_STAGES];
    __shared__ double red[SQ_CONSUMER_WARPS][5];
    __shared__ double sh_sum[SQ_THREADS];
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
    }
    {
        const int* src = reinterpret_cast<const int*>(p.ctrl);
        int* dst = reinterpret_cast<int*>(&cs);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctrl) / sizeof(int)); i += SQ_THREADS) dst[i] = __ldcg(src + i);
    }
    __syncthreads();

    const long long u_begin = (long long)b * p.U / G, u_end = (long long)(b + 1) * p.U / G;
    const int n_units = (int)(u_end - u_begin);

    // ring state: lives across segments AND steps (the mbarrier phases simply keep alternating)
    int ld_s = 0;
    uint32_t ld_ph = 0;
    long long ld_total = 0;          // producer (warp 0): loads issued since the kernel began
    int s = 0;
    uint32_t ph = 0;                 // consumers
    unsigned epoch = 0;
    unsigned long long step_ns = 0;

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
        unsigned long long t_start = 0;
        if (b == 0 && threadIdx.x == 0) t_start = globaltimer_ns();

        // ================= MM: this CTA's range of chunk units =================
        int ld_r = 0;                                   // units of this step already requested
        int p_tile = (int)(u_begin / KT), p_kt = (int)(u_begin - (long long)p_tile * KT);
        int2 p_ij = p.tile_map[p_tile];
        auto issue_loads = [&](int upto) {
            while (ld_r < upto) {
                if (ld_total >= SQ_STAGES && !mbar_test(empty0 + 8 * ld_s, ld_ph ^ 1u)) break;
                const uint32_t fb = full0 + 8 * ld_s;
                const uint32_t dstA = smem_base + ld_s * STAGE_BYTES;
                if (elect_one()) {
                    mbar_expect_tx(fb, STAGE_BYTES);
                    tma_load_2d(dstA, tm, p_kt * SQ_BK, p_ij.x * SQ_BM, fb);
                    tma_load_2d(dstA + SQ_PANEL_BYTES, tm, p_kt * SQ_BK, p_ij.y * SQ_BM, fb);
                }
                __syncwarp();
                ++ld_r;
                ++ld_total;
                if (++ld_s == SQ_STAGES) { ld_s = 0; ld_ph ^= 1u; }
                if (++p_kt == KT) {
                    p_kt = 0;
                    ++p_tile;
                    if (ld_r < n_units) p_ij = p.tile_map[p_tile];
                }
            }
        };
        int done = 0;                                   // units of this step already consumed
        auto wait_full = [&](uint32_t bar, uint32_t parity) {
            if (mbar_try(bar, parity)) return;
            if (warp == 0) {
                do { issue_loads(min(n_units, done + SQ_STAGES)); } while (!mbar_test(bar, parity));
            } else {
                mbar_wait_bounded(bar, parity);
            }
        };

        long long u = u_begin;
        while (u < u_end) {
            const int tile = (int)(u / KT);
            const int kt0 = (int)(u - (long long)tile * KT);
            const int len = min(KT - kt0, (int)(u_end - u));
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
            if (warp == 0) issue_loads(min(n_units, done + SQ_STAGES));
            wait_full(full0 + 8 * s, ph);
            uint32_t st = smem_base + s * STAGE_BYTES;
            load_frag(a0, b0, st + rowA, st + rowB, off[0]);
            for (int i = 0; i < len; ++i) {
                if (warp == 0) issue_loads(min(n_units, done + SQ_STAGES));
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
                if (i + 1 < len) wait_full(full0 + 8 * s1, ph1);
                mma_step(a0, b0);
                load_frag(a0, b0, stn + rowA, stn + rowB, off[0]);      // last chunk of a segment: stale, reloaded below
                mma_step(a1, b1);
                __syncwarp();
                if (lane == 0) mbar_arrive(empty0 + 8 * s);
                s = s1; ph = ph1; st = stn;
                ++done;
            }

            if (kt0 != 0 || len != KT) {
                // partial segment: raw accumulators -> workspace slot (2b: continues a tile, 2b+1: starts one)
                double* T = p.ws + (size_t)(kt0 > 0 ? 2 * b : 2 * b + 1) * RS_TILE_ELEMS;
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
            } else {
                // whole tile: the fused epilogue of sym_square_kernel (update, mirror, five partial sums)
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
                            const double2 e01 = __ldcg(reinterpret_cast<const double2*>(E + (size_t)row * ld + col));
                            const double2 e23 = __ldcg(reinterpret_cast<const double2*>(E + (size_t)row * ld + col + 2));
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
        grid_barrier(p.flags, G, epoch);

        // ================= FIX: split tiles, in bands over all CTAs =================
        {
            const double c2 = cs.coef.c2, c1 = cs.coef.c1, c0 = cs.coef.c0;
            for (int q = b; q < p.n_split * RS_BANDS; q += G) resident_fixup_band(p, q, G, E, Out, rec, c2, c1, c0, tsm, red);
        }
        grid_barrier(p.flags, G, epoch);

        // ================= CTL: the same sums, the same decision, in every CTA =================
        {
            const int n_rec = p.n_tiles + RS_BANDS * p.n_split;
            const double t1 = block_sum_strided_cg(rec + 0, n_rec, SQ_NPART, sh_sum);
            const double s1 = block_sum_strided_cg(rec + 1, n_rec, SQ_NPART, sh_sum);
            const double e2 = block_sum_strided_cg(rec + 2, n_rec, SQ_NPART, sh_sum);
            if (threadIdx.x == 0) control_update(&cs, t1, s1, e2);
            __syncthreads();
        }
        if (b == 0 && threadIdx.x == 0) step_ns += globaltimer_ns() - t_start;
    }

    if (b == 0) {
        const int* src = reinterpret_cast<const int*>(&cs);
        int* dst = reinterpret_cast<int*>(p.ctrl);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctrl) / sizeof(int)); i += SQ_THREADS) dst[i] = src[i];
        if (threadIdx.x == 0) p.timing[0] = step_ns;
    }
}

}  // namespace rfoe
