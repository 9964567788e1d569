// The whole recursion in ONE persistent launch (rows A3-A6 of DESIGN.md for H^p small enough to stay on chip).
//
// A recursion step of a small problem is short -- k=2048: 250 us of tensor work, k=1024: 30 us -- so the launch-per-step
// path spends its time elsewhere: a host round trip per step (the one scalar of A3), two kernel boundaries, and, at
// k=2048, 136 equal tiles on 148 SMs (one wave, 12 SMs idle).  Here a cooperative grid of G <= 148 CTAs (one per SM)
// stays resident for the whole expansion and runs, per step:
//   MM   the step's work is the stream of U = n_tiles x KT "chunk units" (tile, 16-wide slice of the contraction) in
//        tile order; CTA b takes a contiguous range of it, all ranges costing the same (stream-K; where a CTA holds
//        several whole tiles their register epilogues are counted in, as epi_cost units each).  Units arrive by TMA
//        through the same 6-stage mbarrier ring as sym_square_kernel, which keeps running across tile boundaries: no
//        pipeline refill between segments.  A tile that lies wholly in one range gets the fused epilogue of
//        sym_square.cuh straight from registers; the (at most two) partial segments at the ends of a range go to a
//        workspace as raw accumulators.
//   --   grid barrier (a flag per CTA, release / acquire, no atomics)
//   FIX  every split tile is finished in 8 bands of 16 rows, ONE WARP per band, spread over all warps of all CTAs (no
//        block-level synchronisation, so the L2 round trips of the 8 warps of an SM overlap): its segments are added in
//        ascending order of the contraction index (fixed order: reproducible bits), then exactly the fused epilogue --
//        update c2 C + c1 X + c0 I, mirror (through the warp's patch of shared memory: 128-byte runs both ways), the five
//        partial sums, gathered into one record per CTA.
//   --   grid barrier
//   CTL  EVERY CTA sums all records in the same fixed order and takes the step's decision (control_update) on its own
//        shared-memory copy of the control block: identical inputs, identical code, identical decisions -- no broadcast,
//        no third barrier.  CTA 0 writes the history back at the end.
// The host is not in the loop: it enqueues bounds, affine map, first decision, this kernel and the output pass, and
// synchronises once.  Cross-CTA data (X_n written by other SMs, raw segments, records) is read through L2
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
constexpr int RS_EPI_COST = 10;                      // a register epilogue in chunk units (~39k cycles / 4096 per chunk)
constexpr int RS_FLAG_WORDS = 256 + 256 * SQ_CONSUMER_WARPS;   // grid-barrier flags + donation flags (resident_fin.cuh)
constexpr int RS_FIN_MIN_RANGE_TENTHS = 7;           // finisher form (resident_fin.cuh) when a CTA's range of the unit stream is between
constexpr int RS_FIN_MAX_RANGE_TENTHS = 20;          //   0.7 and 2.0 tiles long (k = 1792 ... 2816 on 148 SMs): measured window, DESIGN.md section 13
constexpr int RS_TW_PITCH = 129;                     // row pitch (doubles) of a warp's 16 x 128 transposition patch

struct ResidentPlan {
    int n, ld, kvalid, KT;        // padded size, row pitch, true size, chunks per tile (n / 16)
    int n_tiles, n_split, G, tile_cost;   // tile_cost = KT + epi_cost (epi_cost = 0 when nearly every tile is split)
    long long cost_total;         // n_tiles * tile_cost
    const int2* tile_map;         // (I, J) of every upper-triangle tile, the usual order
    const int4* split;            // per split tile: (tile, first CTA holding a segment of it, number of segments, 0)
    double* W0;                   // the two work matrices (ping-pong by step parity)
    double* W1;
    double* ws;                   // 2 G slots of 128 x 128 raw accumulators (slot 2b: segment that continues a tile, 2b+1: that starts one)
    double* rec0;                 // records of even / odd steps: n_tiles tile records (split tiles' stay zero) + one per CTA (its FIX bands)
    double* rec1;
    unsigned* flags;              // G grid-barrier flags, zero at launch
    unsigned* dflags;             // resident_fin.cuh: G x 8 donation flags (one per CTA and warp), zero at launch
    Ctrl* ctrl;
    unsigned long long* timing;   // CTA 0's %globaltimer, ns: [0] all steps (rfoe_stats_t.square_ms), [1] MM, [2] first barrier, [3] FIX,
                                  // [4] second barrier, [5] CTL
};

__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

__device__ __forceinline__ unsigned ld_volatile_u32(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u32(unsigned* p, unsigned v)
{
    asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// All CTAs of the (cooperative, co-resident) grid: everything written before is visible to everybody after.
// The pattern of cooperative-groups' grid sync with flags instead of an atomic counter: the block barrier orders every
// thread's writes before thread 0's fence + flag store (release); pollers spin on plain volatile loads (an acquire load
// would invalidate the whole L1 on every poll) and fence once when their flag has arrived (acquire); the second block
// barrier hands that to all threads.  Cross-CTA data is then read through L2 only (ld.global.cg / TMA).
__device__ __forceinline__ void grid_barrier(unsigned* flags, int G, unsigned& epoch)
{
    ++epoch;
    __syncthreads();
    if ((int)threadIdx.x < G) {
        if (threadIdx.x == 0) {
            fence_proxy_async_all();      // ordinary stores before later TMA (async proxy) reads of the same data
            __threadfence();
            st_volatile_u32(flags + blockIdx.x, epoch);
        }
        const long long t0 = clock64();
        while ((int)(ld_volatile_u32(flags + threadIdx.x) - epoch) < 0)
            if (clock64() - t0 > 4000000000LL) __trap();      // a lost CTA must not hang the GPU
        __threadfence();
    }
    __syncthreads();
    fence_proxy_async_all();
}

// first chunk unit of CTA b's range (b = G: the end of the stream).  Ranges are equal in COST: chunk units plus
// epi_cost units per tile epilogue, which sits at the tile's end and is never cut.  (rfoe.cu has the host twin.)
__device__ __forceinline__ int rs_boundary(const ResidentPlan& p, int b)
{
    const long long c = (long long)b * p.cost_total / p.G;
    const int tile = (int)(c / p.tile_cost);
    const int off = (int)(c - (long long)tile * p.tile_cost);
    return tile * p.KT + min(off, p.KT);
}

// three fixed-order sums over the tile records in one pass (Tr X_{n+1}, ||X_{n+1}||_F^2, ||X_n^2 - X_n||_F^2): per thread
// strided, then a shuffle tree per warp, then the warps in order.  Reads through L2 (written by other SMs this launch).
__device__ inline void record_sums_cg(const double* __restrict__ rec, int n_rec, double (*sh)[3], double& t1, double& s1, double& e2)
{
    double a = 0.0, c = 0.0, e = 0.0;
    for (int i = threadIdx.x; i < n_rec; i += SQ_THREADS) {
        const double2 x = __ldcg(reinterpret_cast<const double2*>(rec + (size_t)i * SQ_NPART));
        const double y = __ldcg(rec + (size_t)i * SQ_NPART + 2);
        a += x.x; c += x.y; e += y;
    }
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, m);
        c += __shfl_xor_sync(0xffffffffu, c, m);
        e += __shfl_xor_sync(0xffffffffu, e, m);
    }
    if ((threadIdx.x & 31) == 0) { sh[threadIdx.x >> 5][0] = a; sh[threadIdx.x >> 5][1] = c; sh[threadIdx.x >> 5][2] = e; }
    __syncthreads();
    t1 = s1 = e2 = 0.0;
#pragma unroll
    for (int w = 0; w < SQ_CONSUMER_WARPS; ++w) { t1 += sh[w][0]; s1 += sh[w][1]; e2 += sh[w][2]; }
    __syncthreads();
}

// FIX phase, one band (16 rows) of one split tile, by ONE WARP: segments added in ascending order, then the fused
// epilogue.  tw: the warp's 16 x RS_TW_PITCH doubles of shared memory (the operand ring is idle in this phase).
// wsum[5]: the warp's running partial sums of this step in shared memory (Tr Out, ||Out||^2, ||C - X||^2, Tr C, <C, X>).
// Everything arrives BY VALUE (registers): a reference to the kernel's __grid_constant__ plan would turn every field into
// a dependent generic load in this out-of-line function (measured: ~12 us of a 23 us phase).
// meta = (b0 = first CTA holding a segment, nseg, I, J) of the band's tile.
__device__ __noinline__ void resident_fixup_band(int4 meta, int band, const double* __restrict__ ws, int ld, int kvalid,
                                                 const double* __restrict__ E, double* __restrict__ Out, double c2, double c1,
                                                 double c0, double* tw, double* wsum)
{
    const int b0 = meta.x, nseg = meta.y;
    const int I = meta.z, J = meta.w;
    const bool diag = (I == J);
    const int lane = threadIdx.x & 31;
    const int cl = 4 * lane;                                   // this lane's 4 columns of the tile
    const int col = J * SQ_BM + cl;
    constexpr int RB = 4;                                      // rows per batch: 8 (nseg + 1) 16-byte loads in flight per lane
    double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
#pragma unroll 1
    for (int rb = 0; rb < RS_BAND_ROWS; rb += RB) {
        double cv[RB][4], ev[RB][4];
        const int r0 = band * RS_BAND_ROWS + rb;               // first tile row of the batch
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            const double2* e2p = reinterpret_cast<const double2*>(E + (size_t)(I * SQ_BM + r0 + i) * ld + col);
            const double2 x = __ldcg(e2p), y = __ldcg(e2p + 1);
            ev[i][0] = x.x; ev[i][1] = x.y; ev[i][2] = y.x; ev[i][3] = y.y;
        }
        {
            // the first holder's segment starts the tile (slot 2b+1); every later one continues it (slot 2b).  The first two
            // (a split tile has at least two) are fetched together with X_n: one L2 round trip per batch in the common case.
            const double* src0 = ws + (size_t)(2 * b0 + 1) * RS_TILE_ELEMS + r0 * SQ_BM + cl;
            const double* src1 = ws + (size_t)(2 * (b0 + 1)) * RS_TILE_ELEMS + r0 * SQ_BM + cl;
            double cw[RB][4];
#pragma unroll
            for (int i = 0; i < RB; ++i) {
                const double2 x = __ldcg(reinterpret_cast<const double2*>(src0 + i * SQ_BM));
                const double2 y = __ldcg(reinterpret_cast<const double2*>(src0 + i * SQ_BM + 2));
                cv[i][0] = x.x; cv[i][1] = x.y; cv[i][2] = y.x; cv[i][3] = y.y;
            }
#pragma unroll
            for (int i = 0; i < RB; ++i) {
                const double2 x = __ldcg(reinterpret_cast<const double2*>(src1 + i * SQ_BM));
                const double2 y = __ldcg(reinterpret_cast<const double2*>(src1 + i * SQ_BM + 2));
                cw[i][0] = x.x; cw[i][1] = x.y; cw[i][2] = y.x; cw[i][3] = y.y;
            }
#pragma unroll
            for (int i = 0; i < RB; ++i)
#pragma unroll
                for (int u = 0; u < 4; ++u) cv[i][u] += cw[i][u];
        }
        for (int sg = 2; sg < nseg; ++sg) {
            const double* src = ws + (size_t)(2 * (b0 + sg)) * RS_TILE_ELEMS + r0 * SQ_BM + cl;
#pragma unroll
            for (int i = 0; i < RB; ++i) {
                const double2 x = __ldcg(reinterpret_cast<const double2*>(src + i * SQ_BM));
                const double2 y = __ldcg(reinterpret_cast<const double2*>(src + i * SQ_BM + 2));
                cv[i][0] += x.x; cv[i][1] += x.y; cv[i][2] += y.x; cv[i][3] += y.y;
            }
        }
#pragma unroll
        for (int i = 0; i < RB; ++i) {
            const int row = I * SQ_BM + r0 + i;
            double o[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                double v = fma(c2, cv[i][u], c1 * ev[i][u]);
                const double d = cv[i][u] - ev[i][u];
                double w = 1.0;
                if (diag) {
                    const int cc = col + u;
                    w = (cc > row) ? 2.0 : ((cc == row) ? 1.0 : 0.0);
                    if (cc == row) {
                        if (row < kvalid) v += c0;
                        p_tr += v;
                        p_trc += cv[i][u];
                    }
                }
                o[u] = v;
                p_ss = fma(w * v, v, p_ss);
                p_err = fma(w * d, d, p_err);
                p_ce = fma(w * cv[i][u], ev[i][u], p_ce);
            }
            if (!diag) {
                double2* dst = reinterpret_cast<double2*>(Out + (size_t)row * ld + col);
                dst[0] = make_double2(o[0], o[1]);
                dst[1] = make_double2(o[2], o[3]);
            } else {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (col + u >= row) Out[(size_t)row * ld + col + u] = o[u];
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) tw[(rb + i) * RS_TW_PITCH + cl + u] = o[u];
        }
    }
    __syncwarp();
    // mirror: element (row, col) -> (col, row).  Lane = a column cc of the tile: its 16 band rows are 128 contiguous bytes
    // of row J*128 + cc of the output.
#pragma unroll 1
    for (int cc = lane; cc < SQ_BM; cc += 32) {
        const int mrow = J * SQ_BM + cc;
        const int mcol = I * SQ_BM + band * RS_BAND_ROWS;
        double m[RS_BAND_ROWS];
#pragma unroll
        for (int i = 0; i < RS_BAND_ROWS; ++i) m[i] = tw[i * RS_TW_PITCH + cc];
        if (!diag) {
            double2* dst = reinterpret_cast<double2*>(Out + (size_t)mrow * ld + mcol);
#pragma unroll
            for (int i = 0; i < RS_BAND_ROWS / 2; ++i) dst[i] = make_double2(m[2 * i], m[2 * i + 1]);
        } else {
#pragma unroll
            for (int i = 0; i < RS_BAND_ROWS; ++i)
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
    if (lane == 0) { wsum[0] += p_tr; wsum[1] += p_ss; wsum[2] += p_err; wsum[3] += p_trc; wsum[4] += p_ce; }
    __syncwarp();      // tw is reused by this warp's next band
}

__global__ void __launch_bounds__(SQ_THREADS, 1)
resident_recursion_kernel(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1,
                          const __grid_constant__ ResidentPlan p)
{
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[SQ_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[SQ_STAGES];
    __shared__ double red[SQ_CONSUMER_WARPS][5];
    __shared__ double sh3[SQ_CONSUMER_WARPS][3];
    __shared__ __align__(16) Ctrl cs;      // this CTA's copy of the control block
    __shared__ int4 fx_meta[SQ_CONSUMER_WARPS];   // FIX: (first CTA, segments, I, J) of each warp's first band (static over the steps)

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
    if (lane == 0) {
        const int q0 = b + warp * G;
        int4 m4 = make_int4(0, 0, 0, 0);
        if (q0 < p.n_split * RS_BANDS) {
            const int4 sp = p.split[q0 / RS_BANDS];
            const int2 ij = p.tile_map[sp.x];
            m4 = make_int4(sp.y, sp.z, ij.x, ij.y);
        }
        fx_meta[warp] = m4;
    }
    __syncthreads();

    const int u_begin = rs_boundary(p, b), u_end = rs_boundary(p, b + 1);
    const int n_units = u_end - u_begin;

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
        int ld_r = 0;                                   // units of this step already requested
        int p_tile = u_begin / KT, p_kt = u_begin - p_tile * KT;
        int2 p_ij = p.tile_map[n_units > 0 ? p_tile : 0];
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
        // warp 0 is producer and consumer: before it blocks on a stage, the load into that stage must have been issued
        auto ensure_issued = [&](int upto) {
            issue_loads(min(n_units, done + SQ_STAGES));
            while (ld_r < min(n_units, upto)) issue_loads(min(n_units, done + SQ_STAGES));
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
        if (timer) { t_b = globaltimer_ns(); ph_ns[0] += t_b - t_a; t_a = t_b; }
        grid_barrier(p.flags, G, epoch);
        if (timer) { t_b = globaltimer_ns(); ph_ns[1] += t_b - t_a; t_a = t_b; }

        // ================= FIX: split tiles, a band per warp, over all warps of the grid =================
        {
            const double c2 = cs.coef.c2, c1 = cs.coef.c1, c0 = cs.coef.c0;
            double* tw = tsm + warp * (RS_BAND_ROWS * RS_TW_PITCH);
            const int n_q = p.n_split * RS_BANDS;
            if (lane < 5) red[warp][lane] = 0.0;
            __syncwarp();
            int4 meta = fx_meta[warp];                          // this warp's first band: looked up once, at kernel start
            for (int q = b + warp * G; q < n_q; q += SQ_CONSUMER_WARPS * G) {
                if (q >= SQ_CONSUMER_WARPS * G) {               // further bands of large problems: look up now
                    const int4 sp = p.split[q / RS_BANDS];
                    const int2 ij = p.tile_map[sp.x];
                    meta = make_int4(sp.y, sp.z, ij.x, ij.y);
                }
                resident_fixup_band(meta, q % RS_BANDS, p.ws, p.ld, p.kvalid, E, Out, c2, c1, c0, tw, &red[warp][0]);
            }
            // this CTA's bands -> ONE record: a warp's bands in order, then the warps in order (fixed by the plan)
            __syncthreads();
            if (threadIdx.x < 5) {
                double v = 0.0;
#pragma unroll
                for (int w = 0; w < SQ_CONSUMER_WARPS; ++w) v += red[w][threadIdx.x];
                rec[(size_t)(p.n_tiles + b) * SQ_NPART + threadIdx.x] = v;
            }
        }
        if (timer) { t_b = globaltimer_ns(); ph_ns[2] += t_b - t_a; t_a = t_b; }
        grid_barrier(p.flags, G, epoch);
        if (timer) { t_b = globaltimer_ns(); ph_ns[3] += t_b - t_a; t_a = t_b; }

        // ================= CTL: the same sums, the same decision, in every CTA =================
        {
            double t1, s1, e2;
            record_sums_cg(rec, p.n_tiles + G, sh3, t1, s1, e2);
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
