// The whole recursion of a SMALL H^p (k <= 1024) in one persistent launch -- the latency-bound end of resident.cuh.
//
// At k=256 a squaring is 2.5e7 flops: a microsecond of the chip's FP64 tensor pipe, but 33 us on the one SM that owns a
// 128 x 128 tile of sym_square_kernel.  What matters here is the length of the dependent chain of one step, so the
// decomposition is the opposite of the big kernel's: small output tiles with the WHOLE contraction each (no split of the
// contraction index, so no second pass and ONE grid barrier per step), one tile per CTA, all upper-triangle tiles
// resident at once: BM = 32 for k <= 512 (k=256: 36 CTAs, k=512: 136), BM = 64 for k <= 1024 (136 CTAs).  Per step a CTA
//   loads the two BM-row panels of X_n it needs (TMA boxes of BM rows x 128 bytes, 128-byte swizzle) in 64 KiB chunks
//     (BM=32: 128 columns, BM=64: 64) through a 3-stage mbarrier ring (k=256: 2 chunks, all in flight at once),
//   multiplies: 8 warps x (BM/2 x BM/4 outputs), mma.m8n8k4.f64 (SASS DMMA.8x8x4); with BM=32 a warp has only two output
//     blocks, so it keeps two accumulator sets over the even / odd k4-steps (four independent DMMA chains; added at the
//     end: a fixed order),
//   applies the fused epilogue of sym_square.cuh -- X_{n+1} = c2 C + c1 X_n + c0 I to (I,J) and mirrored to (J,I), the
//     five partial sums into one record per tile,
//   passes ONE grid barrier, and takes the step's decision itself: every CTA sums all records in the same fixed order
//     and runs control_update on its own copy of the control block (as in resident.cuh: no broadcast).
#pragma once
#include "resident.cuh"

namespace rfoe {

constexpr int RT_MAX_N = 1024;            // padded size up to which this kernel is used
constexpr int RT_MAX_N32 = 512;           //   ... with 32 x 32 tiles (136 CTAs at 512); above: 64 x 64 (136 CTAs at 1024)
constexpr int RT_STAGES = 3;
constexpr int RT_STAGE_BYTES = 64 * 1024;                         // two panels' chunk
constexpr int RT_PANEL_BYTES = RT_STAGE_BYTES / 2;
constexpr int RT_SMEM_BYTES = RT_STAGES * RT_STAGE_BYTES + 1024;

struct SmallPlan {
    int n, ld, kvalid, mt;        // padded size, row pitch, true size, tiles per side (n / BM)
    int n_tiles, pad0_, pad1_, pad2_;
    double* W0;                   // the two work matrices (ping-pong by step parity)
    double* W1;
    double* rec0;                 // tile records of even / odd steps
    double* rec1;
    unsigned* flags;              // grid-barrier flags, zero at launch
    Ctrl* ctrl;
    unsigned long long* timing;   // CTA 0's %globaltimer, ns: [0] all steps, [1] load + multiply + epilogue, [2] barrier, [3] unused, [4] unused, [5] decision
};

template <int BM>
__global__ void __launch_bounds__(SQ_THREADS, 1)
resident_small_kernel(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1,
                      const __grid_constant__ SmallPlan p)
{
    constexpr int BOX_BYTES = BM * SQ_BK * 8;               // BM rows x 16 doubles
    constexpr int BOXES = RT_PANEL_BYTES / BOX_BYTES;       // boxes per panel chunk (BM=32: 8, BM=64: 4)
    constexpr int KC = BOXES * SQ_BK;                       // contraction columns per stage (128 / 64)
    constexpr int RBW = BM / 16;                            // 8-row output blocks per warp (2 / 4)
    constexpr int CBW = BM / 32;                            // 8-column output blocks per warp (1 / 2)
    constexpr int PAR = (RBW * CBW >= 8) ? 1 : 2;           // accumulator sets over alternating k4-steps
    extern __shared__ uint8_t smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[RT_STAGES];
    __shared__ __align__(8) uint64_t empty_bar[RT_STAGES];
    __shared__ double red[SQ_CONSUMER_WARPS][5];
    __shared__ double sh3[SQ_CONSUMER_WARPS][3];
    __shared__ __align__(16) Ctrl cs;

    const int warp = threadIdx.x >> 5;
    const int lane = threadIdx.x & 31;
    const int b = blockIdx.x, G = gridDim.x;

    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t full0 = smem_u32(&full_bar[0]);
    const uint32_t empty0 = smem_u32(&empty_bar[0]);

    if (threadIdx.x == 0) {
        for (int s = 0; s < RT_STAGES; ++s) {
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

    // this CTA's tile (I <= J) of the BM x BM tiling, row-major over the upper triangle
    int I = 0, J;
    {
        int t = b;
        while (t >= p.mt - I) { t -= p.mt - I; ++I; }
        J = I + t;
    }
    const bool diag = (I == J);
    const int n_chunks = p.n / KC;

    // warp geometry: 2 x 4 warps of (BM/2) x (BM/4) outputs; lane (r = lane / 4, kk = lane % 4) holds A[r][kk], B[kk][r]
    // and C[r][2 kk .. 2 kk + 1] of every 8 x 8 x 4 block
    const int warp_m = warp >> 2, warp_n = warp & 3;
    const int r = lane >> 2, kk = lane & 3;
    // byte offset of element (row, column c of a 16-column box) inside a box: row * 128 + swizzled 16-byte chunk
    uint32_t offA[RBW][4], offB[CBW][4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
        const int c = 4 * ks + kk;
#pragma unroll
        for (int rb = 0; rb < RBW; ++rb) {
            const int row = warp_m * (BM / 2) + rb * 8 + r;
            offA[rb][ks] = (uint32_t)(row * 128 + ((((c >> 1) ^ (row & 7))) << 4) + (c & 1) * 8);
        }
#pragma unroll
        for (int cb = 0; cb < CBW; ++cb) {
            const int row = warp_n * (BM / 4) + cb * 8 + r;
            offB[cb][ks] = (uint32_t)(row * 128 + ((((c >> 1) ^ (row & 7))) << 4) + (c & 1) * 8) + (uint32_t)RT_PANEL_BYTES;
        }
    }

    int ld_s = 0;
    uint32_t ld_ph = 0;
    long long ld_total = 0;
    int s = 0;
    uint32_t ph = 0;
    unsigned epoch = 0;
    unsigned long long step_ns = 0, ph_ns[3] = {0, 0, 0};
    const bool timer = (b == 0 && threadIdx.x == 0);

    while (cs.action == ACT_SP2) {
        const int cur = cs.step & 1;
        const CUtensorMap* tm = cur ? &tm1 : &tm0;
        const double* __restrict__ E = cur ? p.W1 : p.W0;
        double* __restrict__ Out = cur ? p.W0 : p.W1;
        double* __restrict__ rec = cur ? p.rec1 : p.rec0;
        unsigned long long t_start = 0, t_a = 0, t_b = 0;
        if (timer) t_start = t_a = globaltimer_ns();

        int ld_r = 0;
        auto issue_loads = [&](int upto) {
            while (ld_r < upto) {
                if (ld_total >= RT_STAGES && !mbar_test(empty0 + 8 * ld_s, ld_ph ^ 1u)) break;
                const uint32_t fb = full0 + 8 * ld_s;
                const uint32_t dst = smem_base + ld_s * RT_STAGE_BYTES;
                if (elect_one()) {
                    mbar_expect_tx(fb, RT_STAGE_BYTES);
#pragma unroll
                    for (int bx = 0; bx < BOXES; ++bx) {
                        tma_load_2d(dst + bx * BOX_BYTES, tm, ld_r * KC + bx * SQ_BK, I * BM, fb);
                        tma_load_2d(dst + RT_PANEL_BYTES + bx * BOX_BYTES, tm, ld_r * KC + bx * SQ_BK, J * BM, fb);
                    }
                }
                __syncwarp();
                ++ld_r;
                ++ld_total;
                if (++ld_s == RT_STAGES) { ld_s = 0; ld_ph ^= 1u; }
            }
        };

        double acc[RBW][CBW][PAR][2];
#pragma unroll
        for (int rb = 0; rb < RBW; ++rb)
#pragma unroll
            for (int cb = 0; cb < CBW; ++cb)
#pragma unroll
                for (int par = 0; par < PAR; ++par) acc[rb][cb][par][0] = acc[rb][cb][par][1] = 0.0;

        for (int ch = 0; ch < n_chunks; ++ch) {
            if (warp == 0) {
                issue_loads(min(n_chunks, ch + RT_STAGES));
                while (ld_r < ch + 1) issue_loads(min(n_chunks, ch + RT_STAGES));   // the producer never blocks on a chunk it has not issued
            }
            mbar_wait_safe(full0 + 8 * s, ph);
            const uint32_t st = smem_base + s * RT_STAGE_BYTES;
#pragma unroll
            for (int bx = 0; bx < BOXES; ++bx) {
                const uint32_t base = st + bx * BOX_BYTES;
#pragma unroll
                for (int ks = 0; ks < 4; ++ks) {
                    double af[RBW], bf[CBW];
#pragma unroll
                    for (int rb = 0; rb < RBW; ++rb) af[rb] = lds_f64(base + offA[rb][ks]);
#pragma unroll
                    for (int cb = 0; cb < CBW; ++cb) bf[cb] = lds_f64(base + offB[cb][ks]);
#pragma unroll
                    for (int rb = 0; rb < RBW; ++rb)
#pragma unroll
                        for (int cb = 0; cb < CBW; ++cb)
                            dmma_8x8x4(acc[rb][cb][ks & (PAR - 1)][0], acc[rb][cb][ks & (PAR - 1)][1], af[rb], bf[cb]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty0 + 8 * s);
            if (++s == RT_STAGES) { s = 0; ph ^= 1u; }
        }

        // ---- fused epilogue on the warp's (BM/2) x (BM/4) outputs
        {
            const double c2 = cs.coef.c2, c1 = cs.coef.c1, c0 = cs.coef.c0;
            const int ld = p.ld;
            double p_tr = 0.0, p_ss = 0.0, p_err = 0.0, p_trc = 0.0, p_ce = 0.0;
#pragma unroll
            for (int rb = 0; rb < RBW; ++rb) {
                const int row = I * BM + warp_m * (BM / 2) + rb * 8 + r;
#pragma unroll
                for (int cb = 0; cb < CBW; ++cb) {
                    const int col = J * BM + warp_n * (BM / 4) + cb * 8 + 2 * kk;
                    double cv[2];
                    if (PAR == 2) {
                        cv[0] = acc[rb][cb][0][0] + acc[rb][cb][PAR - 1][0];
                        cv[1] = acc[rb][cb][0][1] + acc[rb][cb][PAR - 1][1];
                    } else {
                        cv[0] = acc[rb][cb][0][0];
                        cv[1] = acc[rb][cb][0][1];
                    }
                    const double2 e2 = __ldcg(reinterpret_cast<const double2*>(E + (size_t)row * ld + col));
                    const double ev[2] = {e2.x, e2.y};
                    double o[2];
#pragma unroll
                    for (int u = 0; u < 2; ++u) {
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
                        *reinterpret_cast<double2*>(Out + (size_t)row * ld + col) = make_double2(o[0], o[1]);
                        Out[(size_t)col * ld + row] = o[0];
                        Out[(size_t)(col + 1) * ld + row] = o[1];
                    } else {
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            if (col + u >= row) Out[(size_t)row * ld + col + u] = o[u];
                            if (col + u > row) Out[(size_t)(col + u) * ld + row] = o[u];
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
                rec[(size_t)b * SQ_NPART + threadIdx.x] = v;
            }
        }
        if (timer) { t_b = globaltimer_ns(); ph_ns[0] += t_b - t_a; t_a = t_b; }
        grid_barrier(p.flags, G, epoch);
        if (timer) { t_b = globaltimer_ns(); ph_ns[1] += t_b - t_a; t_a = t_b; }
        {
            double t1, s1, e2;
            record_sums_cg(rec, p.n_tiles, sh3, t1, s1, e2);
            if (threadIdx.x == 0) control_update(&cs, t1, s1, e2);
            __syncthreads();
        }
        if (timer) { t_b = globaltimer_ns(); ph_ns[2] += t_b - t_a; step_ns += t_b - t_start; }
    }

    if (b == 0) {
        const int* src = reinterpret_cast<const int*>(&cs);
        int* dst = reinterpret_cast<int*>(p.ctrl);
        for (int i = threadIdx.x; i < (int)(sizeof(Ctrl) / sizeof(int)); i += SQ_THREADS) dst[i] = src[i];
        if (threadIdx.x == 0) {
            p.timing[0] = step_ns;
            p.timing[1] = ph_ns[0]; p.timing[2] = ph_ns[1]; p.timing[3] = 0; p.timing[4] = 0; p.timing[5] = ph_ns[2];
        }
    }
}

}  // namespace rfoe
