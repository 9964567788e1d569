// librfoe -- C ABI (include/rfoe.h) over the sm_100a kernels.  Host logic only: argument checks,
// workspace management, TMA descriptors, the launch sequence of one expansion and the one-word-per-step
// read from mapped pinned memory.  Every arithmetic step of the path runs in the kernels.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <atomic>
#include <mutex>
#include <new>
#include <thread>
#include <vector>

#include "../../include/rfoe.h"
#include "control.cuh"
#include "hbm_kernels.cuh"
#include "lanczos.cuh"
#include "probe.cuh"
#include "resident.cuh"
#include "resident_fin.cuh"
#include "resident_small.cuh"
#include "shard.cuh"
#include "subspace.cuh"
#include "sym_square.cuh"
#include "sym_square_reduced.cuh"
#include "sym_square_reduced_pair.cuh"
#include "tail.cuh"

using namespace rfoe;

static_assert(RFOE_MAX_STEPS == CTRL_MAX_STEPS, "header / control history size mismatch");

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct HostPage {          // mapped pinned memory
    volatile int word;     // next action, written by control_kernel
    int sym_flag;
    double bounds[2];
    double scalars[8];
    Ctrl ctrl;             // staging copy of the device control block
};

struct rfoe_handle_s {
    int device = 0;
    int sm_count = 148;
    int64_t k_max = 0;
    int ld_max = 0;
    double* W[3] = {nullptr, nullptr, nullptr};
    tq_elem_t* F[2] = {nullptr, nullptr};   // hi / lo parts (FP16, scaled) of X_n - (Tr X_n / k) I for the reduced-precision squaring (lazy)
    double* part[2] = {nullptr, nullptr};
    double* rows[2] = {nullptr, nullptr};
    double* d_bounds = nullptr;
    double* d_scalars = nullptr;
    int* d_flag = nullptr;
    Ctrl* d_ctrl = nullptr;
    int2* d_tiles = nullptr;
    int2* d_pairs = nullptr;   // reduced-precision kernel: (I, J0) of every 2-CTA cluster (tiles (I,J0), (I,J0+1))
    int n_pairs = 0;
    int tiles_m = 0;       // tile-grid size the tile map was built for
    int n_tiles = 0;
    HostPage* hp = nullptr;
    int* d_word = nullptr; // device alias of hp->word
    // the whole recursion in one persistent launch (resident.cuh)
    int coop_ok = 0;           // cooperative launch supported and one CTA of the kernel fits an SM
    int side_by_side = 0;      // set by rfoe_expand_many while several handles work side by side (see expand_impl)
    int rs_m = 0, rs_G = 0, rs_n_split = 0, rs_tile_cost = 0;   // the plan the split list / records were set up for
    int4* d_split = nullptr;
    double* d_rec[2] = {nullptr, nullptr};
    unsigned* d_flags = nullptr;
    int rs_rec_dirty = 0;          // the finisher form has written tile records the band form expects to be zero
    unsigned long long* d_timing = nullptr;
    // sharded expansion over peer memory (rfoe_shard_set_peers / rfoe_shard_ipc_import)
    int p2p_world = 0, p2p_rank = 0;
    double* peer_W[2][SQ_MAX_PEERS] = {};
    double* peer_rec[2][SQ_MAX_PEERS] = {};   // records double-buffered by step parity: a fast rank's step n+1 must not
                                              // overwrite the records its peer's control kernel of step n still reads
    PeerSet* d_peers = nullptr;   // [2]: destinations of a step that writes W[0] / W[1] (device copy for the MODE 3 kernel)
    void* ipc_opened[4 * SQ_MAX_PEERS] = {};
    int n_ipc_opened = 0;
    double* sh_send = nullptr; // sharded expansion: [c tiles | c records] to send, g such blocks received,
    double* sh_recv = nullptr; //   and the records in global tile order (allocated on the first sharded call)
    double* sh_parts = nullptr;
    size_t sh_bytes = 0;
    double* lz_vec = nullptr;  // Lanczos bounds: v, v_prev, w (ld_max doubles each) + block partials
    LanczosState* lz_state = nullptr;
    int lanczos_steps = 0;     // RFOE_OPT_LANCZOS_STEPS: 0 = Gershgorin bounds in rfoe_expand
    double* ws = nullptr;      // scratch of the projection / density steps (grown on demand)
    size_t ws_bytes = 0;
    double* stage_H = nullptr;
    double* stage_P = nullptr;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    cudaEvent_t sq_ev[4 * RFOE_MAX_STEPS] = {};   // begin/end pairs around every squaring launch of an expansion
    int sq_n = 0;
    EncodeTiledFn encode = nullptr;
    // options
    int stop_rule = 0, max_iter = 100, check_sym = 1, trunc_steps = 30, resident = 1, reduced_pair = 1;
    double eps_min = NAN, eps_max = NAN, mixed_head = 0.0, mixed_reltr = 5e-4, homo = NAN, lumo = NAN;
    rfoe_stats_t stats;
    int64_t launches = 0;
};

#define CK(call)                                                     \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) {                                     \
            h->stats.cuda_error = (int)e_;                           \
            h->stats.status = RFOE_ERR_CUDA;                         \
            return RFOE_ERR_CUDA;                                    \
        }                                                            \
    } while (0)

static int round_up(int64_t v, int m) { return (int)((v + m - 1) / m * m); }

static int hbm_grid(const rfoe_handle_s* h, int rows)
{
    int want = (rows + HBM_WARPS - 1) / HBM_WARPS;
    int cap = h->sm_count * 8;
    return want < cap ? (want < 1 ? 1 : want) : cap;
}

// Upper-triangle tile order: strips of G tile rows, each walked COLUMN by column (j outer, i inner).  The ~148 CTAs resident
// at any time then cover G rows x ~12.3 consecutive columns wherever the window falls: 2 G + 0.3 row panels streamed
// through L2 together.  (Round 1 walked G x G super-blocks row-major; a window straddling two super-blocks touched up to
// 36 panels instead of 24, which is the 34.7 GB of DRAM reads per squaring ncu showed at k=16384 against a 22.9 GB floor.)
static void build_tile_order(int m, std::vector<int2>& out)
{
    const int G = 12;
    out.clear();
    out.reserve((size_t)m * (m + 1) / 2);
    for (int SI = 0; SI < m; SI += G)
        for (int j = SI; j < m; ++j)
            for (int i = SI; i < SI + G && i <= j; ++i) out.push_back(make_int2(i, j));
}

static int ensure_tiles(rfoe_handle_s* h, int m, cudaStream_t st)
{
    if (h->tiles_m == m) return RFOE_OK;
    std::vector<int2> order, pairs;
    build_tile_order(m, order);
    for (const int2& t : order)      // row pairs in the same L2-friendly order: tiles (i, j), (i, j+1) with j - i even
        if (((t.y - t.x) & 1) == 0) pairs.push_back(t);
    CK(cudaMemcpyAsync(h->d_tiles, order.data(), order.size() * sizeof(int2), cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(h->d_pairs, pairs.data(), pairs.size() * sizeof(int2), cudaMemcpyHostToDevice, st));
    CK(cudaStreamSynchronize(st));   // the vectors are pageable and die here
    h->tiles_m = m;
    h->n_tiles = (int)order.size();
    h->n_pairs = (int)pairs.size();
    return RFOE_OK;
}

static int make_map(rfoe_handle_s* h, CUtensorMap* map, double* base, int n, int ld, int box_rows = SQ_BM)
{
    cuuint64_t dims[2] = {(cuuint64_t)n, (cuuint64_t)n};
    cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(double)};
    cuuint32_t box[2] = {(cuuint32_t)SQ_BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = h->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->stats.cuda_error = (int)cudaErrorInvalidValue;
        return RFOE_ERR_CUDA;
    }
    return RFOE_OK;
}

static int make_map_parts(rfoe_handle_s* h, CUtensorMap* map, tq_elem_t* base, int n, int ld32)
{
    cuuint64_t dims[2] = {(cuuint64_t)n, (cuuint64_t)n};
    cuuint64_t strides[1] = {(cuuint64_t)ld32 * sizeof(tq_elem_t)};
    cuuint32_t box[2] = {(cuuint32_t)TQ_BK, (cuuint32_t)(TQ_BM / 2)};   // half panels: 64 rows x 128 bytes
    cuuint32_t estr[2] = {1, 1};
    CUresult r = h->encode(map, sizeof(tq_elem_t) == 2 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, base, dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        h->stats.cuda_error = (int)cudaErrorInvalidValue;
        return RFOE_ERR_CUDA;
    }
    return RFOE_OK;
}

static int ensure_parts(rfoe_handle_s* h)
{
    const size_t ld = (size_t)h->ld_max;
    for (tq_elem_t*& p : h->F)
        if (!p && cudaMalloc(&p, ld * (ld + TQ_PAD) * sizeof(tq_elem_t)) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    return RFOE_OK;
}

// reduced-precision step: split X (FP64, in Xin) into its hi / lo parts, then the tcgen05 squaring with the FP64 epilogue
static cudaError_t launch_square_reduced(rfoe_handle_s* h, const CUtensorMap& hi, const CUtensorMap& lo, const double* Xin,
                                      double* Out, int n, int ld, int k, const double* trace, const StepCoef* coef,
                                      double* partials, cudaStream_t st)
{
    split_parts_kernel<<<hbm_grid(h, n), 256, 0, st>>>(Xin, n, ld, k, trace, h->F[0], h->F[1], n + TQ_PAD);
    h->launches++;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * h->n_pairs);
    cfg.blockDim = dim3(TQ_THREADS);
    cfg.dynamicSmemBytes = h->reduced_pair ? TP_SMEM_BYTES : TQ_SMEM_BYTES;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    h->launches++;
    // CTA-pair form (tcgen05.mma.cta_group::2, sym_square_reduced_pair.cuh) unless RFOE_OPT_REDUCED_PAIR = 0
    if (h->reduced_pair)
        return cudaLaunchKernelEx(&cfg, sym_square_reduced_pair_kernel, hi, lo, Xin, Out, n, ld, k, trace, coef, (const int2*)h->d_pairs,
                                  n / TQ_BM, partials);
    return cudaLaunchKernelEx(&cfg, sym_square_reduced_kernel, hi, lo, Xin, Out, n, ld, k, trace, coef, (const int2*)h->d_pairs,
                              n / TQ_BM, partials);
}

template <bool TWO_OP>
static cudaError_t launch_square(rfoe_handle_s* h, const CUtensorMap& a, const CUtensorMap& b, const double* E, double* Out,
                                 int n, int ld, int k, const StepCoef* coef, double* partials, cudaStream_t st)
{
    sym_square_kernel<TWO_OP ? 1 : 0><<<h->n_tiles, SQ_THREADS, SQ_SMEM_BYTES, st>>>(a, b, E, Out, n, ld, k, coef, h->d_tiles, partials, 0);
    h->launches++;
    return cudaGetLastError();
}

// squaring launch bracketed by its own event pair (summed into stats.square_ms after the expansion)
template <bool TWO_OP>
static cudaError_t timed_square(rfoe_handle_s* h, const CUtensorMap& a, const CUtensorMap& b, const double* E, double* Out,
                                int n, int ld, int k, const StepCoef* coef, double* partials, cudaStream_t st)
{
    cudaError_t e = cudaEventRecord(h->sq_ev[2 * h->sq_n], st);
    if (e != cudaSuccess) return e;
    e = launch_square<TWO_OP>(h, a, b, E, Out, n, ld, k, coef, partials, st);
    if (e != cudaSuccess) return e;
    e = cudaEventRecord(h->sq_ev[2 * h->sq_n + 1], st);
    h->sq_n++;
    return e;
}

// ---------------------------------------------------------------------------------------------
// Tail plan of a squaring launch (tail.cuh): tiles [0, n_main) go to the main kernel in whole waves, the last
// T = n_tiles - n_main tiles are cut into `slices` K-slices of kt_per chunks.  Chosen by a cycle model (a full tile
// costs kt * 4096 DMMA cycles + ~45k of epilogue / launch; a slice CTA kt_per * 4096 + ~20k; the two extra kernel
// boundaries and the fix-up ~60k) and only taken when the model saves >= 1.5 %: measured, k=8192 gains 5.2 % (16.35 ->
// 15.55 ms), k=4096 8.5 %, but at k=16384 the modelled 0.3 % came out as -0.06 % (122.22 vs 122.15 ms), so large
// problems keep the plain launch.  Depends on (n_tiles, kt, SM count) only.
struct TailPlan {
    int n_main, slices, kt_per;
};

static TailPlan plan_tail(int n_tiles, int kt_total, int sm)
{
    TailPlan best = {n_tiles, 1, kt_total};
    const double full = kt_total * 4096.0 + 45000.0;
    const double base = (double)((n_tiles + sm - 1) / sm) * full;
    double best_t = base * (1.0 - 0.015);
    const int r = n_tiles % sm;
    for (int w = 0; w <= 1; ++w) {
        const int T = r + w * sm;
        if (T == 0 || T > n_tiles) continue;
        for (int s = 2; s <= 16; ++s) {
            const int per = (kt_total + s - 1) / s;
            if (per < 16) break;
            const int eff = (kt_total + per - 1) / per;
            const long long ctas = (long long)T * eff;
            const double t = (double)((n_tiles - T) / sm) * full + (double)((ctas + sm - 1) / sm) * (per * 4096.0 + 20000.0) + 60000.0;
            if (t < best_t) { best_t = t; best = {n_tiles - T, eff, per}; }
        }
    }
    return best;
}

// SP2 squaring of tiles [t_begin, t_begin + t_count) of the tile order: main kernel below plan.n_main, split-K tail
// + fix-up above.  rec = partial record of tile t_begin.  peers != nullptr (sharded P2P run): the epilogues store to
// every rank's X_{n+1} (peers->out) and record array (peers->rec, global tile index) instead of Out / rec.
static cudaError_t launch_sp2_range(rfoe_handle_s* h, const CUtensorMap& tm, const double* E, double* Out, int n, int ld, int k,
                                    const StepCoef* coef, double* rec, int t_begin, int t_count, const TailPlan& plan,
                                    cudaStream_t st, const PeerSet* peers = nullptr, PeerSet* d_peers = nullptr)
{
    const int t_end = t_begin + t_count;
    const int main_end = t_end < plan.n_main ? t_end : plan.n_main;
    if (main_end > t_begin) {
        if (peers) {   // d_peers: the same PeerSet in device memory (rec_offset = t_begin), see sym_square.cuh MODE 3
            sym_square_kernel<3><<<main_end - t_begin, SQ_THREADS, SQ_SMEM_BYTES, st>>>(tm, tm, E, reinterpret_cast<double*>(d_peers), n, ld, k,
                                                                                    coef, h->d_tiles + t_begin, nullptr, 0);
        } else {
            sym_square_kernel<0><<<main_end - t_begin, SQ_THREADS, SQ_SMEM_BYTES, st>>>(tm, tm, E, Out, n, ld, k, coef,
                                                                                    h->d_tiles + t_begin, rec, 0);
        }
        h->launches++;
    }
    const int tail_b = t_begin > plan.n_main ? t_begin : plan.n_main;
    const int n_tl = t_end - tail_b;
    if (n_tl > 0) {
        sym_square_kernel<2><<<dim3(n_tl, plan.slices), SQ_THREADS, SQ_SMEM_BYTES, st>>>(tm, tm, nullptr, h->ws, n, SQ_BM, k, nullptr,
                                                                                      h->d_tiles + tail_b, nullptr, plan.kt_per);
        PeerSet ps;
        if (peers) { ps = *peers; ps.rec_offset = tail_b; }
        else { ps = PeerSet{}; ps.n = 1; ps.out[0] = Out; ps.rec[0] = rec + (size_t)(tail_b - t_begin) * SQ_NPART; ps.rec_offset = 0; }
        tail_fixup_kernel<<<n_tl, TAIL_THREADS, 0, st>>>(h->ws, plan.slices, n_tl, h->d_tiles + tail_b, E, ld, k, coef, ps);
        h->launches += 2;
    }
    return cudaGetLastError();
}

static int ensure_tail_ws(rfoe_handle_s* h, int n_tiles, const TailPlan& plan);
static int ensure_ws(rfoe_handle_s* h, size_t bytes);

extern "C" const char* rfoe_strerror(int status)
{
    switch (status) {
        case RFOE_OK: return "ok";
        case RFOE_ERR_INVALID_ARG: return "invalid argument";
        case RFOE_ERR_ALLOC: return "allocation failed";
        case RFOE_ERR_CUDA: return "CUDA error";
        case RFOE_ERR_BAD_BOUNDS: return "spectral bounds are empty or not finite";
        case RFOE_ERR_NOT_SYMMETRIC: return "H^p is not bitwise symmetric";
        case RFOE_ERR_UNSUPPORTED: return "unsupported variant, option or device";
        case RFOE_ERR_NOT_CONVERGED: return "maximum number of recursion steps reached";
        case RFOE_ERR_NO_PEER_ACCESS: return "a peer GPU's buffers cannot be mapped (no P2P access)";
        case RFOE_ERR_STATIC_LIMIT: return "k exceeds RFOE_STATIC_MAX_K, the size of the allocation-free entry point's fixed scratch array";
        default: return "unknown status";
    }
}

extern "C" int rfoe_version(void) { return 201; }

extern "C" int rfoe_destroy(rfoe_handle_t h)
{
    if (!h) return RFOE_OK;
    cudaSetDevice(h->device);
    for (double* p : h->W) cudaFree(p);
    for (tq_elem_t* p : h->F) cudaFree(p);
    for (double* p : h->part) cudaFree(p);
    for (double* p : h->rows) cudaFree(p);
    cudaFree(h->d_bounds); cudaFree(h->d_scalars); cudaFree(h->d_flag); cudaFree(h->d_ctrl); cudaFree(h->d_tiles);
    cudaFree(h->d_pairs);
    cudaFree(h->d_split); cudaFree(h->d_rec[0]); cudaFree(h->d_rec[1]); cudaFree(h->d_flags); cudaFree(h->d_timing);
    cudaFree(h->stage_H); cudaFree(h->stage_P); cudaFree(h->ws); cudaFree(h->lz_vec); cudaFree(h->lz_state);
    cudaFree(h->sh_send); cudaFree(h->sh_recv); cudaFree(h->sh_parts);
    for (int i = 0; i < h->n_ipc_opened; ++i) cudaIpcCloseMemHandle(h->ipc_opened[i]);
    cudaFree(h->d_peers);
    if (h->hp) cudaFreeHost(h->hp);
    if (h->ev0) cudaEventDestroy(h->ev0);
    if (h->ev1) cudaEventDestroy(h->ev1);
    for (cudaEvent_t e : h->sq_ev) if (e) cudaEventDestroy(e);
    delete h;
    return RFOE_OK;
}

extern "C" int rfoe_create(rfoe_handle_t* out, int device, int64_t k_max)
{
    if (!out || k_max < 1 || k_max > (1 << 20)) return RFOE_ERR_INVALID_ARG;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return RFOE_ERR_CUDA;
    if (cudaSetDevice(device) != cudaSuccess) return RFOE_ERR_CUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return RFOE_ERR_CUDA;
    if (prop.major != 10) return RFOE_ERR_UNSUPPORTED;   // sm_100a cubin only; no fallback path
    rfoe_handle_s* h = new (std::nothrow) rfoe_handle_s();
    if (!h) return RFOE_ERR_ALLOC;
    memset(&h->stats, 0, sizeof(h->stats));
    h->device = device;
    h->sm_count = prop.multiProcessorCount;
    h->k_max = k_max;
    h->ld_max = round_up(k_max, SQ_BM);
    const size_t ld = (size_t)h->ld_max;
    const size_t wbytes = ld * (ld + SQ_PAD) * sizeof(double);
    const size_t m = ld / SQ_BM, nt = m * (m + 1) / 2;
    bool ok = true;
    ok = ok && cudaMalloc(&h->W[0], wbytes) == cudaSuccess;
    ok = ok && cudaMalloc(&h->W[1], wbytes) == cudaSuccess;
    ok = ok && cudaMalloc(&h->part[0], (nt + m) * SQ_NPART * sizeof(double)) == cudaSuccess;   // + phantom records
    ok = ok && cudaMalloc(&h->part[1], (nt + m) * SQ_NPART * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->rows[0], ld * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->rows[1], ld * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->d_bounds, 2 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->d_scalars, 8 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->d_flag, sizeof(int)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->d_ctrl, sizeof(Ctrl)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->d_tiles, nt * sizeof(int2)) == cudaSuccess;
    ok = ok && cudaMalloc(&h->d_pairs, nt * sizeof(int2)) == cudaSuccess;
    {
        const size_t mr = (size_t)RS_MAX_N / SQ_BM, nrec = mr * (mr + 1) / 2 + 256;
        ok = ok && cudaMalloc(&h->d_split, RS_MAX_SPLIT * sizeof(int4)) == cudaSuccess;
        ok = ok && cudaMalloc(&h->d_rec[0], nrec * SQ_NPART * sizeof(double)) == cudaSuccess;
        ok = ok && cudaMalloc(&h->d_rec[1], nrec * SQ_NPART * sizeof(double)) == cudaSuccess;
        ok = ok && cudaMalloc(&h->d_flags, RS_FLAG_WORDS * sizeof(unsigned)) == cudaSuccess;
        ok = ok && cudaMalloc(&h->d_timing, 8 * sizeof(unsigned long long)) == cudaSuccess;
    }
    ok = ok && cudaHostAlloc((void**)&h->hp, sizeof(HostPage), cudaHostAllocMapped) == cudaSuccess;
    ok = ok && cudaHostGetDevicePointer((void**)&h->d_word, (void*)&h->hp->word, 0) == cudaSuccess;
    ok = ok && cudaEventCreate(&h->ev0) == cudaSuccess && cudaEventCreate(&h->ev1) == cudaSuccess;
    for (cudaEvent_t& e : h->sq_ev) ok = ok && cudaEventCreate(&e) == cudaSuccess;
    if (!ok) { cudaGetLastError(); rfoe_destroy(h); return RFOE_ERR_ALLOC; }
    cudaDriverEntryPointQueryResult qres;
    void* fn = nullptr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn) {
        rfoe_destroy(h);
        return RFOE_ERR_CUDA;
    }
    h->encode = (EncodeTiledFn)fn;
    if (cudaFuncSetAttribute(sym_square_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, SQ_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(sym_square_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SQ_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(sym_square_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SQ_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(sym_square_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, SQ_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(resident_recursion_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, RS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(resident_finisher_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, RS_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(resident_small_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, RT_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(resident_small_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, RT_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(apply_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, AP_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(sym_square_reduced_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TQ_SMEM_BYTES) != cudaSuccess ||
        cudaFuncSetAttribute(sym_square_reduced_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TP_SMEM_BYTES) != cudaSuccess) {
        rfoe_destroy(h);
        return RFOE_ERR_CUDA;
    }
    {
        int coop = 0, per_sm = 0;
        if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device) == cudaSuccess && coop &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, resident_recursion_kernel, SQ_THREADS, RS_SMEM_BYTES) == cudaSuccess &&
            per_sm >= 1 &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, resident_finisher_kernel, SQ_THREADS, RS_SMEM_BYTES) == cudaSuccess &&
            per_sm >= 1 && h->sm_count <= 256 && (RT_MAX_N / 64) * (RT_MAX_N / 64 + 1) / 2 <= h->sm_count &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, resident_small_kernel<32>, SQ_THREADS, RT_SMEM_BYTES) == cudaSuccess && per_sm >= 1 &&
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, resident_small_kernel<64>, SQ_THREADS, RT_SMEM_BYTES) == cudaSuccess && per_sm >= 1)
            h->coop_ok = 1;
        cudaGetLastError();
    }
    *out = h;
    return RFOE_OK;
}

extern "C" int rfoe_set_option(rfoe_handle_t h, int key, double value)
{
    if (!h) return RFOE_ERR_INVALID_ARG;
    switch (key) {
        case RFOE_OPT_STOP_RULE:
            if (value != 0.0 && value != 1.0) return RFOE_ERR_INVALID_ARG;
            h->stop_rule = (int)value; return RFOE_OK;
        case RFOE_OPT_MAX_ITER:
            if (!(value >= 1.0 && value <= (double)RFOE_MAX_STEPS)) return RFOE_ERR_INVALID_ARG;
            h->max_iter = (int)llround(value); return RFOE_OK;
        case RFOE_OPT_EPS_MIN: h->eps_min = value; return RFOE_OK;
        case RFOE_OPT_EPS_MAX: h->eps_max = value; return RFOE_OK;
        case RFOE_OPT_CHECK_SYMMETRY: h->check_sym = (value != 0.0); return RFOE_OK;
        case RFOE_OPT_MIXED_HEAD:
            if (!(value >= 0.0)) return RFOE_ERR_INVALID_ARG;
            h->mixed_head = value; return RFOE_OK;
        case RFOE_OPT_MIXED_RELTR:
            if (!(value >= 0.0)) return RFOE_ERR_INVALID_ARG;
            h->mixed_reltr = value; return RFOE_OK;
        case RFOE_OPT_LANCZOS_STEPS:
            if (!(value >= 0.0 && value <= (double)LZ_MAX_STEPS)) return RFOE_ERR_INVALID_ARG;
            h->lanczos_steps = (int)llround(value); return RFOE_OK;
        case RFOE_OPT_TRUNC_STEPS:
            if (!(value >= 1.0 && value <= (double)RFOE_MAX_STEPS)) return RFOE_ERR_INVALID_ARG;
            h->trunc_steps = (int)llround(value); return RFOE_OK;
        case RFOE_OPT_RESIDENT:
            if (value != 0.0 && value != 1.0 && value != 2.0) return RFOE_ERR_INVALID_ARG;
            h->resident = (int)value; return RFOE_OK;
        case RFOE_OPT_REDUCED_PAIR:
            if (value != 0.0 && value != 1.0) return RFOE_ERR_INVALID_ARG;
            h->reduced_pair = (int)value; return RFOE_OK;
        case RFOE_OPT_HOMO: h->homo = value; return RFOE_OK;
        case RFOE_OPT_LUMO: h->lumo = value; return RFOE_OK;
        default: return RFOE_ERR_UNSUPPORTED;
    }
}

extern "C" int rfoe_get_stats(rfoe_handle_t h, rfoe_stats_t* out)
{
    if (!h || !out) return RFOE_ERR_INVALID_ARG;
    *out = h->stats;
    return RFOE_OK;
}

// HOMO / LUMO estimates from the history of an SP2 run (host only; rfoe.h, reading R-HL).
// u = image of the LUMO bound (small), v = 1 - image of the HOMO bound (small): both are carried back as distances
// from 0 and from 1, in the cancellation-free forms  1 - sqrt(1 - u) = u / (1 + sqrt(1 - u)).
extern "C" int rfoe_estimate_homo_lumo(const rfoe_stats_t* S, double* homo, double* lumo)
{
    if (!S || !homo || !lumo) return RFOE_ERR_INVALID_ARG;
    const int steps = S->iterations;
    const double width = S->eps_max - S->eps_min;
    if (steps < 1 || steps > RFOE_MAX_STEPS || !(width > 0.0) || !isfinite(width) || S->nocc < 1) return RFOE_ERR_INVALID_ARG;
    if (S->variant != RFOE_VARIANT_SP2 || S->fp32_steps != 0) return RFOE_ERR_UNSUPPORTED;
    for (int j = 0; j < steps; ++j)
        if (S->branch[j] != 'S' && S->branch[j] != 'L') return RFOE_ERR_UNSUPPORTED;
    constexpr double E_FLOOR = 1e-6;
    double u_best = INFINITY, v_best = INFINITY;   // smallest LUMO image / smallest (1 - HOMO image) in X_0
    for (int n = 0; n < steps; ++n) {
        const double e = S->e[n];
        const bool settled = (S->t[n] - S->s[n]) < 3.0 / 16.0 && fabs(S->t[n] - (double)S->nocc) < 0.5;
        if (!settled || !(e >= E_FLOOR) || !(e < 0.25)) continue;
        const double a = 2.0 * e / (1.0 + sqrt(1.0 - 4.0 * e));   // = (1 - sqrt(1 - 4e)) / 2
        double u = a, v = a;
        for (int j = n - 1; j >= 0; --j) {
            if (S->branch[j] == 'S') {            // x' = x^2:           x = sqrt(x'),  1 - x = (1 - x') / (1 + sqrt(x'))
                u = sqrt(u);
                v = v / (1.0 + sqrt(1.0 - v));
            } else {                              // 1 - x' = (1 - x)^2: 1 - x = sqrt(1 - x'),  x = x' / (1 + sqrt(1 - x'))
                u = u / (1.0 + sqrt(1.0 - u));
                v = sqrt(v);
            }
        }
        u_best = fmin(u_best, u);
        v_best = fmin(v_best, v);
    }
    if (!isfinite(u_best) || !isfinite(v_best)) return RFOE_ERR_NOT_CONVERGED;
    // X_0 = (eps_max I - H) / width:  lambda = eps_max - width x
    *lumo = S->eps_max - width * u_best;
    *homo = S->eps_min + width * v_best;          // = eps_max - width (1 - v)
    return RFOE_OK;
}

// ---------------------------------------------------------------------------------------------
// A1: Gershgorin bounds into h->d_bounds (device) -- two launches
static int run_bounds(rfoe_handle_s* h, const double* Hp, int k, cudaStream_t st)
{
    gershgorin_rows_kernel<<<hbm_grid(h, k), HBM_THREADS, 0, st>>>(Hp, k, h->rows[0], h->rows[1]);
    h->launches++;
    CK(cudaGetLastError());
    bounds_reduce_kernel<<<1, 256, 0, st>>>(h->rows[0], h->rows[1], k, h->d_bounds);
    h->launches++;
    CK(cudaGetLastError());
    return RFOE_OK;
}

// A1 (optional): m-step Lanczos bounds into h->d_bounds (device) -- lanczos.cuh
static int run_bounds_lanczos(rfoe_handle_s* h, const double* Hp, int k, int m, cudaStream_t st)
{
    if (m > k) m = k;
    if (m < 1) m = 1;
    const size_t ld = (size_t)h->ld_max;
    if (!h->lz_vec && cudaMalloc(&h->lz_vec, (3 * ld + 4096) * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    if (!h->lz_state && cudaMalloc(&h->lz_state, sizeof(LanczosState)) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    double* v = h->lz_vec, *vp = v + ld, *w = vp + ld, *part = w + ld;
    int nb = (k + 255) / 256;
    if (nb > 2 * h->sm_count) nb = 2 * h->sm_count;
    lanczos_init_kernel<<<nb, 256, 0, st>>>(v, vp, k, part, h->lz_state);
    h->launches++;
    for (int j = 0; j < m; ++j) {
        lanczos_symv_kernel<<<hbm_grid(h, k), HBM_THREADS, 0, st>>>(Hp, k, v, w, h->rows[0], part, nb, j == 0, h->lz_state);
        if (j == 0) { lanczos_normalise_kernel<<<nb, 256, 0, st>>>(v, k, part, nb, h->lz_state); h->launches++; }
        lanczos_update_kernel<<<nb, 256, 0, st>>>(w, v, vp, k, h->rows[0], j, part, h->lz_state);
        lanczos_next_kernel<<<nb, 256, 0, st>>>(v, vp, w, k, part, nb, j, h->lz_state);
        lanczos_flag_kernel<<<1, 1, 0, st>>>(h->lz_state, j);
        h->launches += 4;
    }
    lanczos_bounds_kernel<<<1, 32, 0, st>>>(h->lz_state, h->d_bounds);
    h->launches++;
    CK(cudaGetLastError());
    return RFOE_OK;
}

static int check_common(rfoe_handle_s* h, const void* a, const void* b, int64_t k)
{
    if (!h) return RFOE_ERR_INVALID_ARG;
    if (!a || !b || k < 1 || k > h->k_max) return RFOE_ERR_INVALID_ARG;
    return RFOE_OK;
}

extern "C" int rfoe_bounds(rfoe_handle_t h, const double* Hp, int64_t k, double* eps_min, double* eps_max, rfoe_stream_t stream)
{
    if (!h || !Hp || !eps_min || !eps_max || k < 1 || k > h->k_max) return RFOE_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    h->launches = 0;
    h->stats.cuda_error = 0;
    CK(cudaSetDevice(h->device));
    int rc = run_bounds(h, Hp, (int)k, st);
    if (rc != RFOE_OK) return rc;
    CK(cudaMemcpyAsync((void*)h->hp->bounds, h->d_bounds, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    *eps_min = h->hp->bounds[0];
    *eps_max = h->hp->bounds[1];
    h->stats.gpu_launches = h->launches;
    h->stats.status = RFOE_OK;
    return RFOE_OK;
}

// ---- rfoe_bounds_static: row A1 without a handle and without any allocation (include/rfoe.h) ----------------------
// The per-row disc ends go to a file-scope device array instead of handle memory.  In host code the array's NAME is a
// host-side stand-in, not a device address: the kernels get the address cudaGetSymbolAddress returns, resolved once per
// device with that device current.
static __device__ __align__(256) double g_static_rows[2 * RFOE_STATIC_MAX_K];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDev {
    double* rows = nullptr;   // device address of g_static_rows on this device
    int sm_count = 0;
    int cc_major = 0;
};
StaticDev g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mu;
}  // namespace

extern "C" int rfoe_bounds_static(const double* Hp, int64_t k, double* bounds, rfoe_stream_t stream, int* cuda_error)
{
    if (cuda_error) *cuda_error = 0;
    auto fail = [&](cudaError_t e) {
        if (cuda_error) *cuda_error = (int)e;
        cudaGetLastError();
        return (int)RFOE_ERR_CUDA;
    };
    if (!Hp || !bounds || k < 1) return RFOE_ERR_INVALID_ARG;
    if (k > RFOE_STATIC_MAX_K) return RFOE_ERR_STATIC_LIMIT;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(e);
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) return RFOE_ERR_UNSUPPORTED;
    StaticDev sd;
    {
        std::lock_guard<std::mutex> lock(g_static_mu);
        StaticDev& slot = g_static_dev[dev];
        if (!slot.rows) {                                   // set-up, once per device, that device current
            int sms = 0, major = 0;
            if ((e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev)) != cudaSuccess) return fail(e);
            if (major != 10) return RFOE_ERR_UNSUPPORTED;
            if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return fail(e);
            double* ptr = nullptr;
            if ((e = cudaGetSymbolAddress((void**)&ptr, g_static_rows)) != cudaSuccess || !ptr) return fail(e != cudaSuccess ? e : cudaErrorInvalidSymbol);
            slot.sm_count = sms;
            slot.cc_major = major;
            slot.rows = ptr;
        }
        sd = slot;
    }
    cudaStream_t st = (cudaStream_t)stream;
    double* row_lo = sd.rows;
    double* row_hi = sd.rows + RFOE_STATIC_MAX_K;
    const int want = ((int)k + HBM_WARPS - 1) / HBM_WARPS, cap = sd.sm_count * 8;       // hbm_grid() without a handle
    gershgorin_rows_kernel<<<want < cap ? want : cap, HBM_THREADS, 0, st>>>(Hp, (int)k, row_lo, row_hi);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(e);
    bounds_reduce_kernel<<<1, 256, 0, st>>>(row_lo, row_hi, (int)k, bounds);
    if ((e = cudaGetLastError()) != cudaSuccess) return fail(e);
    return RFOE_OK;
}

extern "C" int rfoe_bounds_lanczos(rfoe_handle_t h, const double* Hp, int64_t k, int m, double* eps_min, double* eps_max,
                                   rfoe_stream_t stream)
{
    if (!h || !Hp || !eps_min || !eps_max || k < 1 || k > h->k_max || m < 1 || m > LZ_MAX_STEPS) return RFOE_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    h->launches = 0;
    h->stats.cuda_error = 0;
    CK(cudaSetDevice(h->device));
    int rc = run_bounds_lanczos(h, Hp, (int)k, m, st);
    if (rc != RFOE_OK) return rc;
    CK(cudaMemcpyAsync((void*)h->hp->bounds, h->d_bounds, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    *eps_min = h->hp->bounds[0];
    *eps_max = h->hp->bounds[1];
    h->stats.gpu_launches = h->launches;
    h->stats.status = RFOE_OK;
    return RFOE_OK;
}

static int ensure_third(rfoe_handle_s* h)
{
    if (h->W[2]) return RFOE_OK;
    const size_t ld = (size_t)h->ld_max;
    if (cudaMalloc(&h->W[2], ld * (ld + SQ_PAD) * sizeof(double)) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    return RFOE_OK;
}

struct ShardCtx {
    int rank, world;
    rfoe_allgather_fn allgather;   // exchange by all-gather (rfoe_expand_sharded) ...
    rfoe_barrier_fn barrier;       // ... or stores to peer memory + a barrier (rfoe_expand_sharded_p2p)
    void* user;
};

extern "C" int rfoe_plan_squaring(int64_t k, int sm_count, int64_t* n_tiles, int64_t* n_main, int* slices, int* kt_per_slice)
{
    if (k < 1 || k > (1 << 20) || sm_count < 1 || !n_tiles || !n_main || !slices || !kt_per_slice) return RFOE_ERR_INVALID_ARG;
    const int n = round_up(k, SQ_BM), m = n / SQ_BM;
    const long long nt = (long long)m * (m + 1) / 2;
    const TailPlan p = plan_tail((int)nt, n / SQ_BK, sm_count);
    *n_tiles = nt; *n_main = p.n_main; *slices = p.slices; *kt_per_slice = p.kt_per;
    return RFOE_OK;
}

extern "C" int rfoe_shard_range(int64_t n_tiles, int rank, int world, int64_t* begin, int64_t* count)
{
    if (n_tiles < 1 || world < 1 || rank < 0 || rank >= world || !begin || !count) return RFOE_ERR_INVALID_ARG;
    const int64_t c = (n_tiles + world - 1) / world;
    int64_t b = (int64_t)rank * c;
    if (b > n_tiles) b = n_tiles;
    int64_t e = b + c;
    if (e > n_tiles) e = n_tiles;
    *begin = b;
    *count = e - b;
    return RFOE_OK;
}

// Plan of the persistent recursion (resident.cuh): G CTAs (one per SM, fewer when there are fewer chunk units than SMs)
// share the n_tiles x KT chunk units of a step in contiguous ranges of equal cost; a tile not wholly inside one range is
// "split" and finished in the FIX phase.  host_boundary is the twin of rs_boundary in resident.cuh.
static int host_boundary(long long cost_total, int tile_cost, int KT, int G, int b)
{
    const long long c = (long long)b * cost_total / G;
    const int tile = (int)(c / tile_cost);
    const int off = (int)(c - (long long)tile * tile_cost);
    return tile * KT + (off < KT ? off : KT);
}

struct ResidentHostPlan {
    int G = 0, tile_cost = 0;
    std::vector<int4> split;     // (tile, first CTA holding a segment of it, number of segments, 0)
};

// pure host arithmetic (no device): also behind rfoe_plan_resident, so that CPU tests can check the partition
static ResidentHostPlan compute_resident_plan(int n_tiles, int KT, int sm_count)
{
    ResidentHostPlan pl;
    const long long U = (long long)n_tiles * KT;
    const int G = (int)(U < sm_count ? U : sm_count);
    // register epilogues are counted into the ranges only where a CTA holds several whole tiles; where nearly every tile
    // is split (FIX finishes those) the ranges are equal in chunk units
    int tile_cost = (U / G >= 2LL * KT) ? KT + RS_EPI_COST : KT;
    for (int attempt = 0; attempt < 2; ++attempt) {
        const long long total = (long long)n_tiles * tile_cost;
        bool empty = false;
        for (int b = 0; b < G && !empty; ++b) empty = host_boundary(total, tile_cost, KT, G, b + 1) <= host_boundary(total, tile_cost, KT, G, b);
        if (empty && tile_cost != KT) { tile_cost = KT; continue; }      // (cannot happen with ranges >= 2 tiles; belt and braces)
        pl.split.clear();
        int b = 0;
        for (int t = 0; t < n_tiles; ++t) {
            const int t0 = t * KT, t1 = t0 + KT;
            while (host_boundary(total, tile_cost, KT, G, b + 1) <= t0) ++b;          // b: the CTA whose range holds unit t0
            if (host_boundary(total, tile_cost, KT, G, b + 1) >= t1) continue;         // whole: register epilogue in MM
            int nseg = 1;
            while (host_boundary(total, tile_cost, KT, G, b + nseg) < t1) ++nseg;      // CTAs b .. b + nseg - 1 hold its segments
            pl.split.push_back(make_int4(t, b, nseg, 0));
        }
        break;
    }
    pl.G = G; pl.tile_cost = tile_cost;
    return pl;
}

static int ensure_resident_plan(rfoe_handle_s* h, int m, int KT, cudaStream_t st)
{
    const long long U = (long long)h->n_tiles * KT;
    const int G = (int)(U < h->sm_count ? U : h->sm_count);
    if (h->rs_m == m && h->rs_G == G) return RFOE_OK;
    const ResidentHostPlan pl = compute_resident_plan(h->n_tiles, KT, h->sm_count);
    const std::vector<int4>& split = pl.split;
    if ((int)split.size() > RS_MAX_SPLIT) return RFOE_ERR_UNSUPPORTED;
    h->rs_m = 0;
    if (!split.empty()) CK(cudaMemcpyAsync(h->d_split, split.data(), split.size() * sizeof(int4), cudaMemcpyHostToDevice, st));
    const size_t nrec = (size_t)h->n_tiles + (size_t)pl.G;
    CK(cudaMemsetAsync(h->d_rec[0], 0, nrec * SQ_NPART * sizeof(double), st));   // the tile records of split tiles stay zero
    CK(cudaMemsetAsync(h->d_rec[1], 0, nrec * SQ_NPART * sizeof(double), st));
    CK(cudaStreamSynchronize(st));   // `split` is pageable and dies here
    h->rs_m = m; h->rs_G = pl.G; h->rs_n_split = (int)split.size(); h->rs_tile_cost = pl.tile_cost;
    return RFOE_OK;
}

extern "C" int rfoe_plan_resident(int64_t k, int sm_count, int* path, int* grid, int* kt, int64_t* n_tiles, int* n_split,
                                  int* boundaries, int* split_tiles)
{
    if (k < 1 || k > (1 << 20) || sm_count < 1 || sm_count > 256 || !path || !grid || !kt || !n_tiles || !n_split) return RFOE_ERR_INVALID_ARG;
    const int n = round_up(k, SQ_BM);
    *kt = 0; *n_split = 0;
    if (n > RS_MAX_N) { *path = 0; *grid = 0; *n_tiles = (int64_t)(n / SQ_BM) * (n / SQ_BM + 1) / 2; return RFOE_OK; }
    if (n <= RT_MAX_N) {
        const int bm = (n <= RT_MAX_N32) ? 32 : 64, mt = n / bm;
        *path = (bm == 32) ? 1 : 2;
        *n_tiles = (int64_t)mt * (mt + 1) / 2;
        *grid = (int)*n_tiles;
        if (*grid > sm_count) { *path = 0; *grid = 0; }      // (the library requires one CTA per tile to be co-resident)
        return RFOE_OK;
    }
    const int m = n / SQ_BM, nt = m * (m + 1) / 2, KT = n / SQ_BK;
    const ResidentHostPlan pl = compute_resident_plan(nt, KT, sm_count);
    *path = 3; *grid = pl.G; *kt = KT; *n_tiles = nt; *n_split = (int)pl.split.size();
    const long long total = (long long)nt * pl.tile_cost;
    if (boundaries)
        for (int b = 0; b <= pl.G; ++b) boundaries[b] = host_boundary(total, pl.tile_cost, KT, pl.G, b);
    if (split_tiles)
        for (size_t i = 0; i < pl.split.size(); ++i) {
            split_tiles[3 * i] = pl.split[i].x; split_tiles[3 * i + 1] = pl.split[i].y; split_tiles[3 * i + 2] = pl.split[i].z;
        }
    return RFOE_OK;
}

static int expand_impl(rfoe_handle_t h, const double* Hp, int64_t k64, int64_t nocc, int variant, double tol, double* P,
                       rfoe_stream_t stream, const ShardCtx* sh)
{
    int rc = check_common(h, Hp, P, k64);
    if (rc != RFOE_OK) return rc;
    rfoe_stats_t& S = h->stats;
    memset(&S, 0, sizeof(S));
    S.variant = variant; S.stop_rule = h->stop_rule; S.k = k64; S.nocc = nocc; S.tol = tol;
    auto fail = [&](int code) { S.status = code; return code; };
    if (!(nocc > 0 && nocc < k64) || !(tol >= 0.0) || !isfinite(tol)) return fail(RFOE_ERR_INVALID_ARG);
    {   // overlap of Hp and P
        const char* a = (const char*)Hp; const char* b = (const char*)P;
        const size_t bytes = (size_t)k64 * k64 * sizeof(double);
        if (a < b + bytes && b < a + bytes) return fail(RFOE_ERR_INVALID_ARG);
    }
    if (variant < RFOE_VARIANT_SP2 || variant > RFOE_VARIANT_TRUNC_MIXED) return fail(RFOE_ERR_UNSUPPORTED);
    const bool is_mixed = (variant == RFOE_VARIANT_SP2_MIXED || variant == RFOE_VARIANT_TRUNC_MIXED);
    const bool is_trunc = (variant == RFOE_VARIANT_TRUNC || variant == RFOE_VARIANT_TRUNC_MIXED);
    S.trunc_steps = is_trunc ? h->trunc_steps : 0;
    if (variant == RFOE_VARIANT_SP2_ACCEL && !(isfinite(h->homo) && isfinite(h->lumo) && h->lumo > h->homo))
        return fail(RFOE_ERR_INVALID_ARG);
    const int k = (int)k64;
    const int n = round_up(k, SQ_BM);      // padded extent of the work matrices
    const int ld = n + SQ_PAD;             // their row pitch (never a power of two: see sym_square.cuh)
    const int m = n / SQ_BM;
    cudaStream_t st = (cudaStream_t)stream;
    h->launches = 0;
    CK(cudaSetDevice(h->device));
    if (variant == RFOE_VARIANT_MCWEENY && (rc = ensure_third(h)) != RFOE_OK) return fail(rc);
    if (is_mixed && (rc = ensure_parts(h)) != RFOE_OK) return fail(rc);
    if ((rc = ensure_tiles(h, m, st)) != RFOE_OK) return fail(rc);
    // sharded run: this rank's contiguous range of the tile order, and the exchange buffers
    int t_begin = 0, t_count = h->n_tiles, c_max = h->n_tiles;
    size_t rank_stride = 0;
    if (sh) {
        if (variant != RFOE_VARIANT_SP2 && variant != RFOE_VARIANT_SP2_ACCEL && variant != RFOE_VARIANT_TRUNC) return fail(RFOE_ERR_UNSUPPORTED);
        int64_t b, c;
        if (rfoe_shard_range(h->n_tiles, sh->rank, sh->world, &b, &c) != RFOE_OK || (!sh->allgather && !sh->barrier))
            return fail(RFOE_ERR_INVALID_ARG);
        t_begin = (int)b; t_count = (int)c;
        c_max = (h->n_tiles + sh->world - 1) / sh->world;
    }
    PeerSet psets[2] = {};
    if (sh && sh->barrier) {
        for (int w = 0; w < 2; ++w) {
            psets[w].n = sh->world;
            psets[w].rec_offset = t_begin;
            for (int d = 0; d < sh->world; ++d) { psets[w].out[d] = h->peer_W[w][d]; psets[w].rec[d] = h->peer_rec[w][d]; }
        }
        if (!h->d_peers && cudaMalloc(&h->d_peers, 2 * sizeof(PeerSet)) != cudaSuccess) { cudaGetLastError(); return fail(RFOE_ERR_ALLOC); }
        CK(cudaMemcpyAsync(h->d_peers, psets, sizeof(psets), cudaMemcpyHostToDevice, st));
        CK(cudaStreamSynchronize(st));   // psets lives on this stack frame
        // entry barrier: this call's first epilogue stores into every peer's W[1] / records, which a peer still inside
        // its previous expansion (control kernel, output pass) may be reading -- nobody stores before everybody is here
        if (sh->barrier(sh->user, stream) != 0) return fail(RFOE_ERR_CUDA);
    }
    if (sh && sh->allgather) {
        rank_stride = (size_t)c_max * (TILE_ELEMS + SQ_NPART);
        const size_t need = rank_stride * sh->world * sizeof(double);
        if (h->sh_bytes < need) {
            cudaFree(h->sh_send); cudaFree(h->sh_recv); cudaFree(h->sh_parts);
            h->sh_send = h->sh_recv = h->sh_parts = nullptr; h->sh_bytes = 0;
            if (cudaMalloc(&h->sh_send, rank_stride * sizeof(double)) != cudaSuccess ||
                cudaMalloc(&h->sh_recv, need) != cudaSuccess ||
                cudaMalloc(&h->sh_parts, (size_t)c_max * sh->world * SQ_NPART * sizeof(double)) != cudaSuccess) {
                cudaGetLastError();
                return fail(RFOE_ERR_ALLOC);
            }
            h->sh_bytes = need;
        }
        CK(cudaMemsetAsync(h->sh_send, 0, rank_stride * sizeof(double), st));   // padding tiles / records of a short last range
    }
    const TailPlan plan = plan_tail(h->n_tiles, n / SQ_BK, h->sm_count);
    if ((rc = ensure_tail_ws(h, h->n_tiles, plan)) != RFOE_OK) return fail(rc);
    CUtensorMap tm[3];
    for (int i = 0; i < 3; ++i)
        if (h->W[i] && (rc = make_map(h, &tm[i], h->W[i], n, ld)) != RFOE_OK) return fail(rc);
    CUtensorMap tmF[2];
    if (is_mixed)
        for (int i = 0; i < 2; ++i)
            if ((rc = make_map_parts(h, &tmF[i], h->F[i], n, n + TQ_PAD)) != RFOE_OK) return fail(rc);

    // the whole recursion in one persistent launch when the problem is small enough to live on chip (resident.cuh)
    // (Several handles side by side, rfoe_expand_many: persistent launches of one CTA per SM cannot overlap, launch-per-step
    // kernels of different handles can and fill each other's idle SMs and sync gaps -- measured at k=2048, 4 handles: 91 against
    // 81 expansions/s.  So mid-size problems keep the launch-per-step path there; the latency-bound sizes do not, the small
    // persistent kernel being 3x faster than anything overlap could recover.)
    const bool use_resident = h->resident && h->coop_ok && !sh && n <= RS_MAX_N && !(h->side_by_side && n > RT_MAX_N) &&
                              (variant == RFOE_VARIANT_SP2 || variant == RFOE_VARIANT_SP2_ACCEL || variant == RFOE_VARIANT_TRUNC);
    const bool use_small = use_resident && n <= RT_MAX_N;      // latency-bound sizes: 32 x 32 tiles, one grid barrier per step
    if (use_resident && !use_small) {
        if ((rc = ensure_resident_plan(h, m, n / SQ_BK, st)) != RFOE_OK) return fail(rc);
        if ((rc = ensure_ws(h, (size_t)2 * h->rs_G * RS_TILE_ELEMS * sizeof(double))) != RFOE_OK) return fail(rc);
    }

    CK(cudaEventRecord(h->ev0, st));
    // --- symmetry check, bounds, affine map, first decision: enqueued back to back, validity settled on the device ----
    h->hp->sym_flag = 0;
    if (h->check_sym) {
        CK(cudaMemsetAsync(h->d_flag, 0, sizeof(int), st));
        const int nts = (k + SYM_T - 1) / SYM_T;
        long long blocks = (long long)nts * nts;
        if (blocks > h->sm_count * 16) blocks = h->sm_count * 16;
        symmetry_check_kernel<<<(int)blocks, 256, 0, st>>>(Hp, k, h->d_flag);
        h->launches++;
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(&h->hp->sym_flag, h->d_flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    }
    const bool override_bounds = isfinite(h->eps_min) && isfinite(h->eps_max);
    if (override_bounds) {
        if (!(h->eps_max > h->eps_min)) return fail(RFOE_ERR_BAD_BOUNDS);
        h->hp->bounds[0] = h->eps_min; h->hp->bounds[1] = h->eps_max;
        CK(cudaMemcpyAsync(h->d_bounds, (void*)h->hp->bounds, 2 * sizeof(double), cudaMemcpyHostToDevice, st));
    } else {
        if ((rc = (h->lanczos_steps > 0 ? run_bounds_lanczos(h, Hp, k, h->lanczos_steps, st) : run_bounds(h, Hp, k, st))) != RFOE_OK)
            return fail(rc);
        CK(cudaMemcpyAsync((void*)h->hp->bounds, h->d_bounds, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    Ctrl& C = h->hp->ctrl;
    memset(&C, 0, sizeof(Ctrl));
    C.variant = variant; C.stop_rule = h->stop_rule; C.max_iter = is_trunc ? h->trunc_steps : h->max_iter; C.kvalid = k;
    C.nocc = (double)nocc; C.tol = tol;
    C.mixed_head = h->mixed_head; C.mixed_reltr = h->mixed_reltr;
    C.mixed_phase = is_mixed ? (h->mixed_head > 0.0 ? 0 : 1) : 2;
    C.reltr_prev = INFINITY;
    if (variant == RFOE_VARIANT_SP2_ACCEL) { C.homo = h->homo; C.lumo = h->lumo; }   // images beta / bbar: control_begin
    CK(cudaMemcpyAsync(h->d_ctrl, &C, sizeof(Ctrl), cudaMemcpyHostToDevice, st));

    affine_map_kernel<<<hbm_grid(h, n), HBM_THREADS, 0, st>>>(Hp, k, n, ld, h->d_bounds, h->W[0], h->rows[0], h->rows[1]);
    h->launches++;
    CK(cudaGetLastError());
    h->hp->word = -1;
    control_kernel<<<1, 256, 0, st>>>(h->d_ctrl, 0, h->rows[0], h->rows[1], k, h->d_word, h->d_bounds);   // stops by itself on bad bounds
    h->launches++;
    CK(cudaGetLastError());
    // what the host makes of the prologue's results, once they are here (both paths)
    auto check_prologue = [&]() -> int {
        if (h->check_sym && h->hp->sym_flag) return RFOE_ERR_NOT_SYMMETRIC;
        const double emin = h->hp->bounds[0], emax = h->hp->bounds[1];
        S.eps_min = emin; S.eps_max = emax;
        if (!(isfinite(emin) && isfinite(emax) && emax > emin)) return RFOE_ERR_BAD_BOUNDS;
        // A-Z-RFOE: estimates outside the bounds would put the scaling factors 2/(2 - beta), 2/(1 + bbar) outside (0, 2)
        if (variant == RFOE_VARIANT_SP2_ACCEL && !(emin <= h->homo && h->lumo <= emax)) return RFOE_ERR_INVALID_ARG;
        return RFOE_OK;
    };
    h->sq_n = 0;
    int cur = 0;

    if (use_resident) {
        // --- the recursion without the host: one cooperative launch runs every step, the output pass picks the buffer by
        //     the parity of the device's step counter, and the host synchronises once, at the end
        ResidentPlan rp = {};
        rp.n = n; rp.ld = ld; rp.kvalid = k; rp.KT = n / SQ_BK;
        rp.n_tiles = h->n_tiles; rp.n_split = h->rs_n_split; rp.G = h->rs_G;
        rp.tile_cost = h->rs_tile_cost;
        rp.cost_total = (long long)h->n_tiles * rp.tile_cost;
        rp.tile_map = h->d_tiles; rp.split = h->d_split;
        rp.W0 = h->W[0]; rp.W1 = h->W[1]; rp.ws = h->ws;
        rp.rec0 = h->d_rec[0]; rp.rec1 = h->d_rec[1];
        rp.flags = h->d_flags; rp.dflags = h->d_flags + 256; rp.ctrl = h->d_ctrl; rp.timing = h->d_timing;
        CK(cudaMemsetAsync(h->d_flags, 0, RS_FLAG_WORDS * sizeof(unsigned), st));
        CK(cudaMemsetAsync(h->d_timing, 0, 8 * sizeof(unsigned long long), st));
        if (use_small) {
            const int bm = (n <= RT_MAX_N32) ? 32 : 64;
            CUtensorMap ts[2];
            for (int i = 0; i < 2; ++i)
                if ((rc = make_map(h, &ts[i], h->W[i], n, ld, bm)) != RFOE_OK) return fail(rc);
            SmallPlan sp = {};
            sp.n = n; sp.ld = ld; sp.kvalid = k; sp.mt = n / bm;
            sp.n_tiles = sp.mt * (sp.mt + 1) / 2;
            sp.W0 = h->W[0]; sp.W1 = h->W[1]; sp.rec0 = h->d_rec[0]; sp.rec1 = h->d_rec[1];
            sp.flags = h->d_flags; sp.ctrl = h->d_ctrl; sp.timing = h->d_timing;
            void* args[3] = {(void*)&ts[0], (void*)&ts[1], (void*)&sp};
            CK(cudaLaunchCooperativeKernel(bm == 32 ? (const void*)resident_small_kernel<32> : (const void*)resident_small_kernel<64>,
                                           dim3(sp.n_tiles), dim3(SQ_THREADS), args, RT_SMEM_BYTES, st));
        } else {
            void* args[3] = {(void*)&tm[0], (void*)&tm[1], (void*)&rp};
            // ranges of about a tile or more: the first holder finishes a cut tile (one grid barrier per step, resident_fin.cuh);
            // shorter ranges (tiles cut into many parts): all parts to the workspace, finished in bands (two barriers, resident.cuh)
            const long long units = (long long)h->n_tiles * rp.KT;
            const long long tile10 = (long long)h->rs_G * rp.KT;          // ten times a range, in tenths of a tile: units * 10 / tile10
            const bool fin = h->resident == 1 && units * 10 >= tile10 * RS_FIN_MIN_RANGE_TENTHS && units * 10 < tile10 * RS_FIN_MAX_RANGE_TENTHS;
            if (fin) {
                // the workspace as a matrix of 128-column tiles, one below the other: donated parts travel through the operand ring
                CUtensorMap tw;
                cuuint64_t dims[2] = {(cuuint64_t)SQ_BM, (cuuint64_t)(2 * h->rs_G) * SQ_BM};
                cuuint64_t strides[1] = {(cuuint64_t)SQ_BM * sizeof(double)};
                cuuint32_t box[2] = {(cuuint32_t)SQ_BK, (cuuint32_t)SQ_BM};
                cuuint32_t estr[2] = {1, 1};
                if (h->encode(&tw, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, h->ws, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                              CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
                    h->stats.cuda_error = (int)cudaErrorInvalidValue;
                    return fail(RFOE_ERR_CUDA);
                }
                void* fargs[4] = {(void*)&tm[0], (void*)&tm[1], (void*)&tw, (void*)&rp};
                h->rs_rec_dirty = 1;
                CK(cudaLaunchCooperativeKernel((const void*)resident_finisher_kernel, dim3(h->rs_G), dim3(SQ_THREADS), fargs, RS_SMEM_BYTES, st));
            } else {
                // band form: the tile records of cut tiles are never written and must read zero (the finisher form writes them)
                if (h->rs_rec_dirty) {
                    const size_t nrec = (size_t)h->n_tiles + (size_t)h->rs_G;
                    CK(cudaMemsetAsync(h->d_rec[0], 0, nrec * SQ_NPART * sizeof(double), st));
                    CK(cudaMemsetAsync(h->d_rec[1], 0, nrec * SQ_NPART * sizeof(double), st));
                    h->rs_rec_dirty = 0;
                }
                CK(cudaLaunchCooperativeKernel((const void*)resident_recursion_kernel, dim3(h->rs_G), dim3(SQ_THREADS), args, RS_SMEM_BYTES, st));
            }
        }
        h->launches++;
        copy_out_select_kernel<<<hbm_grid(h, k), HBM_THREADS, 0, st>>>(h->W[0], h->W[1], &h->d_ctrl->step, k, ld, Hp, P, h->rows[0]);
        h->launches++;
        CK(cudaGetLastError());
        sum_rows_kernel<<<1, 256, 0, st>>>(h->rows[0], k, &h->d_ctrl->tr_PH);
        h->launches++;
        CK(cudaGetLastError());
        CK(cudaEventRecord(h->ev1, st));
        CK(cudaMemcpyAsync(&C, h->d_ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
        CK(cudaMemcpyAsync((void*)h->hp->scalars, h->d_timing, 8 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
        if ((rc = check_prologue()) != RFOE_OK) return fail(rc);
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, h->ev0, h->ev1));
        unsigned long long tim[8];
        memcpy(tim, (const void*)h->hp->scalars, sizeof(tim));
        const unsigned long long step_ns = tim[0];
        for (int i = 0; i < 5; ++i) S.resident_phase_ms[i] = (double)tim[1 + i] * 1e-6;
        S.iterations = C.step; S.multiplications = C.multiplications; S.mcweeny_steps = C.mcweeny_steps;
        S.fp32_steps = C.fp32_steps; S.converged = C.converged; S.tr_PH = C.tr_PH; S.device_ms = ms;
        S.gpu_launches = h->launches;
        S.square_launches = C.step;                  // squarings, all inside the one launch
        S.square_ms = (double)step_ns * 1e-6;        // CTA 0's %globaltimer around the steps
        S.resident = 1;
        const int ns = C.step;
        memcpy(S.t, C.ht, sizeof(double) * (ns + 1));
        memcpy(S.s, C.hs, sizeof(double) * (ns + 1));
        memcpy(S.e, C.he, sizeof(double) * ns);
        memcpy(S.reltr, C.hreltr, sizeof(double) * ns);
        memcpy(S.branch, C.branch, ns);
        S.branch[ns] = 0;
        S.status = C.converged ? RFOE_OK : RFOE_ERR_NOT_CONVERGED;
        return S.status;
    }

    CK(cudaStreamSynchronize(st));
    if ((rc = check_prologue()) != RFOE_OK) return fail(rc);

    // --- the recursion: one scalar (the action word) crosses to the host per step ----------------
    int action = h->hp->word;
    while (action != ACT_STOP) {
        const int nxt = cur ^ 1;
        if (action == ACT_SP2 && sh && sh->barrier) {
            // the epilogues of this rank's tiles store X_{n+1} and the records into EVERY rank's arrays (peer memory);
            // after the barrier every rank holds the whole X_{n+1} and all records in global tile order
            if (t_count > 0) {
                CK(cudaEventRecord(h->sq_ev[2 * h->sq_n], st));
                CK(launch_sp2_range(h, tm[cur], h->W[cur], nullptr, n, ld, k, &h->d_ctrl->coef, nullptr, t_begin, t_count, plan, st,
                                    &psets[nxt], h->d_peers + nxt));
                CK(cudaEventRecord(h->sq_ev[2 * h->sq_n + 1], st));
                h->sq_n++;
            }
            if (sh->barrier(sh->user, stream) != 0) return fail(RFOE_ERR_CUDA);
            control_kernel<<<1, 256, 0, st>>>(h->d_ctrl, 1, h->part[nxt], h->part[nxt], h->n_tiles, h->d_word, nullptr);
        } else if (action == ACT_SP2 && sh) {
            // this rank's tiles (and their mirrors) -> W[nxt]; pack them with their records; ONE all-gather; unpack
            // the foreign tiles; the records, now in global tile order, feed the same control kernel on every rank
            if (t_count > 0) {
                CK(cudaEventRecord(h->sq_ev[2 * h->sq_n], st));
                CK(launch_sp2_range(h, tm[cur], h->W[cur], h->W[nxt], n, ld, k, &h->d_ctrl->coef,
                                    h->sh_send + (size_t)c_max * TILE_ELEMS, t_begin, t_count, plan, st));
                CK(cudaEventRecord(h->sq_ev[2 * h->sq_n + 1], st));
                h->sq_n++;
                pack_tiles_kernel<<<t_count, 256, 0, st>>>(h->W[nxt], ld, h->d_tiles + t_begin, h->sh_send);
                h->launches++;
                CK(cudaGetLastError());
            }
            if (sh->allgather(sh->user, h->sh_send, h->sh_recv, (int64_t)(rank_stride * sizeof(double)), stream) != 0)
                return fail(RFOE_ERR_CUDA);
            unpack_tiles_kernel<<<h->n_tiles, 256, 0, st>>>(h->sh_recv, rank_stride, c_max, h->d_tiles, t_begin, t_count, h->W[nxt], ld,
                                                           h->sh_parts);
            h->launches++;
            CK(cudaGetLastError());
            control_kernel<<<1, 256, 0, st>>>(h->d_ctrl, 1, h->sh_parts, h->sh_parts, h->n_tiles, h->d_word, nullptr);
        } else if (action == ACT_SP2) {
            CK(cudaEventRecord(h->sq_ev[2 * h->sq_n], st));
            CK(launch_sp2_range(h, tm[cur], h->W[cur], h->W[nxt], n, ld, k, &h->d_ctrl->coef, h->part[0], 0, h->n_tiles, plan, st));
            CK(cudaEventRecord(h->sq_ev[2 * h->sq_n + 1], st));
            h->sq_n++;
            control_kernel<<<1, 256, 0, st>>>(h->d_ctrl, 1, h->part[0], h->part[0], h->n_tiles, h->d_word, nullptr);
        } else if (action == ACT_SP2_FP32) {
            CK(cudaEventRecord(h->sq_ev[2 * h->sq_n], st));
            CK(launch_square_reduced(h, tmF[0], tmF[1], h->W[cur], h->W[nxt], n, ld, k, &h->d_ctrl->t, &h->d_ctrl->coef, h->part[0], st));
            CK(cudaEventRecord(h->sq_ev[2 * h->sq_n + 1], st));
            h->sq_n++;
            control_kernel<<<1, 256, 0, st>>>(h->d_ctrl, 1, h->part[0], h->part[0], 2 * h->n_pairs, h->d_word, nullptr);
        } else if (action == ACT_MCWEENY) {
            CK(timed_square<false>(h, tm[cur], tm[cur], h->W[cur], h->W[2], n, ld, k, &h->d_ctrl->coef, h->part[0], st));
            CK(timed_square<true>(h, tm[2], tm[cur], h->W[2], h->W[nxt], n, ld, k, &h->d_ctrl->coef_aux, h->part[1], st));
            control_kernel<<<1, 256, 0, st>>>(h->d_ctrl, 1, h->part[1], h->part[0], h->n_tiles, h->d_word, nullptr);
        } else {
            return fail(RFOE_ERR_UNSUPPORTED);
        }
        h->launches++;
        CK(cudaGetLastError());
        CK(cudaStreamSynchronize(st));
        action = h->hp->word;
        cur = nxt;
    }

    // --- output pass: P and tr(P H) ---------------------------------------------------------------
    copy_out_kernel<<<hbm_grid(h, k), HBM_THREADS, 0, st>>>(h->W[cur], k, ld, Hp, P, h->rows[0]);
    h->launches++;
    CK(cudaGetLastError());
    sum_rows_kernel<<<1, 256, 0, st>>>(h->rows[0], k, &h->d_ctrl->tr_PH);
    h->launches++;
    CK(cudaGetLastError());
    CK(cudaEventRecord(h->ev1, st));
    CK(cudaMemcpyAsync(&C, h->d_ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    float ms = 0.f;
    CK(cudaEventElapsedTime(&ms, h->ev0, h->ev1));

    S.iterations = C.step; S.multiplications = C.multiplications; S.mcweeny_steps = C.mcweeny_steps;
    S.fp32_steps = C.fp32_steps; S.converged = C.converged; S.tr_PH = C.tr_PH; S.device_ms = ms;
    S.gpu_launches = h->launches;
    S.square_launches = h->sq_n;
    for (int i = 0; i < h->sq_n; ++i) {
        float sq = 0.f;
        CK(cudaEventElapsedTime(&sq, h->sq_ev[2 * i], h->sq_ev[2 * i + 1]));
        S.square_ms += sq;
    }
    const int ns = C.step;
    memcpy(S.t, C.ht, sizeof(double) * (ns + 1));
    memcpy(S.s, C.hs, sizeof(double) * (ns + 1));
    memcpy(S.e, C.he, sizeof(double) * ns);
    memcpy(S.reltr, C.hreltr, sizeof(double) * ns);
    memcpy(S.branch, C.branch, ns);
    S.branch[ns] = 0;
    S.status = C.converged ? RFOE_OK : RFOE_ERR_NOT_CONVERGED;
    return S.status;
}

extern "C" int rfoe_expand(rfoe_handle_t h, const double* Hp, int64_t k, int64_t nocc, int variant, double tol, double* P,
                           rfoe_stream_t stream)
{
    return expand_impl(h, Hp, k, nocc, variant, tol, P, stream, nullptr);
}

// Many independent problems on one GPU: one host thread per handle, problems taken from a shared counter (rfoe.h).
extern "C" int rfoe_expand_many(const rfoe_handle_t* handles, const rfoe_stream_t* streams, int n_handles, int n_problems,
                                const double* const* Hp, const int64_t* k, const int64_t* nocc, int variant, const double* tol,
                                double* const* P, int* status, rfoe_stats_t* stats)
{
    if (!handles || !streams || n_handles < 1 || n_problems < 0) return RFOE_ERR_INVALID_ARG;
    if (n_problems > 0 && (!Hp || !k || !nocc || !tol || !P)) return RFOE_ERR_INVALID_ARG;
    for (int i = 0; i < n_handles; ++i) {
        if (!handles[i]) return RFOE_ERR_INVALID_ARG;
        for (int j = 0; j < i; ++j)
            if (handles[j] == handles[i]) return RFOE_ERR_INVALID_ARG;
    }
    std::vector<int> rcs((size_t)n_problems, RFOE_OK);
    std::atomic<int> next(0);
    auto worker = [&](int i) {
        for (;;) {
            const int j = next.fetch_add(1);
            if (j >= n_problems) break;
            rcs[j] = expand_impl(handles[i], Hp[j], k[j], nocc[j], variant, tol[j], P[j], streams[i], nullptr);
            if (stats) stats[j] = handles[i]->stats;
        }
    };
    const int n_threads = n_handles < n_problems ? n_handles : n_problems;
    for (int i = 0; i < n_handles; ++i) handles[i]->side_by_side = (n_threads > 1);
    std::vector<std::thread> pool;
    try {
        for (int i = 1; i < n_threads; ++i) pool.emplace_back(worker, i);
    } catch (...) {
        // fewer threads than asked for: the remaining handles stay idle, the problems are still all taken
    }
    if (n_threads > 0) worker(0);
    for (std::thread& t : pool) t.join();
    for (int i = 0; i < n_handles; ++i) handles[i]->side_by_side = 0;
    int first = RFOE_OK;
    for (int j = 0; j < n_problems; ++j) {
        if (status) status[j] = rcs[j];
        if (first == RFOE_OK && rcs[j] != RFOE_OK) first = rcs[j];
    }
    return first;
}

extern "C" int rfoe_expand_sharded(rfoe_handle_t h, const double* Hp, int64_t k, int64_t nocc, int variant, double tol, double* P,
                                   int rank, int world, rfoe_allgather_fn allgather, void* user, rfoe_stream_t stream)
{
    if (world < 1 || rank < 0 || rank >= world || !allgather) return RFOE_ERR_INVALID_ARG;
    ShardCtx sh = {rank, world, allgather, nullptr, user};
    return expand_impl(h, Hp, k, nocc, variant, tol, P, stream, &sh);
}

// ---- sharded expansion over peer memory ------------------------------------------------------------------
extern "C" int rfoe_shard_local_ptrs(rfoe_handle_t h, void** ptrs)
{
    if (!h || !ptrs) return RFOE_ERR_INVALID_ARG;
    ptrs[0] = h->W[0]; ptrs[1] = h->W[1]; ptrs[2] = h->part[0]; ptrs[3] = h->part[1];
    return RFOE_OK;
}

extern "C" int rfoe_shard_set_peers(rfoe_handle_t h, int rank, int world, void* const* ptrs)
{
    if (!h || !ptrs || world < 1 || world > SQ_MAX_PEERS || rank < 0 || rank >= world) return RFOE_ERR_INVALID_ARG;
    if (ptrs[4 * rank] != h->W[0] || ptrs[4 * rank + 1] != h->W[1] || ptrs[4 * rank + 2] != h->part[0] ||
        ptrs[4 * rank + 3] != h->part[1])
        return RFOE_ERR_INVALID_ARG;
    for (int d = 0; d < world; ++d) {
        for (int q = 0; q < 4; ++q)
            if (!ptrs[4 * d + q]) return RFOE_ERR_INVALID_ARG;
        h->peer_W[0][d] = (double*)ptrs[4 * d];
        h->peer_W[1][d] = (double*)ptrs[4 * d + 1];
        h->peer_rec[0][d] = (double*)ptrs[4 * d + 2];
        h->peer_rec[1][d] = (double*)ptrs[4 * d + 3];
    }
    h->p2p_world = world;
    h->p2p_rank = rank;
    return RFOE_OK;
}

extern "C" int rfoe_shard_ipc_export(rfoe_handle_t h, void* handles)
{
    if (!h || !handles) return RFOE_ERR_INVALID_ARG;
    static_assert(sizeof(cudaIpcMemHandle_t) == RFOE_IPC_HANDLE_BYTES, "IPC handle size");
    cudaIpcMemHandle_t* out = (cudaIpcMemHandle_t*)handles;
    CK(cudaSetDevice(h->device));
    CK(cudaIpcGetMemHandle(&out[0], h->W[0]));
    CK(cudaIpcGetMemHandle(&out[1], h->W[1]));
    CK(cudaIpcGetMemHandle(&out[2], h->part[0]));
    CK(cudaIpcGetMemHandle(&out[3], h->part[1]));
    return RFOE_OK;
}

extern "C" int rfoe_shard_ipc_import(rfoe_handle_t h, int rank, int world, const void* handles)
{
    if (!h || !handles || world < 1 || world > SQ_MAX_PEERS || rank < 0 || rank >= world) return RFOE_ERR_INVALID_ARG;
    const cudaIpcMemHandle_t* in = (const cudaIpcMemHandle_t*)handles;
    CK(cudaSetDevice(h->device));
    for (int i = 0; i < h->n_ipc_opened; ++i) cudaIpcCloseMemHandle(h->ipc_opened[i]);
    h->n_ipc_opened = 0;
    void* ptrs[4 * SQ_MAX_PEERS];
    for (int d = 0; d < world; ++d) {
        if (d == rank) { ptrs[4 * d] = h->W[0]; ptrs[4 * d + 1] = h->W[1]; ptrs[4 * d + 2] = h->part[0]; ptrs[4 * d + 3] = h->part[1]; continue; }
        for (int q = 0; q < 4; ++q) {
            void* p = nullptr;
            cudaError_t e = cudaIpcOpenMemHandle(&p, in[4 * d + q], cudaIpcMemLazyEnablePeerAccess);
            if (e == cudaSuccess) {
                // preflight: the buffer lives on the peer's device; this device must be able to reach it over P2P
                h->ipc_opened[h->n_ipc_opened++] = p;
                cudaPointerAttributes attr;
                int can = 1;
                e = cudaPointerGetAttributes(&attr, p);
                if (e == cudaSuccess && attr.device != h->device) e = cudaDeviceCanAccessPeer(&can, h->device, attr.device);
                if (e == cudaSuccess && !can) e = cudaErrorPeerAccessUnsupported;
            }
            if (e != cudaSuccess) {
                cudaGetLastError();
                for (int i = 0; i < h->n_ipc_opened; ++i) cudaIpcCloseMemHandle(h->ipc_opened[i]);
                h->n_ipc_opened = 0;
                h->p2p_world = 0;
                h->stats.cuda_error = (int)e;
                h->stats.status = RFOE_ERR_NO_PEER_ACCESS;
                return RFOE_ERR_NO_PEER_ACCESS;
            }
            ptrs[4 * d + q] = p;
        }
    }
    return rfoe_shard_set_peers(h, rank, world, ptrs);
}

extern "C" int rfoe_expand_sharded_p2p(rfoe_handle_t h, const double* Hp, int64_t k, int64_t nocc, int variant, double tol, double* P,
                                       rfoe_barrier_fn barrier, void* user, rfoe_stream_t stream)
{
    if (!h || !barrier || h->p2p_world < 1) return RFOE_ERR_INVALID_ARG;
    ShardCtx sh = {h->p2p_rank, h->p2p_world, nullptr, barrier, user};
    return expand_impl(h, Hp, k, nocc, variant, tol, P, stream, &sh);
}

// ---------------------------------------------------------------------------------------------
// FP64 tensor-pipe issue-rate probe (probe.cuh): a short calibration launch sizes the timed one for ~ms milliseconds
extern "C" int rfoe_probe_fp64_peak(rfoe_handle_t h, double ms, double* tflops, rfoe_stream_t stream)
{
    if (!h || !tflops || !(ms >= 1.0 && ms <= 10000.0)) return RFOE_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    h->launches = 0;
    h->stats.cuda_error = 0;
    CK(cudaSetDevice(h->device));
    h->hp->scalars[0] = 1e-3; h->hp->scalars[1] = -1e-3;
    CK(cudaMemcpyAsync(h->d_scalars, (void*)h->hp->scalars, 2 * sizeof(double), cudaMemcpyHostToDevice, st));
    const double flops_per_iter = (double)h->sm_count * (PROBE_THREADS / 32) * PROBE_FLOPS_PER_WARP_ITER;
    long long iters = 4096;
    float t = 0.f;
    for (int pass = 0; pass < 2; ++pass) {
        CK(cudaEventRecord(h->ev0, st));
        fp64_peak_probe_kernel<<<h->sm_count, PROBE_THREADS, 0, st>>>(iters, h->d_scalars, h->d_scalars + 4);
        h->launches++;
        CK(cudaGetLastError());
        CK(cudaEventRecord(h->ev1, st));
        CK(cudaStreamSynchronize(st));
        CK(cudaEventElapsedTime(&t, h->ev0, h->ev1));
        if (pass == 0) {
            if (!(t > 0.f)) return RFOE_ERR_CUDA;
            iters = (long long)((double)iters * ms / (double)t) + 1;
        }
    }
    *tflops = flops_per_iter * (double)iters / ((double)t * 1e-3) / 1e12;
    h->stats.gpu_launches = h->launches;
    h->stats.status = RFOE_OK;
    return RFOE_OK;
}

// ---------------------------------------------------------------------------------------------
// single products (kernel-level entry points for tests and roofline timing)
static int single_product(rfoe_handle_s* h, const double* A, const double* B, int64_t k64, double c2, double c1, double c0,
                          double* Cout, double* scalars, float* kernel_ms, cudaStream_t st, bool reduced = false)
{
    if (!h || !A || !Cout || k64 < 1 || k64 > h->k_max) return RFOE_ERR_INVALID_ARG;
    const bool two = (B != nullptr);
    const int k = (int)k64, n = round_up(k, SQ_BM), ld = n + SQ_PAD, m = n / SQ_BM;
    int rc;
    h->launches = 0;
    h->stats.cuda_error = 0;
    CK(cudaSetDevice(h->device));
    if ((rc = ensure_third(h)) != RFOE_OK) return rc;
    if ((rc = ensure_tiles(h, m, st)) != RFOE_OK) return rc;
    CUtensorMap tm[3], tmF[2];
    for (int i = 0; i < 3; ++i)
        if ((rc = make_map(h, &tm[i], h->W[i], n, ld)) != RFOE_OK) return rc;
    if (reduced) {
        if ((rc = ensure_parts(h)) != RFOE_OK) return rc;
        for (int i = 0; i < 2; ++i)
            if ((rc = make_map_parts(h, &tmF[i], h->F[i], n, n + TQ_PAD)) != RFOE_OK) return rc;
    }
    pad_copy_kernel<<<hbm_grid(h, n), HBM_THREADS, 0, st>>>(A, k, n, ld, h->W[0]);
    h->launches++;
    if (two) {
        pad_copy_kernel<<<hbm_grid(h, n), HBM_THREADS, 0, st>>>(B, k, n, ld, h->W[1]);
        h->launches++;
    }
    CK(cudaGetLastError());
    Ctrl& C = h->hp->ctrl;
    C.coef = StepCoef{c2, c1, c0};
    CK(cudaMemcpyAsync(&h->d_ctrl->coef, &C.coef, sizeof(StepCoef), cudaMemcpyHostToDevice, st));
    CK(cudaEventRecord(h->ev0, st));
    if (reduced) {
        diag_sum_kernel<<<1, 256, 0, st>>>(h->W[0], k, ld, h->d_scalars + 7);      // Tr X for the shift d = Tr X / k
        h->launches++;
        CK(launch_square_reduced(h, tmF[0], tmF[1], h->W[0], h->W[2], n, ld, k, h->d_scalars + 7, &h->d_ctrl->coef, h->part[0], st));
    }
    else if (two) CK(launch_square<true>(h, tm[0], tm[1], h->W[0], h->W[2], n, ld, k, &h->d_ctrl->coef, h->part[0], st));
    else {
        const TailPlan plan = plan_tail(h->n_tiles, n / SQ_BK, h->sm_count);
        if ((rc = ensure_tail_ws(h, h->n_tiles, plan)) != RFOE_OK) return rc;
        CK(launch_sp2_range(h, tm[0], h->W[0], h->W[2], n, ld, k, &h->d_ctrl->coef, h->part[0], 0, h->n_tiles, plan, st));
    }
    CK(cudaEventRecord(h->ev1, st));
    sum_partials_kernel<<<1, 256, 0, st>>>(h->part[0], reduced ? 2 * h->n_pairs : h->n_tiles, h->d_scalars);
    h->launches++;
    copy_out_kernel<<<hbm_grid(h, k), HBM_THREADS, 0, st>>>(h->W[2], k, ld, nullptr, Cout, nullptr);
    h->launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync((void*)h->hp->scalars, h->d_scalars, 5 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (scalars) for (int i = 0; i < 5; ++i) scalars[i] = h->hp->scalars[i];
    if (kernel_ms) CK(cudaEventElapsedTime(kernel_ms, h->ev0, h->ev1));
    h->stats.gpu_launches = h->launches;
    return RFOE_OK;
}

extern "C" int rfoe_square(rfoe_handle_t h, const double* X, int64_t k, double c2, double c1, double c0, double* Xout,
                           double* scalars, float* kernel_ms, rfoe_stream_t stream)
{
    return single_product(h, X, nullptr, k, c2, c1, c0, Xout, scalars, kernel_ms, (cudaStream_t)stream);
}

extern "C" int rfoe_square_reduced(rfoe_handle_t h, const double* X, int64_t k, double c2, double c1, double c0, double* Xout,
                                   double* scalars, float* kernel_ms, rfoe_stream_t stream)
{
    return single_product(h, X, nullptr, k, c2, c1, c0, Xout, scalars, kernel_ms, (cudaStream_t)stream, true);
}

extern "C" int rfoe_symm_product(rfoe_handle_t h, const double* A, const double* B, int64_t k, double c2, double c1, double c0,
                                 double* Cout, double* scalars, float* kernel_ms, rfoe_stream_t stream)
{
    if (!B) return RFOE_ERR_INVALID_ARG;
    return single_product(h, A, B, k, c2, c1, c0, Cout, scalars, kernel_ms, (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------
// steps either side of the expansion (NEXT-4): Rayleigh-Ritz projection before, P applied to the basis after
static int make_map_rect(rfoe_handle_s* h, CUtensorMap* map, const double* base, int64_t M, int64_t k, int64_t ld, int box_rows)
{
    cuuint64_t dims[2] = {(cuuint64_t)M, (cuuint64_t)k};
    cuuint64_t strides[1] = {(cuuint64_t)ld * sizeof(double)};
    cuuint32_t box[2] = {(cuuint32_t)SQ_BK, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = h->encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(base), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);   // out-of-range rows / columns read as zero
    if (r != CUDA_SUCCESS) {
        h->stats.cuda_error = (int)cudaErrorInvalidValue;
        return RFOE_ERR_CUDA;
    }
    return RFOE_OK;
}

static int ensure_ws(rfoe_handle_s* h, size_t bytes)
{
    if (h->ws_bytes >= bytes) return RFOE_OK;
    if (h->ws) { cudaFree(h->ws); h->ws = nullptr; h->ws_bytes = 0; }
    if (cudaMalloc(&h->ws, bytes) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    h->ws_bytes = bytes;
    return RFOE_OK;
}

static int ensure_tail_ws(rfoe_handle_s* h, int n_tiles, const TailPlan& plan)
{
    const size_t T = (size_t)(n_tiles - plan.n_main);
    return T ? ensure_ws(h, T * plan.slices * SQ_BM * SQ_BM * sizeof(double)) : RFOE_OK;
}

static bool rect_args_ok(const rfoe_handle_s* h, const void* a, int64_t k, int64_t M, int64_t ld)
{
    return a && k >= 1 && k <= h->k_max && M >= 1 && M <= (int64_t)1 << 30 && ld >= M && (ld & 1) == 0 &&
           (reinterpret_cast<uintptr_t>(a) & 15) == 0;
}

// number of K-slices: the smallest S <= 16 whose tiles x slices fill the SMs to >= 99 % in whole waves (else the best)
static void choose_slices(int n_tiles, int kt_total, int sm_count, int* n_slices, int* kt_per)
{
    int best_s = 1, best_per = kt_total;
    double best_e = -1.0;
    for (int s = 1; s <= 16; ++s) {
        const int per = (kt_total + s - 1) / s;
        if (s > 1 && per < 32) break;
        const int eff_s = (kt_total + per - 1) / per;
        const long long units = (long long)n_tiles * eff_s;
        const long long waves = (units + sm_count - 1) / sm_count;
        const double e = (double)units / (double)(waves * sm_count);
        if (e > best_e + 1e-12) { best_e = e; best_s = eff_s; best_per = per; }
        if (e >= 0.99) break;
    }
    *n_slices = best_s;
    *kt_per = best_per;
}

extern "C" int rfoe_project(rfoe_handle_t h, const double* Psi, const double* HPsi, int64_t k64, int64_t M, int64_t ld,
                            double* Hp, double* scalars, float* kernel_ms, rfoe_stream_t stream)
{
    if (!h || !Hp || !rect_args_ok(h, Psi, k64, M, ld) || !rect_args_ok(h, HPsi, k64, M, ld)) return RFOE_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int k = (int)k64, n = round_up(k, SQ_BM), m = n / SQ_BM;
    int rc;
    h->launches = 0;
    h->stats.cuda_error = 0;
    CK(cudaSetDevice(h->device));
    if ((rc = ensure_tiles(h, m, st)) != RFOE_OK) return rc;
    const int kt_total = (int)((M + SQ_BK - 1) / SQ_BK);
    int n_slices, kt_per;
    choose_slices(h->n_tiles, kt_total, h->sm_count, &n_slices, &kt_per);
    if ((rc = ensure_ws(h, (size_t)n_slices * h->n_tiles * SQ_BM * SQ_BM * sizeof(double))) != RFOE_OK) return rc;
    CUtensorMap tmA, tmB;
    if ((rc = make_map_rect(h, &tmA, Psi, M, k, ld, SQ_BM)) != RFOE_OK) return rc;
    if ((rc = make_map_rect(h, &tmB, HPsi, M, k, ld, SQ_BM)) != RFOE_OK) return rc;
    CK(cudaEventRecord(h->ev0, st));
    sym_square_kernel<2><<<dim3(h->n_tiles, n_slices), SQ_THREADS, SQ_SMEM_BYTES, st>>>(tmA, tmB, nullptr, h->ws, kt_total * SQ_BK, SQ_BM, k,
                                                                                      nullptr, h->d_tiles, nullptr, kt_per);
    h->launches++;
    CK(cudaGetLastError());
    project_reduce_kernel<<<h->n_tiles, 256, 0, st>>>(h->ws, n_slices, h->n_tiles, h->d_tiles, k, Hp, h->part[0]);
    h->launches++;
    CK(cudaGetLastError());
    CK(cudaEventRecord(h->ev1, st));
    sum_partials_kernel<<<1, 256, 0, st>>>(h->part[0], h->n_tiles, h->d_scalars);
    h->launches++;
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync((void*)h->hp->scalars, h->d_scalars, 5 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (scalars) { scalars[0] = h->hp->scalars[0]; scalars[1] = h->hp->scalars[1]; }
    if (kernel_ms) CK(cudaEventElapsedTime(kernel_ms, h->ev0, h->ev1));
    h->stats.gpu_launches = h->launches;
    h->stats.status = RFOE_OK;
    return RFOE_OK;
}

extern "C" int rfoe_apply(rfoe_handle_t h, const double* P, const double* Psi, int64_t k64, int64_t M, int64_t ld, double* Y,
                          int64_t ldy, double* rho, float* kernel_ms, rfoe_stream_t stream)
{
    if (!h || !P || !Y || !rect_args_ok(h, Psi, k64, M, ld) || ldy < M) return RFOE_ERR_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const int k = (int)k64, n = round_up(k, SQ_BM), ldw = n + SQ_PAD, m = n / SQ_BM;
    const int64_t tiles_m = (M + AP_BN - 1) / AP_BN;
    if (tiles_m > 65535) return RFOE_ERR_INVALID_ARG;
    int rc;
    h->launches = 0;
    h->stats.cuda_error = 0;
    CK(cudaSetDevice(h->device));
    CUtensorMap tmP, tmPsi;
    if ((rc = make_map(h, &tmP, h->W[0], n, ldw)) != RFOE_OK) return rc;
    if ((rc = make_map_rect(h, &tmPsi, Psi, M, k, ld, SQ_BK)) != RFOE_OK) return rc;
    int n_slices = 1, rows_per = k;
    const int64_t col_blocks = (M + 255) / 256;
    if (rho) {
        int64_t want = (h->sm_count * 8 + col_blocks - 1) / col_blocks;
        if (want > 64) want = 64;
        if (want > k) want = k;
        if (want < 1) want = 1;
        rows_per = (int)((k + want - 1) / want);
        n_slices = (k + rows_per - 1) / rows_per;
        if ((rc = ensure_ws(h, (size_t)n_slices * (size_t)M * sizeof(double))) != RFOE_OK) return rc;
    }
    pad_copy_kernel<<<hbm_grid(h, n), HBM_THREADS, 0, st>>>(P, k, n, ldw, h->W[0]);
    h->launches++;
    CK(cudaGetLastError());
    const int vec_ok = ((ldy & 1) == 0) && ((reinterpret_cast<uintptr_t>(Y) & 15) == 0);
    CK(cudaEventRecord(h->ev0, st));
    apply_kernel<<<dim3(m, (unsigned)tiles_m), SQ_THREADS, AP_SMEM_BYTES, st>>>(tmP, tmPsi, Y, k, (long long)M, (long long)ldy, n / SQ_BK, vec_ok);
    h->launches++;
    CK(cudaGetLastError());
    CK(cudaEventRecord(h->ev1, st));
    if (rho) {
        density_partial_kernel<<<dim3((unsigned)col_blocks, n_slices), 256, 0, st>>>(Psi, (long long)ld, Y, (long long)ldy, k, (long long)M,
                                                                                   rows_per, h->ws);
        h->launches++;
        density_reduce_kernel<<<(unsigned)col_blocks, 256, 0, st>>>(h->ws, n_slices, (long long)M, rho);
        h->launches++;
        CK(cudaGetLastError());
    }
    CK(cudaStreamSynchronize(st));
    if (kernel_ms) CK(cudaEventElapsedTime(kernel_ms, h->ev0, h->ev1));
    h->stats.gpu_launches = h->launches;
    h->stats.status = RFOE_OK;
    return RFOE_OK;
}

// ---------------------------------------------------------------------------------------------
// end-to-end entry point with host buffers
extern "C" int rfoe_expand_host(rfoe_handle_t h, const double* Hp_host, int64_t k, int64_t nocc, int variant, double tol,
                                double* P_host, rfoe_stream_t stream)
{
    int rc = check_common(h, Hp_host, P_host, k);
    if (rc != RFOE_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaSetDevice(h->device));
    const size_t cap = (size_t)h->k_max * h->k_max * sizeof(double);
    if (!h->stage_H && cudaMalloc(&h->stage_H, cap) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    if (!h->stage_P && cudaMalloc(&h->stage_P, cap) != cudaSuccess) { cudaGetLastError(); return RFOE_ERR_ALLOC; }
    const size_t bytes = (size_t)k * k * sizeof(double);
    CK(cudaMemcpyAsync(h->stage_H, Hp_host, bytes, cudaMemcpyHostToDevice, st));
    rc = rfoe_expand(h, h->stage_H, k, nocc, variant, tol, h->stage_P, stream);
    if (rc != RFOE_OK && rc != RFOE_ERR_NOT_CONVERGED) return rc;
    CK(cudaMemcpyAsync(P_host, h->stage_P, bytes, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    return rc;
}
