// Tighter spectral bounds than Gershgorin's (row A1, optional; reading R3b): m steps of the Lanczos
// recursion.  The paper only says "spectral bound estimates"; on a dense rotated H^p Gershgorin
// over-estimates the spectral width ~50x at k=16384 (radius ~0.8 sigma sqrt(k)), which costs SP2 about 18 of its 56 squarings;
// emin = theta_min(T_m) - beta_m, emax = theta_max(T_m) + beta_m is within 1.5x of the true width after m = 24
// matrix-vector products (8 k^2 bytes each, HBM-bound).  Everything stays on the device: the recursion's scalars
// live in a small state block, the extreme eigenvalues of T_m come from a bisection on its Sturm count.
//   v_0 = s / ||s||, s_i = hash(i) - 1/2;  w = H v_j;  alpha_j = v_j . w;  w -= alpha_j v_j + beta_j v_{j-1};
//   beta_{j+1} = ||w||;  v_{j+1} = w / beta_{j+1}
#pragma once
#include "hbm_kernels.cuh"

namespace rfoe {

constexpr int LZ_MAX_STEPS = 64;

struct LanczosState {
    double alpha[LZ_MAX_STEPS];
    double beta[LZ_MAX_STEPS + 1];   // beta[0] = 0
    double norm0;                    // ||s||
    int steps;                       // steps completed
    int done;                        // set when beta_{j+1} vanished (invariant subspace): later kernels do nothing
};

__device__ __forceinline__ double lanczos_start(uint32_t i)
{
    uint32_t x = i * 2654435761u + 0x9E3779B9u;
    x ^= x >> 16; x *= 0x85EBCA6Bu; x ^= x >> 13; x *= 0xC2B2AE35u; x ^= x >> 16;
    return (double)x * (1.0 / 4294967296.0) - 0.5;
}

// fixed-order sum of n values by one block (result in every thread)
__device__ inline double lz_block_sum(const double* __restrict__ p, int n, double* sh)
{
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) v += p[i];
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

// v <- s (unnormalised), vp <- 0, part[block] = sum of s_i^2 over the block's elements; state reset by block 0
__global__ void __launch_bounds__(256)
lanczos_init_kernel(double* __restrict__ v, double* __restrict__ vp, int k, double* __restrict__ part, LanczosState* __restrict__ st)
{
    __shared__ double sh[256];
    double acc = 0.0;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < k; i += gridDim.x * 256) {
        const double s = lanczos_start((uint32_t)i);
        v[i] = s;
        vp[i] = 0.0;
        acc = fma(s, s, acc);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int m = 128; m >= 1; m >>= 1) {
        if ((int)threadIdx.x < m) sh[threadIdx.x] += sh[threadIdx.x + m];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        part[blockIdx.x] = sh[0];
        if (blockIdx.x == 0) { st->beta[0] = 0.0; st->steps = 0; st->done = 0; }
    }
}

// w = H (v * scale) with scale = 1 / sqrt(sum part[0..n_part)) on the first step (normalises v_0 on the fly and
// stores the normalised vector back) and 1 afterwards; row_vw[i] = v_i w_i.  One warp per row, 512-byte runs.
__global__ void __launch_bounds__(HBM_THREADS)
lanczos_symv_kernel(const double* __restrict__ H, int k, double* __restrict__ v, double* __restrict__ w,
                    double* __restrict__ row_vw, const double* __restrict__ part, int n_part, int first,
                    const LanczosState* __restrict__ st)
{
    if (st->done) return;
    __shared__ double sh[HBM_THREADS];
    double scale = 1.0;
    if (first) scale = 1.0 / sqrt(lz_block_sum(part, n_part, sh));
    const int lane = threadIdx.x & 31;
    const int wglobal = blockIdx.x * HBM_WARPS + (threadIdx.x >> 5);
    const int wtotal = gridDim.x * HBM_WARPS;
    const bool vec = ((k & 1) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    for (int i = wglobal; i < k; i += wtotal) {
        const double* row = H + (size_t)i * k;
        double r0 = 0.0, r1 = 0.0, r2 = 0.0, r3 = 0.0;
        if (vec) {
            const double2* row2 = reinterpret_cast<const double2*>(row);
            const double2* v2 = reinterpret_cast<const double2*>(v);
            const int n2 = k >> 1;
            int j = lane;
            for (; j + 96 < n2; j += 128) {
                const double2 a = row2[j], b = row2[j + 32], c = row2[j + 64], d = row2[j + 96];
                const double2 va = v2[j], vb = v2[j + 32], vc = v2[j + 64], vd = v2[j + 96];
                r0 = fma(a.x, va.x, fma(a.y, va.y, r0));
                r1 = fma(b.x, vb.x, fma(b.y, vb.y, r1));
                r2 = fma(c.x, vc.x, fma(c.y, vc.y, r2));
                r3 = fma(d.x, vd.x, fma(d.y, vd.y, r3));
            }
            for (; j < n2; j += 32) {
                const double2 a = row2[j], va = v2[j];
                r0 = fma(a.x, va.x, fma(a.y, va.y, r0));
            }
        } else {
            for (int j = lane; j < k; j += 32) r0 = fma(row[j], v[j], r0);
        }
        const double r = warp_sum((r0 + r1) + (r2 + r3)) * scale;
        if (lane == 0) {
            w[i] = r;
            row_vw[i] = (v[i] * scale) * r;
        }
    }
}

// first step only, after the product: v <- v / ||s|| (the product above used the scale on the fly)
__global__ void __launch_bounds__(256)
lanczos_normalise_kernel(double* __restrict__ v, int k, const double* __restrict__ part, int n_part, LanczosState* __restrict__ st)
{
    __shared__ double sh[256];
    const double nrm = sqrt(lz_block_sum(part, n_part, sh));
    for (int i = blockIdx.x * 256 + threadIdx.x; i < k; i += gridDim.x * 256) v[i] = v[i] / nrm;
    if (blockIdx.x == 0 && threadIdx.x == 0) st->norm0 = nrm;
}

// alpha_j = sum_i row_vw[i] (every block computes it, fixed order); w <- (w - alpha v) - beta_j vp;
// part[block] = sum of w_i^2 over the block's elements
__global__ void __launch_bounds__(256)
lanczos_update_kernel(double* __restrict__ w, const double* __restrict__ v, const double* __restrict__ vp, int k,
                      const double* __restrict__ row_vw, int j, double* __restrict__ part, LanczosState* __restrict__ st)
{
    if (st->done) return;
    __shared__ double sh[256];
    const double alpha = lz_block_sum(row_vw, k, sh);
    const double beta = st->beta[j];
    double acc = 0.0;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < k; i += gridDim.x * 256) {
        const double x = (w[i] - alpha * v[i]) - beta * vp[i];
        w[i] = x;
        acc = fma(x, x, acc);
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int m = 128; m >= 1; m >>= 1) {
        if ((int)threadIdx.x < m) sh[threadIdx.x] += sh[threadIdx.x + m];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        part[blockIdx.x] = sh[0];
        if (blockIdx.x == 0) st->alpha[j] = alpha;
    }
}

// beta_{j+1} = sqrt(sum part); vp <- v; v <- w / beta_{j+1}  (or: stop, invariant subspace)
// One block only publishes (the others recompute the same sum): run with a grid, state written by block 0 LAST is
// not needed -- every block derives `stop` from the same numbers, the flag is only for the later kernels.
__global__ void __launch_bounds__(256)
lanczos_next_kernel(double* __restrict__ v, double* __restrict__ vp, const double* __restrict__ w, int k,
                    const double* __restrict__ part, int n_part, int j, LanczosState* __restrict__ st)
{
    if (st->done) return;
    __shared__ double sh[256];
    const double beta1 = sqrt(lz_block_sum(part, n_part, sh));
    const bool stop = !(beta1 > 1e-14 * (fabs(st->alpha[j]) + st->beta[j]));
    if (!stop)
        for (int i = blockIdx.x * 256 + threadIdx.x; i < k; i += gridDim.x * 256) {
            vp[i] = v[i];
            v[i] = w[i] / beta1;
        }
    __syncthreads();
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) {
        st->beta[j + 1] = stop ? 0.0 : beta1;
        st->steps = j + 1;
    }
}

// the `done` flag may only be raised once no block of lanczos_next_kernel still reads it: a separate tiny kernel
__global__ void lanczos_flag_kernel(LanczosState* __restrict__ st, int j)
{
    if (st->done == 0 && st->steps == j + 1 && st->beta[j + 1] == 0.0) st->done = 1;
}

__device__ inline int lz_sturm(const double* a, const double* b, int m, double x)   // eigenvalues of T_m below x
{
    int cnt = 0;
    double q = 1.0;
    for (int i = 0; i < m; ++i) {
        q = a[i] - x - (i == 0 ? 0.0 : b[i] * b[i] / q);
        if (q == 0.0) q = 1e-300;
        if (q < 0.0) ++cnt;
    }
    return cnt;
}

// bounds[0] = theta_min(T) - beta_steps, bounds[1] = theta_max(T) + beta_steps   (threads 0 and 1 bisect)
__global__ void lanczos_bounds_kernel(const LanczosState* __restrict__ st, double* __restrict__ bounds)
{
    const int m = st->steps;
    if (threadIdx.x > 1 || m < 1) return;
    const double* a = st->alpha;
    const double* b = st->beta;
    double lo = a[0], hi = a[0];
    for (int i = 0; i < m; ++i) {
        const double r = (i > 0 ? fabs(b[i]) : 0.0) + (i + 1 < m ? fabs(b[i + 1]) : 0.0);
        lo = fmin(lo, a[i] - r);
        hi = fmax(hi, a[i] + r);
    }
    const int target = (threadIdx.x == 0) ? 1 : m;     // smallest / largest eigenvalue
    for (int it = 0; it < 64; ++it) {    // 64 halvings of an interval a few units wide: below one ulp
        const double mid = 0.5 * (lo + hi);
        if (lz_sturm(a, b, m, mid) >= target) hi = mid; else lo = mid;
    }
    const double theta = 0.5 * (lo + hi);
    bounds[threadIdx.x] = (threadIdx.x == 0) ? theta - b[m] : theta + b[m];
}

}  // namespace rfoe
