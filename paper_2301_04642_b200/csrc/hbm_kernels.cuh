// HBM-bound kernels of the RFOE path (rows A1, A2 and the output pass of DESIGN.md): one warp owns
// one matrix row at a time, lanes stride the row so every load/store instruction is a contiguous
// 256/512-byte run; rows are distributed over a grid sized in multiples of the SM count.
// All row-level results go to per-row arrays and are summed later in a fixed order (no FP atomics).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rfoe {

constexpr int HBM_THREADS = 256;
constexpr int HBM_WARPS = HBM_THREADS / 32;

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int m = 16; m >= 1; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    return v;
}

// A1 -- Gershgorin discs ("spectral bound estimates"; reading R3):
// row_lo[i] = H_ii - r_i, row_hi[i] = H_ii + r_i, r_i = sum_{j != i} |H_ij|.
__global__ void __launch_bounds__(HBM_THREADS)
gershgorin_rows_kernel(const double* __restrict__ H, int k, double* __restrict__ row_lo, double* __restrict__ row_hi)
{
    const int lane = threadIdx.x & 31;
    const int wglobal = blockIdx.x * HBM_WARPS + (threadIdx.x >> 5);
    const int wtotal = gridDim.x * HBM_WARPS;
    const bool vec = ((k & 1) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    for (int i = wglobal; i < k; i += wtotal) {
        const double* row = H + (size_t)i * k;
        double r0 = 0.0, r1 = 0.0, r2 = 0.0, r3 = 0.0;
        if (vec) {
            const double2* row2 = reinterpret_cast<const double2*>(row);
            const int n2 = k >> 1;
            int j = lane;
            for (; j + 96 < n2; j += 128) {
                const double2 a = row2[j], b = row2[j + 32], c = row2[j + 64], d = row2[j + 96];
                r0 += ((2 * j == i) ? 0.0 : fabs(a.x)) + ((2 * j + 1 == i) ? 0.0 : fabs(a.y));
                r1 += ((2 * (j + 32) == i) ? 0.0 : fabs(b.x)) + ((2 * (j + 32) + 1 == i) ? 0.0 : fabs(b.y));
                r2 += ((2 * (j + 64) == i) ? 0.0 : fabs(c.x)) + ((2 * (j + 64) + 1 == i) ? 0.0 : fabs(c.y));
                r3 += ((2 * (j + 96) == i) ? 0.0 : fabs(d.x)) + ((2 * (j + 96) + 1 == i) ? 0.0 : fabs(d.y));
            }
            for (; j < n2; j += 32) {
                const double2 a = row2[j];
                r0 += ((2 * j == i) ? 0.0 : fabs(a.x)) + ((2 * j + 1 == i) ? 0.0 : fabs(a.y));
            }
        } else {
            for (int j = lane; j < k; j += 32) r0 += (j == i) ? 0.0 : fabs(row[j]);
        }
        const double r = warp_sum((r0 + r1) + (r2 + r3));
        if (lane == 0) {
            const double d = row[i];
            row_lo[i] = d - r;
            row_hi[i] = d + r;
        }
    }
}

// A2 -- affine initial map (reading R2; the paper's "begins with X_0 = H"):
// X0 = (emax I - H) / (emax - emin), true division.  X0 is written into the zero-padded n x n
// work matrix (row pitch ld) (rows/cols >= k are set to zero); row_tr[i] = X0_ii, row_ss[i] = sum_j X0_ij^2.
__global__ void __launch_bounds__(HBM_THREADS)
affine_map_kernel(const double* __restrict__ H, int k, int n, int ld, const double* __restrict__ bounds,
                  double* __restrict__ X, double* __restrict__ row_tr, double* __restrict__ row_ss)
{
    const int lane = threadIdx.x & 31;
    const int wglobal = blockIdx.x * HBM_WARPS + (threadIdx.x >> 5);
    const int wtotal = gridDim.x * HBM_WARPS;
    const double emin = bounds[0], emax = bounds[1];
    const double w = emax - emin;
    const bool vec = ((k & 1) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    for (int i = wglobal; i < n; i += wtotal) {
        double* xrow = X + (size_t)i * ld;
        if (i >= k) {
            for (int j = lane * 2; j < n; j += 64) *reinterpret_cast<double2*>(xrow + j) = make_double2(0.0, 0.0);
            continue;
        }
        const double* row = H + (size_t)i * k;
        double ss = 0.0;
        if (vec) {
            // four independent 16-byte loads in flight per lane (512-byte runs per warp instruction)
            auto map2 = [&](double2 h, int j, double2& x) {
                x.x = ((j == i) ? (emax - h.x) : (-h.x)) / w;
                x.y = ((j + 1 == i) ? (emax - h.y) : (-h.y)) / w;
                ss = fma(x.x, x.x, ss);
                ss = fma(x.y, x.y, ss);
            };
            int j = lane * 2;
            for (; j + 192 < k; j += 256) {
                const double2 h0 = *reinterpret_cast<const double2*>(row + j);
                const double2 h1 = *reinterpret_cast<const double2*>(row + j + 64);
                const double2 h2 = *reinterpret_cast<const double2*>(row + j + 128);
                const double2 h3 = *reinterpret_cast<const double2*>(row + j + 192);
                double2 x0, x1, x2, x3;
                map2(h0, j, x0); map2(h1, j + 64, x1); map2(h2, j + 128, x2); map2(h3, j + 192, x3);
                *reinterpret_cast<double2*>(xrow + j) = x0;
                *reinterpret_cast<double2*>(xrow + j + 64) = x1;
                *reinterpret_cast<double2*>(xrow + j + 128) = x2;
                *reinterpret_cast<double2*>(xrow + j + 192) = x3;
            }
            for (; j < k; j += 64) {
                const double2 h = *reinterpret_cast<const double2*>(row + j);
                double2 x;
                map2(h, j, x);
                *reinterpret_cast<double2*>(xrow + j) = x;
            }
        } else {
            for (int j = lane; j < k; j += 32) {
                const double h = row[j];
                const double x = ((j == i) ? (emax - h) : (-h)) / w;
                ss = fma(x, x, ss);
                xrow[j] = x;
            }
        }
        for (int j = k + lane; j < n; j += 32) xrow[j] = 0.0;
        ss = warp_sum(ss);
        if (lane == 0) {
            row_ss[i] = ss;
            row_tr[i] = (emax - row[i]) / w;
        }
    }
}

// pad copy: caller matrix (k x k, ld = k) -> zero-padded work matrix (n x n, row pitch ld)
__global__ void __launch_bounds__(HBM_THREADS)
pad_copy_kernel(const double* __restrict__ src, int k, int n, int ld, double* __restrict__ dst)
{
    const int lane = threadIdx.x & 31;
    const int wglobal = blockIdx.x * HBM_WARPS + (threadIdx.x >> 5);
    const int wtotal = gridDim.x * HBM_WARPS;
    for (int i = wglobal; i < n; i += wtotal) {
        double* drow = dst + (size_t)i * ld;
        if (i < k) {
            const double* srow = src + (size_t)i * k;
            for (int j = lane; j < n; j += 32) drow[j] = (j < k) ? srow[j] : 0.0;
        } else {
            for (int j = lane; j < n; j += 32) drow[j] = 0.0;
        }
    }
}

// Output pass: P (k x k, ld = k) <- work matrix (row pitch ld); row_ph[i] = sum_j P_ij H_ij (band energy
// tr(P H^p)).  H may be null (then only the copy is done).
__device__ __forceinline__ void copy_out_rows(const double* __restrict__ W, int k, int ld, const double* __restrict__ H,
                                              double* __restrict__ P, double* __restrict__ row_ph)
{
    const int lane = threadIdx.x & 31;
    const int wglobal = blockIdx.x * HBM_WARPS + (threadIdx.x >> 5);
    const int wtotal = gridDim.x * HBM_WARPS;
    const bool vec = ((k & 1) == 0) && ((reinterpret_cast<uintptr_t>(P) & 15) == 0) &&
                     (H == nullptr || (reinterpret_cast<uintptr_t>(H) & 15) == 0);
    for (int i = wglobal; i < k; i += wtotal) {
        const double* wrow = W + (size_t)i * ld;
        double* prow = P + (size_t)i * k;
        double acc = 0.0;
        if (vec) {
            for (int j = lane * 2; j < k; j += 64) {
                const double2 x = *reinterpret_cast<const double2*>(wrow + j);
                if (H) {
                    const double2 h = *reinterpret_cast<const double2*>(H + (size_t)i * k + j);
                    acc = fma(x.x, h.x, acc);
                    acc = fma(x.y, h.y, acc);
                }
                *reinterpret_cast<double2*>(prow + j) = x;
            }
        } else {
            for (int j = lane; j < k; j += 32) {
                const double x = wrow[j];
                if (H) acc = fma(x, H[(size_t)i * k + j], acc);
                prow[j] = x;
            }
        }
        acc = warp_sum(acc);
        if (lane == 0 && row_ph) row_ph[i] = acc;
    }
}

__global__ void __launch_bounds__(HBM_THREADS)
copy_out_kernel(const double* __restrict__ W, int k, int ld, const double* __restrict__ H, double* __restrict__ P,
                double* __restrict__ row_ph)
{
    copy_out_rows(W, k, ld, H, P, row_ph);
}

// The same pass when the host does not know which of the two work matrices holds the result (the recursion ran in one
// persistent launch): the parity of the step counter in device memory selects it.
__global__ void __launch_bounds__(HBM_THREADS)
copy_out_select_kernel(const double* __restrict__ W0, const double* __restrict__ W1, const int* __restrict__ step, int k, int ld,
                       const double* __restrict__ H, double* __restrict__ P, double* __restrict__ row_ph)
{
    copy_out_rows((*step & 1) ? W1 : W0, k, ld, H, P, row_ph);
}

// Bitwise symmetry check of a k x k matrix: 64 x 64 tiles of the upper triangle, both tiles read
// row-contiguously (512-byte runs) and compared through shared memory.  *flag is set to 1 on any mismatch.
constexpr int SYM_T = 64;
__global__ void __launch_bounds__(256)
symmetry_check_kernel(const double* __restrict__ H, int k, int* __restrict__ flag)
{
    __shared__ unsigned long long ta[SYM_T][SYM_T + 1];
    const int nt = (k + SYM_T - 1) / SYM_T;
    const unsigned long long* Hb = reinterpret_cast<const unsigned long long*>(H);
    const int tx = threadIdx.x & (SYM_T - 1), ty = threadIdx.x / SYM_T;   // 64 x 4
    for (long long t = blockIdx.x; t < (long long)nt * nt; t += gridDim.x) {
        const int bi = (int)(t / nt), bj = (int)(t % nt);
        if (bj < bi) continue;
        __syncthreads();
#pragma unroll 4
        for (int y = ty; y < SYM_T; y += 4) {
            const int i = bi * SYM_T + y, j = bj * SYM_T + tx;
            ta[y][tx] = (i < k && j < k) ? Hb[(size_t)i * k + j] : 0ull;
        }
        __syncthreads();
        int bad = 0;
#pragma unroll 4
        for (int y = ty; y < SYM_T; y += 4) {
            const int i = bj * SYM_T + y, j = bi * SYM_T + tx;   // element (i, j) of the mirrored tile
            if (i < k && j < k) bad |= (Hb[(size_t)i * k + j] != ta[tx][y]);
        }
        if (bad) atomicExch(flag, 1);
    }
}

}  // namespace rfoe
