// One expansion sharded over g GPUs.
//
// Every rank holds the whole X_n.  The upper-triangle tile list (the L2-friendly order of build_tile_order) is cut
// into g contiguous ranges of c = ceil(n_t / g) tiles; rank r squares only its range with the unchanged squaring
// kernel (grid = its tile count), which writes its tiles and their mirrors into its own X_{n+1}.  The exchange step
// -- the paper's distributed pgemm communicates here too -- is ONE all-gather per recursion step of
// [c tiles of 128 x 128 doubles | c partial records]: thanks to the symmetry each GPU receives 4 n^2 (g-1)/g bytes,
// half of an all-gather of row panels.  unpack_tiles_kernel then writes every foreign tile and its mirror into
// X_{n+1} and lays the partial records out in the global tile order, so control_kernel adds them in exactly the
// order of the single-GPU run: all ranks take the same decisions and P is bitwise the single-GPU P.
#pragma once
#include "sym_square.cuh"

namespace rfoe {

constexpr int TILE_ELEMS = SQ_BM * SQ_BM;

// send[i] <- tile (I, J) = tiles[i] of W (row pitch ld), row-major 128 x 128; one CTA per tile
__global__ void __launch_bounds__(256)
pack_tiles_kernel(const double* __restrict__ W, int ld, const int2* __restrict__ tiles, double* __restrict__ send)
{
    const int2 t = tiles[blockIdx.x];
    const double* src = W + (size_t)t.x * SQ_BM * ld + (size_t)t.y * SQ_BM;
    double2* dst = reinterpret_cast<double2*>(send + (size_t)blockIdx.x * TILE_ELEMS);
    for (int e = threadIdx.x; e < TILE_ELEMS / 2; e += 256) {
        const int r = e >> 6, c2 = e & 63;
        dst[e] = *reinterpret_cast<const double2*>(src + (size_t)r * ld + 2 * c2);
    }
}

// recv = g blocks of rank_stride doubles: [c_max tiles | c_max records of SQ_NPART].  One CTA per GLOBAL tile index:
// copies the record to parts_all[t]; unless the tile is in [own_begin, own_begin + own_count) (already in W), writes
// the tile to (I, J) and, for I < J, its transpose to (J, I) through shared memory (256-byte runs both ways).
__global__ void __launch_bounds__(256)
unpack_tiles_kernel(const double* __restrict__ recv, size_t rank_stride, int c_max, const int2* __restrict__ tile_map,
                    int own_begin, int own_count, double* __restrict__ W, int ld, double* __restrict__ parts_all)
{
    __shared__ double sm[32][33];
    const int t = blockIdx.x;
    const int rk = t / c_max, loc = t - rk * c_max;
    const double* blk = recv + (size_t)rk * rank_stride;
    if (threadIdx.x < SQ_NPART)
        parts_all[(size_t)t * SQ_NPART + threadIdx.x] = blk[(size_t)c_max * TILE_ELEMS + (size_t)loc * SQ_NPART + threadIdx.x];
    if (t >= own_begin && t < own_begin + own_count) return;
    const double* src = blk + (size_t)loc * TILE_ELEMS;
    const int2 tile = tile_map[t];
    const int I = tile.x, J = tile.y;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    double* dir = W + (size_t)I * SQ_BM * ld + (size_t)J * SQ_BM;
    double* mir = W + (size_t)J * SQ_BM * ld + (size_t)I * SQ_BM;
    for (int bi = 0; bi < 4; ++bi)
        for (int bj = 0; bj < 4; ++bj) {
            __syncthreads();
#pragma unroll
            for (int y = ty; y < 32; y += 8) {
                const double v = src[(bi * 32 + y) * SQ_BM + bj * 32 + tx];
                dir[(size_t)(bi * 32 + y) * ld + bj * 32 + tx] = v;
                sm[y][tx] = v;
            }
            __syncthreads();
            if (I != J) {
#pragma unroll
                for (int y = ty; y < 32; y += 8) mir[(size_t)(bj * 32 + y) * ld + bi * 32 + tx] = sm[tx][y];
            }
        }
}

}  // namespace rfoe
