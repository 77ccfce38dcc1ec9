// sg_transpose.cu — `transpose` of a row-major matrix, a pure data mover: 2 x element size bytes per element.
//
// One block moves a TILE x TILE tile through shared memory so that BOTH the reads (along the source rows) and the writes
// (along the destination rows) are contiguous TILE * sizeof(T) byte segments (512 B for fp64, 256 B for fp32): every warp
// access is whole 128-byte lines.  The shared tile is padded by one element per row, which makes the transposed (column)
// read conflict-free: a half-warp of 8-byte accesses with a stride of 65 elements touches 16 distinct bank pairs.  Each
// thread of the 512-thread block issues TILE/ROWS = 8 independent streaming loads before the barrier (32 KB in flight per block,
// 4 blocks per SM), which is what keeps HBM busy; loads and stores are marked streaming (the data is touched once).
// The grid is one-dimensional over the tiles, ordered along the SOURCE rows, so concurrently running blocks read adjacent
// segments of the same source rows (open DRAM pages) and write adjacent destination rows.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sg_kernels.h"

namespace {

constexpr int TILE = 64, ROWS = 8, TBLOCK = TILE * ROWS;      // measured at 16384^2 fp64: ROWS 4 / 8 / 16 -> 0.774 / 0.651 / 0.749 ms
// 4-byte elements run at 0.79 of the measured peak (fp64: 1.01).  128 x 128 tiles (512-byte segments on both sides, like fp64) were
// measured and change nothing (422 vs 415 us at 16384^2 fp32): the fp32 mover is bound by its four 4-byte memory instructions per
// element (LDG, STS, LDS, STG), not by the segment length; the paper's transpose benchmark is DOUBLE.

template <class T>
__global__ void __launch_bounds__(TBLOCK) transpose_tiled(const T* __restrict__ in, int64_t ld_in, int64_t rows, int64_t cols,
                                                          T* __restrict__ out, int64_t ld_out, int64_t tiles_c) {
    __shared__ T tile[TILE][TILE + 1];
    const int tx = threadIdx.x % TILE, ty = threadIdx.x / TILE;
    const int64_t tr = blockIdx.x / tiles_c, tc = blockIdx.x % tiles_c;
    const int64_t r0 = tr * TILE, c0 = tc * TILE;
    const bool full = (r0 + TILE <= rows) && (c0 + TILE <= cols);
    if (full) {
        T x[TILE / ROWS];
#pragma unroll
        for (int i = 0; i < TILE / ROWS; ++i) x[i] = __ldcs(in + (r0 + ty + ROWS * i) * ld_in + c0 + tx);
#pragma unroll
        for (int i = 0; i < TILE / ROWS; ++i) tile[ty + ROWS * i][tx] = x[i];
        __syncthreads();
#pragma unroll
        for (int i = 0; i < TILE / ROWS; ++i) __stcs(out + (c0 + ty + ROWS * i) * ld_out + r0 + tx, tile[tx][ty + ROWS * i]);
    } else {
#pragma unroll
        for (int i = 0; i < TILE / ROWS; ++i) {
            const int64_t r = r0 + ty + ROWS * i, c = c0 + tx;
            if (r < rows && c < cols) tile[ty + ROWS * i][tx] = __ldcs(in + r * ld_in + c);
        }
        __syncthreads();
#pragma unroll
        for (int i = 0; i < TILE / ROWS; ++i) {
            const int64_t c = c0 + ty + ROWS * i, r = r0 + tx;
            if (r < rows && c < cols) __stcs(out + c * ld_out + r, tile[tx][ty + ROWS * i]);
        }
    }
}

}  // namespace

cudaError_t sgk_transpose(const void* in, int64_t ld_in, int64_t rows, int64_t cols, void* out, int64_t ld_out, int elem_size, cudaStream_t stream) {
    if (rows == 0 || cols == 0) return cudaSuccess;
    const int64_t tiles_r = (rows + TILE - 1) / TILE, tiles_c = (cols + TILE - 1) / TILE;
    const int64_t tiles = tiles_r * tiles_c;
    if (tiles > 0x7fffffffll) return cudaErrorInvalidValue;
    if (elem_size == 8)
        transpose_tiled<unsigned long long><<<(unsigned)tiles, TBLOCK, 0, stream>>>((const unsigned long long*)in, ld_in, rows, cols, (unsigned long long*)out, ld_out, tiles_c);
    else if (elem_size == 4)
        transpose_tiled<unsigned int><<<(unsigned)tiles, TBLOCK, 0, stream>>>((const unsigned int*)in, ld_in, rows, cols, (unsigned int*)out, ld_out, tiles_c);
    else
        return cudaErrorInvalidValue;
    return cudaGetLastError();
}
