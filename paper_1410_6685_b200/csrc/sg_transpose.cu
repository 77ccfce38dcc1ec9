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
// 4-byte elements through this kernel run at 0.79 of the measured peak (fp64: 1.01), and 128 x 128 tiles (512-byte segments on both
// sides) change nothing (422 vs 415 us at 16384^2 fp32): that mover is bound by its four 4-byte memory instructions per element (LDG,
// STS, LDS, STG), not by the segment length.  So 4-byte matrices whose rows are 8-byte aligned on both sides take transpose_pairs
// below: every memory instruction moves 8 bytes, as for fp64.

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


// 4-byte elements, 8-byte accesses: a tile is PR x 2 source rows by TILE source columns.  A thread loads the two 8-byte pairs of a
// 2 x 2 block (rows 2q, 2q+1; columns 2t, 2t+1), transposes it in registers and writes the two row-pairs (a[2q][c], a[2q+1][c]) to
// shared memory; even source columns fill the upper half of the shared tile and odd ones the lower half, so a half-warp's 8-byte
// stores are a stride of 65 pairs apart (16 distinct bank pairs).  The destination rows are then read as contiguous pairs and stored
// as PR * 8 = 512-byte segments.  Eight independent 8-byte loads per thread before the barrier, 32 KB per block, as for fp64.
constexpr int PR = 64;                                         // row pairs per tile: 128 source rows x 64 source columns
__global__ void __launch_bounds__(TBLOCK) transpose_pairs(const unsigned int* __restrict__ in, int64_t ld_in, int64_t rows, int64_t cols,
                                                          unsigned int* __restrict__ out, int64_t ld_out, int64_t tiles_c) {
    __shared__ uint2 tile[TILE][PR + 1];
    const int64_t tr = blockIdx.x / tiles_c, tc = blockIdx.x % tiles_c;
    const int64_t r0 = tr * (2 * PR), c0 = tc * TILE;
    if ((r0 + 2 * PR <= rows) && (c0 + TILE <= cols)) {
        const int t = threadIdx.x % (TILE / 2), qy = threadIdx.x / (TILE / 2);        // pair column 0..31, row-pair group 0..15
        constexpr int QS = TBLOCK / (TILE / 2), NQ = PR / QS;                         // 16 row pairs per sweep, 4 sweeps
        uint2 a0[NQ], a1[NQ];
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
            const unsigned int* src = in + (r0 + 2 * (qy + QS * i)) * ld_in + c0 + 2 * t;
            a0[i] = __ldcs(reinterpret_cast<const uint2*>(src));
            a1[i] = __ldcs(reinterpret_cast<const uint2*>(src + ld_in));
        }
#pragma unroll
        for (int i = 0; i < NQ; ++i) {
            tile[t][qy + QS * i] = make_uint2(a0[i].x, a1[i].x);                      // source column 2t
            tile[TILE / 2 + t][qy + QS * i] = make_uint2(a0[i].y, a1[i].y);           // source column 2t + 1
        }
        __syncthreads();
        const int q = threadIdx.x % PR, cy = threadIdx.x / PR;                        // row pair 0..63, destination-row group 0..7
        constexpr int CS = TBLOCK / PR;
#pragma unroll
        for (int j = 0; j < TILE / CS; ++j) {
            const int c = cy + CS * j;
            __stcs(reinterpret_cast<uint2*>(out + (c0 + c) * ld_out + r0 + 2 * q), tile[(c & 1) * (TILE / 2) + (c >> 1)][q]);
        }
    } else {                                                                          // ragged edge tiles: element by element
        for (int e = threadIdx.x; e < 2 * PR * TILE; e += TBLOCK) {
            const int64_t c = c0 + e / (2 * PR), r = r0 + e % (2 * PR);
            if (r < rows && c < cols) out[c * ld_out + r] = in[r * ld_in + c];
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
    else if (elem_size == 4) {
        const bool pairs = ((reinterpret_cast<uintptr_t>(in) | reinterpret_cast<uintptr_t>(out)) % 8 == 0) && ld_in % 2 == 0 && ld_out % 2 == 0;
        const int64_t ptiles = ((rows + 2 * PR - 1) / (2 * PR)) * tiles_c;
        if (pairs && rows >= 2 * PR)
            transpose_pairs<<<(unsigned)ptiles, TBLOCK, 0, stream>>>((const unsigned int*)in, ld_in, rows, cols, (unsigned int*)out, ld_out, tiles_c);
        else
            transpose_tiled<unsigned int><<<(unsigned)tiles, TBLOCK, 0, stream>>>((const unsigned int*)in, ld_in, rows, cols, (unsigned int*)out, ld_out, tiles_c);
    }
    else
        return cudaErrorInvalidValue;
    return cudaGetLastError();
}
