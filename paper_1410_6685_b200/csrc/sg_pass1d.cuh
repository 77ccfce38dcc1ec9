// sg_pass1d.cuh — the fused 1-D pass (SURVEY.md §8(a) a3 map/zip, a4 terminal reductions, a5 quantifier contracts).
//
// One launch per pass: every distinct input is loaded once with 128-bit coalesced loads, the whole op chain is
// evaluated in registers (the paper's merged kernel body, PAPER.md:307-309 — here without the barrier between
// the map and the reduction stage, the map value never leaves registers), materialised outputs are stored,
// and every reduction/quantifier of the pass is accumulated per thread, reduced by warp shuffles and shared
// memory, written as one partial per block and combined in fixed order by the last block to finish.
//
// Two evaluators share this file's structure and epilogue:
//   pass1d_template<P>  — the program P::prog is a compile-time constant: straight-line code, all registers static;
//   pass1d_bytecode     — the same SgProg bytes interpreted at run time (register file selected by uniform switch).
#ifndef SG_PASS1D_CUH_
#define SG_PASS1D_CUH_

#include <utility>

#include "sg_device.cuh"

namespace sgk {

__host__ __device__ constexpr bool out_is_reduction(uint8_t k) { return k >= OUT_SUM && k <= OUT_COUNT; }
__host__ __device__ constexpr bool out_is_pred_reduction(uint8_t k) { return k >= OUT_ALL && k <= OUT_COUNT; }

// ---------------------------------------------------------------------------------------------------------
// epilogue: block reduction of every accumulator cell, one partial per block, last block combines all partials
// in block order (deterministic: no floating-point atomics) and writes the 8-byte results.
// ---------------------------------------------------------------------------------------------------------
template <class T, int NOUT>
__device__ __forceinline__ void block_reduce_cells(Cell (&acc)[NOUT], const uint8_t (&kind)[NOUT], Cell* smem /*[32*NOUT]*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (int)(blockDim.x >> 5);     // any block of whole warps (<= 32)
#pragma unroll
    for (int o = 0; o < NOUT; ++o) {
        if (!out_is_reduction(kind[o])) continue;
#pragma unroll
        for (int d = 16; d >= 1; d >>= 1) {
            Cell other = cell_shfl_down(acc[o], d);
            cell_combine<T>(kind[o], acc[o], other);
        }
        if (lane == 0) smem[warp * NOUT + o] = acc[o];
    }
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int o = 0; o < NOUT; ++o) {
            if (!out_is_reduction(kind[o])) continue;
            Cell c = (lane < nwarps) ? smem[lane * NOUT + o] : cell_identity<T>(kind[o]);
#pragma unroll
            for (int d = 16; d >= 1; d >>= 1) {
                Cell other = cell_shfl_down(c, d);
                cell_combine<T>(kind[o], c, other);
            }
            acc[o] = c;     // valid in thread 0
        }
    }
    __syncthreads();
}

// the 8-byte result of an AXIS_ALL output: the device slot and, when the context gave one, its place in the pinned host mirror —
// written from here the hand-back needs no copy-engine transfer between this kernel and the next one of the stream
__device__ __forceinline__ void store_scalar(const SgArgs& a, int o, unsigned long long r) {
    *reinterpret_cast<unsigned long long*>(a.out_ptr[o]) = r;
    if (a.out_host[o] != nullptr) *reinterpret_cast<volatile unsigned long long*>(a.out_host[o]) = r;
}

template <class T, int NOUT>
__device__ __forceinline__ void epilogue_1d(Cell (&acc)[NOUT], const uint8_t (&kind)[NOUT], const SgArgs& a, bool need_ticket) {
    __shared__ Cell smem[32 * SG_MAX_OUT];
    __shared__ unsigned int s_last;
    if (!need_ticket) return;     // passes with neither reductions nor a dynamic tile counter leave ctrl untouched
    block_reduce_cells<T, NOUT>(acc, kind, smem);
    // Every step below is a round trip to L2 on the pass's critical path (a one-element reduction measured 3.7 us against 0.5 us for an
    // empty dependent launch), so a single-block grid finalises directly: its block IS the last one.
    if (gridDim.x == 1) {
        if (threadIdx.x == 0) {
#pragma unroll
            for (int o = 0; o < NOUT; ++o)
                if (out_is_reduction(kind[o])) store_scalar(a, o, cell_final<T>(kind[o], acc[o]));
            a.ctrl[1] = 0; a.ctrl[2] = 0;
        }
        return;
    }
    Cell* ws = reinterpret_cast<Cell*>(a.workspace);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int o = 0; o < NOUT; ++o)
            if (out_is_reduction(kind[o])) ws[(size_t)blockIdx.x * SG_MAX_OUT + o] = acc[o];
        // release: the partials above are visible to whoever observes this increment (one instruction instead of fence + atomic)
        unsigned int t;
        asm volatile("atom.add.release.gpu.global.u32 %0, [%1], 1;" : "=r"(t) : "l"(&a.ctrl[0]) : "memory");
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();        // acquire side: the other blocks' partials
#pragma unroll
    for (int o = 0; o < NOUT; ++o) {
        if (!out_is_reduction(kind[o])) continue;
        Cell c = cell_identity<T>(kind[o]);
        for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
            Cell other;
            const unsigned long long* src = reinterpret_cast<const unsigned long long*>(&ws[(size_t)b * SG_MAX_OUT + o]);
            other.a = __ldcg(src); other.b = __ldcg(src + 1);
            cell_combine<T>(kind[o], c, other);
        }
        acc[o] = c;
    }
    block_reduce_cells<T, NOUT>(acc, kind, smem);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int o = 0; o < NOUT; ++o)
            if (out_is_reduction(kind[o])) store_scalar(a, o, cell_final<T>(kind[o], acc[o]));
        a.ctrl[0] = 0; a.ctrl[1] = 0; a.ctrl[2] = 0;       // the end of the kernel makes these visible to the next launch
    }
}

// ---------------------------------------------------------------------------------------------------------
// one-element loads/stores of the ragged path (head before the aligned body, tail after the last full tile)
// ---------------------------------------------------------------------------------------------------------
template <class T>
__device__ __forceinline__ T load_elem(uint8_t kind, uint8_t ref, int k, const SgArgs& a, int64_t i) {
    switch (kind) {
        case IN_VEC: return (i < a.in_len[k]) ? reinterpret_cast<const volatile T*>(a.in_ptr[k])[i] : T(0);
        case IN_SHIFT: return (i + 1 < a.in_len[ref]) ? reinterpret_cast<const volatile T*>(a.in_ptr[ref])[i + 1] : T(0);
        case IN_STRIDED: return (i < a.in_len[k]) ? reinterpret_cast<const volatile T*>(a.in_ptr[k])[i * a.in_stride[k]] : T(0);
        case IN_VEC_CVT: return (i < a.in_len[k]) ? load_cvt<T>(a.in_ptr[k], i, ref) : T(0);
        case IN_SCALAR: return *reinterpret_cast<const volatile T*>(a.in_ptr[k]);
        case IN_IMM: { T v; memcpy(&v, &a.imm[k], sizeof(T)); return v; }
        default: return T(0);
    }
}

}  // namespace sgk
#endif  // SG_PASS1D_CUH_
