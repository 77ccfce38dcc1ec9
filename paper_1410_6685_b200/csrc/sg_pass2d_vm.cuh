// sg_pass2d_vm.cuh — pass2d_bytecode: the bytecode evaluator for MATRIX passes that have no precompiled template instance
// (north_star: "a register-resident op-bytecode fallback for long chains" — on the 2-D domain as well, so an unregistered
// matrix chain runs instead of failing).  Same programs, same interpreter core (vm_exec over the shared-memory register file of
// sg_pass1d_vm.cuh) as the 1-D bytecode kernel; the domain is walked row by row:
//
//   * a block owns whole rows r = blockIdx.x, blockIdx.x + gridDim.x, ...; a thread evaluates E = 16 / sizeof(T) consecutive
//     columns per step (one 128-bit cell), column tiles of BLOCK * E columns;
//   * IN_VEC = matrix element (r, c); IN_ROWB = vector[c]; IN_COLB = vector[r]; scalars and immediates are broadcast once;
//   * AXIS_ROWS reductions finish inside the block (it owns the whole row): one block reduction per row;
//   * AXIS_COLS reductions accumulate per block in a workspace slice [block][cols] (column c of a block is always the same
//     thread's: no races), combined over the blocks in block order by the last block to finish — deterministic, no atomics
//     on floating point;
//   * AXIS_ALL reductions and quantifiers use the 1-D epilogue.
// Every access is guarded per element, so any shape, leading dimension and alignment works.  It is the fallback: it moves the
// same bytes as a template instance but spends an interpreter's instructions per element.
#ifndef SG_PASS2D_VM_CUH_
#define SG_PASS2D_VM_CUH_

#include "sg_pass1d_vm.cuh"

namespace sgk {

template <class T> __device__ __forceinline__ void store_final_2dvm(uint8_t kind, void* base, int64_t idx, const Cell& c) {
    const unsigned long long r = cell_final<T>(kind, c);
    if ((kind == OUT_MAX || kind == OUT_MIN) && sizeof(T) == 4) reinterpret_cast<uint32_t*>(base)[idx] = (uint32_t)r;
    else reinterpret_cast<unsigned long long*>(base)[idx] = r;
}

template <class T>
__global__ void __launch_bounds__(BLOCK, 2) pass2d_bytecode(const __grid_constant__ SgProg g, const __grid_constant__ SgArgs a) {
    extern __shared__ __align__(16) unsigned char vm_file2d[];
    __shared__ Cell s_red[32 * SG_MAX_OUT];
    __shared__ unsigned int s_last;
    constexpr int E = VmE<T>::value;
    pdl_wait();
    pdl_trigger();
    const int64_t rows = a.n, cols = a.cols;
    Cell acc[SG_MAX_OUT];           // AXIS_ALL
    uint8_t kind_all[SG_MAX_OUT];   // the AXIS_ALL outputs' kinds (OUT_STORE otherwise): what the 1-D epilogue reduces
    bool has_all = false, has_rows = false, has_cols = false;
#pragma unroll
    for (int o = 0; o < SG_MAX_OUT; ++o) {
        const bool live = o < g.shape.n_out;
        const bool red = live && out_is_reduction(g.out[o].kind);
        kind_all[o] = (red && g.out[o].axis == AXIS_ALL) ? g.out[o].kind : (uint8_t)OUT_STORE;
        acc[o] = cell_identity<T>(kind_all[o]);
        has_all |= red && g.out[o].axis == AXIS_ALL;
        has_rows |= red && g.out[o].axis == AXIS_ROWS;
        has_cols |= red && g.out[o].axis == AXIS_COLS;
    }
    VmRegs<T, E> rf((uint32_t)__cvta_generic_to_shared(vm_file2d));
    for (int k = 0; k < g.shape.n_in; ++k) {
        const SgIn in = g.in[k];
        if (in.kind == IN_SCALAR || in.kind == IN_IMM) {
            T x[E];
            const T s = load_elem<T>(in.kind, in.ref, k, a, 0);
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = s;
            rf.put(in.reg, x);
        }
    }
    // this block's slice of the per-column partials starts from the identity
    if (has_cols)
        for (int o = 0; o < g.shape.n_out; ++o) {
            if (!(out_is_reduction(g.out[o].kind) && g.out[o].axis == AXIS_COLS)) continue;
            Cell* ws = reinterpret_cast<Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]) + (size_t)blockIdx.x * cols;
            for (int64_t c = threadIdx.x; c < cols; c += BLOCK) ws[c] = cell_identity<T>(g.out[o].kind);
        }
    __syncthreads();

    const int64_t tile_cols = (int64_t)BLOCK * E;
    for (int64_t r = blockIdx.x; r < rows; r += gridDim.x) {
        Cell rowc[SG_MAX_OUT];      // AXIS_ROWS partials of this thread for row r
#pragma unroll
        for (int o = 0; o < SG_MAX_OUT; ++o) rowc[o] = cell_identity<T>(o < g.shape.n_out ? g.out[o].kind : (uint8_t)OUT_STORE);
        for (int64_t c0 = 0; c0 < cols; c0 += tile_cols) {
            const int64_t c = c0 + (int64_t)threadIdx.x * E;
            const int nval = (cols - c) >= E ? E : ((cols - c) > 0 ? (int)(cols - c) : 0);
            unsigned int pf = 0;
            for (int k = 0; k < g.shape.n_in; ++k) {
                const SgIn in = g.in[k];
                if (in.kind == IN_SCALAR || in.kind == IN_IMM) continue;
                if (in.kind == IN_BOOLVEC) {        // a stored BOOL matrix: one byte per element, into a predicate register
                    unsigned int bits = 0;
#pragma unroll
                    for (int e = 0; e < E; ++e)
                        if (e < nval) bits |= (unsigned int)(reinterpret_cast<const volatile uint8_t*>(a.in_ptr[k])[r * a.in_stride[k] + c + e] != 0) << e;
                    pf = pput<E>(pf, in.reg, bits);
                    continue;
                }
                T x[E];
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    x[e] = T(0);
                    if (e < nval) {
                        if (in.kind == IN_VEC) x[e] = reinterpret_cast<const volatile T*>(a.in_ptr[k])[r * a.in_stride[k] + c + e];
                        else if (in.kind == IN_ROWB) x[e] = reinterpret_cast<const volatile T*>(a.in_ptr[k])[c + e];
                        else if (in.kind == IN_COLB) x[e] = reinterpret_cast<const volatile T*>(a.in_ptr[k])[r];
                    }
                }
                rf.put(in.reg, x);
            }
            vm_exec<T, E>(g, rf, pf);
            for (int o = 0; o < g.shape.n_out; ++o) {
                const SgOut out = g.out[o];
                if (out.kind == OUT_STORE) {
                    T x[E];
                    rf.get(out.src, x);
                    T* rowp = reinterpret_cast<T*>(a.out_ptr[o]) + r * a.out_len[o];
#pragma unroll
                    for (int e = 0; e < E; ++e)
                        if (e < nval) rowp[c + e] = x[e];
                } else if (out.kind == OUT_STORE_BOOL) {
                    const unsigned int bits = pget<E>(pf, out.src);
                    uint8_t* rowp = reinterpret_cast<uint8_t*>(a.out_ptr[o]) + r * a.out_len[o];
#pragma unroll
                    for (int e = 0; e < E; ++e)
                        if (e < nval) rowp[c + e] = (bits >> e) & 1u;
                } else if (out_is_reduction(out.kind)) {
                    T x[E];
                    unsigned int bits = 0, mask = (1u << E) - 1u;
                    if (out_is_pred_reduction(out.kind)) bits = pget<E>(pf, out.src);
                    else {
                        rf.get(out.src, x);
                        if (out.pred != SG_NO_PRED) mask = pget<E>(pf, out.pred);
                    }
                    Cell* wsc = (out.axis == AXIS_COLS)
                                    ? reinterpret_cast<Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]) + (size_t)blockIdx.x * cols + c
                                    : nullptr;
#pragma unroll
                    for (int e = 0; e < E; ++e) {
                        if (e >= nval) continue;
                        Cell tmp;
                        Cell& dst = (out.axis == AXIS_ALL) ? acc[o] : (out.axis == AXIS_ROWS) ? rowc[o] : tmp;
                        if (out.axis == AXIS_COLS) tmp = wsc[e];
                        if (out_is_pred_reduction(out.kind)) cell_accum_pred(out.kind, dst, (bits >> e) & 1u);
                        else if ((mask >> e) & 1u) {
                            switch (out.kind) {
                                case OUT_SUM: cell_accum_value<T>(OUT_SUM, dst, x[e]); break;
                                case OUT_MAX: cell_accum_value<T>(OUT_MAX, dst, x[e]); break;
                                default: cell_accum_value<T>(OUT_MIN, dst, x[e]); break;
                            }
                        }
                        if (out.axis == AXIS_COLS) wsc[e] = tmp;
                    }
                }
            }
        }
        // the block owns the whole row: its AXIS_ROWS results are final after one block reduction
        if (has_rows) {
            uint8_t kind_rows[SG_MAX_OUT];
#pragma unroll
            for (int o = 0; o < SG_MAX_OUT; ++o)
                kind_rows[o] = (o < g.shape.n_out && out_is_reduction(g.out[o].kind) && g.out[o].axis == AXIS_ROWS) ? g.out[o].kind : (uint8_t)OUT_STORE;
            block_reduce_cells<T, SG_MAX_OUT>(rowc, kind_rows, s_red);
            if (threadIdx.x == 0)
                for (int o = 0; o < g.shape.n_out; ++o)
                    if (out_is_reduction(kind_rows[o])) store_final_2dvm<T>(kind_rows[o], a.out_ptr[o], r, rowc[o]);
        }
    }

    // per-column partials: the last block to finish combines the blocks' slices in block order
    if (has_cols) {
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) s_last = (atomicAdd(&a.ctrl[8], 1u) == gridDim.x - 1);
        __syncthreads();
        if (s_last) {
            __threadfence();
            for (int o = 0; o < g.shape.n_out; ++o) {
                const SgOut out = g.out[o];
                if (!(out_is_reduction(out.kind) && out.axis == AXIS_COLS)) continue;
                const Cell* ws = reinterpret_cast<const Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]);
                for (int64_t c = threadIdx.x; c < cols; c += BLOCK) {
                    Cell acc_c = cell_identity<T>(out.kind);
                    for (unsigned int b = 0; b < gridDim.x; ++b) {
                        Cell other;
                        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(&ws[(size_t)b * cols + c]);
                        other.a = __ldcg(src); other.b = __ldcg(src + 1);
                        switch (out.kind) {
                            case OUT_SUM: cell_combine<T>(OUT_SUM, acc_c, other); break;
                            case OUT_MAX: cell_combine<T>(OUT_MAX, acc_c, other); break;
                            case OUT_MIN: cell_combine<T>(OUT_MIN, acc_c, other); break;
                            case OUT_ALL: cell_combine<T>(OUT_ALL, acc_c, other); break;
                            case OUT_ANY: cell_combine<T>(OUT_ANY, acc_c, other); break;
                            default: cell_combine<T>(OUT_COUNT, acc_c, other); break;
                        }
                    }
                    store_final_2dvm<T>(out.kind, a.out_ptr[o], c, acc_c);
                }
            }
            if (threadIdx.x == 0) a.ctrl[8] = 0;
        }
    }
    epilogue_1d<T, SG_MAX_OUT>(acc, kind_all, a, has_all);
}

}  // namespace sgk
#endif  // SG_PASS2D_VM_CUH_
