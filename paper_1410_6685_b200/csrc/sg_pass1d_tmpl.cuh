// sg_pass1d_tmpl.cuh — pass1d_template<P>: the fused 1-D pass with the program as a compile-time constant.
// "Each method is associated with a kernel template, which the library instantiates"; here the
// template is instantiated ahead of time over a whole merged chain instead of per method.
#ifndef SG_PASS1D_TMPL_CUH_
#define SG_PASS1D_TMPL_CUH_

#include "sg_pass1d.cuh"

namespace sgk {

__host__ __device__ constexpr bool prog_has_float_sum(const SgProg& g) {
    for (int o = 0; o < g.shape.n_out; ++o)
        if (g.out[o].kind == OUT_SUM && (g.shape.dtype == DT_F32 || g.shape.dtype == DT_F64)) return true;
    return false;
}
#ifndef SG_WARP_CONTIG
#define SG_WARP_CONTIG 2      // 0: block-interleaved tile layout, 1: warp-contiguous for passes with a neighbour operand, 2: for every pass
#endif
__host__ __device__ constexpr bool prog_has_shift(const SgProg& g) {
    for (int k = 0; k < g.shape.n_in; ++k)
        if (g.in[k].kind == IN_SHIFT) return true;
    return false;
}
__host__ __device__ constexpr bool prog_has_reduction(const SgProg& g) {
    for (int o = 0; o < g.shape.n_out; ++o)
        if (out_is_reduction(g.out[o].kind)) return true;
    return false;
}

template <class P> struct Meta1D {
    static constexpr SgShape S = P::prog.shape;
    typedef typename TypeOf<S.dtype>::type T;
    typedef typename Traits<T>::vec VEC;
    static constexpr int V = Traits<T>::V;
    static constexpr int U = P::unroll;                 // 128-bit loads per input per thread per tile
    static constexpr int E = U * V;                     // elements per thread per tile
    static constexpr int TILE = BLOCK * E;
    static constexpr int NV = S.n_vreg > 0 ? S.n_vreg : 1;
    static constexpr int NP = S.n_preg > 0 ? S.n_preg : 1;
    static constexpr int NOUT = S.n_out > 0 ? S.n_out : 1;
    static constexpr bool early_exit = (S.flags & PF_EARLY_EXIT) != 0;
    // Tile layout: warp w owns the U consecutive runs of 32 vectors [w*U*32, (w+1)*U*32) of the tile (2 KiB of fp32 at U = 4), access u
    // of lane l is vector (w*U + u)*32 + l.  Round 1 interleaved the warps (vector k -> thread k % BLOCK, access k / BLOCK).  With a
    // warp-contiguous layout the element after lane 31's vector is lane 0's vector of the warp's NEXT access — a neighbour operand
    // (IN_SHIFT) is a shuffle, and one scalar load per warp and tile instead of one per access: config 3's body + contracts in one
    // pass (sum + for_all + is_sorted, 2^28 fp32) 0.1815 -> 0.1615 ms = the time of the body alone.  It also serves the other passes
    // better (same-run A/B against the interleaved layout): config 1 at 2^28 0.3434 -> 0.3392 ms, x := 2x to a second buffer
    // 0.3318 -> 0.3134 ms, sqrt 0.0815 -> 0.0808 ms, int64 sum/max/min 0.1529 -> 0.1543 ms (the one that loses).
    static constexpr bool warp_contig = SG_WARP_CONTIG == 2 || (SG_WARP_CONTIG == 1 && prog_has_shift(P::prog));
    __device__ static __forceinline__ int vidx(int u) {
        return warp_contig ? (((int)(threadIdx.x >> 5) * U + u) * 32 + (int)(threadIdx.x & 31)) : (u * BLOCK + (int)threadIdx.x);
    }
    static constexpr bool has_reduction = prog_has_reduction(P::prog);
    static constexpr bool tickets = has_reduction && !early_exit && !prog_has_float_sum(P::prog);      // see the ticket loop of pass1d_template
};

// ---- compile-time body: one fold over the instruction list, every register index is a constant --------
// index of the IN_IMM input that lives in V register `reg`, or -1 (input registers are never recycled)
template <class P> __host__ __device__ constexpr int imm_input_of_reg(int reg) {
    for (int k = 0; k < P::prog.shape.n_in; ++k)
        if (P::prog.in[k].kind == IN_IMM && P::prog.in[k].reg == reg) return k;
    return -1;
}

template <class P, class T, int NV, int NP, int E, int I>
__device__ __forceinline__ void exec_instr(T (&v)[NV][E], bool (&p)[NP][E], const SgArgs& a) {
    constexpr SgInstr ins = P::prog.code[I];
    constexpr int immk = (ins.op == OP_MOD || ins.op == OP_DIV) ? imm_input_of_reg<P>(ins.b) : -1;
    if constexpr (immk >= 0 && sizeof(T) == 4 && !Traits<T>::is_float) {
        // x MOD d / x DIV d with an immediate divisor: multiply-high by the host-computed magic instead of dividing
        if (a.imm_div[immk].valid) {        // |d| > 1 (uniform)
#pragma unroll
            for (int e = 0; e < E; ++e)
                v[ins.dst][e] = (T)(ins.op == OP_MOD ? magic_mod_i32((int32_t)v[ins.a][e], a.imm_div[immk]) : magic_div_i32((int32_t)v[ins.a][e], a.imm_div[immk]));
            return;
        }
    }
#pragma unroll
    for (int e = 0; e < E; ++e) {
        if constexpr (op_is_value(ins.op)) v[ins.dst][e] = value_op<T>(ins.op, v[ins.a][e], v[ins.b][e]);
        else if constexpr (op_is_compare(ins.op)) p[ins.dst][e] = compare_op<T>(ins.op, v[ins.a][e], v[ins.b][e]);
        else p[ins.dst][e] = logic_op(ins.op, p[ins.a][e], p[ins.b][e]);
    }
}
template <class P, class T, int NV, int NP, int E, int... I>
__device__ __forceinline__ void exec_body(T (&v)[NV][E], bool (&p)[NP][E], const SgArgs& a, std::integer_sequence<int, I...>) {
    (exec_instr<P, T, NV, NP, E, I>(v, p, a), ...);
}

// ---- inputs of one full tile ---------------------------------------------------------------------------
template <class P, int K>
__device__ __forceinline__ void load_input_full(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][Meta1D<P>::E],
                                                bool (&p)[Meta1D<P>::NP][Meta1D<P>::E], const SgArgs& a, int64_t base) {
    typedef Meta1D<P> M;
    typedef typename M::T T;
    typedef typename M::VEC VEC;
    constexpr SgIn in = P::prog.in[K];
    if constexpr (in.kind == IN_VEC) {
        const VEC* src = reinterpret_cast<const VEC*>(reinterpret_cast<const T*>(a.in_ptr[K]) + base);
#pragma unroll
        for (int u = 0; u < M::U; ++u) {
            VEC x = in.pad ? ld_stream_rw(src + M::vidx(u)) : ld_stream(src + M::vidx(u));
            const T* xe = reinterpret_cast<const T*>(&x);
#pragma unroll
            for (int e = 0; e < M::V; ++e) v[in.reg][u * M::V + e] = xe[e];
        }
    } else if constexpr (in.kind == IN_VEC_CVT) {
        // a collection of another element type S, converted as it is loaded: V source elements (V * sizeof(S) bytes) per vector
        typedef typename TypeOf<in.ref>::type S;
        const S* src = reinterpret_cast<const S*>(a.in_ptr[K]) + base;
#pragma unroll
        for (int u = 0; u < M::U; ++u) {
            S x[M::V];
            ld_stream_bytes<M::V * (int)sizeof(S)>(src + (size_t)M::vidx(u) * M::V, x);
#pragma unroll
            for (int e = 0; e < M::V; ++e) v[in.reg][u * M::V + e] = cvt_elem<T, S>(x[e]);
        }
    } else if constexpr (in.kind == IN_SHIFT) {
        // x[i+1]: own vector shifted by one, last element from the next lane, lane 31 reads one scalar
        constexpr int rr = P::prog.in[in.ref].reg;
        const T* src = reinterpret_cast<const T*>(a.in_ptr[in.ref]) + base;
#pragma unroll
        for (int u = 0; u < M::U; ++u) {
#pragma unroll
            for (int e = 0; e + 1 < M::V; ++e) v[in.reg][u * M::V + e] = v[rr][u * M::V + e + 1];
            T nxt = __shfl_down_sync(0xffffffffu, v[rr][u * M::V], 1);
            if constexpr (M::warp_contig) {
                if (u + 1 < M::U) {
                    const T first_next = __shfl_sync(0xffffffffu, v[rr][(u + 1 < M::U ? u + 1 : u) * M::V], 0);
                    if ((threadIdx.x & 31) == 31) nxt = first_next;
                } else if ((threadIdx.x & 31) == 31) nxt = __ldg(src + (size_t)(M::vidx(u) + 1) * M::V);
            } else {
                if ((threadIdx.x & 31) == 31) nxt = __ldg(src + (size_t)(M::vidx(u) + 1) * M::V);
            }
            v[in.reg][u * M::V + M::V - 1] = nxt;
        }
    } else if constexpr (in.kind == IN_STRIDED) {
        const T* src = reinterpret_cast<const T*>(a.in_ptr[K]);
#pragma unroll
        for (int u = 0; u < M::U; ++u)
#pragma unroll
            for (int e = 0; e < M::V; ++e)
                v[in.reg][u * M::V + e] = __ldg(src + (base + (int64_t)M::vidx(u) * M::V + e) * a.in_stride[K]);
    } else if constexpr (in.kind == IN_BOOLVEC) {
        const uint8_t* src = reinterpret_cast<const uint8_t*>(a.in_ptr[K]) + base;
#pragma unroll
        for (int u = 0; u < M::U; ++u)
#pragma unroll
            for (int e = 0; e < M::V; ++e) p[in.reg][u * M::V + e] = src[(size_t)M::vidx(u) * M::V + e] != 0;
    }
    // IN_SCALAR / IN_IMM are broadcast once before the tile loop
}
template <class P, int... K>
__device__ __forceinline__ void load_inputs_full(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][Meta1D<P>::E],
                                                 bool (&p)[Meta1D<P>::NP][Meta1D<P>::E], const SgArgs& a, int64_t base,
                                                 std::integer_sequence<int, K...>) {
    (load_input_full<P, K>(v, p, a, base), ...);
}

template <class P, int E, int K>
__device__ __forceinline__ void bcast_input(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][E], const SgArgs& a) {
    typedef typename Meta1D<P>::T T;
    constexpr SgIn in = P::prog.in[K];
    if constexpr (in.kind == IN_SCALAR || in.kind == IN_IMM) {
        T s = load_elem<T>(in.kind, in.ref, K, a, 0);
#pragma unroll
        for (int e = 0; e < E; ++e) v[in.reg][e] = s;
    }
}
template <class P, int E, int... K>
__device__ __forceinline__ void bcast_inputs(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][E], const SgArgs& a, std::integer_sequence<int, K...>) {
    (bcast_input<P, E, K>(v, a), ...);
}

// ---- outputs of one full tile --------------------------------------------------------------------------
template <class P, int O>
__device__ __forceinline__ void emit_output_full(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][Meta1D<P>::E],
                                                 bool (&p)[Meta1D<P>::NP][Meta1D<P>::E], Cell (&acc)[Meta1D<P>::NOUT],
                                                 const SgArgs& a, int64_t base) {
    typedef Meta1D<P> M;
    typedef typename M::T T;
    typedef typename M::VEC VEC;
    constexpr SgOut out = P::prog.out[O];
    if constexpr (out.kind == OUT_STORE) {
        VEC* dst = reinterpret_cast<VEC*>(reinterpret_cast<T*>(a.out_ptr[O]) + base);
#pragma unroll
        for (int u = 0; u < M::U; ++u) {
            VEC x;
            T* xe = reinterpret_cast<T*>(&x);
#pragma unroll
            for (int e = 0; e < M::V; ++e) xe[e] = v[out.src][u * M::V + e];
            st_stream(dst + M::vidx(u), x);
        }
    } else if constexpr (out.kind == OUT_STORE_BOOL) {
        uint8_t* dst = reinterpret_cast<uint8_t*>(a.out_ptr[O]) + base;
#pragma unroll
        for (int u = 0; u < M::U; ++u)
#pragma unroll
            for (int e = 0; e < M::V; ++e) dst[(size_t)M::vidx(u) * M::V + e] = p[out.src][u * M::V + e];
    } else if constexpr (out_is_pred_reduction(out.kind)) {
#pragma unroll
        for (int e = 0; e < M::E; ++e) cell_accum_pred(out.kind, acc[O], p[out.src][e]);
    } else if constexpr (out_is_reduction(out.kind)) {
#pragma unroll
        for (int e = 0; e < M::E; ++e) {
            if constexpr (out.pred == SG_NO_PRED) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]);
            else if (p[out.pred][e]) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]);
        }
    }
}
template <class P, int... O>
__device__ __forceinline__ void emit_outputs_full(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][Meta1D<P>::E],
                                                  bool (&p)[Meta1D<P>::NP][Meta1D<P>::E], Cell (&acc)[Meta1D<P>::NOUT],
                                                  const SgArgs& a, int64_t base, std::integer_sequence<int, O...>) {
    (emit_output_full<P, O>(v, p, acc, a, base), ...);
}

// ---- one ragged element (head / tail), E = 1 -----------------------------------------------------------
template <class P, int K>
__device__ __forceinline__ void load_input_one(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][1], bool (&p)[Meta1D<P>::NP][1],
                                               const SgArgs& a, int64_t i) {
    typedef typename Meta1D<P>::T T;
    constexpr SgIn in = P::prog.in[K];
    if constexpr (in.kind == IN_BOOLVEC) p[in.reg][0] = (i < a.in_len[K]) && reinterpret_cast<const volatile uint8_t*>(a.in_ptr[K])[i] != 0;
    else if constexpr (in.kind != IN_SCALAR && in.kind != IN_IMM) v[in.reg][0] = load_elem<T>(in.kind, in.ref, K, a, i);
}
template <class P, int O>
__device__ __forceinline__ void emit_output_one(typename Meta1D<P>::T (&v)[Meta1D<P>::NV][1], bool (&p)[Meta1D<P>::NP][1],
                                                Cell (&acc)[Meta1D<P>::NOUT], const SgArgs& a, int64_t i) {
    typedef typename Meta1D<P>::T T;
    constexpr SgOut out = P::prog.out[O];
    if (i >= a.out_len[O]) return;
    if constexpr (out.kind == OUT_STORE) reinterpret_cast<T*>(a.out_ptr[O])[i] = v[out.src][0];
    else if constexpr (out.kind == OUT_STORE_BOOL) reinterpret_cast<uint8_t*>(a.out_ptr[O])[i] = p[out.src][0];
    else if constexpr (out_is_pred_reduction(out.kind)) cell_accum_pred(out.kind, acc[O], p[out.src][0]);
    else if constexpr (out_is_reduction(out.kind)) {
        if constexpr (out.pred == SG_NO_PRED) cell_accum_value<T>(out.kind, acc[O], v[out.src][0]);
        else if (p[out.pred][0]) cell_accum_value<T>(out.kind, acc[O], v[out.src][0]);
    }
}
template <class P, int... K, int... I, int... O>
__device__ __forceinline__ void ragged_range(Cell (&acc)[Meta1D<P>::NOUT], const SgArgs& a, int64_t lo, int64_t hi, int64_t start,
                                             int64_t step, std::integer_sequence<int, K...> ks, std::integer_sequence<int, I...> is,
                                             std::integer_sequence<int, O...>) {
    typedef Meta1D<P> M;
    typename M::T v[M::NV][1];
    bool p[M::NP][1];
    bcast_inputs<P, 1>(v, a, ks);
    for (int64_t i = lo + start; i < hi; i += step) {
        (load_input_one<P, K>(v, p, a, i), ...);
        exec_body<P, typename M::T, M::NV, M::NP, 1>(v, p, a, is);
        (emit_output_one<P, O>(v, p, acc, a, i), ...);
    }
}

// ---- the kernel ----------------------------------------------------------------------------------------
template <class P>
__global__ void __launch_bounds__(BLOCK, P::min_blocks) pass1d_template(const __grid_constant__ SgArgs a) {
    typedef Meta1D<P> M;
    typedef typename M::T T;
    constexpr auto KS = std::make_integer_sequence<int, M::S.n_in>{};
    constexpr auto IS = std::make_integer_sequence<int, M::S.n_instr>{};
    constexpr auto OS = std::make_integer_sequence<int, M::S.n_out>{};

    constexpr SgProg g = P::prog;     // local constant copy: indexable inside unrolled loops
    pdl_wait();
    pdl_trigger();
    Cell acc[M::NOUT];
    uint8_t kind[M::NOUT];
    bool has_reduction = false;
#pragma unroll
    for (int o = 0; o < M::NOUT; ++o) {
        kind[o] = (o < M::S.n_out) ? g.out[o].kind : (uint8_t)OUT_STORE;
        acc[o] = cell_identity<T>(kind[o]);
        has_reduction |= out_is_reduction(kind[o]);
    }
    unsigned int need_mask = 0, flagged = 0;
    __shared__ unsigned int s_decided;          // early-exit passes: the decided word as warp 0 last saw it
    if constexpr (M::early_exit) {
#pragma unroll
        for (int o = 0; o < M::S.n_out; ++o) need_mask |= 1u << o;
        if (threadIdx.x == 0) s_decided = 0;
        __syncthreads();
    }

    {
        T v[M::NV][M::E];
        bool p[M::NP][M::E];
        bcast_inputs<P, M::E>(v, a, KS);
        unsigned int it = 0;
        for (int64_t tile = blockIdx.x; tile < a.static_tiles; tile += gridDim.x, ++it) {
            // every POLL-th tile the decided word is requested BEHIND the tile's loads and examined after the tile is processed, so the
            // poll costs no round trip of its own.  ONE warp per block asks and passes what it saw to the block through shared memory;
            // the other warps read it at their own next poll point (no barrier: a stale value only delays the exit).  Measured on
            // config 3 (2^28 fp32, 740 blocks, 16 KiB tiles, warp-contiguous layout), clean pass / time to answer for a violation at
            // n/64, 20 %, n/2 of the vector:
            //   every warp polls, load in front of the tile's loads, every 2nd / 4th / 8th tile / never:  0.193 / 0.171 / 0.162 / 0.160 ms
            //   one warp per block, in front of the loads, every 2nd tile:                                0.177 ms / 17, 43, 86 us
            //   one warp per block, behind the loads, every 2nd / 3rd / 4th / 6th tile:                   0.168 / 0.167 / 0.166 / 0.166 ms,
            //                                                                  to answer 17, 40, 82 / 21, 41, 86 / 25, 48, 86 / 33, 50, 97 us
            // (a load in front of the tile's loads holds the warp's tile loads back by one L2 round trip per poll, and that warp then
            // finishes last; ld.relaxed.gpu and ld.global.cg cost the same)
#ifndef SG_POLL
#define SG_POLL 2
#endif
            constexpr unsigned int POLL = SG_POLL;
            unsigned int decided_word = 0;
            const bool poll = M::early_exit && !a.no_early_exit && (it % POLL) == 0;
            const int64_t base = a.head + tile * M::TILE;
            load_inputs_full<P>(v, p, a, base, KS);
            if constexpr (M::early_exit) {
                if (poll && threadIdx.x < 32) decided_word = ld_relaxed_u32(&a.ctrl[1]);
            }
            exec_body<P, T, M::NV, M::NP, M::E>(v, p, a, IS);
            emit_outputs_full<P>(v, p, acc, a, base, OS);
            if constexpr (M::early_exit) {
                if (poll) {
#pragma unroll
                    for (int o = 0; o < M::S.n_out; ++o) {
                        bool decided = (kind[o] == OUT_ALL) ? (acc[o].a == 0) : (acc[o].a != 0);
                        if (!(flagged & (1u << o)) && __any_sync(0xffffffffu, decided)) {
                            flagged |= 1u << o;
                            if ((threadIdx.x & 31) == 0) atomicOr(&a.ctrl[1], 1u << o);
                        }
                    }
                    if (threadIdx.x < 32) {
                        if (decided_word != 0 && threadIdx.x == 0) *reinterpret_cast<volatile unsigned int*>(&s_decided) = decided_word;
                    } else decided_word = *reinterpret_cast<volatile unsigned int*>(&s_decided);
                    if ((decided_word & need_mask) == need_mask || (decided_word & a.exit_any) != 0) break;
                }
            }
        }
        // The tiles after static_tiles are handed out one by one through a ticket on ctrl[2], fetched one tile ahead by thread 0
        // behind the tile's own loads.  Equal static shares finish at different times on this part (read-only stream over 592
        // blocks: the median block is done 10 us before the last of 156 us; a 1R+1W stream: 100 us of 372 us, SM pairs differ 2x in
        // write throughput), tickets over the last part of the body let every block finish together (profiles/r02_grid_shape.md).
        // Which block gets which of these tiles differs from run to run, so the host enables tickets only for passes whose
        // reductions are exact in any order (integer sums, max/min, counts, quantifiers) and that have no early exit; a pass with a
        // floating-point sum keeps the static order and returns the same bits on every run (sg_kernels.cu has the measurements of
        // both, and of per-ticket partial cells that would make the sums order-independent: they cost what the tickets gain).
        if constexpr (M::tickets) {
            if (a.static_tiles < a.n_full_tiles) {
                __shared__ long long s_tile[2];
                if (threadIdx.x == 0) s_tile[0] = a.static_tiles + atomicAdd(&a.ctrl[2], 1u);
                __syncthreads();
                for (int buf = 0;; buf ^= 1) {
                    const int64_t tile = s_tile[buf];
                    if (tile >= a.n_full_tiles) break;
                    const int64_t base = a.head + tile * M::TILE;
                    load_inputs_full<P>(v, p, a, base, KS);
                    unsigned int ticket = 0;
                    if (threadIdx.x == 0) ticket = atomicAdd(&a.ctrl[2], 1u);
                    exec_body<P, T, M::NV, M::NP, M::E>(v, p, a, IS);
                    emit_outputs_full<P>(v, p, acc, a, base, OS);
                    if (threadIdx.x == 0) s_tile[buf ^ 1] = a.static_tiles + ticket;
                    __syncthreads();
                }
            }
        }
    }
    // ragged head [0, head) and tail [head + full tiles, n): spread over the grid's threads
    {
        const int64_t gtid = (int64_t)blockIdx.x * BLOCK + threadIdx.x, gstep = (int64_t)gridDim.x * BLOCK;
        ragged_range<P>(acc, a, 0, a.head, gtid, gstep, KS, IS, OS);
        ragged_range<P>(acc, a, a.head + a.n_full_tiles * M::TILE, a.n, gtid, gstep, KS, IS, OS);
    }
    epilogue_1d<T, M::NOUT>(acc, kind, a, has_reduction);
}

}  // namespace sgk
#endif  // SG_PASS1D_TMPL_CUH_
