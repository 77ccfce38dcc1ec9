// sg_filter.cuh — stream-compacting filter pass (filter).
//
// One pass over the input: the predicate chain is evaluated in registers, kept elements are ranked by a
// warp-ballot prefix inside the tile and by a decoupled look-back over per-tile aggregates across tiles, and
// written in ascending index order (STABLE, R3).  Count and any reductions over the kept values
// (masked reductions) are produced by the same pass.
//
// Tile layout: warp-blocked.  A tile is BLOCK*U*W elements; warp w owns U*32*W consecutive elements, and in
// step u lane l owns the W consecutive elements at  tile + w*U*32*W + u*32*W + l*W  — so the order
// (warp, u, lane, e) is memory order and a ballot over lanes ranks them.
// Tile ids are handed out by an atomic counter (a tile is only claimed by a running block: forward progress).
// Tile state word: [63:62] flag (1 aggregate, 2 inclusive prefix) | [61:40] launch epoch | [39:0] count.
#ifndef SG_FILTER_CUH_
#define SG_FILTER_CUH_

#include "sg_pass1d_tmpl.cuh"
#include "sg_pass1d_vm.cuh"

namespace sgk {

constexpr unsigned long long ST_AGG = 1ull << 62, ST_INC = 2ull << 62, ST_FLAGS = 3ull << 62;
constexpr unsigned long long ST_VAL = (1ull << 40) - 1;

__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_state(unsigned long long* p, unsigned long long v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// ---- evaluators: produce, for the FW elements at index i, the candidate values and the keep bits ----------
template <class P> struct FilterTemplateEval {
    typedef Meta1D<P> M;
    typedef typename M::T T;
    static constexpr int NOUT = M::NOUT;
    static constexpr int U = 4;                          // steps per tile
    static constexpr int FW = 16 / (int)sizeof(T);       // elements per thread per step (one 128-bit access)

    template <int K>
    __device__ __forceinline__ static void load_k(T (&v)[M::NV][FW], bool (&p)[M::NP][FW], const SgArgs& a, int64_t i, bool full) {
        typedef typename M::VEC VEC;
        constexpr SgIn in = P::prog.in[K];
        if constexpr (in.kind == IN_SCALAR || in.kind == IN_IMM) {
            T s = load_elem<T>(in.kind, in.ref, K, a, 0);
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = s;
        } else if constexpr (in.kind == IN_BOOLVEC) {
#pragma unroll
            for (int e = 0; e < FW; ++e) p[in.reg][e] = (i + e < a.in_len[K]) && reinterpret_cast<const volatile uint8_t*>(a.in_ptr[K])[i + e] != 0;
        } else {
            if (in.kind == IN_VEC && full) {
                const VEC* src = reinterpret_cast<const VEC*>(reinterpret_cast<const T*>(a.in_ptr[K]) + i);
#pragma unroll
                for (int u = 0; u < FW / M::V; ++u) {
                    VEC w = ld_stream(src + u);
                    const T* we = reinterpret_cast<const T*>(&w);
#pragma unroll
                    for (int e = 0; e < M::V; ++e) v[in.reg][u * M::V + e] = we[e];
                }
            } else {
#pragma unroll
                for (int e = 0; e < FW; ++e) v[in.reg][e] = load_elem<T>(in.kind, in.ref, K, a, i + e);
            }
        }
    }
    template <int O>
    __device__ __forceinline__ static void out_o(T (&v)[M::NV][FW], bool (&p)[M::NP][FW], const SgArgs& a, int64_t i, T (&val)[FW],
                                                 unsigned int& keep, Cell (&acc)[NOUT]) {
        constexpr SgOut out = P::prog.out[O];
#pragma unroll
        for (int e = 0; e < FW; ++e) {
            const bool in_range = i + e < a.out_len[O];
            if constexpr (out.kind == OUT_FILTER) {
                val[e] = v[out.src][e];
                keep |= (unsigned int)(in_range && p[out.pred][e]) << e;
            } else if constexpr (out_is_pred_reduction(out.kind)) {
                if (in_range) cell_accum_pred(out.kind, acc[O], p[out.src][e]);
            } else if constexpr (out_is_reduction(out.kind)) {
                if constexpr (out.pred == SG_NO_PRED) { if (in_range) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]); }
                else { if (in_range && p[out.pred][e]) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]); }
            }
        }
    }
    template <int... K, int... I, int... O>
    __device__ __forceinline__ static void run_(const SgArgs& a, int64_t i, bool full, T (&val)[FW], unsigned int& keep, Cell (&acc)[NOUT],
                                                std::integer_sequence<int, K...>, std::integer_sequence<int, I...> is, std::integer_sequence<int, O...>) {
        T v[M::NV][FW];
        bool p[M::NP][FW];
        (load_k<K>(v, p, a, i, full), ...);
        exec_body<P, T, M::NV, M::NP, FW>(v, p, a, is);
        keep = 0;
        (out_o<O>(v, p, a, i, val, keep, acc), ...);
    }
    __device__ __forceinline__ static void run(const SgProg*, const SgArgs& a, int64_t i, bool full, T (&val)[FW], unsigned int& keep, Cell (&acc)[NOUT]) {
        run_(a, i, full, val, keep, acc, std::make_integer_sequence<int, M::S.n_in>{}, std::make_integer_sequence<int, M::S.n_instr>{},
             std::make_integer_sequence<int, M::S.n_out>{});
    }
    __device__ __forceinline__ static uint8_t out_kind(const SgProg*, int o) {
        constexpr SgProg g = P::prog;
        return o < M::S.n_out ? g.out[o].kind : (uint8_t)OUT_STORE;
    }
};

template <class TT> struct FilterBytecodeEval {
    typedef TT T;
    static constexpr int NOUT = SG_MAX_OUT;
    static constexpr int U = 4;                          // steps per tile
    static constexpr int FW = 16 / (int)sizeof(T);       // elements per thread per step (one 128-bit access)
    __device__ __forceinline__ static void run(const SgProg* g, const SgArgs& a, int64_t i, bool full, T (&val)[FW], unsigned int& keep, Cell (&acc)[NOUT]) {
        VmRegs<T, FW> rf;
        unsigned int pf = 0;
        for (int k = 0; k < g->shape.n_in; ++k) {
            const SgIn in = g->in[k];
            if (in.kind == IN_SCALAR || in.kind == IN_IMM) {
                T x[FW];
                const T s = load_elem<T>(in.kind, in.ref, k, a, 0);
#pragma unroll
                for (int e = 0; e < FW; ++e) x[e] = s;
                rf.put(in.reg, x);
            } else vm_load<T, FW>(*g, a, k, i, full, rf, pf);
        }
        vm_exec<T, FW>(*g, rf, pf);
        keep = 0;
        for (int o = 0; o < g->shape.n_out; ++o) {
            const SgOut out = g->out[o];
            if (out.kind != OUT_FILTER) continue;
            rf.get(out.src, val);
            const unsigned int bits = pget<FW>(pf, out.pred);
#pragma unroll
            for (int e = 0; e < FW; ++e) keep |= (unsigned int)((i + e < a.out_len[o]) && ((bits >> e) & 1u)) << e;
        }
        vm_emit<T, FW>(*g, a, i, a.n, false, rf, pf, acc);     // reductions only: OUT_FILTER is not a reduction/store kind there
    }
    __device__ __forceinline__ static uint8_t out_kind(const SgProg* g, int o) { return o < g->shape.n_out ? g->out[o].kind : (uint8_t)OUT_STORE; }
};

// ---- the kernel body -------------------------------------------------------------------------------------
// Per tile: evaluate -> ballot ranks -> barrier -> scatter kept items into a shared-memory tile (tile-local order)
// while warp 0 runs the look-back -> barrier -> coalesced copy of the compacted tile to its global position.
// The id of the next tile is fetched (atomicAdd) at the start of the current one, so its latency is hidden.
template <class EV>
__device__ __forceinline__ void filter_body(const SgProg* g, const SgArgs& a) {
    typedef typename EV::T T;
    constexpr int U = EV::U, FW = EV::FW;
    constexpr int TILE = BLOCK * U * FW;
    constexpr int NOUT = EV::NOUT;
    __shared__ T s_vals[TILE];
    __shared__ int s_tile[2];
    __shared__ unsigned int s_warp_total[WARPS];
    __shared__ unsigned long long s_tile_excl;

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int lt_mask = (1u << lane) - 1u;
    Cell acc[NOUT];
    uint8_t kind[NOUT];
    int fo = 0;     // index of the OUT_FILTER output
#pragma unroll
    for (int o = 0; o < NOUT; ++o) {
        kind[o] = EV::out_kind(g, o);
        acc[o] = cell_identity<T>(kind[o]);
        if (kind[o] == OUT_FILTER) fo = o;
    }
    T* const dst = reinterpret_cast<T*>(a.out_ptr[fo]);
    const long long cap = a.out_cap[fo];
    unsigned long long* const state = a.tile_state;
    const unsigned long long ep = ((unsigned long long)(a.epoch & 0x3fffffu)) << 40;
    const bool all_vec = (a.vec_ok >> 31) & 1;

    if (a.n_tiles == 0 && blockIdx.x == 0 && threadIdx.x == 0) *reinterpret_cast<long long*>(a.out_aux[fo]) = 0;

    if (threadIdx.x == 0) s_tile[0] = (int)atomicAdd(&a.ctrl[2], 1u);
    __syncthreads();
    for (int it = 0;; ++it) {
        const int tile = s_tile[it & 1];
        if (tile >= a.n_tiles) break;
        int next_tile = 0;
        if (threadIdx.x == 0) next_tile = (int)atomicAdd(&a.ctrl[2], 1u);      // consumed just before the first barrier
        const int64_t tbase = (int64_t)tile * TILE;
        const bool full = all_vec && (tbase + TILE <= a.n);

        T val[U][FW];
        unsigned int keep[U], off[U];
        unsigned int running = 0;
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int64_t i = tbase + (int64_t)warp * (U * 32 * FW) + u * (32 * FW) + lane * FW;
            EV::run(g, a, i, full, val[u], keep[u], acc);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            // exclusive prefix over lanes of the per-thread keep count (0..4) from three bit-plane ballots
            const unsigned int c = __popc(keep[u]);
            const unsigned int b0 = __ballot_sync(0xffffffffu, c & 1u), b1 = __ballot_sync(0xffffffffu, c & 2u), b2 = __ballot_sync(0xffffffffu, c & 4u);
            off[u] = running + __popc(b0 & lt_mask) + 2 * __popc(b1 & lt_mask) + 4 * __popc(b2 & lt_mask);
            running += __popc(b0) + 2 * __popc(b1) + 4 * __popc(b2);
        }
        if (lane == 0) s_warp_total[warp] = running;
        if (threadIdx.x == 0) s_tile[(it + 1) & 1] = next_tile;
        __syncthreads();
        unsigned int warp_excl = 0, tile_total = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
            const unsigned int t = s_warp_total[w];
            if (w < warp) warp_excl += t;
            tile_total += t;
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            unsigned int pos = warp_excl + off[u];
#pragma unroll
            for (int e = 0; e < FW; ++e)
                if ((keep[u] >> e) & 1u) s_vals[pos++] = val[u][e];
        }
        // decoupled look-back by warp 0 (the other warps are already at the barrier below)
        if (warp == 0) {
            unsigned long long excl = 0;
            if (tile == 0) {
                if (lane == 0) st_state(&state[0], ST_INC | ep | (unsigned long long)tile_total);
            } else {
                if (lane == 0) st_state(&state[tile], ST_AGG | ep | (unsigned long long)tile_total);
                int look = tile - 1;
                for (;;) {
                    const int idx = look - lane;
                    unsigned long long w = (idx >= 0) ? ld_state(&state[idx]) : (ST_INC | ep);   // virtual tile -1: inclusive prefix 0
                    const bool valid = ((w & ST_FLAGS) != 0) && ((w & (0x3fffffull << 40)) == ep);
                    const bool inc = valid && ((w & ST_FLAGS) == ST_INC);
                    const unsigned int vmask = __ballot_sync(0xffffffffu, valid), imask = __ballot_sync(0xffffffffu, inc);
                    const int first_invalid = (~vmask) ? (__ffs(~vmask) - 1) : 32;
                    const int first_inc = imask ? (__ffs(imask) - 1) : 32;
                    if (first_inc < first_invalid) {
                        unsigned long long x = (lane <= first_inc) ? (w & ST_VAL) : 0ull;
#pragma unroll
                        for (int d = 16; d >= 1; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
                        excl += x;
                        break;
                    } else if (first_invalid == 32) {
                        unsigned long long x = w & ST_VAL;
#pragma unroll
                        for (int d = 16; d >= 1; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
                        excl += x;
                        look -= 32;
                    }   // else: a predecessor has not published yet — poll the same window again
                }
                if (lane == 0) st_state(&state[tile], ST_INC | ep | (excl + tile_total));
            }
            if (lane == 0) {
                s_tile_excl = excl;
                if (tile == a.n_tiles - 1) *reinterpret_cast<long long*>(a.out_aux[fo]) = (long long)(excl + tile_total);
            }
        }
        __syncthreads();
        const long long tile_excl = (long long)s_tile_excl;
        bool overflow = false;
        for (unsigned int i = threadIdx.x; i < tile_total; i += BLOCK) {
            const long long pos = tile_excl + i;
            if (pos < cap) dst[pos] = s_vals[i]; else overflow = true;
        }
        if (overflow) a.ctrl[3] = 1u;
        // no third barrier: the next tile's first barrier separates this copy-out from the next scatter
    }
    epilogue_1d<T, NOUT>(acc, kind, a, true);
}

template <class P>
__global__ void __launch_bounds__(BLOCK, P::min_blocks) filter1d_template(const __grid_constant__ SgArgs a) {
    filter_body<FilterTemplateEval<P>>(nullptr, a);
}
template <class T>
__global__ void __launch_bounds__(BLOCK) filter1d_bytecode(const __grid_constant__ SgProg g, const __grid_constant__ SgArgs a) {
    filter_body<FilterBytecodeEval<T>>(&g, a);
}

}  // namespace sgk
#endif  // SG_FILTER_CUH_
