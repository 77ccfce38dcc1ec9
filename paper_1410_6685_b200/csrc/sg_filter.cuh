// sg_filter.cuh — stream-compacting filter pass (filter).
//
// One pass over the input: the predicate chain is evaluated in registers, kept elements are ranked by a
// warp-ballot prefix inside the tile and by a decoupled look-back over per-tile aggregates across tiles, and
// written in ascending index order (STABLE, R3).  Count and any reductions over the kept values
// (masked reductions) are produced by the same pass.
//
// Tile layout: warp-blocked.  A tile is BLOCK*U*FW elements (32 KiB for one input); warp w owns U*32*FW
// consecutive elements, and in step u lane l owns the FW consecutive elements at
//     tile + w*U*32*FW + u*32*FW + l*FW
// so the order (warp, u, lane, e) is memory order and a ballot over lanes ranks them.
//
// Staging: full tiles of 16-byte aligned inputs are brought into an NS-stage shared-memory ring by ONE bulk
// asynchronous copy per input per tile (cp.async.bulk, the TMA engine; completion on an mbarrier), issued
// NS-2 tiles ahead by thread 0 — the bytes in flight do not depend on which phase (evaluate / rank / look-back /
// copy-out) the block is in.  The kept values are compacted IN PLACE into the stage they came from (every
// thread holds its elements in registers by then) and copied out coalesced.
//
// Look-back: at B200 rates a tile completes every few nanoseconds chip-wide, so a window of 32 predecessors per
// L2 round trip never catches up with the tiles in flight, and under a saturated memory system one round trip
// costs microseconds (measured: 17 us per tile with the textbook one-warp, one-window-at-a-time look-back).
// Warp 0 therefore requests LB = 8 windows (256 tile states) at once and examines them ONE TILE LATER: the
// round trip overlaps the evaluation of the block's next tile (software pipeline, see filter_body).
//
// Tile ids are handed out by an atomic counter, NS tiles ahead per block; a block processes its claims in
// increasing order, so the smallest unpublished tile is always held by a running block (forward progress).
// Tile state word: [63:62] flag (1 aggregate, 2 inclusive prefix) | [61:40] launch epoch | [39:0] count.
#ifndef SG_FILTER_CUH_
#define SG_FILTER_CUH_

#include "sg_bulk.cuh"
#include "sg_pass1d_tmpl.cuh"
#include "sg_pass1d_vm.cuh"

namespace sgk {

constexpr unsigned long long ST_AGG = 1ull << 62, ST_INC = 2ull << 62, ST_FLAGS = 3ull << 62;
constexpr unsigned long long ST_VAL = (1ull << 40) - 1;
constexpr int LB = 8;       // look-back windows (of 32 tile states) requested per round trip

__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_state(unsigned long long* p, unsigned long long v) {
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// load modes of one step: guarded element loads (ragged / misaligned), 128-bit global loads, shared-memory stage
enum { FM_GUARDED = 0, FM_GLOBAL = 1, FM_STAGED = 2 };

// ---- evaluators: produce, for the FW elements at index i, the candidate values and the keep bits ----------
template <class P> struct FilterTemplateEval {
    typedef Meta1D<P> M;
    typedef typename M::T T;
    static constexpr int NOUT = M::NOUT;
    static constexpr int FW = 16 / (int)sizeof(T);       // elements per thread per step (one 128-bit access)
    static constexpr int count_vec() {
        int n = 0;
        for (int k = 0; k < M::S.n_in; ++k) n += (P::prog.in[k].kind == IN_VEC);
        return n;
    }
    static constexpr int NVEC_REAL = count_vec();
    static constexpr int U = NVEC_REAL <= 1 ? 4 * P::unroll : 4;     // steps per tile: 16 KiB per step-quadruple and input
    static constexpr int TILE = BLOCK * U * FW;
    static constexpr int NS = P::row_unroll >= 3 ? P::row_unroll : 3;   // buffers in the ring (the pipeline needs >= 3)
    static constexpr bool STAGED = NVEC_REAL >= 1 && (size_t)NS * NVEC_REAL * TILE * sizeof(T) <= 200 * 1024;
    static constexpr int NVEC = STAGED ? NVEC_REAL : 1;
    static constexpr size_t SMEM = (size_t)NS * NVEC * TILE * sizeof(T) + NS * sizeof(uint64_t);
    __host__ __device__ static constexpr int vec_slot(int K) {
        int n = 0;
        for (int k = 0; k < K; ++k) n += (P::prog.in[k].kind == IN_VEC);
        return n;
    }

    // thread 0: one bulk copy per IN_VEC input for tile t into stage buffer `dst` ([NVEC][TILE])
    template <int... K>
    __device__ __forceinline__ static void issue_(const SgArgs& a, int64_t tbase, T* dst, uint64_t* bar, std::integer_sequence<int, K...>) {
        mbar_expect_tx(bar, (uint32_t)(NVEC_REAL * TILE * sizeof(T)));
        ((P::prog.in[K].kind == IN_VEC
              ? bulk_g2s(dst + (size_t)vec_slot(K) * TILE, reinterpret_cast<const T*>(a.in_ptr[K]) + tbase, (uint32_t)(TILE * sizeof(T)), bar)
              : (void)0),
         ...);
    }
    __device__ __forceinline__ static void issue(const SgProg*, const SgArgs& a, int64_t tbase, T* dst, uint64_t* bar) {
        issue_(a, tbase, dst, bar, std::make_integer_sequence<int, M::S.n_in>{});
    }

    template <int MODE, int K>
    __device__ __forceinline__ static void load_k(T (&v)[M::NV][FW], bool (&p)[M::NP][FW], const SgArgs& a, int64_t i, const T* stage, int toff) {
        typedef typename M::VEC VEC;
        constexpr SgIn in = P::prog.in[K];
        if constexpr (in.kind == IN_SCALAR || in.kind == IN_IMM) {
            T s = load_elem<T>(in.kind, in.ref, K, a, 0);
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = s;
        } else if constexpr (in.kind == IN_BOOLVEC) {
#pragma unroll
            for (int e = 0; e < FW; ++e) p[in.reg][e] = (i + e < a.in_len[K]) && reinterpret_cast<const volatile uint8_t*>(a.in_ptr[K])[i + e] != 0;
        } else if constexpr (in.kind == IN_VEC && MODE != FM_GUARDED) {
            VEC w;
            if constexpr (MODE == FM_STAGED) w = *reinterpret_cast<const VEC*>(stage + (size_t)vec_slot(K) * TILE + toff);
            else w = ld_stream(reinterpret_cast<const VEC*>(reinterpret_cast<const T*>(a.in_ptr[K]) + i));
            const T* we = reinterpret_cast<const T*>(&w);
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = we[e];
        } else {
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = load_elem<T>(in.kind, in.ref, K, a, i + e);
        }
    }
    template <int MODE, int O>
    __device__ __forceinline__ static void out_o(T (&v)[M::NV][FW], bool (&p)[M::NP][FW], const SgArgs& a, int64_t i, T (&val)[FW],
                                                 unsigned int& keep, Cell (&acc)[NOUT]) {
        constexpr SgOut out = P::prog.out[O];
#pragma unroll
        for (int e = 0; e < FW; ++e) {
            const bool in_range = (MODE != FM_GUARDED) || (i + e < a.out_len[O]);     // full tiles lie inside every output's length
            if constexpr (out.kind == OUT_FILTER) {
                val[e] = v[out.src][e];
                keep |= (unsigned int)(in_range && p[out.pred][e]) << e;
            } else if constexpr (out_is_pred_reduction(out.kind)) {
                if (in_range) cell_accum_pred(out.kind, acc[O], p[out.src][e]);
            } else if constexpr (out_is_reduction(out.kind)) {
                if constexpr (out.pred == SG_NO_PRED) { if (in_range) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]); }
                else if constexpr (out.kind == OUT_SUM && !Traits<T>::is_float) {
                    // masked integer sum as one widening multiply-add: acc += x * (0 or 1)
                    acc[O].a += (unsigned long long)((long long)v[out.src][e] * (long long)(int)(in_range && p[out.pred][e]));
                } else { if (in_range && p[out.pred][e]) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]); }
            }
        }
    }
    template <int MODE, int... K, int... I, int... O>
    __device__ __forceinline__ static void run_(const SgArgs& a, int64_t i, const T* stage, int toff, T (&val)[FW], unsigned int& keep, Cell (&acc)[NOUT],
                                                std::integer_sequence<int, K...>, std::integer_sequence<int, I...> is, std::integer_sequence<int, O...>) {
        T v[M::NV][FW];
        bool p[M::NP][FW];
        (load_k<MODE, K>(v, p, a, i, stage, toff), ...);
        exec_body<P, T, M::NV, M::NP, FW>(v, p, a, is);
        keep = 0;
        (out_o<MODE, O>(v, p, a, i, val, keep, acc), ...);
    }
    template <int MODE>
    __device__ __forceinline__ static void run(const SgProg*, const SgArgs& a, int64_t i, const T* stage, int toff, T (&val)[FW], unsigned int& keep,
                                               Cell (&acc)[NOUT]) {
        run_<MODE>(a, i, stage, toff, val, keep, acc, std::make_integer_sequence<int, M::S.n_in>{}, std::make_integer_sequence<int, M::S.n_instr>{},
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
    static constexpr int TILE = BLOCK * U * FW;
    static constexpr int NVEC = 1, NS = 3;
    static constexpr bool STAGED = false;
    static constexpr size_t SMEM = (size_t)NS * TILE * sizeof(T) + NS * sizeof(uint64_t);
    __device__ __forceinline__ static void issue(const SgProg*, const SgArgs&, int64_t, T*, uint64_t*) {}
    template <int MODE>
    __device__ __forceinline__ static void run(const SgProg* g, const SgArgs& a, int64_t i, const T*, int, T (&val)[FW], unsigned int& keep, Cell (&acc)[NOUT]) {
        const bool full = MODE != FM_GUARDED;
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
// Software pipeline over the tiles a block claims (iteration `it` uses stage it % NS):
//   wait for the stage -> evaluate -> ballot ranks -> barrier 1 -> thread 0 refills the stage freed in the previous
//   iteration; warp 0 PUBLISHES this tile's aggregate, RESOLVES the look-back of the PREVIOUS tile from the tile
//   states it requested one iteration ago, and REQUESTS this tile's LB windows; every warp scatters its kept items in
//   place (tile-local order) -> barrier 2 -> coalesced copy-out of the PREVIOUS tile at its now known global offset.
// The look-back round trip (several microseconds under a saturated memory system) is thus overlapped with a whole
// tile of work, and an aggregate is published without waiting for any predecessor.
template <class EV, int MODE>
__device__ __forceinline__ void filter_eval_tile(const SgProg* g, const SgArgs& a, int64_t tbase, const typename EV::T* stage,
                                                 typename EV::T (&val)[EV::U][EV::FW], unsigned int (&keep)[EV::U], Cell (&acc)[EV::NOUT]) {
    constexpr int U = EV::U, FW = EV::FW;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int u = 0; u < U; ++u) {
        const int toff = warp * (U * 32 * FW) + u * (32 * FW) + lane * FW;
        EV::template run<MODE>(g, a, tbase + toff, stage, toff, val[u], keep[u], acc);
    }
}

template <class EV>
__device__ __forceinline__ void filter_body(const SgProg* g, const SgArgs& a) {
    typedef typename EV::T T;
    constexpr int U = EV::U, FW = EV::FW, TILE = EV::TILE, NOUT = EV::NOUT, NS = EV::NS, NVEC = EV::NVEC;
    extern __shared__ __align__(128) unsigned char dyn_smem[];
    T* const stage_base = reinterpret_cast<T*>(dyn_smem);                                   // [NS][NVEC][TILE]
    uint64_t* const full_bar = reinterpret_cast<uint64_t*>(dyn_smem + (size_t)NS * NVEC * TILE * sizeof(T));
    __shared__ int s_tile[NS];
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
    const bool staged = EV::STAGED && all_vec;

    if (a.n_tiles == 0 && blockIdx.x == 0 && threadIdx.x == 0) *reinterpret_cast<long long*>(a.out_aux[fo]) = 0;

    // claim NS tiles; their bulk copies are in flight before the first one is touched
    if (threadIdx.x == 0) {
        if (staged) {
            for (int s = 0; s < NS; ++s) mbar_init(&full_bar[s], 1);
            mbar_fence_init();
        }
        for (int s = 0; s < NS; ++s) {
            const int t = (int)atomicAdd(&a.ctrl[2], 1u);
            s_tile[s] = t;
            if (staged && t < a.n_full_tiles) EV::issue(g, a, (int64_t)t * TILE, stage_base + (size_t)s * NVEC * TILE, &full_bar[s]);
        }
    }
    __syncthreads();

    // state of the previous tile (resolved and copied out one iteration later)
    int prev_tile = -1;
    unsigned int prev_total = 0;
    T* prev_cbuf = nullptr;
    unsigned long long lbw[LB];         // warp 0: tile states requested for the previous tile's look-back
#pragma unroll
    for (int j = 0; j < LB; ++j) lbw[j] = 0;

    for (int it = 0;; ++it) {
        const int s = it % NS;
        const int tile = s_tile[s];
        const bool active = tile < a.n_tiles;
        if (!active && prev_tile < 0) break;
        T* const cbuf = stage_base + (size_t)s * NVEC * TILE;    // this tile's stage; slot 0 becomes the compaction buffer

        T val[U][FW];
        unsigned int keep[U], off[U];
        unsigned int running = 0;
        if (active) {
            const int64_t tbase = (int64_t)tile * TILE;
            const bool full = all_vec && tile < a.n_full_tiles;  // inside every operand's and output's length
            if (staged && full) {
                mbar_wait(&full_bar[s], (uint32_t)((it / NS) & 1));
                filter_eval_tile<EV, FM_STAGED>(g, a, tbase, cbuf, val, keep, acc);
            } else if (full) {
                filter_eval_tile<EV, FM_GLOBAL>(g, a, tbase, cbuf, val, keep, acc);
            } else {
                filter_eval_tile<EV, FM_GUARDED>(g, a, tbase, cbuf, val, keep, acc);
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
        }
        __syncthreads();        // 1: this tile's stage has been read into registers; warp totals visible; the previous
                                //    iteration's copy-out (of tile it-2's ... it-1's predecessor stage) is complete
        // the stage of tile it-2 was copied out during iteration it-1: refill it for iteration it+NS-2
        if (threadIdx.x == 0 && it >= 2) {
            const int sr = (it - 2) % NS;
            const int t = (int)atomicAdd(&a.ctrl[2], 1u);
            s_tile[sr] = t;                                     // read at the top of iteration it+NS-2, behind barrier 2
            if (staged && t < a.n_full_tiles) {
                fence_proxy_async();
                EV::issue(g, a, (int64_t)t * TILE, stage_base + (size_t)sr * NVEC * TILE, &full_bar[sr]);
            }
        }
        unsigned int warp_excl = 0, tile_total = 0;
        if (active) {
#pragma unroll
            for (int w = 0; w < WARPS; ++w) {
                const unsigned int t = s_warp_total[w];
                if (w < warp) warp_excl += t;
                tile_total += t;
            }
        }
        if (warp == 0) {
            // (a) publish this tile's aggregate: it never waits for a predecessor
            if (active && lane == 0) st_state(&state[tile], (tile == 0 ? ST_INC : ST_AGG) | ep | (unsigned long long)tile_total);
            // (b) resolve the previous tile's look-back from the states requested one iteration ago
            if (prev_tile >= 0) {
                unsigned long long excl = 0;
                if (prev_tile != 0) {
                    int look = prev_tile - 1;
                    for (;;) {
                        // ballots of all LB windows first (independent), then ONE position search and ONE warp sum
                        int p_inc = LB * 32, p_inv = LB * 32;       // first inclusive prefix / first unpublished state, in (window, lane) order
#pragma unroll
                        for (int j = LB - 1; j >= 0; --j) {
                            const unsigned long long w = lbw[j];
                            const bool valid = ((w & ST_FLAGS) != 0) && ((w & (0x3fffffull << 40)) == ep);
                            const bool inc = valid && ((w & ST_FLAGS) == ST_INC);
                            const unsigned int vmask = __ballot_sync(0xffffffffu, valid), imask = __ballot_sync(0xffffffffu, inc);
                            if (imask) p_inc = 32 * j + __ffs(imask) - 1;
                            if (~vmask) p_inv = 32 * j + __ffs(~vmask) - 1;
                        }
                        // contributing states: up to and including the first inclusive prefix, else every state before the first unpublished one
                        const bool done = p_inc < p_inv;
                        const int upto = done ? p_inc + 1 : p_inv;
                        unsigned long long x = 0;
#pragma unroll
                        for (int j = 0; j < LB; ++j)
                            if (32 * j + lane < upto) x += lbw[j] & ST_VAL;
#pragma unroll
                        for (int d = 16; d >= 1; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
                        excl += x;
                        if (done) break;
                        look -= upto;       // go deeper, or poll again from the predecessor that has not published yet
#pragma unroll
                        for (int j = 0; j < LB; ++j) {
                            const int idx = look - lane - 32 * j;
                            lbw[j] = (idx >= 0) ? ld_state(&state[idx]) : (ST_INC | ep);
                        }
                    }
                    if (lane == 0) st_state(&state[prev_tile], ST_INC | ep | (excl + prev_total));
                }
                if (lane == 0) {
                    s_tile_excl = excl;
                    if (prev_tile == a.n_tiles - 1) *reinterpret_cast<long long*>(a.out_aux[fo]) = (long long)(excl + prev_total);
                }
            }
            // (c) request this tile's LB windows of predecessor states; they are examined in the next iteration
            if (active) {
#pragma unroll
                for (int j = 0; j < LB; ++j) {
                    const int idx = tile - 1 - lane - 32 * j;
                    lbw[j] = (idx >= 0) ? ld_state(&state[idx]) : (ST_INC | ep);    // virtual tile -1: inclusive prefix 0
                }
            }
        }
        if (active) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                unsigned int pos = warp_excl + off[u];
#pragma unroll
                for (int e = 0; e < FW; ++e)
                    if ((keep[u] >> e) & 1u) cbuf[pos++] = val[u][e];
            }
        }
        __syncthreads();        // 2: the previous tile's global offset is known (and this tile is compacted)
        if (prev_tile >= 0) {
            const long long tile_excl = (long long)s_tile_excl;
            bool overflow = false;
            for (unsigned int i = threadIdx.x; i < prev_total; i += BLOCK) {
                const long long pos = tile_excl + i;
                if (pos < cap) dst[pos] = prev_cbuf[i]; else overflow = true;
            }
            if (overflow) a.ctrl[3] = 1u;
        }
        prev_tile = active ? tile : -1;
        prev_total = tile_total;
        prev_cbuf = cbuf;
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
