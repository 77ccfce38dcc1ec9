// sg_filter.cuh — stream-compacting filter pass (filter).
//
// One pass over the input: the predicate chain is evaluated in registers, kept elements are ranked inside the tile
// by a per-thread count + warp scan and across tiles by a decoupled look-back over per-tile aggregates, and written
// in ascending index order (STABLE, R3).  Count and reductions over the kept values are produced by the
// same pass.
//
// Tile = 256 rows of 128 bytes (32 KiB per input).  Thread t of the 256 compute threads owns ROW t: its EPT = 32
// (4-byte types) or 16 (8-byte types) elements are CONSECUTIVE in memory, so one popc of its keep mask and one warp
// scan rank the whole tile (no per-element ballots), and it appends its kept values in order.
//
// Staging: full tiles of 16-byte aligned inputs are brought into a 2-stage shared-memory ring by ONE TMA tensor
// copy per input per tile (cp.async.bulk.tensor.2d, completion on an mbarrier), issued two tiles ahead by thread 0.
// The tensor map views the input as rows of 128 bytes and applies the 128-byte swizzle: the 16-byte chunk j of row r
// lands at chunk (j ^ (r & 7)), so thread t reads its own row with conflict-free 128-bit shared loads.  Ragged or
// misaligned tiles are filled cooperatively (coalesced guarded loads, same swizzled layout).
//
// Block = 8 compute warps + 1 look-back warp (warp specialisation).  Kept values go into a shared-memory RING that
// is decoupled from the input stages; a tile waits there until its global offset is known, while the compute warps
// go on with the next tiles.  A block claims RUNS of consecutive tiles: only the first tile of a run needs a
// look-back (the others add the run's local prefix), and once the run's offset is known the later tiles publish
// their inclusive prefix directly.  The look-back warp requests LB = 8 windows (256 tile states) per round trip:
// under a saturated memory system one round trip costs more than a microsecond (measured), and at B200 rates a
// 32-state window never catches up with the tiles in flight.
//
// Tile ids are handed out by an atomic counter; a block processes its claims in increasing order, so the smallest
// unpublished tile is always held by a running block (forward progress).
// Tile state word: [63:62] flag (1 aggregate, 2 inclusive prefix) | [61:40] launch epoch | [39:0] count.
#ifndef SG_FILTER_CUH_
#define SG_FILTER_CUH_

#include "sg_bulk.cuh"
#include "sg_pass1d_tmpl.cuh"
#include "sg_pass1d_vm.cuh"

namespace sgk {

constexpr unsigned long long ST_AGG = 1ull << 62, ST_INC = 2ull << 62, ST_FLAGS = 3ull << 62;
constexpr unsigned long long ST_VAL = (1ull << 40) - 1;
// tuning knobs (overridable at compile time for sweeps; measured on cfg2, 2^27 int32, 1/7 kept — profiles/r02_filter_sweep.md):
//   RUN = 1 / 2 / 3 / 4 / 5 / 6 tiles per run: 167 / 157 / 155 / 154 / 157 / 166 us.  A run is only taken at full length while its
//   kept values fill at most 2/3 of the ring (SG_F_RULE 3/2); round 1's factor 2 silently turned RUN = 4 into RUN = 1 at this
//   selectivity (4 * 1170 * 2 > 8192), which is the 168 us it measured.
//   LB = 2 / 4 / 8 look-back windows per round trip: 154.3 / 154.8 / 155.3 us;  COPY_BATCH 1..4 and the poll back-off: no effect.
#ifndef SG_F_LB
#define SG_F_LB 4
#endif
#ifndef SG_F_RUN
#define SG_F_RUN 4
#endif
#ifndef SG_F_COPY_BATCH
#define SG_F_COPY_BATCH 3
#endif
#ifndef SG_F_RULE_NUM
#define SG_F_RULE_NUM 3
#define SG_F_RULE_DEN 2
#endif
#ifndef SG_F_SLEEP
#define SG_F_SLEEP 500
#endif
constexpr int LB = SG_F_LB;               // look-back windows (of 32 tile states) requested per round trip
constexpr int F_ROWS = 256;         // rows of 128 bytes per tile
constexpr int F_TILE_BYTES = F_ROWS * 128;              // 32 KiB per staged input
constexpr int F_TILE_CHUNKS = F_TILE_BYTES / 16;        // 16-byte chunks per tile
constexpr int RUN = SG_F_RUN;              // consecutive tiles a block claims at once while few values are kept (else 1); one look-back per run
constexpr int NR = 16;              // runs of one block whose offset may be outstanding (ring of run slots)
constexpr int NP = 8;               // tiles of one block that may wait for their global offset (each may be a run of its own: NP < NR)
constexpr int COPY_BATCH = SG_F_COPY_BATCH;       // pending tiles with a known offset are copied out once this many have gathered (or the ring / queue fills)

__device__ __forceinline__ unsigned long long ld_state(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_state(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// byte offset, inside a staged tile, of 16-byte chunk j of row r (128-byte swizzle)
__device__ __forceinline__ uint32_t swz(uint32_t r, uint32_t j) { return r * 128u + ((j ^ (r & 7u)) << 4); }

// ---- evaluators: produce, for the FW elements of one chunk starting at index i, the candidate values and keep bits ----
template <class P> struct FilterTemplateEval {
    typedef Meta1D<P> M;
    typedef typename M::T T;
    typedef typename M::VEC VEC;
    static constexpr int NOUT = M::NOUT;
    static constexpr int FW = 16 / (int)sizeof(T);       // elements per 16-byte chunk
    static constexpr int CT = 128 * P::unroll;           // compute threads: 512 = two per row (16 compute warps), 256 = one per row
    static constexpr int CPT = F_TILE_CHUNKS / CT;       // consecutive 16-byte chunks per thread per tile
    static constexpr int EPT = CPT * FW;                 // consecutive elements per thread per tile
    static constexpr int TILE = F_TILE_BYTES / (int)sizeof(T);
    static constexpr int RC = TILE;                      // elements of the compaction ring (a power of two, >= one tile)
    static_assert(CT == 256 || CT == 512, "filter instances: unroll 2 or 4");
    static constexpr int NS = (P::row_unroll >= 1 && P::row_unroll <= 3) ? P::row_unroll : 2;    // input stages
    __host__ __device__ static constexpr int count_vec() {
        int n = 0;
        for (int k = 0; k < M::S.n_in; ++k) n += (P::prog.in[k].kind == IN_VEC);
        return n;
    }
    static constexpr int NSTG = count_vec() < SG_MAX_TMAP ? count_vec() : SG_MAX_TMAP;   // inputs staged through shared memory (the rest: element loads)
    static constexpr size_t STAGE_BYTES = (size_t)NS * NSTG * F_TILE_BYTES;
    static constexpr size_t SMEM = STAGE_BYTES + (size_t)RC * sizeof(T) + NS * sizeof(uint64_t);
    __host__ __device__ static constexpr int vec_slot(int K) {      // index of IN_VEC input K among the IN_VEC inputs
        int n = 0;
        for (int k = 0; k < K; ++k) n += (P::prog.in[k].kind == IN_VEC);
        return n;
    }
    __host__ __device__ static constexpr bool staged_input(int K) { return P::prog.in[K].kind == IN_VEC && vec_slot(K) < NSTG; }
    __host__ __device__ static constexpr int filter_out() {
        for (int o = 0; o < M::S.n_out; ++o)
            if (P::prog.out[o].kind == OUT_FILTER) return o;
        return 0;
    }
    // reductions over exactly the kept values (same source register, same predicate as the filter) are accumulated when
    // the compacted values are copied out: one visit per KEPT element instead of one per element
    __host__ __device__ static constexpr bool kept_reduction(int O) {
        const SgOut f = P::prog.out[filter_out()], out = P::prog.out[O];
        return (out.kind == OUT_SUM || out.kind == OUT_MAX || out.kind == OUT_MIN) && out.src == f.src && out.pred == f.pred;
    }
    template <int O>
    __device__ __forceinline__ static void accum_kept_o(T x, Cell (&acc)[NOUT]) {
        constexpr SgOut out = P::prog.out[O];
        if constexpr (kept_reduction(O)) cell_accum_value<T>(out.kind, acc[O], x);
    }
    template <int... O>
    __device__ __forceinline__ static void accum_kept_(T x, Cell (&acc)[NOUT], std::integer_sequence<int, O...>) {
        (accum_kept_o<O>(x, acc), ...);
    }
    __device__ __forceinline__ static void accum_kept(const SgProg*, T x, Cell (&acc)[NOUT]) {
        accum_kept_(x, acc, std::make_integer_sequence<int, M::S.n_out>{});
    }

    // thread 0: one TMA tensor copy per staged input: rows [row0, row0+256) -> stage (shared-window address)
    template <int K>
    __device__ __forceinline__ static void issue_k(const SgArgs& a, int row0, uint32_t stage, uint64_t* bar) {
        if constexpr (staged_input(K)) {
            constexpr int slot = vec_slot(K);
            tma_load_2d(stage + (uint32_t)slot * F_TILE_BYTES, a.tmap[slot], 0, row0, bar);
        }
    }
    template <int... K>
    __device__ __forceinline__ static void issue_(const SgArgs& a, int row0, uint32_t stage, uint64_t* bar, std::integer_sequence<int, K...>) {
        mbar_expect_tx(bar, (uint32_t)(NSTG * F_TILE_BYTES));
        (issue_k<K>(a, row0, stage, bar), ...);
    }
    __device__ __forceinline__ static void issue(const SgProg*, const SgArgs& a, int row0, uint32_t stage, uint64_t* bar) {
        issue_(a, row0, stage, bar, std::make_integer_sequence<int, M::S.n_in>{});
    }
    // all compute threads: cooperative fill of the staged inputs of one tile (coalesced, guarded), same swizzled layout
    template <int K>
    __device__ __forceinline__ static void fill_k(const SgArgs& a, int64_t tbase, unsigned char* stage) {
        if constexpr (staged_input(K)) {
            constexpr int slot = vec_slot(K);
            unsigned char* dstb = stage + (size_t)slot * F_TILE_BYTES;
            const T* src = reinterpret_cast<const T*>(a.in_ptr[K]);
            const bool vec = (a.vec_ok >> 31) & 1;                  // every vector operand 16-byte aligned
#pragma unroll
            for (int q = 0; q < CPT; ++q) {
                const int c = threadIdx.x + CT * q;                 // chunk of the tile, in memory order
                const int64_t i = tbase + (int64_t)c * FW;
                VEC w;
                T* we = reinterpret_cast<T*>(&w);
                if (vec && i + FW <= a.in_len[K]) w = ld_stream(reinterpret_cast<const VEC*>(src + i));
                else {
#pragma unroll
                    for (int e = 0; e < FW; ++e) we[e] = load_elem<T>(IN_VEC, 0, K, a, i + e);
                }
                *reinterpret_cast<VEC*>(dstb + swz((uint32_t)c >> 3, (uint32_t)c & 7u)) = w;
            }
        }
    }
    template <int... K>
    __device__ __forceinline__ static void fill_(const SgArgs& a, int64_t tbase, unsigned char* stage, std::integer_sequence<int, K...>) {
        (fill_k<K>(a, tbase, stage), ...);
    }
    __device__ __forceinline__ static void fill(const SgProg*, const SgArgs& a, int64_t tbase, unsigned char* stage) {
        fill_(a, tbase, stage, std::make_integer_sequence<int, M::S.n_in>{});
    }

    // one chunk: FW consecutive elements starting at index i; staged inputs come from the stage at byte offset choff
    template <bool GUARDED, int K>
    __device__ __forceinline__ static void load_k(T (&v)[M::NV][FW], bool (&p)[M::NP][FW], const SgArgs& a, int64_t i, const unsigned char* stage, uint32_t choff) {
        constexpr SgIn in = P::prog.in[K];
        if constexpr (in.kind == IN_SCALAR || in.kind == IN_IMM) {
            T s = load_elem<T>(in.kind, in.ref, K, a, 0);
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = s;
        } else if constexpr (in.kind == IN_BOOLVEC) {
#pragma unroll
            for (int e = 0; e < FW; ++e) p[in.reg][e] = (i + e < a.in_len[K]) && reinterpret_cast<const volatile uint8_t*>(a.in_ptr[K])[i + e] != 0;
        } else if constexpr (staged_input(K)) {
            constexpr int slot = vec_slot(K);
            const VEC w = *reinterpret_cast<const VEC*>(stage + (size_t)slot * F_TILE_BYTES + choff);
            const T* we = reinterpret_cast<const T*>(&w);
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = we[e];
        } else {
#pragma unroll
            for (int e = 0; e < FW; ++e) v[in.reg][e] = load_elem<T>(in.kind, in.ref, K, a, i + e);
        }
    }
    template <bool GUARDED, int O>
    __device__ __forceinline__ static void out_o(T (&v)[M::NV][FW], bool (&p)[M::NP][FW], const SgArgs& a, int64_t i, T (&val)[FW],
                                                 unsigned int& keep, Cell (&acc)[NOUT]) {
        constexpr SgOut out = P::prog.out[O];
#pragma unroll
        for (int e = 0; e < FW; ++e) {
            const bool in_range = !GUARDED || (i + e < a.out_len[O]);       // full tiles lie inside every output's length
            if constexpr (out.kind == OUT_FILTER) {
                val[e] = v[out.src][e];
                keep |= (unsigned int)(in_range && p[out.pred][e]) << e;
            } else if constexpr (out_is_pred_reduction(out.kind)) {
                if (in_range) cell_accum_pred(out.kind, acc[O], p[out.src][e]);
            } else if constexpr (kept_reduction(O)) {
                // accumulated at copy-out (accum_kept)
            } else if constexpr (out_is_reduction(out.kind)) {
                if constexpr (out.pred == SG_NO_PRED) { if (in_range) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]); }
                else { if (in_range && p[out.pred][e]) cell_accum_value<T>(out.kind, acc[O], v[out.src][e]); }
            }
        }
    }
    template <bool GUARDED, int... K, int... I, int... O>
    __device__ __forceinline__ static void run_(const SgArgs& a, int64_t i, const unsigned char* stage, uint32_t choff, T (&val)[FW], unsigned int& keep,
                                                Cell (&acc)[NOUT], std::integer_sequence<int, K...>, std::integer_sequence<int, I...> is,
                                                std::integer_sequence<int, O...>) {
        T v[M::NV][FW];
        bool p[M::NP][FW];
        (load_k<GUARDED, K>(v, p, a, i, stage, choff), ...);
        exec_body<P, T, M::NV, M::NP, FW>(v, p, a, is);
        keep = 0;
        (out_o<GUARDED, O>(v, p, a, i, val, keep, acc), ...);
    }
    template <bool GUARDED>
    __device__ __forceinline__ static void run(const SgProg*, const SgArgs& a, int64_t i, const unsigned char* stage, uint32_t choff, T (&val)[FW],
                                               unsigned int& keep, Cell (&acc)[NOUT]) {
        run_<GUARDED>(a, i, stage, choff, val, keep, acc, std::make_integer_sequence<int, M::S.n_in>{}, std::make_integer_sequence<int, M::S.n_instr>{},
                      std::make_integer_sequence<int, M::S.n_out>{});
    }
    __device__ __forceinline__ static uint8_t out_kind(const SgProg*, int o) {
        constexpr SgProg g = P::prog;
        return o < M::S.n_out ? g.out[o].kind : (uint8_t)OUT_STORE;
    }
};

// bytecode evaluator: nothing is staged (every operand is loaded per chunk from global memory); same tile geometry
template <class TT> struct FilterBytecodeEval {
    typedef TT T;
    static constexpr int NOUT = SG_MAX_OUT;
    static constexpr int FW = 16 / (int)sizeof(T);
    static constexpr int CT = BLOCK, CPT = F_TILE_CHUNKS / CT;
    static constexpr int EPT = CPT * FW;
    static constexpr int TILE = F_TILE_BYTES / (int)sizeof(T);
    static constexpr int RC = TILE, NS = 2, NSTG = 0;
    static constexpr size_t STAGE_BYTES = VM_FILE_BYTES;     // no input is staged: the stage area holds the VM's shared-memory register file
    static constexpr size_t SMEM = STAGE_BYTES + (size_t)RC * sizeof(T) + NS * sizeof(uint64_t);
    __device__ __forceinline__ static void issue(const SgProg*, const SgArgs&, int, uint32_t, uint64_t*) {}
    __device__ __forceinline__ static void fill(const SgProg*, const SgArgs&, int64_t, unsigned char*) {}
    __device__ __forceinline__ static void accum_kept(const SgProg*, T, Cell (&)[NOUT]) {}      // masked reductions are accumulated per element
    template <bool GUARDED>
    __device__ __forceinline__ static void run(const SgProg* g, const SgArgs& a, int64_t i, const unsigned char* vm_file, uint32_t, T (&val)[FW], unsigned int& keep,
                                               Cell (&acc)[NOUT]) {
        VmRegs<T, FW> rf(smem_u32(vm_file));
        unsigned int pf = 0;
        for (int k = 0; k < g->shape.n_in; ++k) {
            const SgIn in = g->in[k];
            if (in.kind == IN_SCALAR || in.kind == IN_IMM) {
                T x[FW];
                const T s = load_elem<T>(in.kind, in.ref, k, a, 0);
#pragma unroll
                for (int e = 0; e < FW; ++e) x[e] = s;
                rf.put(in.reg, x);
            } else vm_load<T, FW>(*g, a, k, i, !GUARDED && ((a.vec_ok >> 31) & 1), rf, pf);
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

// look-back warp: exclusive prefix of `tile` (sum of the kept counts of all tiles before it).  The tile's AGGREGATE has
// already been published by the compute warps — at once, so that no other block's look-back waits for this warp's backlog.
__device__ __forceinline__ unsigned long long filter_lookback(unsigned long long* state, unsigned long long ep, int tile, unsigned int tile_total, int lane) {
    if (tile == 0) return 0;        // its inclusive prefix was published with the aggregate
    unsigned long long excl = 0;
    int look = tile - 1;
    for (;;) {
        unsigned long long lbw[LB];
        // cheap poll: wait until the nearest window has no unpublished state in front of its first inclusive prefix
        for (;;) {
            const int idx = look - lane;
            lbw[0] = (idx >= 0) ? ld_state(&state[idx]) : (ST_INC | ep);    // virtual tile -1: inclusive prefix 0
            const bool valid = ((lbw[0] & ST_FLAGS) != 0) && ((lbw[0] & (0x3fffffull << 40)) == ep);
            const bool inc = valid && ((lbw[0] & ST_FLAGS) == ST_INC);
            const unsigned int vmask = __ballot_sync(0xffffffffu, valid), imask = __ballot_sync(0xffffffffu, inc);
            const unsigned int before_inc = imask ? ((imask & (0u - imask)) - 1u) : 0xffffffffu;    // lanes in front of the first inclusive prefix
            if ((~vmask & before_inc) == 0u) break;
            __nanosleep(SG_F_SLEEP);       // a near predecessor has not published yet: do not hammer the state words (nor this SM's issue slots)
        }
#pragma unroll
        for (int j = 1; j < LB; ++j) {
            const int idx = look - lane - 32 * j;
            lbw[j] = (idx >= 0) ? ld_state(&state[idx]) : (ST_INC | ep);
        }
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
    }
    if (lane == 0) st_state(&state[tile], ST_INC | ep | (excl + tile_total));
    return excl;
}



// appends the kept elements of one thread's row (keep bits in `mask`, element k = val[k / FW][k % FW]) at `addr`
template <class T, int FW, int CPT, int... K>
__device__ __forceinline__ void scatter_row(uint32_t& addr, unsigned int mask, T (&val)[CPT][FW], std::integer_sequence<int, K...>) {
    (sts_append_if<T, K>(addr, mask, val[K / FW][K % FW]), ...);
}

// ---- the kernel body -------------------------------------------------------------------------------------
template <class EV>
__device__ __forceinline__ void filter_body(const SgProg* g, const SgArgs& a) {
    typedef typename EV::T T;
    constexpr int FW = EV::FW, EPT = EV::EPT, TILE = EV::TILE, NOUT = EV::NOUT, NS = EV::NS, NSTG = EV::NSTG, RC = EV::RC;
    constexpr int CT = EV::CT, CW = CT / 32, CPT = EV::CPT;       // compute threads / warps, chunks per thread
    static_assert(NP < NR, "a run slot must not be reused while one of its tiles is pending");
    extern __shared__ __align__(1024) unsigned char dyn_smem[];
    unsigned char* const stage_base = dyn_smem;                                             // [NS][NSTG][F_TILE_BYTES], 1024-byte aligned (swizzle)
    const uint32_t ring = pin_reg(smem_u32(dyn_smem + EV::STAGE_BYTES));                             // [RC] compacted values awaiting their offset (shared-window address)
    uint64_t* const full_bar = reinterpret_cast<uint64_t*>(dyn_smem + EV::STAGE_BYTES + (size_t)RC * sizeof(T));
    __shared__ int s_tile[NS + 1];                      // tile id of iteration it at [it % (NS+1)]
    __shared__ unsigned int s_warp_total[2][CW];     // double-buffered: a warp may run one barrier ahead
    __shared__ int s_ready[2];                          // thread 0 -> all: pending tiles whose offset is known (polled before the barrier)
    __shared__ int s_q_tile[NP];                        // pending tile queue: tile id,
    __shared__ unsigned int s_q_total[NP];              //   kept count,
    __shared__ unsigned int s_q_lpre[NP];               //   kept count of the earlier tiles of its run,
    __shared__ int s_q_run[NP];                         //   run number (of this block)
    __shared__ int s_r_tile[NR];                        // compute -> look-back warp: first tile of the run (-1: no more runs)
    __shared__ unsigned int s_r_total[NR];              //                            its kept count
    __shared__ unsigned long long s_r_excl[NR];         // look-back warp -> compute: global offset of the run's first tile
    __shared__ uint64_t run_posted[NR], run_resolved[NR];   // mbarriers, one arrival each
    __shared__ volatile int s_resolved;                 // look-back warp -> thread 0: runs 0 .. s_resolved-1 of this block have their offset
                                                        // (runs resolve in order; ONE shared load replaces a chain of mbarrier polls,
                                                        // ~150 cycles each, that sat on warp 0's path to the per-tile barrier)

    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
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
    const bool use_tma = NSTG > 0 && ((a.vec_ok >> 30) & 1);       // tensor maps encoded: 16-byte aligned inputs, >= 1 full tile

    if (a.n_tiles == 0 && blockIdx.x == 0 && threadIdx.x == 0) *reinterpret_cast<long long*>(a.out_aux[fo]) = 0;

    // thread 0 hands out this block's tile sequence: runs of consecutive tiles claimed with one atomic each.  A run is RUN
    // tiles while a run's kept values fit comfortably in the ring, else ONE tile: a tile that cannot enter the ring waits
    // for its run's offset, and with long runs that wait would chain from block to block.  Entries: (tile << 1) | first-of-run.
    // The atomic of the NEXT run is issued one call before its result is needed, so its latency never stalls warp 0.
    int seq_base = 0, seq_j = 0, seq_len = 0;   // thread 0 only: current run, position in it, its length
    int nxt_base = 0, nxt_len = 0;              // thread 0 only: the run claimed ahead
    unsigned int last_total = (unsigned int)RC; // thread 0 only: kept count of the latest tile (pessimistic until one is known)
    auto claim_ahead = [&]() {                  // thread 0 only
        nxt_len = (last_total * (unsigned int)RUN * (unsigned int)SG_F_RULE_NUM <= (unsigned int)RC * (unsigned int)SG_F_RULE_DEN) ? RUN : 1;
        nxt_base = (int)atomicAdd(&a.ctrl[2], (unsigned int)nxt_len);
    };
    auto next_tile = [&]() -> int {             // thread 0 only
        if (seq_j == seq_len) { seq_base = nxt_base; seq_len = nxt_len; seq_j = 0; }
        const int first = (seq_j == 0);
        const int t = seq_base + seq_j++;
        if (seq_j == seq_len) claim_ahead();
        return t >= 0x3fffffff ? 0x7ffffffe : ((t << 1) | first);
    };
    if (threadIdx.x == 0) {
        for (int r = 0; r < NR; ++r) {
            mbar_init(&run_posted[r], 1);
            mbar_init(&run_resolved[r], 1);
        }
        for (int s = 0; s < NS; ++s) mbar_init(&full_bar[s], 1);
        mbar_fence_init();
        s_resolved = 0;
        claim_ahead();
        for (int s = 0; s < NS; ++s) {          // the first NS tiles: their copies are in flight before the first one is touched
            const int tv = next_tile();
            s_tile[s] = tv;
            const int t = tv >> 1;
            if (use_tma && t < a.n_full_tiles) EV::issue(g, a, t * F_ROWS, smem_u32(stage_base + (size_t)s * NSTG * F_TILE_BYTES), &full_bar[s]);
        }
    }
    __syncthreads();

    if (warp == CW) {
        // ---------------- look-back warp: one message per run, in order ----------------
        for (int r = 0;; ++r) {
            const int rs = r % NR;
            mbar_wait(&run_posted[rs], (uint32_t)((r / NR) & 1));
            const int tile = s_r_tile[rs];
            if (tile < 0) break;
            const unsigned int total = s_r_total[rs];
            const unsigned long long excl = filter_lookback(state, ep, tile, total, lane);
            if (lane == 0) {
                s_r_excl[rs] = excl;
                __threadfence_block();          // the offset is visible before the count that announces it
                s_resolved = r + 1;
                mbar_arrive(&run_resolved[rs]);
            }
        }
    } else {
        // ---------------- compute warps ----------------
        // Pending tiles (compacted into the ring, offset not yet known) form a queue in processing order; every compute
        // thread tracks the same queue state in registers.  A tile's offset = its run's offset + the kept counts of the
        // run's earlier tiles (local prefix), so only the FIRST tile of a run needs a look-back; once the run's offset is
        // known, later tiles of the run publish their INCLUSIVE prefix directly — other blocks' look-backs end there.
        int q_head = 0, q_count = 0;
        unsigned int ring_head = 0, ring_tail = 0;
        int run_no = -1;                        // number of the current run of this block
        unsigned int run_lpre = 0;              // kept count of the current run's earlier tiles
        bool overflow = false;
        // copies out the k oldest pending tiles.  Tiles of one run are adjacent in the ring AND in the output, so each
        // run's share goes out in ONE coalesced loop (one wait, one address computation, one set of uniform checks).
        auto copy_out = [&](int k) {
            while (k > 0) {
                const int e0 = q_head % NP;
                const int r = s_q_run[e0];
                mbar_wait(&run_resolved[r % NR], (uint32_t)((r / NR) & 1));
                unsigned int total = s_q_total[e0];
                int m = 1;
                while (m < k && s_q_run[(q_head + m) % NP] == r) { total += s_q_total[(q_head + m) % NP]; ++m; }
                const long long base = (long long)(s_r_excl[r % NR] + s_q_lpre[e0]);
                const unsigned int r0 = ring_tail & (RC - 1);
                if (base + (long long)total <= cap && r0 + total <= (unsigned int)RC) {
                    // common case (uniform): inside the output's capacity, no wrap-around in the ring
                    T* const d0 = dst + base;
                    for (unsigned int i = threadIdx.x; i < total; i += CT) {
                        const T v = lds_elem<T>(ring, r0 + i);
                        EV::accum_kept(g, v, acc);
                        d0[i] = v;
                    }
                } else {
                    for (unsigned int i = threadIdx.x; i < total; i += CT) {
                        const long long pos = base + i;
                        const T v = lds_elem<T>(ring, (ring_tail + i) & (RC - 1));
                        EV::accum_kept(g, v, acc);
                        if (pos < cap) dst[pos] = v; else overflow = true;
                    }
                }
                if (threadIdx.x == 0 && s_q_tile[(q_head + m - 1) % NP] == a.n_tiles - 1) *reinterpret_cast<long long*>(a.out_aux[fo]) = base + (long long)total;
                ring_tail += total;
                q_head += m;
                q_count -= m;
                k -= m;
            }
        };
        int it = 0;
        for (;; ++it) {
            const int s = it % NS;
            const int tv = s_tile[it % (NS + 1)];
            const int tile = tv >> 1;
            const bool first = tv & 1;          // first tile of a run
            if (tile >= a.n_tiles) break;
            if (first) { ++run_no; run_lpre = 0; }
            const int rs = run_no % NR;
            // thread 0 fetches the tile of iteration it+NS now (a new run costs one atomic, whose latency hides behind the
            // evaluation), makes the id visible before this iteration's barrier, and issues its copy right after the barrier
            // into THIS stage, which every thread has read into registers by then
            int tv_next = 0x7ffffffe;
            if (threadIdx.x == 0) tv_next = next_tile();

            const int64_t tbase = (int64_t)tile * TILE;
            const bool full = tile < a.n_full_tiles;            // inside every operand's and output's length: no range checks
            unsigned char* const stg = stage_base + (size_t)s * NSTG * F_TILE_BYTES;
            if (NSTG > 0) {
                if (use_tma && full) mbar_wait(&full_bar[s], (uint32_t)((it / NS) & 1));
                else {
                    EV::fill(g, a, tbase, stg);
                    named_bar_sync<2, CT>();
                }
            }
            T val[CPT][FW];
            unsigned int mask = 0;                              // keep bits of this thread's EPT consecutive elements
#pragma unroll
            for (int j = 0; j < CPT; ++j) {
                unsigned int kj;
                const int64_t i = tbase + (int64_t)threadIdx.x * EPT + j * FW;
                const uint32_t gc = threadIdx.x * CPT + j;      // chunk of the tile: row gc / 8, chunk gc % 8 of the row
                if (full) EV::template run<false>(g, a, i, stg, swz(gc >> 3, gc & 7u), val[j], kj, acc);
                else EV::template run<true>(g, a, i, stg, swz(gc >> 3, gc & 7u), val[j], kj, acc);
                mask |= kj << (j * FW);
            }
            // rank: the thread's elements are consecutive, so one popc and one warp scan order the tile
            const unsigned int cnt = __popc(mask);
            unsigned int incl = cnt;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned int t = __shfl_up_sync(0xffffffffu, incl, d);
                if (lane >= d) incl += t;
            }
            if (lane == 31) s_warp_total[it & 1][warp] = incl;
            bool run_known = false;         // thread 0: the current run's offset has been resolved already
            if (threadIdx.x == 0) {
                s_tile[(it + NS) % (NS + 1)] = tv_next;
                const int resolved = s_resolved;        // runs [0, resolved) of this block have their offset
                int ready = 0;      // how many of the oldest pending tiles already have their offset (never blocks)
                for (; ready < q_count; ++ready)
                    if (s_q_run[(q_head + ready) % NP] >= resolved) break;
                s_ready[it & 1] = ready;
                if (!first) run_known = run_no < resolved;
            }
            named_bar_sync<1, CT>();     // the stage is in registers; warp totals, next tile id and the ready count are visible
            unsigned int warp_excl = 0, tile_total = 0;
#pragma unroll
            for (int w = 0; w < CW; ++w) {
                const unsigned int t = s_warp_total[it & 1][w];
                if (w < warp) warp_excl += t;
                tile_total += t;
            }
            if (threadIdx.x == 0) {
                // publish at once: the inclusive prefix if it is known (tile 0, or the run's offset is resolved), else the aggregate
                if (tile == 0) st_state(&state[0], ST_INC | ep | (unsigned long long)tile_total);
                else if (run_known) st_state(&state[tile], ST_INC | ep | (s_r_excl[rs] + run_lpre + tile_total));
                else st_state(&state[tile], ST_AGG | ep | (unsigned long long)tile_total);
                const int e = it % NP;
                s_q_tile[e] = tile;
                s_q_total[e] = tile_total;
                s_q_lpre[e] = run_lpre;
                s_q_run[e] = run_no;
                last_total = tile_total;
                if (first) {                // first tile of a run: hand it to the look-back warp
                    s_r_tile[rs] = tile;
                    s_r_total[rs] = tile_total;
                    mbar_arrive(&run_posted[rs]);
                }
                if (use_tma && (tv_next >> 1) < a.n_full_tiles) {
                    fence_proxy_async();
                    EV::issue(g, a, (tv_next >> 1) * F_ROWS, smem_u32(stg), &full_bar[s]);
                }
            }
            int copied = 0;
            if (ring_head - ring_tail + tile_total > (unsigned int)RC) {
                // rare: the ring cannot take this tile yet — wait for the oldest offsets first
                while (ring_head - ring_tail + tile_total > (unsigned int)RC) { copy_out(1); ++copied; }
                named_bar_sync<2, CT>();
            }
            {
                const unsigned int pos = ring_head + warp_excl + (incl - cnt);
                if (((ring_head & (RC - 1)) + tile_total) <= (unsigned int)RC) {
                    // the tile does not wrap around the ring (uniform): plain appends
                    uint32_t addr = ring + (pos & (RC - 1)) * (uint32_t)sizeof(T);
                    scatter_row<T, FW, CPT>(addr, mask, val, std::make_integer_sequence<int, CPT * FW>{});
                } else {
                    unsigned int q = pos;
#pragma unroll
                    for (int j = 0; j < CPT; ++j)
#pragma unroll
                        for (int e = 0; e < FW; ++e)
                            if ((mask >> (j * FW + e)) & 1u) sts_elem<T>(ring, (q++) & (RC - 1), val[j][e]);
                }
            }
            ring_head += tile_total;
            run_lpre += tile_total;
            ++q_count;
            // copy out the tiles whose offset was known at the poll (never blocks) — a few at a time: a call costs every thread some
            // eighty instructions before its first element (queue entries, the run's offset, the uniform checks), tiles of one run
            // then go out in ONE loop — and as many as the queue bound demands
            int k = s_ready[it & 1] - copied;
            if (k < COPY_BATCH && ring_head - ring_tail + (unsigned int)TILE / 2u <= (unsigned int)RC) k = 0;
            if (k < q_count - (NP - 1)) k = q_count - (NP - 1);
            if (k > 0) copy_out(k);
        }
        if (threadIdx.x == 0) {             // no run follows: release the look-back warp
            const int rs = (run_no + 1) % NR;
            s_r_tile[rs] = -1;
            mbar_arrive(&run_posted[rs]);
        }
        named_bar_sync<1, CT>();         // the last tile's queue entry (written by thread 0 after its barrier) is visible
        copy_out(q_count);
        if (overflow) a.ctrl[3] = 1u;
    }
    epilogue_1d<T, NOUT>(acc, kind, a, true);
}

template <class P>
__global__ void __launch_bounds__(FilterTemplateEval<P>::CT + 32, P::min_blocks) filter1d_template(const __grid_constant__ SgArgs a) {
    pdl_wait();
    pdl_trigger();
    filter_body<FilterTemplateEval<P>>(nullptr, a);
}
template <class T>
__global__ void __launch_bounds__(BLOCK + 32) filter1d_bytecode(const __grid_constant__ SgProg g, const __grid_constant__ SgArgs a) {
    pdl_wait();
    pdl_trigger();
    filter_body<FilterBytecodeEval<T>>(&g, a);
}

}  // namespace sgk
#endif  // SG_FILTER_CUH_
