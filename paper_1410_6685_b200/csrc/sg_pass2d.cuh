// sg_pass2d.cuh — the fused matrix pass: elementwise chain over a rows x cols row-major
// domain with ROW-/COL-broadcast vector operands, in-place store, and per-row / per-column /
// whole-matrix reductions in the same pass.  The Gaussian-elimination row update of Listing 5 (PAPER.md:315-322,
// 337-356) for ALL rows j > k is one launch of this kernel — the paper's per-row launches are what made that
// benchmark slow.
//
// Tiling: block (strip s, chunk ch) owns columns [s*SW, (s+1)*SW) and rows [ch*rpc, (ch+1)*rpc).  A thread owns
// E = U*V fixed columns (128-bit accesses) for every row of the chunk, so ROW-broadcast operands and per-column
// accumulators live in registers for the whole chunk.  Rows are staged through shared memory: thread 0 issues one
// bulk asynchronous copy (cp.async.bulk, the TMA engine) per row, NS stages of RU rows ahead of the consumers.
// Per-column partials are combined over chunks by the last block of the strip, per-row partials over strips by
// the last block of the chunk, both in fixed order (deterministic; no floating-point atomics).
#ifndef SG_PASS2D_CUH_
#define SG_PASS2D_CUH_

#include "sg_bulk.cuh"
#include "sg_pass1d_tmpl.cuh"

namespace sgk {

constexpr int RB = 32;      // rows per batch between the two barriers of the per-row combine

template <class T> __device__ __forceinline__ void store_final(uint8_t kind, void* base, int64_t idx, const Cell& c) {
    const unsigned long long r = cell_final<T>(kind, c);
    if ((kind == OUT_MAX || kind == OUT_MIN) && sizeof(T) == 4) reinterpret_cast<uint32_t*>(base)[idx] = (uint32_t)r;
    else reinterpret_cast<unsigned long long*>(base)[idx] = r;
}
__device__ __forceinline__ Cell ldcg_cell(const Cell* p) {
    Cell c;
    const unsigned long long* s = reinterpret_cast<const unsigned long long*>(p);
    c.a = __ldcg(s); c.b = __ldcg(s + 1);
    return c;
}

struct Slots2D { int vec[SG_MAX_IN]; int row[SG_MAX_OUT]; int colb[SG_MAX_IN]; };

template <class P> struct Meta2D : Meta1D<P> {
    typedef Meta1D<P> B;
    static constexpr int RU = P::row_unroll;
    static constexpr int SW = BLOCK * B::E;     // strip width in columns
    static constexpr int count_kind(uint8_t kind) {
        int n = 0;
        for (int k = 0; k < B::S.n_in; ++k) n += (P::prog.in[k].kind == kind);
        return n;
    }
    static constexpr int NVECINREAL = count_kind(IN_VEC);
    static constexpr int NCOLBREAL = count_kind(IN_COLB);
    static constexpr int NVECIN = NVECINREAL > 0 ? NVECINREAL : 1;
    static constexpr int NS = P::stages;            // shared-memory stages in flight
    static constexpr size_t SMEM = (size_t)NS * NVECIN * RU * SW * sizeof(typename B::T) + NS * sizeof(uint64_t);
    static constexpr int colb_slot(int K) {
        int n = 0;
        for (int k = 0; k < K; ++k) n += (P::prog.in[k].kind == IN_COLB);
        return n;
    }
    static constexpr int vec_slot(int K) {
        int n = 0;
        for (int k = 0; k < K; ++k) n += (P::prog.in[k].kind == IN_VEC);
        return n;
    }
    static constexpr int count_axis(uint8_t axis) {
        int n = 0;
        for (int o = 0; o < B::S.n_out; ++o) n += (out_is_reduction(P::prog.out[o].kind) && P::prog.out[o].axis == axis);
        return n;
    }
    static constexpr int NROWS = count_axis(AXIS_ROWS) > 0 ? count_axis(AXIS_ROWS) : 1;
    static constexpr int row_slot(int O) {
        int n = 0;
        for (int o = 0; o < O; ++o) n += (out_is_reduction(P::prog.out[o].kind) && P::prog.out[o].axis == AXIS_ROWS);
        return n;
    }
    static constexpr bool has_axis(uint8_t axis) { return count_axis(axis) > 0; }
    static constexpr Slots2D slots() {
        Slots2D s{};
        for (int k = 0; k < SG_MAX_IN; ++k) s.vec[k] = k < B::S.n_in ? vec_slot(k) : 0;
        for (int k = 0; k < SG_MAX_IN; ++k) s.colb[k] = k < B::S.n_in ? colb_slot(k) : 0;
        for (int o = 0; o < SG_MAX_OUT; ++o) s.row[o] = o < B::S.n_out ? row_slot(o) : 0;
        return s;
    }
    static constexpr Slots2D SLOTS = slots();
    static constexpr bool HAS_ROWS = has_axis(AXIS_ROWS), HAS_COLS = has_axis(AXIS_COLS);
};

// Warp reduction of R per-row partials at once (R a power of two <= 32).  A butterfly per row costs 5 combines per lane and
// row; here the first log2(R) exchange steps HALVE the number of rows a lane still holds (a lane sends the half it gives up
// and combines the half it keeps), so R rows cost R-1 + (5 - log2 R) combines per lane instead of 5R — the double-double
// combine (11 fp64 operations) is what bounds a row-sum pass otherwise.  Afterwards c[0] of the lanes whose low
// (5 - log2 R) bits are zero holds the total of row `warp_row_of_lane<R>(lane)`.  Fixed combine order: deterministic.
template <class T, int R>
__device__ __forceinline__ void warp_reduce_rows(uint8_t kind, Cell (&c)[R], int lane) {
    static_assert(R >= 1 && R <= 32 && (R & (R - 1)) == 0, "rows in flight must be a power of two <= 32");
    int d = 16;
#pragma unroll
    for (int h = R / 2; h >= 1; h >>= 1) {
        const bool upper = (lane & d) != 0;
#pragma unroll
        for (int i = 0; i < h; ++i) {
            const Cell send = upper ? c[i] : c[i + h];
            Cell keep = upper ? c[i + h] : c[i];
            const Cell recv = cell_shfl_xor_kind<T>(kind, send, d);
            cell_combine<T>(kind, keep, recv);
            c[i] = keep;
        }
        d >>= 1;
    }
#pragma unroll
    for (; d >= 1; d >>= 1) {
        const Cell other = cell_shfl_xor_kind<T>(kind, c[0], d);
        cell_combine<T>(kind, c[0], other);
    }
}
template <int R> __device__ __forceinline__ int warp_row_of_lane(int lane) {
    int row = 0, d = 16;
#pragma unroll
    for (int h = R / 2; h >= 1; h >>= 1) { if (lane & d) row += h; d >>= 1; }
    return row;
}
template <int R> __device__ __forceinline__ bool warp_row_owner(int lane) {
    int low = 31;
#pragma unroll
    for (int h = R / 2; h >= 1; h >>= 1) low >>= 1;
    return (lane & low) == 0;
}

// ALIGNED: every row of every matrix operand starts on a 16-byte boundary and holds a whole number of 128-bit vectors (base,
// leading dimension and column count): rows are staged by bulk copies and stored with 128-bit accesses.  Otherwise (odd column
// counts or leading dimensions, PAPER.md:209-219 puts no condition on a matrix's shape) the block fills the stage cooperatively
// with element loads in the same layout, and ROW-broadcast loads, stores and reductions are guarded per ELEMENT.
template <class P, bool ALIGNED>
__device__ __forceinline__ void pass2d_body(const SgArgs& a) {
    typedef Meta2D<P> M;
    typedef typename M::T T;
    typedef typename M::VEC VEC;
    constexpr int U = M::U, V = M::V, E = M::E, RU = M::RU, NOUT = M::NOUT;
    constexpr auto IS = std::make_integer_sequence<int, M::S.n_instr>{};
    constexpr SgProg g = P::prog;                 // local constant copy: indexable inside unrolled loops
    constexpr Slots2D slots = M::SLOTS;

    __shared__ Cell s_row[M::NROWS][WARPS][RB];

    const int strip = blockIdx.x % a.n_strips, chunk = blockIdx.x / a.n_strips;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t r_begin = (int64_t)chunk * a.rows_per_chunk;
    const int64_t r_end = (r_begin + a.rows_per_chunk < a.n) ? (r_begin + a.rows_per_chunk) : a.n;
    int64_t col[U];
    int nval[U];                // valid columns of the thread's vector u: 0 or V when ALIGNED, 0..V otherwise
    bool cvalid[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        col[u] = (int64_t)strip * M::SW + (int64_t)(u * BLOCK + threadIdx.x) * V;
        const int64_t left = a.cols - col[u];
        nval[u] = left >= V ? V : (left > 0 ? (int)left : 0);
        cvalid[u] = ALIGNED ? (left >= V) : (left > 0);
    }
    // element e of vector u takes part?  (compile-time true inside valid vectors of the aligned form)
    auto evalid = [&](int u, int e) { return ALIGNED ? true : e < nval[u]; };

    T v[M::NV][E];
    bool p[M::NP][E];
    Cell acc[NOUT];             // AXIS_ALL
    Cell acc_col[NOUT][E];      // AXIS_COLS (unused entries are dead code)
    uint8_t kind[NOUT];
    bool has_all = false;
#pragma unroll
    for (int o = 0; o < NOUT; ++o) {
        kind[o] = (o < M::S.n_out && g.out[o].axis == AXIS_ALL) ? g.out[o].kind : (uint8_t)OUT_STORE;
        acc[o] = cell_identity<T>(kind[o]);
        has_all |= out_is_reduction(kind[o]);
#pragma unroll
        for (int e = 0; e < E; ++e) acc_col[o][e] = cell_identity<T>(o < M::S.n_out ? g.out[o].kind : (uint8_t)OUT_STORE);
    }

    // operands that do not depend on the row: immediates, device scalars, ROW-broadcast vectors
#pragma unroll
    for (int k = 0; k < M::S.n_in; ++k) {
        const SgIn in = g.in[k];
        if (in.kind == IN_SCALAR || in.kind == IN_IMM) {
            const T s = load_elem<T>(in.kind, in.ref, k, a, 0);
#pragma unroll
            for (int e = 0; e < E; ++e) v[in.reg][e] = s;
        } else if (in.kind == IN_ROWB) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                VEC x = VEC();
                T* xw = reinterpret_cast<T*>(&x);
                if (ALIGNED) { if (cvalid[u]) x = *reinterpret_cast<const VEC*>(reinterpret_cast<const T*>(a.in_ptr[k]) + col[u]); }
                else {
#pragma unroll
                    for (int e = 0; e < V; ++e)
                        if (e < nval[u]) xw[e] = reinterpret_cast<const T*>(a.in_ptr[k])[col[u] + e];
                }
                const T* xe = reinterpret_cast<const T*>(&x);
#pragma unroll
                for (int e = 0; e < V; ++e) v[in.reg][u * V + e] = xe[e];
            }
        }
    }

    // ---- staged row loop: RS rows per stage, NS stages in flight (bulk copies issued by thread 0) -----------------
    constexpr int RS = RU, NS = M::NS;
    extern __shared__ __align__(1024) unsigned char dyn_smem[];     // same declaration as sg_filter.cuh (one symbol per translation unit)
    T* const stage_base = reinterpret_cast<T*>(dyn_smem);
    uint64_t* const full = reinterpret_cast<uint64_t*>(dyn_smem + (size_t)NS * M::NVECIN * RS * M::SW * sizeof(T));
    const int64_t c0 = (int64_t)strip * M::SW;
    const uint32_t row_bytes = (uint32_t)(((a.cols - c0) < M::SW ? (a.cols - c0) : M::SW) * sizeof(T));
    const int64_t n_rows = r_end - r_begin;
    const int64_t nb = (n_rows + RS - 1) / RS;
    auto issue = [&](int64_t b) {
        const int s = (int)(b % NS);
        const int64_t r0 = r_begin + b * RS;
        const int nr = (int)((r_end - r0) < RS ? (r_end - r0) : RS);
        mbar_expect_tx(&full[s], (uint32_t)(nr * M::NVECINREAL) * row_bytes);
#pragma unroll
        for (int k = 0; k < M::S.n_in; ++k) {
            if (g.in[k].kind != IN_VEC) continue;
            T* dst = stage_base + ((size_t)s * M::NVECIN + slots.vec[k]) * RS * M::SW;
            const T* src = reinterpret_cast<const T*>(a.in_ptr[k]) + r0 * a.in_stride[k] + c0;
            for (int j = 0; j < nr; ++j) bulk_g2s(dst + (size_t)j * M::SW, src + (size_t)j * a.in_stride[k], row_bytes, &full[s]);
        }
    };
    // unaligned rows: the whole block copies the rows of batch b into stage b % NS with element loads (same layout)
    auto fill = [&](int64_t b) {
        const int s = (int)(b % NS);
        const int64_t r0 = r_begin + b * RS;
        const int nr = (int)((r_end - r0) < RS ? (r_end - r0) : RS);
        const int row_elems = (int)(row_bytes / sizeof(T));
#pragma unroll
        for (int k = 0; k < M::S.n_in; ++k) {
            if (g.in[k].kind != IN_VEC) continue;
            T* dst = stage_base + ((size_t)s * M::NVECIN + slots.vec[k]) * RS * M::SW;
            const volatile T* src = reinterpret_cast<const volatile T*>(a.in_ptr[k]) + r0 * a.in_stride[k] + c0;
            for (int j = 0; j < nr; ++j)
                for (int c = threadIdx.x; c < row_elems; c += BLOCK) dst[(size_t)j * M::SW + c] = src[(size_t)j * a.in_stride[k] + c];
        }
    };
    if (ALIGNED) {
        if (threadIdx.x == 0) {
            for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
            mbar_fence_init();
        }
        __syncthreads();
        if (threadIdx.x == 0)
            for (int64_t b = 0; b < NS && b < nb; ++b) issue(b);
    }

    // COL-broadcast operands (one value per row, e.g. the elimination factors f_j): the values of batch b+1 are requested while batch b
    // is processed — loaded right before their first use they cost a full global-memory round trip per stage (ncu on config 4's pass:
    // 45 % of the stall samples were `long scoreboard` on the first multiplication by f_j)
    constexpr int NCOLB = M::NCOLBREAL > 0 ? M::NCOLBREAL : 1;
    T colb_next[NCOLB][RS];
    auto fetch_colb = [&](int64_t b, T (&dst)[NCOLB][RS]) {
        const int64_t r0 = r_begin + b * RS;
        int slot = 0;
#pragma unroll
        for (int k = 0; k < M::S.n_in; ++k) {
            if (g.in[k].kind != IN_COLB) continue;
#pragma unroll
            for (int j = 0; j < RS; ++j) dst[slot][j] = (r0 + j < r_end) ? __ldg(reinterpret_cast<const T*>(a.in_ptr[k]) + r0 + j) : T(0);
            ++slot;
        }
    };
    if (M::NCOLBREAL > 0 && nb > 0) fetch_colb(0, colb_next);

    for (int64_t b = 0; b < nb; ++b) {
        const int s = (int)(b % NS);
        const int64_t r0 = r_begin + b * RS;
        const int64_t rb = r_begin + (b * RS) / RB * RB;                // start of the current RB-row batch of the per-row combine
        T colb[NCOLB][RS];
        if (M::NCOLBREAL > 0) {
#pragma unroll
            for (int q = 0; q < NCOLB; ++q)
#pragma unroll
                for (int j = 0; j < RS; ++j) colb[q][j] = colb_next[q][j];
            if (b + 1 < nb) fetch_colb(b + 1, colb_next);
        }
        if (ALIGNED) mbar_wait(&full[s], (uint32_t)((b / NS) & 1));
        else { fill(b); __syncthreads(); }
        Cell rowc[M::NROWS][RS];                 // per-thread partials of the AXIS_ROWS outputs, one per row of the stage
#pragma unroll
        for (int o = 0; o < M::S.n_out; ++o)
            if (out_is_reduction(g.out[o].kind) && g.out[o].axis == AXIS_ROWS) {
#pragma unroll
                for (int j = 0; j < RS; ++j) rowc[slots.row[o]][j] = cell_identity<T>(g.out[o].kind);
            }
#pragma unroll
        for (int j = 0; j < RS; ++j) {
            const int64_t r = r0 + j;
            if (r >= r_end) break;
#pragma unroll
            for (int k = 0; k < M::S.n_in; ++k) {
                const SgIn in = g.in[k];
                if (in.kind == IN_VEC) {
                    const T* srow = stage_base + (((size_t)s * M::NVECIN + slots.vec[k]) * RS + j) * M::SW;
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const VEC x = *reinterpret_cast<const VEC*>(srow + (u * BLOCK + threadIdx.x) * V);
                        const T* xe = reinterpret_cast<const T*>(&x);
#pragma unroll
                        for (int e = 0; e < V; ++e) v[in.reg][u * V + e] = xe[e];
                    }
                } else if (in.kind == IN_COLB) {
                    const T sc = colb[slots.colb[k]][j];
#pragma unroll
                    for (int e = 0; e < E; ++e) v[in.reg][e] = sc;
                }
            }
            exec_body<P, T, M::NV, M::NP, E>(v, p, a, IS);
#pragma unroll
            for (int o = 0; o < M::S.n_out; ++o) {
                const SgOut out = g.out[o];
                if (out.kind == OUT_STORE) {
                    T* rowp = reinterpret_cast<T*>(a.out_ptr[o]) + r * a.out_len[o];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        if (!cvalid[u]) continue;
                        if (ALIGNED) {
                            VEC x;
                            T* xe = reinterpret_cast<T*>(&x);
#pragma unroll
                            for (int e = 0; e < V; ++e) xe[e] = v[out.src][u * V + e];
                            st_stream(reinterpret_cast<VEC*>(rowp + col[u]), x);
                        } else {
#pragma unroll
                            for (int e = 0; e < V; ++e)
                                if (e < nval[u]) rowp[col[u] + e] = v[out.src][u * V + e];
                        }
                    }
                } else if (out_is_reduction(out.kind)) {
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        if (!cvalid[u]) continue;
#pragma unroll
                        for (int e = 0; e < V; ++e) {
                            if (!evalid(u, e)) continue;
                            const int ee = u * V + e;
                            Cell& dstc = (out.axis == AXIS_ALL) ? acc[o] : (out.axis == AXIS_COLS) ? acc_col[o][ee] : rowc[out.axis == AXIS_ROWS ? slots.row[o] : 0][j];
                            if (out_is_pred_reduction(out.kind)) cell_accum_pred(out.kind, dstc, p[out.src][ee]);
                            else if (out.pred == SG_NO_PRED || p[out.pred == SG_NO_PRED ? 0 : out.pred][ee]) cell_accum_value<T>(out.kind, dstc, v[out.src][ee]);
                        }
                    }
                }
            }
        }
        // the RS rows of the stage are reduced across the warp together (see warp_reduce_rows)
#pragma unroll
        for (int o = 0; o < M::S.n_out; ++o) {
            const SgOut out = g.out[o];
            if (!(out_is_reduction(out.kind) && out.axis == AXIS_ROWS)) continue;
            warp_reduce_rows<T, RS>(out.kind, rowc[slots.row[o]], lane);
            const int64_t r = r0 + warp_row_of_lane<RS>(lane);
            if (warp_row_owner<RS>(lane) && r < r_end) s_row[slots.row[o]][warp][(int)(r - rb)] = rowc[slots.row[o]][0];
        }
        __syncthreads();                        // every thread is done with stage s (and with this batch's s_row writes)
        if (ALIGNED && threadIdx.x == 0 && b + NS < nb) { fence_proxy_async(); issue(b + NS); }
        const int64_t done_rows = (b + 1) * RS < n_rows ? (b + 1) * RS : n_rows;
        if (M::HAS_ROWS && (done_rows % RB == 0 || done_rows == n_rows)) {
            const int64_t rb_end = r_begin + done_rows;
            if ((int64_t)threadIdx.x < rb_end - rb) {
#pragma unroll
                for (int o = 0; o < M::S.n_out; ++o) {
                    const SgOut out = g.out[o];
                    if (!(out_is_reduction(out.kind) && out.axis == AXIS_ROWS)) continue;
                    Cell c = s_row[slots.row[o]][0][threadIdx.x];
#pragma unroll
                    for (int w = 1; w < WARPS; ++w) cell_combine<T>(out.kind, c, s_row[slots.row[o]][w][threadIdx.x]);
                    Cell* ws = reinterpret_cast<Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]);
                    ws[(size_t)strip * a.n + rb + threadIdx.x] = c;
                }
            }
            __syncthreads();
        }
    }

    // per-column partials of this chunk
    if (M::HAS_COLS) {
#pragma unroll
        for (int o = 0; o < M::S.n_out; ++o) {
            const SgOut out = g.out[o];
            if (!(out_is_reduction(out.kind) && out.axis == AXIS_COLS)) continue;
            Cell* ws = reinterpret_cast<Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]);
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (!cvalid[u]) continue;
#pragma unroll
                for (int e = 0; e < V; ++e)
                    if (evalid(u, e)) ws[(size_t)chunk * a.cols + col[u] + e] = acc_col[o][u * V + e];
            }
        }
    }

    // tickets: last block of the strip combines the chunks, last block of the chunk combines the strips
    if (M::HAS_COLS || M::HAS_ROWS) {
        __shared__ unsigned int s_flags;
        unsigned int* ctrl2 = a.ctrl + 8;
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned int f = 0;
            if (M::HAS_COLS && atomicAdd(&ctrl2[strip], 1u) == (unsigned int)a.n_chunks - 1) f |= 1u;
            if (M::HAS_ROWS && atomicAdd(&ctrl2[a.n_strips + chunk], 1u) == (unsigned int)a.n_strips - 1) f |= 2u;
            s_flags = f;
        }
        __syncthreads();
        const unsigned int f = s_flags;
        if (f) __threadfence();
        if (f & 1u) {
#pragma unroll
            for (int o = 0; o < M::S.n_out; ++o) {
                const SgOut out = g.out[o];
                if (!(out_is_reduction(out.kind) && out.axis == AXIS_COLS)) continue;
                const Cell* ws = reinterpret_cast<const Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]);
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    if (!cvalid[u]) continue;
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        if (!evalid(u, e)) continue;
                        Cell c = cell_identity<T>(out.kind);
                        for (int ch = 0; ch < a.n_chunks; ++ch) cell_combine<T>(out.kind, c, ldcg_cell(&ws[(size_t)ch * a.cols + col[u] + e]));
                        store_final<T>(out.kind, a.out_ptr[o], col[u] + e, c);
                    }
                }
            }
            if (threadIdx.x == 0) ctrl2[strip] = 0;
        }
        if (f & 2u) {
#pragma unroll
            for (int o = 0; o < M::S.n_out; ++o) {
                const SgOut out = g.out[o];
                if (!(out_is_reduction(out.kind) && out.axis == AXIS_ROWS)) continue;
                const Cell* ws = reinterpret_cast<const Cell*>(reinterpret_cast<char*>(a.workspace) + a.ws_off[o]);
                for (int64_t r = r_begin + threadIdx.x; r < r_end; r += BLOCK) {
                    Cell c = cell_identity<T>(out.kind);
                    for (int s = 0; s < a.n_strips; ++s) cell_combine<T>(out.kind, c, ldcg_cell(&ws[(size_t)s * a.n + r]));
                    store_final<T>(out.kind, a.out_ptr[o], r, c);
                }
            }
            if (threadIdx.x == 0) ctrl2[a.n_strips + chunk] = 0;
        }
    }
    epilogue_1d<T, NOUT>(acc, kind, a, has_all);
}

template <class P>
__global__ void __launch_bounds__(BLOCK, P::min_blocks) pass2d_template(const __grid_constant__ SgArgs a) {
    pdl_wait();
    pdl_trigger();
    if ((a.vec_ok >> 29) & 1) pass2d_body<P, false>(a);     // bit 29: rows are not 16-byte aligned (uniform)
    else pass2d_body<P, true>(a);
}

}  // namespace sgk

#include "sg_pass2d_tile.cuh"
#endif  // SG_PASS2D_CUH_
