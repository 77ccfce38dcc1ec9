// sg_plan.cpp — the plan builder and flush.
//
// "Before generating kernels, the optimizer constructs an execution plan from the pending operations.  The plan
// takes the form of a DAG ... The optimizer then traverses the DAG, merging kernel vertices and collapsing
// intermediate dependencies where possible".  Here: liveness decides which data nodes are
// materialised (a live user handle) and which collapse into registers (anonymous intermediates);
// kernel nodes are merged greedily into PASSES — one fused launch each — under three kinds of edge:
//   register edges  (producer and consumer may share a pass),
//   scalar edges    (a reduction result consumed elementwise: consumer pass > producer pass),
//   memory edges    (RAW / WAR / WAW on overlapping storage of in-place operations and views).
// SG_FLAG_UNFUSED turns every pending operation into its own pass with a materialised result: the naive
// "one kernel per method call" plan of PAPER.md:282, kept as the measurement baseline.
#include <stdio.h>
#include <string.h>
#include <time.h>

#include <algorithm>
#include <map>

#include "sg_ctx.h"

sg_status sg_build_pass(sg_ctx* c, Pass& P, std::vector<char*>& temps, std::string& dump);   // sg_build.cpp

namespace {

int es_of(const Value& v) { return dtype_size(v.dtype); }

MemRange range_of(const Value& v, bool exact = true) {
    MemRange r;
    r.exact = exact && v.kind != VK_SCALAR;
    const int64_t es = es_of(v);
    r.ptr = v.ptr; r.stride = v.stride; r.ld = v.ld; r.rows = v.rows; r.cols = v.cols;
    r.lo = v.ptr;
    if (v.kind == VK_MAT) r.hi = v.ptr + ((v.rows > 0 ? (v.rows - 1) * v.ld : 0) + v.cols) * es;
    else if (v.kind == VK_SCALAR) r.hi = v.ptr + es;
    else r.hi = v.ptr + ((v.cols > 0 ? (v.cols - 1) * v.stride : 0) + 1) * es;
    return r;
}
bool overlaps(const MemRange& a, const MemRange& b) { return a.lo < b.hi && b.lo < a.hi; }
bool same_view(const MemRange& a, const MemRange& b) {
    return a.ptr == b.ptr && a.stride == b.stride && a.ld == b.ld && a.rows == b.rows && a.cols == b.cols;
}
// may a pass that reads `r` also write `w` in place?  Only when the read is index-for-index over the very same view: then every
// element is read by the thread that writes it, before it writes it.  A shifted read (x[i+1] belongs to another thread, warp or
// block), a broadcast or a scalar read of storage the pass overwrites would see a mix of old and new values.
bool read_is_private_to_writer(const MemRange& w, const MemRange& r) { return r.exact && same_view(w, r); }

bool pending(const sg_ctx* c, const Value& v) { return v.node >= 0 && !c->nodes[v.node].done; }

}  // namespace

namespace {

// The signature of the pending list (PlanMemo, sg_ctx.h): everything the pass assignment reads, as bytes.  Values are numbered in
// order of first appearance (table slots differ from step to step), described once: kind, dtype, shape, address, liveness, producer.
// Immediates are left out: they decide nothing in the assignment (a build that then fails a limit falls back to the full planner).
std::string plan_signature(const sg_ctx* c, bool unfused) {
    const std::vector<Node>& N = c->nodes;
    const std::vector<Value>& V = c->values;
    // upper bound of the key: per operation a head + two operands + two results, each value described at most once per mention
    constexpr size_t VAL = 4 + 8 * 4 + 5 * 8, NODE = 12 * 4 + 16 + 2 * 8 + 4 * VAL;
    std::string key;
    key.resize(16 + N.size() * NODE + c->contracts.size() * (VAL + 4));
    char* w = &key[0];
    const auto put = [&](const void* p, size_t n) { memcpy(w, p, n); w += n; };
    const auto put32 = [&](int32_t x) { memcpy(w, &x, 4); w += 4; };
    // value numbering by first appearance: a small open-addressed table keyed by the table slot
    size_t cap = 64;
    while (cap < 8 * N.size() + 16) cap <<= 1;
    std::vector<int32_t> slot_key(cap, -1), slot_id(cap, 0);
    int32_t next_id = 0;
    const auto value = [&](int vi) {
        size_t h = ((size_t)vi * 0x9E3779B1u) & (cap - 1);
        while (slot_key[h] >= 0 && slot_key[h] != vi) h = (h + 1) & (cap - 1);
        if (slot_key[h] == vi) { put32(slot_id[h]); return; }
        slot_key[h] = vi; slot_id[h] = next_id;
        const Value& v = V[vi];
        put32(-1 - next_id);                            // first appearance: the description follows
        ++next_id;
        const int32_t head[8] = {v.kind, v.dtype, (v.node >= 0 && !N[v.node].done) ? v.node : -1, v.materialised, v.slot >= 0, v.user_refs > 0, v.count_known, 0};
        put(head, sizeof(head));
        const int64_t shape[5] = {(int64_t)(uintptr_t)v.ptr, v.stride, v.ld, v.rows, v.cols};
        put(shape, sizeof(shape));
    };
    put32((int32_t)N.size());
    put32(unfused ? 1 : 0);
    for (const Node& n : N) {
        const int32_t head[12] = {n.kind, n.op, n.n_opd, n.axis, n.dtype, n.src_dtype, n.is2d, n.inplace, n.needed, n.post, n.done, 0};
        put(head, sizeof(head));
        const int64_t dom[2] = {n.rows, n.cols};
        put(dom, sizeof(dom));
        for (int j = 0; j < n.n_opd; ++j) {
            put32(n.opd[j].kind); put32(n.opd[j].bcast);
            if (n.opd[j].kind != OPD_IMM) value(n.opd[j].value);
        }
        if (n.out >= 0) value(n.out); else put32(0x7fffffff);
        if (n.out2 >= 0) value(n.out2); else put32(0x7fffffff);
    }
    put32((int32_t)c->contracts.size());
    for (const Contract& k : c->contracts) { value(k.value); put32(k.kind); }
    key.resize((size_t)(w - key.data()));
    return key;
}

// quantifier outputs of a pass that may end early at a violated contract (PF_EARLY_EXIT with registered for_all contracts)
struct ExitMember { int value; uint8_t kind; bool is_contract; };
typedef std::vector<std::vector<ExitMember>> ExitGroups;

// Plans and launches everything pending.  *executed = number of passes whose kernels were queued on the stream when the
// function returned (all of them on success).  On failure the caller rolls the context back (retire_nodes).
sg_status flush_body(sg_ctx* c, int* executed, ExitGroups* exit_groups) {
    bool unfused = c->flags & SG_FLAG_UNFUSED;
    struct FlagGuard { sg_ctx* c; uint32_t flags; ~FlagGuard() { c->flags = flags; } } flag_guard{c, c->flags};   // the last-resort lowering below sets SG_FLAG_UNFUSED for this flush only
    std::vector<Node>& N = c->nodes;
    std::vector<Value>& V = c->values;
    int64_t launches_total = c->stats.launches_total;
    memset(&c->stats, 0, sizeof(c->stats));
    c->stats.launches_total = launches_total;
    c->dumps.clear();

    // ---- 1. liveness: which pending operations are needed at all ----------------------------------------
    std::vector<int> work;
    auto need = [&](int i) { if (i >= 0 && !N[i].done && !N[i].needed) { N[i].needed = true; work.push_back(i); } };
    for (size_t i = 0; i < N.size(); ++i) {
        if (N[i].done) continue;
        const bool live = (N[i].out >= 0 && V[N[i].out].user_refs > 0) || (N[i].out2 >= 0 && V[N[i].out2].user_refs > 0) || N[i].inplace;
        if (live) need((int)i);
    }
    for (const Contract& k : c->contracts) need(V[k.value].node);
    while (!work.empty()) {
        const int i = work.back(); work.pop_back();
        for (int j = 0; j < N[i].n_opd; ++j)
            if (N[i].opd[j].kind != OPD_IMM) need(V[N[i].opd[j].value].node);
    }
    // values that will exist in memory after this flush (live handle or caller-provided storage)
    auto materialises = [&](const Node& n) {
        if (n.kind != NK_MAP) return false;
        return unfused || n.inplace || V[n.out].user_refs > 0;
    };
    // ---- 2. POST contracts read stored results (R17): mark their predicate cone ----------------
    std::vector<int> post_group(N.size(), -1);
    std::vector<std::vector<int>> post_leaves(c->contracts.size());
    for (size_t ki = 0; ki < c->contracts.size(); ++ki) {
        const Contract& k = c->contracts[ki];
        if (k.kind != SG_CONTRACT_POST) continue;
        std::vector<int> st{V[k.value].node};
        while (!st.empty()) {
            const int i = st.back(); st.pop_back();
            if (i < 0 || N[i].done || N[i].post) continue;
            N[i].post = true;
            post_group[i] = (int)ki;
            for (int j = 0; j < N[i].n_opd; ++j) {
                if (N[i].opd[j].kind == OPD_IMM) continue;
                const Value& v = V[N[i].opd[j].value];
                if (!pending(c, v)) continue;
                if (materialises(N[v.node])) { post_leaves[ki].push_back(v.node); continue; }   // leaf: read back from memory
                st.push_back(v.node);
            }
        }
    }

    // ---- 3. pass assignment ------------------------------------------------------------------------------
    // A pass holds at most SG_MAX_OUT outputs.  Stores and reductions are counted when an operation joins a pass, but an intermediate
    // that joined as a register value becomes one more output LATER, when a consumer ends up in a later pass (a spill) — so the first
    // assignment may overfill a pass.  Then the assignment is repeated with outputs held in reserve for such spills (2, 4, 6, 7 of the
    // 8), and as the last resort with the unfused lowering, which always fits (one operation, one output per pass).
    std::vector<Pass> passes;
    std::vector<char> spill;                    // value must be stored because a later pass consumes it
    auto pass_outputs = [&](const Pass& P) {
        int outs = 0;
        for (int k : P.nodes) outs += (N[k].kind != NK_MAP) || materialises(N[k]) || spill[N[k].out];
        return outs;
    };
    // The other limits of a pass (distinct inputs, registers of the evaluator, instructions) are only known once its program is built:
    // a build that fails on one of them also repeats the assignment, with fewer operations per pass.
    static const int reserves[] = {0, 2, 4, 6, 7}, node_limits[] = {SG_MAX_INSTR, SG_MAX_INSTR, 16, 8, 4};
    std::vector<char*> temps;
    const sg_stats stats0 = c->stats;
    // plan cache: the same pending list (signature) was assigned before — take that assignment, under the limits it succeeded with
    // (a loop whose pending lists never repeat — other buffers or views every step, like Listing 5 written over host-issued row
    // operations — would only pay for signatures: after 16 misses in a row the cache sits out the next 64 flushes, then tries again)
    bool use_cache = !(c->flags & SG_FLAG_NO_PLAN_CACHE);
    if (use_cache && c->plan_cache_pause > 0) { c->plan_cache_pause--; use_cache = false; }
    std::string signature;
    const PlanMemo* memo = nullptr;
    if (use_cache) {
        signature = plan_signature(c, unfused);
        for (const PlanMemo& m : c->plan_cache)
            if (m.key == signature) { memo = &m; break; }
        if (memo) { c->plan_cache_hits++; c->plan_cache_miss_streak = 0; }
        else {
            c->plan_cache_misses++;
            if (++c->plan_cache_miss_streak >= 16) { c->plan_cache_pause = 64; c->plan_cache_miss_streak = 8; }
        }
    }
    for (int attempt = memo ? memo->attempt : 0;; ++attempt) {
    if (attempt >= 5) { unfused = true; c->flags |= SG_FLAG_UNFUSED; }
    const int out_limit = SG_MAX_OUT - reserves[attempt < 5 ? attempt : 0];
    const int node_limit = node_limits[attempt < 5 ? attempt : 0];
    passes.clear();
    spill.assign(V.size(), 0);
    c->stats = stats0;
    c->dumps.clear();
    for (Node& n : N) {
        if (n.done) continue;
        n.pass = -1;
        if (n.out >= 0 && V[n.out].user_refs < 0) V[n.out].user_refs = 0;       // spill marks of an abandoned attempt
    }
    if (memo) {
        passes = memo->passes;
        for (size_t i = 0; i < N.size(); ++i) {
            N[i].pass = memo->node_pass[i];
            if (memo->node_spill[i]) spill[N[i].out] = 1;
        }
    } else
    for (size_t i = 0; i < N.size(); ++i) {
        Node& X = N[i];
        if (X.done || !X.needed) continue;
        int lb = 0, forced = -1;
        std::vector<MemRange> reads, writes;
        std::vector<std::pair<int, bool>> reg_producers;     // (producer, the operand is read index-for-index)
        for (int j = 0; j < X.n_opd; ++j) {
            if (X.opd[j].kind == OPD_IMM) continue;
            const Value& v = V[X.opd[j].value];
            if (pending(c, v) && N[v.node].needed) {
                const Node& Y = N[v.node];
                if (Y.kind == NK_MAP) {
                    // a neighbour operand and the operand of a dtype conversion are read back from memory: a pass has ONE value
                    // file, the conversion happens as the operand is loaded (IN_VEC_CVT)
                    const bool from_memory = X.opd[j].kind == OPD_SHIFT || (X.kind == NK_MAP && X.op == NODE_OP_CAST);
                    const bool via_memory = unfused || (X.post && materialises(Y)) || from_memory;
                    lb = std::max(lb, Y.pass + (via_memory ? 1 : 0));
                    const bool exact = X.opd[j].kind != OPD_SHIFT && X.opd[j].bcast == SG_BCAST_NONE;
                    if (!via_memory) reg_producers.push_back({v.node, exact});
                    if (from_memory) spill[X.opd[j].value] = 1;
                    // A pending IN-PLACE result read from memory by a later pass is a read of the caller's buffer: a later in-place
                    // writer of overlapping storage (another view of it) must not share that pass (WAR).  Spilled temporaries have
                    // storage of their own and need no such edge.
                    if (via_memory && Y.inplace && V[Y.out].ptr) reads.push_back(range_of(V[Y.out], exact));
                } else if (Y.kind == NK_REDUCE) {
                    lb = std::max(lb, Y.pass + 1);
                } else {    // NK_FILTER: only a reduction over the kept values may follow, in the same pass
                    if (X.kind != NK_REDUCE) return sg_fail(c, SG_ERR_UNSUPPORTED, "operation on a pending filter output");
                    forced = Y.pass;
                }
            } else {
                if (!v.materialised && v.slot < 0) return sg_fail(c, SG_ERR_ARG, "operand has neither storage nor a pending producer");
                if (v.slot >= 0) continue;                      // scalar slot written by an earlier flush
                reads.push_back(range_of(v, X.opd[j].kind != OPD_SHIFT && X.opd[j].bcast == SG_BCAST_NONE));
            }
        }
        if (X.post && post_group[i] >= 0)       // the whole predicate of a POST contract runs after the results it reads are stored
            for (int y : post_leaves[post_group[i]])
                if (N[y].pass >= 0) lb = std::max(lb, N[y].pass + 1);
        if (X.kind == NK_MAP && X.inplace) writes.push_back(range_of(V[X.out]));
        if (X.kind == NK_FILTER && X.inplace) writes.push_back(range_of(V[X.out]));
        for (size_t q = 0; q < passes.size(); ++q) {
            for (const MemRange& r : reads)
                for (const MemRange& w : passes[q].writes)
                    if (overlaps(r, w)) lb = std::max(lb, (int)q + 1);                          // RAW through memory
            for (const MemRange& w : writes) {
                for (const MemRange& w2 : passes[q].writes)
                    if (overlaps(w, w2)) lb = std::max(lb, (int)q + 1);                         // WAW
                for (const MemRange& r : passes[q].reads)
                    if (overlaps(w, r)) lb = std::max(lb, (int)q + (read_is_private_to_writer(w, r) ? 0 : 1));  // WAR: same pass only index-for-index
            }
        }
        // within this very operation: an in-place result may alias an operand only index-for-index
        for (const MemRange& w : writes)
            for (const MemRange& r : reads)
                if (overlaps(w, r) && !read_is_private_to_writer(w, r)) return sg_fail(c, SG_ERR_ALIAS, "in-place operation reads a shifted or overlapping view of its destination");

        const bool stores = materialises(X);
        const int xdt = (X.dtype == SG_BOOL) ? -1 : X.dtype;
        auto compatible = [&](const Pass& P) {
            if (unfused) return false;
            if (P.is2d != X.is2d) return false;
            if (X.is2d) { if (P.rows != X.rows || P.cols != X.cols) return false; }
            else if (std::llabs((long long)(P.cols - X.cols)) > 1024) return false;
            if (xdt >= 0 && P.dtype >= 0 && P.dtype != xdt) return false;
            if (X.kind == NK_FILTER && (P.has_filter || P.has_store || X.is2d)) return false;
            if (stores && P.has_filter) return false;
            if ((int)P.nodes.size() + 1 > node_limit) return false;
            if (pass_outputs(P) + 1 > out_limit) return false;
            return true;
        };
        int p = -1;
        if (forced >= 0) {
            if (lb > forced) return sg_fail(c, SG_ERR_UNSUPPORTED, "reduction over a filter output cannot share the filter's pass");
            p = forced;
        } else {
            for (size_t q = (size_t)lb; q < passes.size(); ++q)
                if (compatible(passes[q])) { p = (int)q; break; }
            if (p < 0) {
                passes.emplace_back();
                p = (int)passes.size() - 1;
                passes[p].is2d = X.is2d; passes[p].rows = X.rows; passes[p].cols = X.cols;
            }
        }
        Pass& P = passes[p];
        X.pass = p;
        P.nodes.push_back((int)i);
        if (!X.is2d) P.cols = std::max(P.cols, X.cols);
        if (xdt >= 0 && P.dtype < 0) P.dtype = xdt;
        P.has_filter |= (X.kind == NK_FILTER);
        P.has_store |= stores;
        for (const MemRange& r : reads) P.reads.push_back(r);
        for (const MemRange& w : writes) P.writes.push_back(w);
        for (const auto& yp : reg_producers) {
            const int y = yp.first;
            if (N[y].pass < p) {                                // register edge became a cross-pass edge: spill the value
                spill[N[y].out] = 1;
                if (passes[N[y].pass].has_filter) return sg_fail(c, SG_ERR_UNSUPPORTED, "a filter pass cannot materialise an intermediate");
                passes[N[y].pass].has_store = true;
                if (N[y].inplace && V[N[y].out].ptr) P.reads.push_back(range_of(V[N[y].out], yp.second));     // (see above: the caller's buffer is read here)
            }
        }
    }
    bool fits = true;
    for (const Pass& P : passes) fits = fits && pass_outputs(P) <= SG_MAX_OUT;
    if (!fits && attempt < 5) {
        if (memo) { c->plan_cache.erase(c->plan_cache.begin() + (memo - c->plan_cache.data())); memo = nullptr; }
        continue;
    }
    if (passes.size() > 256) return sg_fail(c, SG_ERR_CAPACITY, "more than 256 passes in one flush");     // (sg_stats describes the first 16)

    // ---- 4. programs, outputs, geometry ------------------------------------------------------------------
    // spilled intermediates become context-owned temporaries, released after the launches are queued
    const auto build_all = [&]() -> sg_status {
    c->stats.n_passes = (int32_t)passes.size();
    for (const Node& n : N) c->stats.n_nodes += (!n.done && n.needed);
    std::vector<char> spill_copy = spill;
    for (size_t pi = 0; pi < passes.size(); ++pi) {
        Pass& P = passes[pi];
        // mark spilled values by giving them a (hidden) reference for the duration of the build
        for (int k : P.nodes)
            if (N[k].kind == NK_MAP && spill_copy[N[k].out] && V[N[k].out].user_refs == 0) V[N[k].out].user_refs = -1;
        std::string dump;
        sg_status s = sg_build_pass(c, P, temps, dump);
        if (s != SG_OK) return s;
        c->dumps.push_back(P.prog);
        char err[256] = {0};
        int rc = sgk_plan(P.prog, P.args, (c->flags & SG_FLAG_FORCE_BYTECODE) ? 1 : 0, c->sm_count, c->plan_only ? 0 : 1, &P.geom, err, sizeof(err));
        if (rc != 0) return sg_fail(c, (sg_status)rc, err);
        P.args.no_early_exit = (c->flags & SG_FLAG_NO_EARLY_EXIT) ? 1 : 0;
        if (pi < 16) {
            c->stats.pass_n_in[pi] = P.n_mem_in;
            c->stats.pass_n_instr[pi] = P.prog.shape.n_instr;
            c->stats.pass_n_out[pi] = P.prog.shape.n_out;
            c->stats.pass_n_args[pi] = P.n_mem_in + P.n_scalar_in + P.prog.shape.n_out;
            c->stats.pass_kernel[pi] = P.geom.template_id;
        }
        c->stats.bytes_min += P.bytes;
        if (P.geom.template_id > 0) c->stats.n_template++; else c->stats.n_bytecode++;
    }
    return SG_OK;
    };
    const sg_status built = build_all();
    if (built == SG_ERR_CAPACITY && attempt < 5) {
        if (memo) {         // (immediates are not part of the signature: this list needs tighter limits than the remembered one)
            c->plan_cache.erase(c->plan_cache.begin() + (memo - c->plan_cache.data()));
            memo = nullptr;
        }
        continue;
    }
    if (built != SG_OK) return built;
    if (use_cache && !memo) {
        PlanMemo m;
        m.key = std::move(signature);
        m.attempt = attempt;
        m.node_pass.resize(N.size());
        m.node_spill.assign(N.size(), 0);
        for (size_t i = 0; i < N.size(); ++i) {
            m.node_pass[i] = N[i].pass;
            m.node_spill[i] = (N[i].out >= 0 && N[i].kind == NK_MAP && N[i].needed) ? spill[N[i].out] : 0;
        }
        m.passes.reserve(passes.size());
        for (const Pass& P : passes) {
            Pass q;
            q.is2d = P.is2d; q.has_filter = P.has_filter; q.has_store = P.has_store; q.dtype = P.dtype; q.rows = P.rows; q.cols = P.cols; q.nodes = P.nodes;
            m.passes.push_back(std::move(q));
        }
        if (c->plan_cache.size() < 8) c->plan_cache.push_back(std::move(m));
        else { c->plan_cache[c->plan_cache_next % 8] = std::move(m); c->plan_cache_next++; }
    }
    break;
    }

    // ---- 5. resources and launches -----------------------------------------------------------------------
    c->last.clear();
    if (!c->plan_only) {
        size_t ws = 0, st = 0; int cw = 0;
        for (const Pass& P : passes) { ws = std::max(ws, P.geom.ws_bytes); st = std::max(st, P.geom.state_words); cw = std::max(cw, P.geom.ctrl_words); }
        if (cw + 8 > c->ctrl_words) return sg_fail(c, SG_ERR_CAPACITY, "matrix pass needs more ticket words than the control block holds");
        if (ws > c->workspace_bytes) {
            cudaStreamSynchronize(c->stream);
            if (c->workspace) cudaFree(c->workspace);
            c->workspace_bytes = ws + ws / 4;
            if (cudaMalloc((void**)&c->workspace, c->workspace_bytes) != cudaSuccess) { c->workspace = nullptr; c->workspace_bytes = 0; cudaGetLastError(); return sg_fail(c, SG_ERR_OOM, "workspace allocation failed"); }
        }
        if (st > c->tile_state_words) {
            cudaStreamSynchronize(c->stream);
            if (c->tile_state) cudaFree(c->tile_state);
            c->tile_state_words = st + st / 4;
            if (cudaMalloc((void**)&c->tile_state, 8 * c->tile_state_words) != cudaSuccess || cudaMemset(c->tile_state, 0, 8 * c->tile_state_words) != cudaSuccess) {
                c->tile_state = nullptr; c->tile_state_words = 0; cudaGetLastError();
                return sg_fail(c, SG_ERR_OOM, "tile-state allocation failed");
            }
        }
        cudaEvent_t t0 = c->ev_t0, t1 = c->ev_t1;
        if (c->timing) {            // timed region: this flush gets its own event pair, read back at sg_timing_end
            std::pair<cudaEvent_t, cudaEvent_t> pr{nullptr, nullptr};
            if (!c->timing_pool.empty()) { pr = c->timing_pool.back(); c->timing_pool.pop_back(); }
            else if (cudaEventCreate(&pr.first) != cudaSuccess || cudaEventCreate(&pr.second) != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, "event creation failed");
            c->timing_events.push_back(pr);
            t0 = pr.first; t1 = pr.second;
        }
        cudaEventRecord(t0, c->stream);
        for (Pass& P : passes) {
            P.args.workspace = c->workspace;
            P.args.tile_state = c->tile_state;
            P.args.ctrl = c->ctrl;
            if (P.prog.shape.flags & PF_FILTER) {
                if (++c->epoch > 0x3ffff0u) {       // epoch tag about to wrap: clear the states once
                    cudaMemsetAsync(c->tile_state, 0, 8 * c->tile_state_words, c->stream);
                    c->epoch = 1;
                }
                P.args.epoch = c->epoch;
            }
            cudaError_t e = sgk_launch(P.prog, P.args, P.geom, c->stream);
            if (e != cudaSuccess) {
                c->stats.launches_total = launches_total;
                return sg_fail(c, SG_ERR_CUDA, std::string("kernel launch failed: ") + cudaGetErrorString(e));
            }
            c->last.push_back({P.prog, P.args, P.geom});
            launches_total++;
            ++*executed;
        }
        cudaEventRecord(t1, c->stream);
        // a8: hand the flush's scalars back.  The reductions' last blocks have written their results to the pinned mirror themselves
        // (SgArgs.out_host); whatever else the flush produced in the slab (filter counts, one-element passes) goes back in one copy
        int64_t lo = c->slab_slots, hi = -1;
        auto written_by_kernel = [&](int64_t slot) {
            for (const Pass& P : passes)
                for (int o = 0; o < P.prog.shape.n_out; ++o)
                    if (P.args.out_host[o] == (void*)(c->slab_host + 8 * slot)) return true;
            return false;
        };
        for (const Node& n : N) {
            if (n.done || !n.needed) continue;
            for (int o : {n.out, n.out2})
                if (o >= 0 && V[o].kind == VK_SCALAR && V[o].slot >= 0 && !written_by_kernel(V[o].slot)) { lo = std::min(lo, V[o].slot); hi = std::max(hi, V[o].slot); }
        }
        if (hi >= lo) {
            if (cudaMemcpyAsync(c->slab_host + 8 * lo, c->slab + 8 * lo, 8 * (size_t)(hi - lo + 1), cudaMemcpyDeviceToHost, c->stream) != cudaSuccess)
                return sg_fail(c, SG_ERR_CUDA, "scalar hand-back failed");
        }
        cudaEventRecord(c->ev_done, c->stream);
        // storage released since the previous flush goes back now; this flush's temporaries stay until the next
        // flush so that sg_replay_last can re-run the same launches
        for (char* t : c->deferred_free) sg_dev_free(c, t);
        c->deferred_free = temps;
    } else {
        for (Pass& P : passes) c->last.push_back({P.prog, P.args, P.geom});
        *executed = (int)passes.size();
    }
    c->stats.launches_total = launches_total;
    // quantifier passes that may end early at a violated contract: remember their members for the contract check
    for (const Pass& P : passes) {
        if (!(P.prog.shape.flags & PF_EARLY_EXIT) || !P.args.exit_any || P.args.no_early_exit) continue;
        std::vector<ExitMember> grp;
        for (int k : P.nodes) {
            const Node& n = N[k];
            if (n.kind != NK_REDUCE || (n.op != OUT_ALL && n.op != OUT_ANY)) continue;
            bool is_contract = false;
            for (const Contract& ct : c->contracts) is_contract |= (ct.value == n.out && n.op == OUT_ALL);
            grp.push_back({n.out, n.op, is_contract});
        }
        exit_groups->push_back(grp);
    }

    return SG_OK;
}

// Retires the pending list.  Operations of the first `executed` passes ran (their kernels are queued): their results have
// storage now.  Everything else — operations no live handle needed, and after a failed flush the operations that were never
// launched — is DISCARDED: storage this flush allocated for their results is given back, their result handles name no data
// (a discarded filter output is empty) until they are released.  In-place destinations keep their previous contents.
void retire_nodes(sg_ctx* c, int executed) {
    std::vector<Node>& N = c->nodes;
    std::vector<Value>& V = c->values;
    for (Node& n : N) {
        if (n.done) continue;
        n.done = true;
        const bool ran = n.needed && n.pass >= 0 && n.pass < executed;
        for (int o : {n.out, n.out2}) {
            if (o < 0) continue;
            Value& v = V[o];
            if (v.user_refs < 0) v.user_refs = 0;
            if (v.node >= 0 && &N[v.node] == &n) v.node = -1;
            if (!ran) {
                if (v.fresh_alloc && v.ptr) { sg_dev_free(c, v.ptr); v.ptr = nullptr; v.owned = false; }
                if (!n.inplace && v.kind != VK_SCALAR) v.materialised = false;
                if (!v.count_known) { v.count_known = true; v.cols = 0; v.ld = 0; }
            }
            v.fresh_alloc = false;
        }
    }
    for (int i : c->live) { Value& v = V[i]; if (v.node >= 0 && N[v.node].done) v.node = -1; }
    N.clear();
    size_t keep = 0;
    for (int i : c->live) {         // unreferenced results die with the flush
        Value& v = V[i];
        if (v.alive && v.user_refs <= 0) {
            if (v.owned && v.ptr) { c->deferred_free.push_back(v.ptr); v.ptr = nullptr; v.owned = false; }
            if (v.kind == VK_SCALAR && v.slot >= 0) {
                bool contract = false;
                for (const Contract& k : c->contracts) contract |= (&V[k.value] == &v);
                if (!contract) { c->slab_free.push_back(v.slot); v.slot = -1; v.alive = false; }
            } else v.alive = false;
        }
        if (v.alive) c->live[keep++] = i;
        else c->free_values.push_back(i);       // the pending list is empty: nothing names this slot any more
    }
    c->live.resize(keep);
}

}  // namespace

// The flush is transactional: if planning fails (unsupported chain, too many passes, aliasing, allocation), nothing was launched,
// the error is reported and the pending list is discarded, so the context stays usable for later work.  If a launch fails, the
// passes already queued count as executed and the rest is discarded.
sg_status sg_flush_impl(sg_ctx* c) {
    if (c->nodes.empty()) return SG_OK;
    std::vector<Value>& V = c->values;
    int executed = 0;
    ExitGroups exit_groups;
    const sg_status s = flush_body(c, &executed, &exit_groups);
    if (s != SG_OK) {
        const std::string why = c->err;
        c->contracts.clear();               // before retire_nodes: contract scalars of a discarded list give their slots back
        retire_nodes(c, executed);
        c->err = why + (executed ? " (later passes discarded)" : " (pending operations discarded)");
        return s;
    }
    // ---- 6. commit: results now have storage; the pending list is consumed -------------------------------
    retire_nodes(c, 1 << 30);

    // ---- 7. contracts: evaluated on the device with the data; read with the scalars ----
    sg_status result = SG_OK;
    if (!c->contracts.empty()) {
        if (!c->plan_only && cudaEventSynchronize(c->ev_done) != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, "event sync failed");
        for (const Contract& k : c->contracts) {
            const Value& v = V[k.value];
            bool ok = true;
            if (!c->plan_only && v.slot >= 0) ok = c->slab_host[8 * v.slot] != 0;
            if (!ok && result == SG_OK) {
                result = SG_ERR_CONTRACT;
                c->err = std::string(k.kind == SG_CONTRACT_PRE ? "precondition" : "postcondition") + " violated: " + k.tag;
            }
        }
        // A pass of quantifiers ends as soon as one of its registered for_all contracts is violated (early exit).  The other
        // quantifiers of that pass were then evaluated on a PREFIX of the data: one that was decided on the prefix (a for_all
        // already false, an exists already true) is final, the others are not evaluated and reading them is an error.
        if (result == SG_ERR_CONTRACT && !c->plan_only)
            for (const auto& grp : exit_groups) {
                bool violated = false;
                for (const ExitMember& m : grp)
                    if (m.is_contract && V[m.value].slot >= 0 && c->slab_host[8 * V[m.value].slot] == 0) violated = true;
                if (!violated) continue;
                for (const ExitMember& m : grp) {
                    Value& v = V[m.value];
                    if (v.slot < 0) continue;
                    const bool t = c->slab_host[8 * v.slot] != 0;
                    if ((m.kind == OUT_ALL && t) || (m.kind == OUT_ANY && !t)) v.undecided = true;
                }
            }
        c->contracts.clear();
    }
    if (!c->plan_only) {
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, cudaGetErrorString(e));
    }
    return result;
}

extern "C" sg_status sg_plan_cache_stats(sg_ctx* c, int64_t* hits, int64_t* misses) {
    if (!c || !hits || !misses) return SG_ERR_ARG;
    *hits = c->plan_cache_hits;
    *misses = c->plan_cache_misses;
    return SG_OK;
}

extern "C" sg_status sg_last_flush_ms(sg_ctx* c, float* ms) {
    if (!c || !ms) return SG_ERR_ARG;
    if (c->plan_only) { *ms = 0.f; return SG_OK; }
    if (cudaEventSynchronize(c->ev_t1) != cudaSuccess || cudaEventElapsedTime(ms, c->ev_t0, c->ev_t1) != cudaSuccess) {
        cudaGetLastError();
        return sg_fail(c, SG_ERR_CUDA, "no timed flush");
    }
    return SG_OK;
}

extern "C" sg_status sg_timing_begin(sg_ctx* c) {
    if (!c) return SG_ERR_ARG;
    for (auto& pr : c->timing_events) c->timing_pool.push_back(pr);
    c->timing_events.clear();
    c->timing = true;
    return SG_OK;
}

extern "C" sg_status sg_timing_end(sg_ctx* c, float* total_ms, int32_t* n_flushes) {
    if (!c || !total_ms || !n_flushes) return SG_ERR_ARG;
    c->timing = false;
    *total_ms = 0.f;
    *n_flushes = (int32_t)c->timing_events.size();
    if (c->plan_only) return SG_OK;
    for (auto& pr : c->timing_events) {
        float ms = 0.f;
        if (cudaEventSynchronize(pr.second) != cudaSuccess || cudaEventElapsedTime(&ms, pr.first, pr.second) != cudaSuccess) {
            cudaGetLastError();
            return sg_fail(c, SG_ERR_CUDA, "timed flush not complete");
        }
        *total_ms += ms;
        c->timing_pool.push_back(pr);
    }
    c->timing_events.clear();
    return SG_OK;
}

extern "C" sg_status sg_replay_last(sg_ctx* c, int32_t reps, float* ms_per_rep) {
    if (!c || !ms_per_rep || reps <= 0) return SG_ERR_ARG;
    SgDeviceScope dev_scope(c);
    if (c->plan_only) { *ms_per_rep = 0.f; return SG_OK; }
    if (c->last.empty()) return sg_fail(c, SG_ERR_ARG, "nothing to replay");
    cudaEventRecord(c->ev_t0, c->stream);
    for (int r = 0; r < reps; ++r)
        for (Launch& l : c->last) {
            if (l.prog.shape.flags & PF_FILTER) {
                if (++c->epoch > 0x3ffff0u) { cudaMemsetAsync(c->tile_state, 0, 8 * c->tile_state_words, c->stream); c->epoch = 1; }
                l.args.epoch = c->epoch;
            }
            cudaError_t e = sgk_launch(l.prog, l.args, l.geom, c->stream);
            if (e != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, cudaGetErrorString(e));
            c->stats.launches_total++;
        }
    cudaEventRecord(c->ev_t1, c->stream);
    float ms = 0.f;
    if (cudaEventSynchronize(c->ev_t1) != cudaSuccess || cudaEventElapsedTime(&ms, c->ev_t0, c->ev_t1) != cudaSuccess)
        return sg_fail(c, SG_ERR_CUDA, cudaGetErrorString(cudaGetLastError()));
    *ms_per_rep = ms / reps;
    return SG_OK;
}

// The last flush's launch sequence captured ONCE into a CUDA graph and replayed `reps` times: the launch-inclusive measurement of
// short passes (SURVEY.md §8(d) note iii).  device_ms: CUDA events around the replays; wall_ms: host clock from the first
// cudaGraphLaunch to the stream's completion, both per replay.
extern "C" sg_status sg_replay_last_graph(sg_ctx* c, int32_t reps, float* device_ms_per_rep, float* wall_ms_per_rep) {
    if (!c || !device_ms_per_rep || !wall_ms_per_rep || reps <= 0) return SG_ERR_ARG;
    SgDeviceScope dev_scope(c);
    if (c->plan_only) { *device_ms_per_rep = *wall_ms_per_rep = 0.f; return SG_OK; }
    if (c->last.empty()) return sg_fail(c, SG_ERR_ARG, "nothing to replay");
    for (const Launch& l : c->last)
        if (l.prog.shape.flags & PF_FILTER) return sg_fail(c, SG_ERR_UNSUPPORTED, "a filter pass tags its tile states with a per-launch epoch: not replayable from a graph");
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    auto fail = [&](const char* what) {
        const cudaError_t e = cudaGetLastError();
        if (exec) cudaGraphExecDestroy(exec);
        if (graph) cudaGraphDestroy(graph);
        return sg_fail(c, SG_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
    };
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return fail("stream sync");
    // captured on a stream of its own (the context's stream may be the legacy default stream, which cannot capture); the graph
    // is then launched on the context's stream like every other piece of work
    cudaStream_t cap = nullptr;
    if (cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) != cudaSuccess) return fail("capture stream");
    if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { cudaStreamDestroy(cap); return fail("begin capture"); }
    // ALL `reps` repetitions go into ONE graph: the device then runs them back to back without the host in between (a graph launch
    // per repetition would measure the host's launch rate, ~4 us per cudaGraphLaunch, not the passes)
    bool ok = true;
    for (int r = 0; r < reps && ok; ++r)
        for (Launch& l : c->last) ok = ok && sgk_launch(l.prog, l.args, l.geom, cap) == cudaSuccess;
    const bool ended = cudaStreamEndCapture(cap, &graph) == cudaSuccess;
    cudaStreamDestroy(cap);
    if (!ended || !ok || !graph) return fail("capture");
    if (cudaGraphInstantiate(&exec, graph, 0) != cudaSuccess) return fail("graph instantiate");
    cudaGraphLaunch(exec, c->stream);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return fail("graph warm-up");
    const int graph_launches = 3;
    timespec w0, w1;
    clock_gettime(CLOCK_MONOTONIC, &w0);
    cudaEventRecord(c->ev_t0, c->stream);
    for (int r = 0; r < graph_launches; ++r) cudaGraphLaunch(exec, c->stream);
    cudaEventRecord(c->ev_t1, c->stream);
    if (cudaStreamSynchronize(c->stream) != cudaSuccess) return fail("graph replay");
    clock_gettime(CLOCK_MONOTONIC, &w1);
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->ev_t0, c->ev_t1) != cudaSuccess) return fail("event");
    *device_ms_per_rep = ms / (reps * graph_launches);
    *wall_ms_per_rep = (float)(((w1.tv_sec - w0.tv_sec) * 1e3 + (w1.tv_nsec - w0.tv_nsec) * 1e-6) / (reps * graph_launches));
    c->stats.launches_total += (int64_t)reps * (graph_launches + 1) * (int64_t)c->last.size();
    cudaGraphExecDestroy(exec);
    cudaGraphDestroy(graph);
    return SG_OK;
}
