// sg_api.cpp — the C ABI of include/sg.h: context, collections, views and the enqueue side of deferred
// execution.  Nothing here launches a kernel: operations are appended to the pending list
// after their scalar contracts (count / shape / dtype equality) are checked.
#include <stdio.h>
#include <string.h>

#include "sg_ctx.h"

#define CK(c) do { if (!(c)) return SG_ERR_ARG; } while (0)

sg_status sg_fail(sg_ctx* c, sg_status code, const std::string& msg) {
    if (c) c->err = msg;
    return code;
}

// A handle is (generation << 32) | (slot + 1).  Slots of dead values are recycled (retire_nodes puts them on free_values once no
// pending operation can name them), so a long-running loop's table stays as large as its high-water mark of live handles; the
// generation makes a handle that was released, and whose slot now holds another value, an unknown handle instead of an alias.
static inline int hidx(sg_handle h) { return (int)(h & 0xffffffffll) - 1; }
static inline sg_handle hnd(const sg_ctx* c, int idx) { return ((sg_handle)c->values[idx].gen << 32) | (sg_handle)(idx + 1); }
static Value* val(sg_ctx* c, sg_handle h) {
    const int64_t slot = (h & 0xffffffffll) - 1;
    if (h <= 0 || slot < 0 || (size_t)slot >= c->values.size()) return nullptr;
    Value& v = c->values[slot];
    if (!v.alive || (sg_handle)v.gen != (h >> 32)) return nullptr;
    return &v;
}
static sg_handle new_value(sg_ctx* c, const Value& v) {
    int idx;
    if (!c->free_values.empty()) {
        idx = c->free_values.back(); c->free_values.pop_back();
        const uint32_t gen = (c->values[idx].gen + 1) & 0x7fffffffu;
        c->values[idx] = v;
        c->values[idx].gen = gen;
    } else {
        c->values.push_back(v);
        idx = (int)c->values.size() - 1;
    }
    c->live.push_back(idx);
    return hnd(c, idx);
}

void* sg_dev_alloc(sg_ctx* c, size_t bytes) {
    if (bytes == 0) bytes = 16;
    if (c->plan_only) { uintptr_t p = c->fake_next; c->fake_next += (bytes + 511) / 512 * 512; return (void*)p; }
    if (c->has_alloc) return c->alloc.alloc(c->alloc.user, bytes);
    void* p = nullptr;
    if (cudaMallocAsync(&p, bytes, c->stream) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return p;
}
void sg_dev_free(sg_ctx* c, void* p) {
    if (!p || c->plan_only) return;
    if (c->has_alloc) c->alloc.free(c->alloc.user, p);
    else cudaFreeAsync(p, c->stream);
}
int64_t sg_slot_alloc(sg_ctx* c) {
    if (!c->slab_free.empty()) { int64_t s = c->slab_free.back(); c->slab_free.pop_back(); return s; }
    if (c->slab_next >= c->slab_slots) return -1;
    return c->slab_next++;
}

extern "C" {

const char* sg_version(void) { return "safegpu-b200 0.1 (sm_100a)"; }
int32_t sg_template_count(void) { return sgk_template_count(); }
const char* sg_template_name(int32_t k) { return sgk_template_name(k); }
const char* sg_last_error(sg_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

sg_status sg_ctx_create(sg_ctx** out, int device, void* cuda_stream, const sg_alloc* alloc_or_null) {
    CK(out);
    sg_ctx* c = new sg_ctx();
    c->device = device;
    c->plan_only = device < 0;
    c->stream = (cudaStream_t)cuda_stream;
    if (alloc_or_null) { c->alloc = *alloc_or_null; c->has_alloc = true; }
    c->slab_slots = 1 << 16;
    if (!c->plan_only) {
        // the product path has no CPU fallback: without a usable device every entry point fails loudly
        int prev = -1, sms = 0;
        cudaGetDevice(&prev);
        if (cudaSetDevice(device) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device) != cudaSuccess) {
            cudaGetLastError();
            if (prev >= 0) cudaSetDevice(prev);
            delete c;
            return SG_ERR_CUDA;
        }
        struct Restore { int d; ~Restore() { if (d >= 0) cudaSetDevice(d); } } restore{prev};   // the caller's current device is left as it was
        c->sm_count = sms;
        c->ctrl_words = 1 << 14;
        bool ok = cudaMalloc((void**)&c->ctrl, sizeof(unsigned int) * c->ctrl_words) == cudaSuccess &&
                  cudaMemset(c->ctrl, 0, sizeof(unsigned int) * c->ctrl_words) == cudaSuccess &&
                  cudaMalloc((void**)&c->slab, 8 * c->slab_slots) == cudaSuccess &&
                  cudaMemset(c->slab, 0, 8 * c->slab_slots) == cudaSuccess &&
                  cudaMallocHost((void**)&c->slab_host, 8 * c->slab_slots) == cudaSuccess &&
                  cudaEventCreateWithFlags(&c->ev_done, cudaEventDisableTiming) == cudaSuccess &&
                  cudaEventCreate(&c->ev_t0) == cudaSuccess && cudaEventCreate(&c->ev_t1) == cudaSuccess;
        if (!ok) { cudaGetLastError(); delete c; return SG_ERR_CUDA; }
        memset(c->slab_host, 0, 8 * c->slab_slots);
    } else {
        c->slab = (char*)(uintptr_t)0x1000;
    }
    *out = c;
    return SG_OK;
}

sg_status sg_ctx_destroy(sg_ctx* c) {
    SgDeviceScope dev_scope(c);
    CK(c);
    if (!c->plan_only) {
        cudaStreamSynchronize(c->stream);
        for (auto& v : c->values)
            if (v.alive && v.owned && v.ptr) sg_dev_free(c, v.ptr);
        for (char* p : c->deferred_free) sg_dev_free(c, p);
        cudaStreamSynchronize(c->stream);
        if (c->workspace) cudaFree(c->workspace);
        if (c->tile_state) cudaFree(c->tile_state);
        if (c->ctrl) cudaFree(c->ctrl);
        if (c->slab) cudaFree(c->slab);
        if (c->slab_host) cudaFreeHost(c->slab_host);
        if (c->ev_done) cudaEventDestroy(c->ev_done);
        for (auto* v : {&c->timing_events, &c->timing_pool})
            for (auto& pr : *v) { cudaEventDestroy(pr.first); cudaEventDestroy(pr.second); }
        if (c->ev_t0) cudaEventDestroy(c->ev_t0);
        if (c->ev_t1) cudaEventDestroy(c->ev_t1);
    }
    delete c;
    return SG_OK;
}

sg_status sg_ctx_set_flags(sg_ctx* c, uint32_t flags) { CK(c); c->flags = flags; return SG_OK; }

static sg_status make_collection(sg_ctx* c, int kind, sg_dtype dtype, int64_t rows, int64_t cols, int64_t ld, void* dev_ptr, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    if (dtype < SG_F32 || dtype > SG_BOOL || rows < 0 || cols < 0 || ld < cols) return sg_fail(c, SG_ERR_ARG, "bad dtype or shape");
    Value v;
    v.kind = kind; v.dtype = dtype; v.rows = rows; v.cols = cols; v.ld = ld; v.stride = 1;
    v.materialised = true; v.user_refs = 1;
    if (dev_ptr) v.ptr = (char*)dev_ptr;
    else {
        v.ptr = (char*)sg_dev_alloc(c, (size_t)rows * ld * dtype_size(dtype));
        if (!v.ptr) return sg_fail(c, SG_ERR_OOM, "device allocation failed");
        v.owned = true;
    }
    *out = new_value(c, v);
    return SG_OK;
}
sg_status sg_vec_create(sg_ctx* c, sg_dtype dtype, int64_t n, void* dev_ptr, sg_handle* out) {
    return make_collection(c, VK_VEC, dtype, 1, n, n, dev_ptr, out);
}
sg_status sg_mat_create(sg_ctx* c, sg_dtype dtype, int64_t rows, int64_t cols, int64_t ld, void* dev_ptr, sg_handle* out) {
    return make_collection(c, VK_MAT, dtype, rows, cols, ld, dev_ptr, out);
}

// A view needs storage: a pending collection is executed first (trigger (2)).
static sg_status need_storage(sg_ctx* c, sg_handle h, Value** out) {
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    if (!v->materialised || v->node >= 0) {
        sg_status s = sg_flush_impl(c);
        if (s != SG_OK) return s;
        v = val(c, h);
    }
    if (!v->materialised) return sg_fail(c, SG_ERR_ARG, "collection has no storage");
    *out = v;
    return SG_OK;
}

static sg_status resolve_count(sg_ctx* c, Value* v) {
    if (v->count_known) return SG_OK;
    if (c->plan_only) { v->count_known = true; return SG_OK; }
    if (cudaEventSynchronize(c->ev_done) != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, "event sync failed");
    int64_t n = 0;
    memcpy(&n, c->slab_host + 8 * v->count_slot, 8);
    if (n > v->cols) {                  // the caller's buffer was too small: kept items beyond it were dropped
        v->ld = v->cols; v->count_known = true;
        return sg_fail(c, SG_ERR_CAPACITY, "filter output exceeded the caller's capacity");
    }
    v->cols = n; v->ld = n; v->count_known = true;
    return SG_OK;
}

sg_status sg_vec_subset(sg_ctx* c, sg_handle h, int64_t start, int64_t finish, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s = need_storage(c, h, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_VEC) return sg_fail(c, SG_ERR_ARG, "subset needs a vector");
    if ((s = resolve_count(c, v)) != SG_OK) return s;
    if (start < 0 || finish < start || finish > v->cols) return sg_fail(c, SG_ERR_ARG, "subset range out of bounds");
    Value w = *v;
    w.ptr = v->ptr + start * v->stride * dtype_size(v->dtype);
    w.cols = finish - start; w.ld = w.cols; w.owned = false; w.user_refs = 1; w.node = -1; w.count_slot = -1;
    *out = new_value(c, w);
    return SG_OK;
}
sg_status sg_mat_row(sg_ctx* c, sg_handle m, int64_t i, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s = need_storage(c, m, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_MAT || i < 0 || i >= v->rows) return sg_fail(c, SG_ERR_ARG, "row index out of bounds");
    Value w = *v;
    w.kind = VK_VEC; w.ptr = v->ptr + i * v->ld * dtype_size(v->dtype); w.rows = 1; w.ld = w.cols; w.stride = 1;
    w.owned = false; w.user_refs = 1; w.node = -1;
    *out = new_value(c, w);
    return SG_OK;
}
sg_status sg_mat_rows(sg_ctx* c, sg_handle m, int64_t r0, int64_t r1, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s = need_storage(c, m, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_MAT || r0 < 0 || r1 < r0 || r1 > v->rows) return sg_fail(c, SG_ERR_ARG, "row range out of bounds");
    Value w = *v;
    w.ptr = v->ptr + r0 * v->ld * dtype_size(v->dtype); w.rows = r1 - r0;
    w.owned = false; w.user_refs = 1; w.node = -1;
    *out = new_value(c, w);
    return SG_OK;
}
sg_status sg_mat_elem(sg_ctx* c, sg_handle m, int64_t i, int64_t j, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s = need_storage(c, m, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_MAT || i < 0 || i >= v->rows || j < 0 || j >= v->cols) return sg_fail(c, SG_ERR_ARG, "element index out of bounds");
    Value w = *v;
    w.kind = VK_SCALAR; w.ptr = v->ptr + (i * v->ld + j) * dtype_size(v->dtype); w.rows = 1; w.cols = 1; w.ld = 1;
    w.owned = false; w.user_refs = 1; w.node = -1;
    *out = new_value(c, w);
    return SG_OK;
}

static uint64_t imm_bits(int dtype, const sg_operand& o) {
    // immediates are converted to the collection's dtype at enqueue (DESIGN.md R-imm)
    const bool is_f = o.kind == SG_OPERAND_IMM_F64;
    uint64_t bits = 0;
    switch (dtype) {
        case SG_F32: { float f = is_f ? (float)o.f : (float)o.i; memcpy(&bits, &f, 4); break; }
        case SG_F64: { double d = is_f ? o.f : (double)o.i; memcpy(&bits, &d, 8); break; }
        case SG_I32: { int32_t v = is_f ? (int32_t)o.f : (int32_t)o.i; memcpy(&bits, &v, 4); break; }
        default: { int64_t v = is_f ? (int64_t)o.f : o.i; memcpy(&bits, &v, 8); break; }
    }
    return bits;
}

// the pending value behind a handle must have a known length before it can be an operand
static sg_status operand_value(sg_ctx* c, sg_handle h, Value** out) {
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown operand handle");
    if (!v->count_known) {      // output of a pending filter: the domain changes — flush, then read the count
        sg_status s = sg_flush_impl(c);
        if (s != SG_OK) return s;
        v = val(c, h);
        if ((s = resolve_count(c, v)) != SG_OK) return s;
    }
    *out = v;
    return SG_OK;
}

static sg_status append_map(sg_ctx* c, uint8_t op, int n_opd, const Operand* opd, int opd_dtype, bool is2d, int64_t rows, int64_t cols,
                            sg_handle dst, sg_handle* out, int src_dtype = -1) {
    Node nd;
    nd.kind = NK_MAP; nd.op = op; nd.n_opd = n_opd; nd.src_dtype = src_dtype;
    for (int i = 0; i < n_opd; ++i) nd.opd[i] = opd[i];
    nd.dtype = opd_dtype; nd.is2d = is2d; nd.rows = rows; nd.cols = cols;
    const bool to_bool = (op >= OP_EQ && op <= OP_NOT);
    const int out_dtype = to_bool ? SG_BOOL : opd_dtype;
    if (dst) {
        Value* d = val(c, dst);
        if (!d || !d->materialised) return sg_fail(c, SG_ERR_ARG, "dst must be a collection with storage");
        if (d->dtype != out_dtype) return sg_fail(c, SG_ERR_DTYPE, "dst dtype differs from the result dtype");
        if (d->rows != rows || d->cols != cols || (d->kind == VK_MAT) != is2d) return sg_fail(c, SG_ERR_SHAPE, "dst shape differs from the result shape");
        if (d->stride != 1) return sg_fail(c, SG_ERR_UNSUPPORTED, "strided dst");
        // Aliases.  ANOTHER handle whose pending in-place result lives in storage this operation overwrites (the same view created twice,
        // an overlapping subset, the whole vector and a slice of it) keeps naming that storage: read after this point it must give
        // what the memory holds once the writes have landed in program order — not its own pending result, which this operation is
        // about to overwrite (in part).  Its pending result lives on as an anonymous version (still written to the buffer by its
        // producer, still read by the operations enqueued so far); the handle itself goes back to being plain memory, so later
        // readers are ordered behind both writers by the plan builder's RAW edges.
        {
            const auto span = [](const Value& v, const char** lo, const char** hi) {
                const int64_t es = dtype_size(v.dtype);
                *lo = v.ptr;
                *hi = v.kind == VK_MAT ? v.ptr + ((v.rows > 0 ? (v.rows - 1) * v.ld : 0) + v.cols) * es
                                       : v.ptr + ((v.cols > 0 ? (v.cols - 1) * v.stride : 0) + 1) * es;
            };
            const char *dlo, *dhi;
            span(*d, &dlo, &dhi);
            const size_t n_live = c->live.size();
            for (size_t li = 0; li < n_live; ++li) {
                const int ai = c->live[li];
                if (ai == hidx(dst)) continue;
                const Value& A = c->values[ai];
                if (!A.alive || A.kind == VK_SCALAR || !A.ptr || A.node < 0 || c->nodes[A.node].done) continue;
                if (!c->nodes[A.node].inplace || c->nodes[A.node].out != ai) continue;
                const char *alo, *ahi;
                span(A, &alo, &ahi);
                if (!(alo < dhi && dlo < ahi)) continue;
                Value prev = A;
                prev.user_refs = 0;
                prev.owned = false;
                const int prev_id = hidx(new_value(c, prev));       // may move the table: no reference into it is held here
                for (auto& n : c->nodes)
                    if (!n.done)
                        for (int i = 0; i < n.n_opd; ++i)
                            if (n.opd[i].kind != OPD_IMM && n.opd[i].value == ai) n.opd[i].value = prev_id;
                for (int i = 0; i < n_opd; ++i)                      // this operation reads it as it is now: the pending result
                    if (nd.opd[i].kind != OPD_IMM && nd.opd[i].value == ai) nd.opd[i].value = prev_id;
                c->nodes[c->values[ai].node].out = prev_id;
                c->values[ai].node = -1;
            }
            d = val(c, dst);
            // The handle's own pending in-place result is about to be superseded (its store is dropped, the value lives on in
            // registers).  That is only sound if nobody reads the buffer in between through ANOTHER handle: such a reader — enqueued
            // after the pending result, or this very operation — must find the pending result in memory.  Rare enough to take the
            // simple way: run what is pending first (eager execution is always right), then enqueue this operation.
            if (d->node >= 0 && !c->nodes[d->node].done && c->nodes[d->node].inplace) {
                const auto reads_alias = [&](const Node& n) {
                    for (int i = 0; i < n.n_opd; ++i) {
                        if (n.opd[i].kind == OPD_IMM) continue;
                        const Value& w = c->values[n.opd[i].value];
                        if (!w.ptr || (w.node >= 0 && !c->nodes[w.node].done)) continue;      // (an element view is a one-element range)
                        const char *wlo, *whi;
                        span(w, &wlo, &whi);
                        if (wlo < dhi && dlo < whi) return true;
                    }
                    return false;
                };
                bool alias_reader = reads_alias(nd);
                for (size_t k = (size_t)d->node + 1; k < c->nodes.size() && !alias_reader; ++k)
                    alias_reader = !c->nodes[k].done && reads_alias(c->nodes[k]);
                if (alias_reader) {
                    const sg_status fs = sg_flush_impl(c);
                    if (fs != SG_OK) return fs;
                    d = val(c, dst);
                    if (!d) return sg_fail(c, SG_ERR_ARG, "dst released");
                }
            }
        }
        // the handle keeps naming the same storage; its value is now the pending result (SSA over buffers)
        Value old = *d;
        old.user_refs = 0;                      // the previous contents stay reachable for already-enqueued readers
        old.owned = false;                      // the handle keeps owning the storage
        if (d->node >= 0 && !c->nodes[d->node].done) {
            // the previous contents are themselves a PENDING in-place result that this operation supersedes: that value never reaches
            // the buffer (a dead store) and lives on as an anonymous intermediate.  It must not keep the buffer's address: if a later
            // pass reads it, it is spilled to storage of its own — spilled into the buffer it would be overwritten by the new result
            old.ptr = nullptr;
            old.materialised = false;
        }
        const int old_id = hidx(new_value(c, old));
        d = val(c, dst);
        for (int i = 0; i < n_opd; ++i)         // this operation itself reads the previous contents
            if (nd.opd[i].kind != OPD_IMM && nd.opd[i].value == hidx(dst)) nd.opd[i].value = old_id;
        for (auto& n : c->nodes)                // earlier pending readers of this handle read the previous contents
            if (!n.done)
                for (int i = 0; i < n.n_opd; ++i)
                    if (n.opd[i].kind != OPD_IMM && n.opd[i].value == hidx(dst)) n.opd[i].value = old_id;
        for (auto& n : c->nodes)
            if (!n.done && n.out == hidx(dst)) {
                // an earlier pending in-place result is superseded: it becomes an anonymous intermediate version
                // (row.divided_by(p) then row.in_place_minus(q) -> one expression)
                n.out = old_id;
                n.inplace = false;
            }
        for (auto& k : c->contracts)
            if (k.value == hidx(dst)) k.value = old_id;
        d->node = (int)c->nodes.size();
        nd.out = hidx(dst); nd.inplace = true;
        c->nodes.push_back(nd);
        *out = dst;
        return SG_OK;
    }
    Value v;
    v.kind = is2d ? VK_MAT : VK_VEC; v.dtype = out_dtype; v.rows = rows; v.cols = cols; v.ld = cols; v.stride = 1;
    v.materialised = false; v.user_refs = 1; v.node = (int)c->nodes.size();
    nd.out = hidx(new_value(c, v));
    c->nodes.push_back(nd);
    *out = hnd(c, nd.out);
    return SG_OK;
}

// The dtype-changing projection: element i of the result is element i of v converted to `to`.
sg_status sg_cast(sg_ctx* c, sg_handle h, sg_dtype to, sg_handle dst, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s = operand_value(c, h, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_VEC) return sg_fail(c, SG_ERR_UNSUPPORTED, "sg_cast needs a vector");
    if (v->dtype == SG_BOOL || to < SG_F32 || to > SG_I64) return sg_fail(c, SG_ERR_DTYPE, "sg_cast converts between F32, F64, I32 and I64");
    Operand opd[2];
    opd[0].kind = OPD_VALUE; opd[0].value = hidx(h); opd[1] = opd[0];
    if ((int)to == v->dtype) return append_map(c, OP_MOV, 1, opd, v->dtype, false, 1, v->cols, dst, out);     // same type: a copy
    if (v->stride != 1) return sg_fail(c, SG_ERR_UNSUPPORTED, "sg_cast of a strided view");
    return append_map(c, NODE_OP_CAST, 1, opd, (int)to, false, 1, v->cols, dst, out, v->dtype);
}

sg_status sg_enqueue(sg_ctx* c, sg_op op, const sg_operand* ops, int32_t n, sg_handle dst, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && ops && out);
    // `c.project (agent (a: INT): DOUBLE do Result := sqrt (a) end)`: the square root of an INTEGER vector is
    // a DOUBLE collection — the conversion happens as the integers are loaded, in the same pass as the square root (R20)
    if (op == SG_SQRT && n == 1 && ops[0].kind == SG_OPERAND_HANDLE) {
        Value* iv = val(c, ops[0].h);
        if (iv && iv->kind == VK_VEC && (iv->dtype == SG_I32 || iv->dtype == SG_I64)) {
            sg_handle as_f64 = 0;
            sg_status s = sg_cast(c, ops[0].h, SG_F64, 0, &as_f64);
            if (s != SG_OK) return s;
            sg_operand o = ops[0];
            o.h = as_f64;
            s = sg_enqueue(c, SG_SQRT, &o, 1, dst, out);
            sg_release(c, as_f64);              // anonymous intermediate: never stored
            return s;
        }
    }
    if (op < SG_ADD || (op > SG_NOT && op != SG_SQRT)) return sg_fail(c, SG_ERR_ARG, "unknown op");
    const bool unary = (op == SG_NEG || op == SG_ABS || op == SG_NOT || op == SG_SQRT);
    if (n != (unary ? 1 : 2)) return sg_fail(c, SG_ERR_ARG, "wrong operand count");
    const bool logic = (op >= SG_AND && op <= SG_NOT);
    Value* vv[2] = {nullptr, nullptr};
    int dtype = -1;
    for (int i = 0; i < n; ++i) {
        if (ops[i].kind == SG_OPERAND_HANDLE) {
            sg_status s = operand_value(c, ops[i].h, &vv[i]);
            if (s != SG_OK) return s;
            if (dtype < 0) dtype = vv[i]->dtype;
            else if (dtype != vv[i]->dtype) return sg_fail(c, SG_ERR_DTYPE, "operand dtypes differ");
        } else if (ops[i].kind != SG_OPERAND_IMM_F64 && ops[i].kind != SG_OPERAND_IMM_I64) return sg_fail(c, SG_ERR_ARG, "bad operand kind");
    }
    if (dtype < 0) return sg_fail(c, SG_ERR_ARG, "at least one operand must be a collection");
    if (logic != (dtype == SG_BOOL)) return sg_fail(c, SG_ERR_DTYPE, logic ? "logical ops need BOOL operands" : "arithmetic on BOOL");
    if (op == SG_MOD && (dtype == SG_F32 || dtype == SG_F64)) return sg_fail(c, SG_ERR_DTYPE, "MOD needs an integer dtype");
    if (op == SG_SQRT && dtype != SG_F32 && dtype != SG_F64) return sg_fail(c, SG_ERR_DTYPE, "SQRT needs a float collection or an integer vector");
    // iteration domain: a matrix operand fixes a 2-D domain; vectors may broadcast along it
    bool is2d = false; int64_t rows = 1, cols = -1; bool have_coll = false;
    for (int i = 0; i < n; ++i)
        if (vv[i] && vv[i]->kind == VK_MAT) { is2d = true; rows = vv[i]->rows; cols = vv[i]->cols; }
    if (!is2d) {
        int64_t rb = -1, cb = -1;
        for (int i = 0; i < n; ++i) {
            if (!vv[i] || vv[i]->kind != VK_VEC) continue;
            if (ops[i].bcast == SG_BCAST_ROW) cb = vv[i]->cols;
            else if (ops[i].bcast == SG_BCAST_COL) rb = vv[i]->cols;
        }
        if (rb >= 0 && cb >= 0) { is2d = true; rows = rb; cols = cb; }      // outer combination of a COL and a ROW vector
        else if (rb >= 0 || cb >= 0) return sg_fail(c, SG_ERR_SHAPE, "a broadcast vector needs a matrix (or the other broadcast) operand");
    }
    Operand opd[2];
    for (int i = 0; i < n; ++i) {
        if (!vv[i]) { opd[i].kind = OPD_IMM; opd[i].imm = imm_bits(dtype, ops[i]); continue; }
        opd[i].kind = OPD_VALUE; opd[i].value = hidx(ops[i].h); opd[i].bcast = SG_BCAST_NONE;
        if (vv[i]->kind == VK_SCALAR) continue;
        have_coll = true;
        if (is2d) {
            if (vv[i]->kind == VK_MAT) {
                if (vv[i]->rows != rows || vv[i]->cols != cols) return sg_fail(c, SG_ERR_SHAPE, "matrix dimensions differ");
            } else {
                if (ops[i].bcast == SG_BCAST_ROW) { if (vv[i]->cols != cols) return sg_fail(c, SG_ERR_SHAPE, "ROW-broadcast vector length != columns"); }
                else if (ops[i].bcast == SG_BCAST_COL) { if (vv[i]->cols != rows) return sg_fail(c, SG_ERR_SHAPE, "COL-broadcast vector length != rows"); }
                else return sg_fail(c, SG_ERR_SHAPE, "vector operand of a matrix operation needs a broadcast kind");
                opd[i].bcast = ops[i].bcast;
            }
        } else {
            if (cols < 0) cols = vv[i]->cols;
            else if (cols != vv[i]->cols) return sg_fail(c, SG_ERR_SHAPE, "vector counts differ");
        }
    }
    if (!have_coll) {
        // only device scalars (and immediates): a one-element domain, e.g. avg = sum / count computed on the
        // device from the deferred sum without a host round trip
        bool have_scalar = false;
        for (int i = 0; i < n; ++i) have_scalar |= (vv[i] && vv[i]->kind == VK_SCALAR);
        if (!have_scalar || is2d) return sg_fail(c, SG_ERR_ARG, "at least one operand must be a vector, matrix or device scalar");
        cols = 1;
    }
    if (unary) { opd[1] = opd[0]; }
    return append_map(c, (uint8_t)op, unary ? 1 : 2, opd, dtype, is2d, rows, cols, dst, out);
}

sg_status sg_mat_transpose(sg_ctx* c, sg_handle m, void* dev_out, int64_t ld_out, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s;
    // trigger (2): the kernel below is not part of the pending list, so EVERYTHING pending runs first — a pending operation may
    // write m's memory (or read the output buffer) through another handle or view of the same storage
    if (!c->nodes.empty() && (s = sg_flush_impl(c)) != SG_OK) return s;
    if ((s = need_storage(c, m, &v)) != SG_OK) return s;
    if (v->kind != VK_MAT) return sg_fail(c, SG_ERR_ARG, "transpose needs a matrix");
    const int es = dtype_size(v->dtype);
    if (es != 4 && es != 8) return sg_fail(c, SG_ERR_DTYPE, "transpose of a BOOL matrix");
    const int64_t rows = v->rows, cols = v->cols, ld_in = v->ld;
    const char* src = v->ptr;
    if (ld_out == 0) ld_out = rows;
    if (ld_out < rows) return sg_fail(c, SG_ERR_ARG, "leading dimension of the transpose is smaller than its column count");
    if (dev_out) {
        const char* a0 = src; const char* a1 = src + (size_t)rows * ld_in * es;
        const char* b0 = (const char*)dev_out; const char* b1 = b0 + (size_t)cols * ld_out * es;
        if (a0 < b1 && b0 < a1) return sg_fail(c, SG_ERR_ALIAS, "transpose output overlaps its input");
    }
    sg_handle h;
    s = sg_mat_create(c, (sg_dtype)v->dtype, cols, rows, ld_out, dev_out, &h);      // may reallocate the handle table: v is stale now
    if (s != SG_OK) return s;
    if (!c->plan_only) {
        if (sgk_transpose(src, ld_in, rows, cols, val(c, h)->ptr, ld_out, es, c->stream) != cudaSuccess) {
            cudaGetLastError();
            sg_release(c, h);
            return sg_fail(c, SG_ERR_CUDA, "transpose launch failed");
        }
    }
    c->stats.launches_total++;
    *out = h;
    return SG_OK;
}

sg_status sg_mat_col(sg_ctx* c, sg_handle m, int64_t j, int64_t r0, int64_t r1, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v;
    sg_status s = need_storage(c, m, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_MAT || j < 0 || j >= v->cols || r0 < 0 || r1 < r0 || r1 > v->rows) return sg_fail(c, SG_ERR_ARG, "column range out of bounds");
    // a strided view of the column, then a deferred copy into new storage
    Value w = *v;
    w.kind = VK_VEC; w.ptr = v->ptr + (r0 * v->ld + j) * dtype_size(v->dtype); w.rows = 1; w.cols = r1 - r0; w.stride = v->ld; w.ld = w.cols;
    w.owned = false; w.user_refs = 0; w.node = -1;
    const int view = hidx(new_value(c, w));
    Operand opd[2];
    opd[0].kind = OPD_VALUE; opd[0].value = view; opd[1] = opd[0];
    return append_map(c, OP_MOV, 1, opd, w.dtype, false, 1, w.cols, 0, out);
}

static sg_status append_reduce(sg_ctx* c, uint8_t kind, sg_handle h, int axis, int result_dtype, sg_handle* out) {
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    // a reduction over the output of a PENDING filter joins the filter's pass as a masked reduction
    const bool on_pending_filter = !v->count_known && v->node >= 0 && axis == AXIS_ALL;
    if (!on_pending_filter) {
        sg_status s = operand_value(c, h, &v);
        if (s != SG_OK) return s;
    }
    if (v->kind == VK_SCALAR) return sg_fail(c, SG_ERR_ARG, "reduction of a scalar");
    const bool is2d = v->kind == VK_MAT;
    if (!is2d && axis != AXIS_ALL) return sg_fail(c, SG_ERR_ARG, "axis reductions need a matrix");
    if ((kind == OUT_MAX || kind == OUT_MIN) && (v->rows * v->cols == 0)) return sg_fail(c, SG_ERR_EMPTY, "max/min of an empty collection");
    Node nd;
    nd.kind = NK_REDUCE; nd.op = kind; nd.n_opd = 1; nd.axis = axis;
    nd.opd[0].kind = OPD_VALUE; nd.opd[0].value = hidx(h);
    nd.dtype = v->dtype; nd.is2d = is2d; nd.rows = v->rows; nd.cols = v->cols;
    Value r;
    r.dtype = result_dtype; r.materialised = false; r.user_refs = 1; r.node = (int)c->nodes.size();
    if (axis == AXIS_ALL) {
        r.kind = VK_SCALAR; r.rows = 1; r.cols = 1; r.ld = 1;
        r.slot = sg_slot_alloc(c);
        if (r.slot < 0) return sg_fail(c, SG_ERR_OOM, "out of scalar slots");
    } else {
        r.kind = VK_VEC; r.rows = 1; r.cols = (axis == AXIS_ROWS) ? v->rows : v->cols; r.ld = r.cols;
    }
    nd.out = hidx(new_value(c, r));
    c->nodes.push_back(nd);
    *out = hnd(c, nd.out);
    return SG_OK;
}

sg_status sg_reduce(sg_ctx* c, sg_handle h, sg_red kind, int32_t acc, sg_axis axis, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    if (axis < SG_AXIS_ALL || axis > SG_AXIS_COLS) return sg_fail(c, SG_ERR_ARG, "bad axis");
    const bool is_f = v->dtype == SG_F32 || v->dtype == SG_F64;
    // accumulator / result dtype: SG_ACC_DEFAULT or exactly the one the semantics fix (include/sg.h); a narrower accumulator
    // could not meet the sum tolerances stated against the long-double oracle (R1), so it is rejected, not emulated
    const int natural = (kind == SG_SUM) ? (is_f ? SG_F64 : SG_I64) : (kind == SG_COUNT) ? SG_I64 : v->dtype;
    if (acc != SG_ACC_DEFAULT && acc != natural) return sg_fail(c, SG_ERR_DTYPE, "unsupported accumulator dtype for this reduction");
    switch (kind) {
        case SG_SUM:
            if (v->dtype == SG_BOOL) return sg_fail(c, SG_ERR_DTYPE, "SUM of BOOL: use COUNT");
            return append_reduce(c, OUT_SUM, h, axis, is_f ? SG_F64 : SG_I64, out);
        case SG_RMAX: case SG_RMIN:
            if (v->dtype == SG_BOOL) return sg_fail(c, SG_ERR_DTYPE, "MAX/MIN of BOOL");
            return append_reduce(c, kind == SG_RMAX ? OUT_MAX : OUT_MIN, h, axis, v->dtype, out);
        case SG_COUNT:
            if (v->dtype != SG_BOOL) return sg_fail(c, SG_ERR_DTYPE, "COUNT needs a BOOL collection");
            return append_reduce(c, OUT_COUNT, h, axis, SG_I64, out);
        default: return sg_fail(c, SG_ERR_ARG, "unknown reduction");
    }
}
static sg_status quantifier(sg_ctx* c, uint8_t kind, sg_handle h, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    if (v->dtype != SG_BOOL) return sg_fail(c, SG_ERR_DTYPE, "for_all / exists need a BOOL collection");
    return append_reduce(c, kind, h, AXIS_ALL, SG_BOOL, out);
}
sg_status sg_forall(sg_ctx* c, sg_handle h, sg_handle* out) { return quantifier(c, OUT_ALL, h, out); }
sg_status sg_exists(sg_ctx* c, sg_handle h, sg_handle* out) { return quantifier(c, OUT_ANY, h, out); }

sg_status sg_forall_adjacent(sg_ctx* c, sg_handle h, sg_op cmp, sg_handle* out) {
    SgDeviceScope dev_scope(c);
    CK(c && out);
    if (cmp < SG_EQ || cmp > SG_GE) return sg_fail(c, SG_ERR_ARG, "adjacent predicate needs a comparison");
    Value* v;
    sg_status s = operand_value(c, h, &v);
    if (s != SG_OK) return s;
    if (v->kind != VK_VEC || v->dtype == SG_BOOL) return sg_fail(c, SG_ERR_ARG, "adjacent predicate needs a numeric vector");
    // b_i = v_i cmp v_{i+1}, i in [0, n-2]: the zip of subset(0,n-1) with subset(1,n)
    Operand opd[2];
    opd[0].kind = OPD_VALUE; opd[0].value = hidx(h);
    opd[1].kind = OPD_SHIFT; opd[1].value = hidx(h);
    sg_handle b;
    const int64_t m = v->cols > 0 ? v->cols - 1 : 0;
    s = append_map(c, (uint8_t)cmp, 2, opd, v->dtype, false, 1, m, 0, &b);
    if (s != SG_OK) return s;
    s = quantifier(c, OUT_ALL, b, out);
    val(c, b)->user_refs = 0;       // anonymous intermediate
    return s;
}

sg_status sg_filter(sg_ctx* c, sg_handle values, sg_handle mask, void* dev_out, int64_t capacity, sg_handle* out_vec, sg_handle* out_count) {
    SgDeviceScope dev_scope(c);
    CK(c && out_vec && out_count);
    Value *v, *m;
    sg_status s = operand_value(c, values, &v);
    if (s != SG_OK) return s;
    if ((s = operand_value(c, mask, &m)) != SG_OK) return s;
    if (v->kind != VK_VEC || m->kind != VK_VEC) return sg_fail(c, SG_ERR_ARG, "filter needs vectors");
    if (m->dtype != SG_BOOL || v->dtype == SG_BOOL) return sg_fail(c, SG_ERR_DTYPE, "filter needs numeric values and a BOOL mask");
    if (v->cols != m->cols) return sg_fail(c, SG_ERR_SHAPE, "values and mask counts differ");
    if (dev_out && capacity < 0) return sg_fail(c, SG_ERR_ARG, "negative capacity");
    Node nd;
    nd.kind = NK_FILTER; nd.n_opd = 2;
    nd.opd[0].kind = OPD_VALUE; nd.opd[0].value = hidx(values);
    nd.opd[1].kind = OPD_VALUE; nd.opd[1].value = hidx(mask);
    nd.dtype = v->dtype; nd.rows = 1; nd.cols = v->cols;
    Value cnt;
    cnt.kind = VK_SCALAR; cnt.dtype = SG_I64; cnt.rows = cnt.cols = cnt.ld = 1; cnt.user_refs = 1; cnt.node = (int)c->nodes.size();
    cnt.slot = sg_slot_alloc(c);
    if (cnt.slot < 0) return sg_fail(c, SG_ERR_OOM, "out of scalar slots");
    Value r;
    r.kind = VK_VEC; r.dtype = v->dtype; r.rows = 1; r.cols = dev_out ? capacity : v->cols; r.ld = r.cols;
    r.user_refs = 1; r.node = (int)c->nodes.size(); r.count_known = false; r.count_slot = cnt.slot;
    if (dev_out) r.ptr = (char*)dev_out;
    nd.inplace = dev_out != nullptr;
    nd.out = hidx(new_value(c, r));
    nd.out2 = hidx(new_value(c, cnt));
    c->nodes.push_back(nd);
    *out_vec = hnd(c, nd.out);
    *out_count = hnd(c, nd.out2);
    return SG_OK;
}

sg_status sg_contract(sg_ctx* c, sg_handle h, int32_t kind, const char* tag) {
    CK(c);
    Value* v = val(c, h);
    if (!v || v->kind != VK_SCALAR || v->dtype != SG_BOOL) return sg_fail(c, SG_ERR_ARG, "a contract is a BOOL scalar");
    if (kind != SG_CONTRACT_PRE && kind != SG_CONTRACT_POST) return sg_fail(c, SG_ERR_ARG, "bad contract kind");
    c->contracts.push_back({hidx(h), kind, tag ? tag : ""});
    return SG_OK;
}

sg_status sg_flush(sg_ctx* c) {
    CK(c);
    SgDeviceScope dev_scope(c);
    return sg_flush_impl(c);
}

// Listing 5's whole loop for steps [k0, k1): one persistent cooperative kernel (sg_ge.cu), no host in the loop.
sg_status sg_mat_ge_steps(sg_ctx* c, sg_handle m, sg_handle det, sg_handle minpiv, double eps, int64_t k0, int64_t k1) {
    CK(c);
    SgDeviceScope dev_scope(c);
    sg_status s;
    // like sg_mat_transpose, the kernel is not part of the pending list: everything pending runs first (trigger (2))
    if (!c->nodes.empty() && (s = sg_flush_impl(c)) != SG_OK) return s;
    Value* vm = val(c, m);
    Value* vd = val(c, det);
    Value* vp = val(c, minpiv);
    if (!vm || !vd || !vp) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    if (vm->kind != VK_MAT || !vm->materialised || !vd->materialised || !vp->materialised) return sg_fail(c, SG_ERR_ARG, "sg_mat_ge_steps: a matrix and two vectors with storage");
    if (vm->dtype != SG_F64 || vd->dtype != SG_F64 || vp->dtype != SG_F64) return sg_fail(c, SG_ERR_DTYPE, "sg_mat_ge_steps: F64 only");
    if (vm->rows != vm->cols) return sg_fail(c, SG_ERR_SHAPE, "sg_mat_ge_steps: square matrix expected");
    if (vd->rows * vd->cols != 1 || vp->rows * vp->cols != 1) return sg_fail(c, SG_ERR_SHAPE, "sg_mat_ge_steps: det and minpiv are one-element vectors");
    const int64_t n = vm->rows;
    if (k0 < 0 || k1 > n || k0 > k1) return sg_fail(c, SG_ERR_ARG, "sg_mat_ge_steps: step range");
    if (!(eps >= 0.0)) return sg_fail(c, SG_ERR_ARG, "sg_mat_ge_steps: eps must be >= 0");
    if (k0 == k1) return SG_OK;
    if (c->plan_only) { c->stats.launches_total++; return SG_OK; }
    unsigned int* ready = c->ctrl + 4;          // control words 4..7 are not used by the pass kernels
    if (cudaMemsetAsync(ready, 0, sizeof(unsigned int), c->stream) != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, cudaGetErrorString(cudaGetLastError()));
    int grid = 0;
    const cudaError_t e = sgk_ge_loop((double*)vm->ptr, n, vm->ld, (double*)vd->ptr, (double*)vp->ptr, eps, k0, k1, ready, c->sm_count, c->stream, &grid);
    if (e != cudaSuccess) { cudaGetLastError(); return sg_fail(c, SG_ERR_CUDA, std::string("determinant loop launch failed: ") + cudaGetErrorString(e)); }
    c->stats.launches_total++;
    return SG_OK;
}

// Listing 3 as a library composite: one segmented three-way partition launch per recursion level (sg_sort.cu).
sg_status sg_vec_quicksort(sg_ctx* c, sg_handle v, void* dev_out, sg_handle* out) {
    CK(c && out);
    SgDeviceScope dev_scope(c);
    sg_status s;
    if (!c->nodes.empty() && (s = sg_flush_impl(c)) != SG_OK) return s;     // not part of the pending list: everything pending runs first
    Value* a;
    if ((s = need_storage(c, v, &a)) != SG_OK) return s;
    if ((s = resolve_count(c, a)) != SG_OK) return s;
    if (a->kind != VK_VEC || a->stride != 1) return sg_fail(c, SG_ERR_ARG, "quicksort needs a unit-stride vector");
    if (a->dtype == SG_BOOL) return sg_fail(c, SG_ERR_DTYPE, "quicksort of a BOOL collection");
    const int64_t n = a->cols;
    if (n <= 0) return sg_fail(c, SG_ERR_EMPTY, "quicksort: require a.count > 0 (PAPER.md:248)");
    const int es = dtype_size(a->dtype);
    const char* src = a->ptr;
    const int dtype = a->dtype;
    if (dev_out) {
        const char* b0 = (const char*)dev_out;
        if (src < b0 + (size_t)n * es && b0 < src + (size_t)n * es) return sg_fail(c, SG_ERR_ALIAS, "quicksort output overlaps its input");
    }
    sg_handle h;
    if ((s = sg_vec_create(c, (sg_dtype)dtype, n, dev_out, &h)) != SG_OK) return s;     // may reallocate the handle table: `a` is stale now
    if (c->plan_only) { c->stats.launches_total += 2; *out = h; return SG_OK; }
    const size_t ws_bytes = sgk_quicksort_workspace_bytes(n, es);
    void* ws = sg_dev_alloc(c, ws_bytes);
    if (!ws) { sg_release(c, h); return sg_fail(c, SG_ERR_OOM, "quicksort workspace allocation failed"); }
    const int64_t slot = sg_slot_alloc(c);          // four pinned 8-byte slots' worth of read-back words
    int64_t slots[4] = {slot, -1, -1, -1};
    bool contiguous = slot >= 0;
    for (int i = 1; i < 4 && contiguous; ++i) { slots[i] = sg_slot_alloc(c); contiguous = slots[i] == slot + i; }
    unsigned int* host_flag = contiguous ? reinterpret_cast<unsigned int*>(c->slab_host + 8 * slot) : nullptr;
    unsigned int local_flag[8] = {0};
    int launches = 0;
    unsigned int error = 0;
    const cudaError_t e = sgk_quicksort(dtype, src, val(c, h)->ptr, n, ws, c->sm_count, host_flag ? host_flag : local_flag, c->stream, &launches, &error);
    for (int i = 0; i < 4; ++i)
        if (slots[i] >= 0) c->slab_free.push_back(slots[i]);
    c->deferred_free.push_back((char*)ws);
    c->stats.launches_total += launches;
    if (e != cudaSuccess) { cudaGetLastError(); sg_release(c, h); return sg_fail(c, SG_ERR_CUDA, std::string("quicksort failed: ") + cudaGetErrorString(e)); }
    if (error & 2u) { sg_release(c, h); return sg_fail(c, SG_ERR_CAPACITY, "quicksort: segment table overflow"); }
    if (error & 1u) {
        sg_release(c, h);
        return sg_fail(c, SG_ERR_CONTRACT, "postcondition violated: Result.count = a.count (a key is neither <, = nor > its pivot: NaN)");
    }
    *out = h;
    return SG_OK;
}

sg_status sg_scalar_dtype(sg_ctx* c, sg_handle h, int32_t* dtype) {
    CK(c && dtype);
    Value* v = val(c, h);
    if (!v || v->kind != VK_SCALAR) return sg_fail(c, SG_ERR_ARG, "not a scalar handle");
    *dtype = v->dtype;
    return SG_OK;
}

// does a pending in-place operation write storage that `v` names (through another handle: a view of it, the vector it is a view of)?
static bool pending_writer_overlaps(const sg_ctx* c, const Value& v) {
    if (!v.ptr) return false;              // (an element view, sg_mat_elem, is a one-element range)
    const auto span = [](const Value& x, const char** lo, const char** hi) {
        const int64_t es = dtype_size(x.dtype);
        *lo = x.ptr;
        *hi = x.kind == VK_MAT ? x.ptr + ((x.rows > 0 ? (x.rows - 1) * x.ld : 0) + x.cols) * es : x.ptr + ((x.cols > 0 ? (x.cols - 1) * x.stride : 0) + 1) * es;
    };
    const char *vlo, *vhi;
    span(v, &vlo, &vhi);
    for (const Node& n : c->nodes) {
        if (n.done || !n.inplace || n.out < 0) continue;
        const Value& w = c->values[n.out];
        if (!w.ptr || w.kind == VK_SCALAR) continue;
        const char *wlo, *whi;
        span(w, &wlo, &whi);
        if (wlo < vhi && vlo < whi) return true;
    }
    return false;
}

sg_status sg_scalar_get(sg_ctx* c, sg_handle h, void* host_out, size_t bytes) {
    SgDeviceScope dev_scope(c);
    CK(c && host_out);
    Value* v = val(c, h);
    if (!v || v->kind != VK_SCALAR) return sg_fail(c, SG_ERR_ARG, "not a scalar handle");
    // trigger (1), PAPER.md:284 — also for an element view (sg_mat_elem) whose matrix has a pending in-place result
    if (v->node >= 0 || (v->slot < 0 && pending_writer_overlaps(c, *v))) {
        sg_status s = sg_flush_impl(c);
        if (s != SG_OK && s != SG_ERR_CONTRACT) return s;
        v = val(c, h);
    }
    if (v->undecided) return sg_fail(c, SG_ERR_CONTRACT, "quantifier not evaluated: its pass ended early at a violated contract");
    const size_t sz = dtype_size(v->dtype);
    if (bytes < sz) return sg_fail(c, SG_ERR_ARG, "host buffer too small");
    if (c->plan_only) { memset(host_out, 0, sz); return SG_OK; }
    if (v->slot >= 0) {
        if (cudaEventSynchronize(c->ev_done) != cudaSuccess) return sg_fail(c, SG_ERR_CUDA, "event sync failed");
        memcpy(host_out, c->slab_host + 8 * v->slot, sz);
        return SG_OK;
    }
    if (!v->ptr) return sg_fail(c, SG_ERR_ARG, "scalar has no storage");
    if (cudaMemcpyAsync(host_out, v->ptr, sz, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess)
        return sg_fail(c, SG_ERR_CUDA, cudaGetErrorString(cudaGetLastError()));
    return SG_OK;
}

sg_status sg_vec_count(sg_ctx* c, sg_handle h, int64_t* n) {
    SgDeviceScope dev_scope(c);
    CK(c && n);
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    if (!v->count_known) {
        if (v->node >= 0) { sg_status s = sg_flush_impl(c); if (s != SG_OK && s != SG_ERR_CONTRACT) return s; v = val(c, h); }
        sg_status s = resolve_count(c, v);
        if (s != SG_OK) return s;
    }
    *n = v->rows * v->cols;     // count is a scalar contract: O(1)
    return SG_OK;
}

sg_status sg_vec_data(sg_ctx* c, sg_handle h, void** dev_ptr) {
    SgDeviceScope dev_scope(c);
    CK(c && dev_ptr);
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    // trigger (2): the collection's own pending result, or a pending in-place result in the same storage under another handle
    if (v->node >= 0 || !v->materialised || pending_writer_overlaps(c, *v)) { sg_status s = sg_flush_impl(c); if (s != SG_OK && s != SG_ERR_CONTRACT) return s; v = val(c, h); }
    if (!v->materialised) return sg_fail(c, SG_ERR_ARG, "collection has no storage");
    *dev_ptr = v->ptr;
    return SG_OK;
}

sg_status sg_vec_read(sg_ctx* c, sg_handle h, void* host_out, size_t bytes) {
    SgDeviceScope dev_scope(c);
    CK(c && host_out);
    void* p = nullptr;
    sg_status s = sg_vec_data(c, h, &p);
    if (s != SG_OK) return s;
    int64_t n = 0;
    if ((s = sg_vec_count(c, h, &n)) != SG_OK) return s;
    Value* v = val(c, h);
    if (v->stride != 1 || (v->kind == VK_MAT && v->ld != v->cols)) return sg_fail(c, SG_ERR_UNSUPPORTED, "to_array of a strided view");
    const size_t need = (size_t)n * dtype_size(v->dtype);
    if (bytes < need) return sg_fail(c, SG_ERR_ARG, "host buffer too small");
    if (c->plan_only || need == 0) return SG_OK;
    if (cudaMemcpyAsync(host_out, p, need, cudaMemcpyDeviceToHost, c->stream) != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess)
        return sg_fail(c, SG_ERR_CUDA, cudaGetErrorString(cudaGetLastError()));
    return SG_OK;
}

sg_status sg_release(sg_ctx* c, sg_handle h) {
    CK(c);
    Value* v = val(c, h);
    if (!v) return sg_fail(c, SG_ERR_ARG, "unknown handle");
    if (v->user_refs > 0) v->user_refs--;
    if (v->user_refs == 0 && v->node < 0) {      // nothing pending produces it
        // ... but a pending operation may still READ it (y = x + 1; release(x); flush): then only the reference goes now, the
        // flush that consumes the readers gives the storage and the scalar slot back (retire_nodes frees unreferenced values)
        for (auto& n : c->nodes)
            if (!n.done)
                for (int i = 0; i < n.n_opd; ++i)
                    if (n.opd[i].kind != OPD_IMM && n.opd[i].value == hidx(h)) return SG_OK;
        for (auto& k : c->contracts)
            if (k.value == hidx(h)) return SG_OK;
        if (v->owned && v->ptr) { c->deferred_free.push_back(v->ptr); v->ptr = nullptr; v->owned = false; }
        if (v->slot >= 0 && v->kind == VK_SCALAR) { c->slab_free.push_back(v->slot); v->slot = -1; }
        v->alive = false;
    }
    return SG_OK;
}

sg_status sg_plan_stats(sg_ctx* c, sg_stats* out) { CK(c && out); *out = c->stats; return SG_OK; }

int64_t sg_plan_dump(sg_ctx* c, int32_t pass, char* buf, int64_t cap) {
    if (!c || pass < 0 || (size_t)pass >= c->dumps.size()) return -1;
    const std::string s = sg_dump_prog(c->dumps[pass]);
    if (buf && cap > 0) { int64_t n = (int64_t)s.size() < cap - 1 ? (int64_t)s.size() : cap - 1; memcpy(buf, s.data(), n); buf[n] = 0; }
    return (int64_t)s.size() + 1;
}

}  // extern "C"
