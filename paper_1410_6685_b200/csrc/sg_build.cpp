// sg_build.cpp — lowers one pass (a group of merged pending operations) to its canonical SgProg + SgArgs.
// This is the paper's "kernel generation on the basis of the optimized DAG" without a compiler in
// the loop: the result is plain data that either matches a precompiled template instance or is interpreted.
// Merged elementwise bodies need no barrier (X[i]+Y[i] becomes a*X[i]+Y[i]; PAPER.md:322:
// (A[i]/pivot) - A[step]); scalars and immediates simply become extra kernel arguments.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <map>

#include "sg_ctx.h"

namespace {

// where the last block of a reduction pass writes an AXIS_ALL result besides its device slot: the slot's place in the pinned host
// mirror (SgArgs.out_host).  SAFEGPU_DIRECT_SCALARS=0 turns the write-through off (every scalar then goes back through the copy
// after the flush's last pass): the A/B switch of the measurement in DESIGN.md.
void* scalar_host_slot(const sg_ctx* c, int64_t slot) {
    static const bool direct = [] { const char* e = getenv("SAFEGPU_DIRECT_SCALARS"); return !(e && e[0] == '0'); }();
    return (!direct || c->plan_only || !c->slab_host || slot < 0) ? nullptr : (void*)(c->slab_host + 8 * slot);
}

struct Builder {
    sg_ctx* c;
    Pass& P;
    std::vector<PassInput> inputs;
    std::map<int, int> vreg_of, preg_of;        // value id -> register (computed in this pass or loaded)
    std::vector<char> vfree, pfree;              // register free lists (true = free)
    int n_vreg = 0, n_preg = 0;
    std::string err;

    Builder(sg_ctx* ctx, Pass& p) : c(ctx), P(p) {}

    int alloc_v() {
        for (size_t i = 0; i < vfree.size(); ++i) if (vfree[i]) { vfree[i] = 0; return (int)i; }
        vfree.push_back(0);
        return n_vreg++;
    }
    int alloc_p() {
        for (size_t i = 0; i < pfree.size(); ++i) if (pfree[i]) { pfree[i] = 0; return (int)i; }
        pfree.push_back(0);
        return n_preg++;
    }
    int add_input(uint8_t kind, const char* ptr, int64_t stride, uint64_t imm, int ref, bool boolvec, bool* fresh) {
        for (size_t k = 0; k < inputs.size(); ++k) {
            const PassInput& in = inputs[k];
            if (in.kind != kind) continue;
            if (kind == IN_IMM ? in.imm == imm : kind == IN_SHIFT ? in.value == ref : (in.ptr == ptr && in.stride == stride)) { *fresh = false; return (int)k; }
        }
        PassInput in{};
        in.kind = kind; in.ptr = ptr; in.stride = stride; in.imm = imm; in.value = ref; in.boolvec = boolvec;
        // An input lives in its register from the START of the program (every input of a tile is loaded before the first instruction
        // runs), so it must never take a register that an earlier temporary has used and given back: `(a+b)*(c+d) + e` would load e
        // into the register c+d is then computed in.  Inputs always get a register of their own.
        if (boolvec) { pfree.push_back(0); in.reg = n_preg++; }
        else { vfree.push_back(0); in.reg = n_vreg++; }
        inputs.push_back(in);
        *fresh = true;
        return (int)inputs.size() - 1;
    }
};

const char* op_name(uint8_t op) {
    static const char* n[] = {"OP_ADD", "OP_SUB", "OP_MUL", "OP_DIV", "OP_MIN", "OP_MAX", "OP_MOD", "OP_NEG", "OP_ABS", "OP_EQ", "OP_NE",
                              "OP_LT", "OP_LE", "OP_GT", "OP_GE", "OP_AND", "OP_OR", "OP_NOT", "OP_MOV", "OP_SQRT"};
    return op < OP_COUNT_ ? n[op] : "?";
}
const char* in_name(uint8_t k) {
    static const char* n[] = {"IN_VEC", "IN_SHIFT", "IN_STRIDED", "IN_SCALAR", "IN_IMM", "IN_ROWB", "IN_COLB", "IN_BOOLVEC", "IN_VEC_CVT"};
    return k < 9 ? n[k] : "?";
}
const char* out_name(uint8_t k) {
    static const char* n[] = {"OUT_STORE", "OUT_STORE_BOOL", "OUT_SUM", "OUT_MAX", "OUT_MIN", "OUT_ALL", "OUT_ANY", "OUT_COUNT", "OUT_FILTER"};
    return k < 9 ? n[k] : "?";
}
const char* dt_name(uint8_t d) {
    static const char* n[] = {"DT_F32", "DT_F64", "DT_I32", "DT_I64"};
    return d < 4 ? n[d] : "?";
}

// Signed magic number for truncating int32 division by d, |d| >= 2 (multiply-high scheme; the device side is
// magic_div_i32 in sg_device.cuh).  valid == 0 for |d| <= 1.
SgDiv i32_magic(int32_t d) {
    SgDiv m{};
    const uint32_t two31 = 0x80000000u;
    const uint32_t ad = d < 0 ? 0u - (uint32_t)d : (uint32_t)d;
    if (ad <= 1) return m;
    const uint32_t t = two31 + ((uint32_t)d >> 31);
    const uint32_t anc = t - 1 - t % ad;
    int p = 31;
    uint32_t q1 = two31 / anc, r1 = two31 - q1 * anc, q2 = two31 / ad, r2 = two31 - q2 * ad, delta;
    do {
        ++p;
        q1 *= 2; r1 *= 2;
        if (r1 >= anc) { ++q1; r1 -= anc; }
        q2 *= 2; r2 *= 2;
        if (r2 >= ad) { ++q2; r2 -= ad; }
        delta = ad - r2;
    } while (q1 < delta || (q1 == delta && r1 == 0));
    uint32_t M = q2 + 1;
    if (d < 0) M = 0u - M;
    m.M = (int32_t)M;
    m.addsel = (d > 0 && (int32_t)M < 0) ? 1 : (d < 0 && (int32_t)M > 0) ? -1 : 0;
    m.s = p - 32;
    m.neg_d = (int32_t)(0u - (uint32_t)d);
    m.valid = 1;
    return m;
}

std::string dump_prog(const SgProg& g) {
    char b[256];
    std::string s = "{";
    snprintf(b, sizeof(b), "{%s, %d, %d, %d, %d, %d, %d, 0},\n  {", dt_name(g.shape.dtype), g.shape.flags, g.shape.n_in, g.shape.n_instr, g.shape.n_out,
             g.shape.n_vreg, g.shape.n_preg);
    s += b;
    for (int k = 0; k < g.shape.n_in; ++k) {
        snprintf(b, sizeof(b), "%s{%s,%d,%d,%d}", k ? "," : "", in_name(g.in[k].kind), g.in[k].ref, g.in[k].reg, g.in[k].pad);
        s += b;
    }
    s += "},\n  {";
    for (int k = 0; k < g.shape.n_instr; ++k) {
        snprintf(b, sizeof(b), "%s{%s,%d,%d,%d}", k ? "," : "", op_name(g.code[k].op), g.code[k].dst, g.code[k].a, g.code[k].b);
        s += b;
    }
    s += "},\n  {";
    for (int k = 0; k < g.shape.n_out; ++k) {
        snprintf(b, sizeof(b), "%s{%s,%d,%d,%d}", k ? "," : "", out_name(g.out[k].kind), g.out[k].src, g.out[k].pred, g.out[k].axis);
        s += b;
    }
    s += "}}";
    return s;
}

}  // namespace

std::string sg_dump_prog(const SgProg& g) { return dump_prog(g); }

sg_status sg_build_pass(sg_ctx* c, Pass& P, std::vector<char*>& temps, std::string& dump) {
    std::vector<Node>& N = c->nodes;
    std::vector<Value>& V = c->values;
    const bool unfused = c->flags & SG_FLAG_UNFUSED;
    Builder B(c, P);
    SgProg& g = P.prog;
    SgArgs& a = P.args;
    memset(&g, 0, sizeof(g));
    memset(&a, 0, sizeof(a));
    const int dtype = P.dtype >= 0 ? P.dtype : SG_I32;      // a pass of pure BOOL logic has an unused V file
    const int64_t es = dtype_size(dtype);
    g.shape.dtype = (uint8_t)dtype;
    g.shape.flags = (P.is2d ? PF_2D : 0) | (P.has_filter ? PF_FILTER : 0);
    a.n = P.is2d ? P.rows : P.cols;
    a.cols = P.is2d ? P.cols : 0;

    auto stored = [&](const Node& n) { return n.kind == NK_MAP && (unfused || n.inplace || V[n.out].user_refs != 0); };

    // liveness inside the pass: last use of every value; values feeding an output stay to the end
    std::map<int, int> last_use;
    std::map<int, char> pinned;
    for (size_t i = 0; i < P.nodes.size(); ++i) {
        const Node& X = N[P.nodes[i]];
        for (int j = 0; j < X.n_opd; ++j)
            if (X.opd[j].kind != OPD_IMM) {
                last_use[X.opd[j].value] = (int)i;
                if (X.kind != NK_MAP) pinned[X.opd[j].value] = 1;
            }
        if (stored(X)) pinned[X.out] = 1;
    }
    std::map<int, std::pair<int, int>> filter_regs;     // filter output value -> (values reg, mask reg)
    std::map<int, int64_t> filter_len;                  // filter output value -> length of the filter's SOURCE (the domain of reductions over the kept values)
    int n_out = 0, n_instr = 0;
    bool only_quant = true;

    // operand -> register (loading it as an input if it is not computed in this pass)
    auto resolve = [&](const Node& X, const Operand& o, bool want_pred, int* reg) -> sg_status {
        bool fresh = false;
        if (o.kind == OPD_IMM) {
            const int k = B.add_input(IN_IMM, nullptr, 0, o.imm, -1, false, &fresh);
            if (fresh) P.n_scalar_in++;
            *reg = B.inputs[k].reg;
            return SG_OK;
        }
        const Value& v = V[o.value];
        const bool in_pass = v.node >= 0 && !N[v.node].done && N[v.node].needed && N[v.node].pass == X.pass && N[v.node].kind == NK_MAP;
        const bool via_memory = unfused || (X.post && in_pass && stored(N[v.node])) || o.kind == OPD_SHIFT;
        if (in_pass && !via_memory) {
            auto& m = want_pred ? B.preg_of : B.vreg_of;
            auto it = m.find(o.value);
            if (it == m.end()) return sg_fail(c, SG_ERR_ARG, "internal: operand register missing");
            *reg = it->second;
            return SG_OK;
        }
        if (in_pass && via_memory) return sg_fail(c, SG_ERR_ARG, "internal: memory operand produced in the same pass");
        const char* ptr = v.ptr;
        if (v.kind == VK_SCALAR && v.slot >= 0) ptr = c->slab + 8 * v.slot;
        if (!ptr) return sg_fail(c, SG_ERR_ARG, "operand has no storage");
        auto& m = want_pred ? B.preg_of : B.vreg_of;
        // register cache key: the value, its shifted form, or its converted form (a conversion never shares a register with the raw value:
        // they live in passes of different dtypes anyway)
        const int key = o.kind == OPD_SHIFT ? -2 - o.value : o.value;
        auto it = m.find(key);
        if (it != m.end()) { *reg = it->second; return SG_OK; }
        int k;
        if (v.kind == VK_SCALAR) {
            if (want_pred) return sg_fail(c, SG_ERR_UNSUPPORTED, "BOOL scalar operand");
            k = B.add_input(IN_SCALAR, ptr, 0, 0, -1, false, &fresh);
        } else if (X.kind == NK_MAP && X.op == NODE_OP_CAST) {
            // dtype-changing projection: the operand is converted to the pass dtype as it is loaded
            if (P.is2d || v.kind != VK_VEC || v.stride != 1) return sg_fail(c, SG_ERR_UNSUPPORTED, "dtype conversion of a matrix or strided view");
            k = B.add_input(IN_VEC_CVT, ptr, 1, 0, -1, false, &fresh);
            if (fresh) { P.n_mem_in++; P.bytes += v.cols * dtype_size(v.dtype); B.inputs[k].src_dtype = (uint8_t)v.dtype; }
            fresh = false;
        } else if (o.kind == OPD_SHIFT) {
            int base = B.add_input(IN_VEC, ptr, v.stride, 0, -1, false, &fresh);
            if (fresh) { P.n_mem_in++; P.bytes += v.cols * es; }
            if (v.stride != 1) return sg_fail(c, SG_ERR_UNSUPPORTED, "neighbour predicate on a strided view");
            k = B.add_input(IN_SHIFT, nullptr, 0, 0, base, false, &fresh);
            fresh = false;
        } else if (want_pred) {
            if (v.stride != 1 || (P.is2d && v.kind != VK_MAT)) return sg_fail(c, SG_ERR_UNSUPPORTED, "strided or broadcast BOOL operand read from memory");
            // a BOOL matrix (a mask somebody kept) is read back by the 2-D bytecode evaluator: in_stride = its leading dimension
            k = B.add_input(IN_BOOLVEC, ptr, P.is2d ? v.ld : 1, 0, -1, true, &fresh);
            if (fresh) { P.n_mem_in++; P.bytes += v.rows * v.cols; }
            fresh = false;
        } else if (P.is2d && v.kind == VK_VEC) {
            if (v.stride != 1) return sg_fail(c, SG_ERR_UNSUPPORTED, "strided broadcast vector");
            k = B.add_input(o.bcast == SG_BCAST_ROW ? IN_ROWB : IN_COLB, ptr, 1, 0, -1, false, &fresh);
            if (fresh) { P.n_mem_in++; P.bytes += v.cols * es; }
            fresh = false;
        } else if (P.is2d) {
            k = B.add_input(IN_VEC, ptr, v.ld, 0, -1, false, &fresh);
            if (fresh) { P.n_mem_in++; P.bytes += v.rows * v.cols * es; }
            fresh = false;
        } else {
            k = B.add_input(v.stride == 1 ? IN_VEC : IN_STRIDED, ptr, v.stride, 0, -1, false, &fresh);
            if (fresh) { P.n_mem_in++; P.bytes += v.cols * es; }
            fresh = false;
        }
        if (fresh && v.kind == VK_SCALAR) P.n_scalar_in++;
        B.inputs[k].len = std::max<int64_t>(B.inputs[k].len, v.kind == VK_MAT ? v.rows * v.cols : v.cols);
        if (o.kind == OPD_SHIFT) { B.inputs[B.inputs[k].value].len = v.cols; a.n = std::max<int64_t>(a.n, v.cols); }
        m[key] = B.inputs[k].reg;
        *reg = B.inputs[k].reg;
        return SG_OK;
    };

    for (size_t i = 0; i < P.nodes.size(); ++i) {
        Node& X = N[P.nodes[i]];
        const bool opd_pred = (X.dtype == SG_BOOL);
        int r[2] = {0, 0};
        if (X.kind == NK_REDUCE && V[X.opd[0].value].node >= 0 && !N[V[X.opd[0].value].node].done && N[V[X.opd[0].value].node].kind == NK_FILTER) {
            // reduction over the kept values of this pass's filter: a masked reduction of the filter's source
            auto it = filter_regs.find(X.opd[0].value);
            if (it == filter_regs.end()) return sg_fail(c, SG_ERR_ARG, "internal: filter registers missing");
            if (n_out >= SG_MAX_OUT) return sg_fail(c, SG_ERR_CAPACITY, "too many outputs in one pass");
            g.out[n_out] = {X.op, (uint8_t)it->second.first, (uint8_t)it->second.second, AXIS_ALL};
            a.out_ptr[n_out] = c->slab + 8 * V[X.out].slot;
            a.out_host[n_out] = scalar_host_slot(c, V[X.out].slot);
            a.out_len[n_out] = filter_len[X.opd[0].value];      // masked reduction over the SOURCE elements (X.cols is the output's capacity: a tight caller buffer would cut the sum short)
            only_quant = false;
            ++n_out;
            continue;
        }
        for (int j = 0; j < X.n_opd; ++j) {
            const bool want_pred = (X.kind == NK_FILTER) ? (j == 1) : opd_pred;
            sg_status s = resolve(X, X.opd[j], want_pred, &r[j]);
            if (s != SG_OK) return s;
        }
        // operands whose last use is this node give their registers back (inputs are never recycled)
        for (int j = 0; j < X.n_opd; ++j) {
            if (X.opd[j].kind != OPD_VALUE) continue;
            const int vid = X.opd[j].value;
            if (last_use[vid] != (int)i || pinned.count(vid)) continue;
            const bool is_pred = (X.kind == NK_FILTER) ? (j == 1) : opd_pred;
            auto& m = is_pred ? B.preg_of : B.vreg_of;
            auto it = m.find(vid);
            if (it == m.end()) continue;
            bool is_input = false;
            for (const PassInput& in : B.inputs) is_input |= (in.boolvec == is_pred && in.reg == it->second);
            if (!is_input) (is_pred ? B.pfree : B.vfree)[it->second] = 1;
        }
        if (X.kind == NK_MAP) {
            if (n_instr >= SG_MAX_INSTR) return sg_fail(c, SG_ERR_CAPACITY, "too many operations in one pass");
            const bool to_pred = X.op >= OP_EQ && X.op <= OP_NOT;
            const int d = to_pred ? B.alloc_p() : B.alloc_v();
            (to_pred ? B.preg_of : B.vreg_of)[X.out] = d;
            const uint8_t opc = X.op == NODE_OP_CAST ? (uint8_t)OP_MOV : X.op;
            g.code[n_instr++] = {opc, (uint8_t)d, (uint8_t)r[0], (uint8_t)(X.n_opd > 1 ? r[1] : r[0])};
            if (stored(X)) {
                if (n_out >= SG_MAX_OUT) return sg_fail(c, SG_ERR_CAPACITY, "too many outputs in one pass");
                Value& ov = V[X.out];
                const int64_t oes = dtype_size(ov.dtype);
                if (!ov.ptr) {
                    ov.ptr = (char*)sg_dev_alloc(c, (size_t)(ov.rows * ov.cols * oes));
                    if (!ov.ptr) return sg_fail(c, SG_ERR_OOM, "device allocation failed");
                    ov.owned = true; ov.fresh_alloc = true; ov.ld = ov.cols; ov.stride = 1;
                }
                ov.materialised = true;
                g.out[n_out] = {(uint8_t)(to_pred ? OUT_STORE_BOOL : OUT_STORE), (uint8_t)d, SG_NO_PRED, AXIS_ALL};
                a.out_ptr[n_out] = ov.ptr;
                a.out_len[n_out] = P.is2d ? ov.ld : X.cols;
                P.bytes += ov.rows * ov.cols * oes;
                only_quant = false;
                ++n_out;
            }
        } else if (X.kind == NK_REDUCE) {
            if (n_out >= SG_MAX_OUT) return sg_fail(c, SG_ERR_CAPACITY, "too many outputs in one pass");
            Value& ov = V[X.out];
            g.out[n_out] = {X.op, (uint8_t)r[0], SG_NO_PRED, (uint8_t)X.axis};
            if (X.axis == AXIS_ALL) {
                a.out_ptr[n_out] = c->slab + 8 * ov.slot;
                a.out_host[n_out] = scalar_host_slot(c, ov.slot);
            } else {
                const int64_t oes = dtype_size(ov.dtype);
                if (!ov.ptr) {
                    ov.ptr = (char*)sg_dev_alloc(c, (size_t)(ov.cols * oes));
                    if (!ov.ptr) return sg_fail(c, SG_ERR_OOM, "device allocation failed");
                    ov.owned = true; ov.fresh_alloc = true;
                }
                ov.materialised = true;
                a.out_ptr[n_out] = ov.ptr;
                P.bytes += ov.cols * oes;
            }
            a.out_len[n_out] = X.cols;
            if (X.op != OUT_ALL && X.op != OUT_ANY) only_quant = false;
            if (X.op == OUT_ALL)
                for (const Contract& k : c->contracts)
                    if (k.value == X.out) a.exit_any |= 1u << n_out;
            ++n_out;
        } else {    // NK_FILTER
            if (n_out >= SG_MAX_OUT) return sg_fail(c, SG_ERR_CAPACITY, "too many outputs in one pass");
            Value& ov = V[X.out];
            if (!ov.ptr) {
                ov.ptr = (char*)sg_dev_alloc(c, (size_t)(ov.cols * es));
                if (!ov.ptr) return sg_fail(c, SG_ERR_OOM, "device allocation failed");
                ov.owned = true; ov.fresh_alloc = true;
            }
            ov.materialised = true;
            filter_regs[X.out] = {r[0], r[1]};
            filter_len[X.out] = X.cols;
            g.out[n_out] = {OUT_FILTER, (uint8_t)r[0], (uint8_t)r[1], AXIS_ALL};
            a.out_ptr[n_out] = ov.ptr;
            a.out_len[n_out] = X.cols;
            a.out_cap[n_out] = ov.cols;
            a.out_aux[n_out] = c->slab + 8 * V[X.out2].slot;
            only_quant = false;
            ++n_out;
        }
    }
    (void)temps;
    if (B.inputs.size() > SG_MAX_IN) return sg_fail(c, SG_ERR_CAPACITY, "too many distinct inputs in one pass");
    if (B.n_vreg > SG_MAX_VREG || B.n_preg > SG_MAX_PREG) return sg_fail(c, SG_ERR_CAPACITY, "fused chain needs too many registers");
    for (size_t k = 0; k < B.inputs.size(); ++k) {
        const PassInput& in = B.inputs[k];
        g.in[k].kind = in.kind;
        g.in[k].ref = in.kind == IN_SHIFT ? (uint8_t)in.value : in.kind == IN_VEC_CVT ? in.src_dtype : 0;
        g.in[k].reg = (uint8_t)in.reg;
        a.in_ptr[k] = in.ptr;
        a.in_stride[k] = in.stride;
        a.in_len[k] = in.len;
        a.imm[k] = in.imm;
        if (in.kind == IN_IMM && dtype == SG_I32) {
            int32_t d; memcpy(&d, &in.imm, 4);
            a.imm_div[k] = i32_magic(d);
        }
        // an input whose storage this pass also writes must not go through the read-only path
        if (in.ptr)
            for (int o = 0; o < n_out; ++o)
                if ((g.out[o].kind == OUT_STORE || g.out[o].kind == OUT_STORE_BOOL) && a.out_ptr[o] == (void*)in.ptr) g.in[k].pad = 1;
    }
    g.shape.n_in = (uint8_t)B.inputs.size();
    g.shape.n_instr = (uint8_t)n_instr;
    g.shape.n_out = (uint8_t)n_out;
    g.shape.n_vreg = (uint8_t)B.n_vreg;
    g.shape.n_preg = (uint8_t)B.n_preg;
    if (only_quant && n_out > 0 && !P.is2d) g.shape.flags |= PF_EARLY_EXIT;
    (void)dump;      // the text form is produced on demand (sg_dump_prog): it costs more than the plan itself
    return SG_OK;
}
