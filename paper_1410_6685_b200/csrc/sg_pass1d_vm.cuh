// sg_pass1d_vm.cuh — pass1d_bytecode: the register-resident op-bytecode evaluator for chains that have no
// precompiled template instance.  The SgProg bytes are interpreted per tile; control flow is warp-uniform (every
// thread runs the same program), each decoded instruction is applied to a register-resident vector of E elements,
// and the value register file is addressed by uniform switches so that it never spills to local memory.
#ifndef SG_PASS1D_VM_CUH_
#define SG_PASS1D_VM_CUH_

#include "sg_pass1d.cuh"

namespace sgk {

constexpr int VM_VREG = 16;     // value registers of the bytecode evaluator (plan builder reuses dead registers)
// elements per thread per tile: one 128-bit access per operand
template <class T> struct VmE { static constexpr int value = 16 / (int)sizeof(T); };

// Configurations of the 1-D bytecode kernel: (threads per block, cells per value register and thread).  One decoded micro-op is
// applied to C cells = C * 16 bytes per thread, so the dispatch (a compare-and-branch tree: nvcc emits no indexed branch for the
// opcode switch) is paid once per C * E elements; the register file costs (R * C + I) cells of VB * 16 bytes of shared memory, where R
// = registers the chain computes or loads per element and I = registers that hold ONE value for the whole pass (immediates, device
// scalars: a single broadcast cell each).  The widest configuration whose file still lets three blocks share an SM is chosen.
struct VmConfig { int threads, cells; };
// Eight cells were measured and rejected: 128 registers with 558 local-memory instructions and 70 k SASS instructions (the unrolled case
// bodies overflow the instruction cache): 369 us on config 1's chain against 347 us for two cells.
__host__ __device__ constexpr VmConfig vm_config(int cfg) { return cfg == 2 ? VmConfig{128, 4} : cfg == 1 ? VmConfig{256, 2} : VmConfig{256, 1}; }
constexpr int VM_NCFG = 3;
constexpr size_t VM_MAX_FILE_BYTES = (size_t)SG_MAX_VREG * 256u * 16u;     // the narrowest configuration with every register in use (96 KiB)
__host__ __device__ constexpr size_t vm_file_bytes_cfg(int r, int i, int cfg) {
    return (size_t)((r > 0 ? r : 1) * vm_config(cfg).cells + i) * (size_t)vm_config(cfg).threads * 16u;
}
// R and I of a program (see above)
__host__ __device__ inline void vm_count_regs(const SgProg& g, int* r, int* i) {
    bool single[SG_MAX_VREG] = {};
    for (int k = 0; k < g.shape.n_in; ++k)
        if ((g.in[k].kind == IN_SCALAR || g.in[k].kind == IN_IMM) && g.in[k].reg < SG_MAX_VREG) single[g.in[k].reg] = true;
    int ni = 0;
    for (int k = 0; k < g.shape.n_vreg && k < SG_MAX_VREG; ++k) ni += single[k];
    *i = ni; *r = g.shape.n_vreg - ni;
}
__host__ __device__ inline int vm_pick_config(const SgProg& g) {
    int r, i;
    vm_count_regs(g, &r, &i);
#ifndef SG_VM_MAXCFG
#define SG_VM_MAXCFG (VM_NCFG - 1)
#endif
    for (int cfg = SG_VM_MAXCFG; cfg > 0; --cfg)
        if (vm_file_bytes_cfg(r, i, cfg) <= 72u * 1024u) return cfg;
    return 0;
}
__host__ __device__ inline int vm_tile_cfg(int elem_size, int cfg) { return vm_config(cfg).threads * (16 / elem_size) * vm_config(cfg).cells; }

// The value register file lives in SHARED memory: register k of thread t is the 16-byte cell at
//     base + k * VM_REG_STRIDE + t * 16
// (consecutive threads -> consecutive cells: conflict-free 128-bit accesses).  A register number is then just an
// address offset — no per-register switch, about forty hardware registers per thread instead of 160+, so three
// blocks run per SM where one did.  VM_FILE_BYTES of dynamic shared memory per block.
constexpr uint32_t VM_CELL_STRIDE = BLOCK * 16;      // bytes between the cells of one register (one cell per thread)
constexpr size_t VM_FILE_BYTES = (size_t)VM_VREG * VM_CELL_STRIDE;       // single-cell file of the filter evaluator

template <class T, int E> struct VmRegs {
    static_assert(E * sizeof(T) == 16, "one 128-bit cell per register");
    uint32_t base;      // shared-window address of this thread's cell of register 0
    uint32_t stride;    // bytes between registers = cells * VM_CELL_STRIDE
    VmRegs() = default;
    __device__ __forceinline__ explicit VmRegs(uint32_t file_base, int cell = 0, int cells = 1)
        : base(file_base + (uint32_t)cell * VM_CELL_STRIDE + (threadIdx.x & (BLOCK - 1)) * 16u), stride((uint32_t)cells * VM_CELL_STRIDE) {}
    __device__ __forceinline__ void get(uint8_t k, T (&o)[E]) const {
        uint32_t w[4];
        asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(base + k * stride) : "memory");
        memcpy(o, w, 16);
    }
    __device__ __forceinline__ void put(uint8_t k, const T (&o)[E]) {
        uint32_t w[4];
        memcpy(w, o, 16);
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(base + k * stride), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
    }
};

// predicate file: SG_MAX_PREG registers x E bits packed in one 32-bit word (E <= 4)
template <int E> __device__ __forceinline__ unsigned int pget(unsigned int pf, uint8_t k) { return (pf >> (k * E)) & ((1u << E) - 1u); }
template <int E> __device__ __forceinline__ unsigned int pput(unsigned int pf, uint8_t k, unsigned int bits) {
    const unsigned int m = ((1u << E) - 1u) << (k * E);
    return (pf & ~m) | ((bits << (k * E)) & m);
}

// One decode per instruction, applied to C independent cells (2 x the elements per decode, 2 x the ILP).  The result of the
// previous value instruction stays in hardware registers: an operand that names it is not re-read from shared memory.
template <class T, int E, int C>
__device__ __forceinline__ void vm_exec(const SgProg& g, VmRegs<T, E> (&rf)[C], unsigned int (&pf)[C]) {
    T last[C][E];
    int last_dst = -1;
#pragma unroll
    for (int c = 0; c < C; ++c)
#pragma unroll
        for (int e = 0; e < E; ++e) last[c][e] = T(0);
    for (int i = 0; i < g.shape.n_instr; ++i) {
        const SgInstr ins = g.code[i];
        if (op_is_value(ins.op) || op_is_compare(ins.op)) {
            T x[C][E], y[C][E];
            const bool fa = ins.a == last_dst, fb = ins.b == last_dst;      // uniform
#pragma unroll
            for (int c = 0; c < C; ++c) {
                if (fa) { _Pragma("unroll") for (int e = 0; e < E; ++e) x[c][e] = last[c][e]; } else rf[c].get(ins.a, x[c]);
                if (fb) { _Pragma("unroll") for (int e = 0; e < E; ++e) y[c][e] = last[c][e]; } else rf[c].get(ins.b, y[c]);
            }
            if (op_is_value(ins.op)) {
                switch (ins.op) {
#define VOP(OPC) case OPC: _Pragma("unroll") for (int c = 0; c < C; ++c) _Pragma("unroll") for (int e = 0; e < E; ++e) last[c][e] = value_op<T>(OPC, x[c][e], y[c][e]); break;
                    VOP(OP_ADD) VOP(OP_SUB) VOP(OP_MUL) VOP(OP_DIV) VOP(OP_MIN) VOP(OP_MAX) VOP(OP_MOD) VOP(OP_NEG) VOP(OP_ABS) VOP(OP_SQRT)
#undef VOP
                    default: _Pragma("unroll") for (int c = 0; c < C; ++c) _Pragma("unroll") for (int e = 0; e < E; ++e) last[c][e] = x[c][e]; break;
                }
                last_dst = ins.dst;
#pragma unroll
                for (int c = 0; c < C; ++c) rf[c].put(ins.dst, last[c]);
            } else {
#pragma unroll
                for (int c = 0; c < C; ++c) {
                    unsigned int bits = 0;
                    switch (ins.op) {
#define COP(OPC) case OPC: _Pragma("unroll") for (int e = 0; e < E; ++e) bits |= (unsigned int)compare_op<T>(OPC, x[c][e], y[c][e]) << e; break;
                        COP(OP_EQ) COP(OP_NE) COP(OP_LT) COP(OP_LE) COP(OP_GT)
#undef COP
                        default: _Pragma("unroll") for (int e = 0; e < E; ++e) bits |= (unsigned int)(x[c][e] >= y[c][e]) << e; break;
                    }
                    pf[c] = pput<E>(pf[c], ins.dst, bits);
                }
            }
        } else {
#pragma unroll
            for (int c = 0; c < C; ++c) {
                const unsigned int x = pget<E>(pf[c], ins.a), y = pget<E>(pf[c], ins.b);
                const unsigned int z = ins.op == OP_AND ? (x & y) : ins.op == OP_OR ? (x | y) : ~x;
                pf[c] = pput<E>(pf[c], ins.dst, z);
            }
        }
    }
}
// single-cell form (filter evaluator)
template <class T, int E>
__device__ __forceinline__ void vm_exec(const SgProg& g, VmRegs<T, E>& rf, unsigned int& pf) {
    VmRegs<T, E> r1[1] = {rf};
    unsigned int p1[1] = {pf};
    vm_exec<T, E, 1>(g, r1, p1);
    pf = p1[0];
}

// load input k for E consecutive elements starting at i (guarded: elements >= limit read as zero)
template <class T, int E, class RF>
__device__ __forceinline__ void vm_load(const SgProg& g, const SgArgs& a, int k, int64_t i, bool full, RF& rf, unsigned int& pf) {
    typedef typename Traits<T>::vec VEC;
    constexpr int V = Traits<T>::V;
    const SgIn in = g.in[k];
    T x[E];
    if (in.kind == IN_VEC && full && ((a.vec_ok >> k) & 1)) {
        const VEC* src = reinterpret_cast<const VEC*>(reinterpret_cast<const T*>(a.in_ptr[k]) + i);
#pragma unroll
        for (int u = 0; u < E / V; ++u) {
            VEC w = ld_stream_rw(src + u);
            const T* we = reinterpret_cast<const T*>(&w);
#pragma unroll
            for (int e = 0; e < V; ++e) x[u * V + e] = we[e];
        }
        rf.put(in.reg, x);
    } else if (in.kind == IN_BOOLVEC) {
        unsigned int bits = 0;
#pragma unroll
        for (int e = 0; e < E; ++e)
            if (i + e < a.in_len[k]) bits |= (unsigned int)(reinterpret_cast<const volatile uint8_t*>(a.in_ptr[k])[i + e] != 0) << e;
        pf = pput<E>(pf, in.reg, bits);
    } else if (in.kind != IN_SCALAR && in.kind != IN_IMM) {
#pragma unroll
        for (int e = 0; e < E; ++e) x[e] = load_elem<T>(in.kind, in.ref, k, a, i + e);
        rf.put(in.reg, x);
    }
}

template <class T, int E, class RF>
__device__ __forceinline__ void vm_emit(const SgProg& g, const SgArgs& a, int64_t i, int64_t hi, bool full, const RF& rf, unsigned int pf,
                                        Cell (&acc)[SG_MAX_OUT]) {
    typedef typename Traits<T>::vec VEC;
    constexpr int V = Traits<T>::V;
#pragma unroll
    for (int o = 0; o < SG_MAX_OUT; ++o) {
        if (o >= g.shape.n_out) break;
        const SgOut out = g.out[o];
        if (out.kind == OUT_FILTER) continue;      // handled by the compaction kernel
        const int64_t len = a.out_len[o] < hi ? a.out_len[o] : hi;   // hi: end of the head range, or n
        if (out_is_pred_reduction(out.kind) || out.kind == OUT_STORE_BOOL) {
            const unsigned int bits = pget<E>(pf, out.src);
#pragma unroll
            for (int e = 0; e < E; ++e) {
                if (i + e >= len) break;
                if (out.kind == OUT_STORE_BOOL) reinterpret_cast<uint8_t*>(a.out_ptr[o])[i + e] = (bits >> e) & 1u;
                else cell_accum_pred(out.kind, acc[o], (bits >> e) & 1u);
            }
        } else {
            T x[E];
            rf.get(out.src, x);
            if (out.kind == OUT_STORE) {
                if (full && ((a.vec_ok >> (16 + o)) & 1)) {
                    VEC* dst = reinterpret_cast<VEC*>(reinterpret_cast<T*>(a.out_ptr[o]) + i);
#pragma unroll
                    for (int u = 0; u < E / V; ++u) st_stream(dst + u, *reinterpret_cast<const VEC*>(&x[u * V]));
                } else {
#pragma unroll
                    for (int e = 0; e < E; ++e)
                        if (i + e < len) reinterpret_cast<T*>(a.out_ptr[o])[i + e] = x[e];
                }
            } else {
                const unsigned int mask = out.pred == SG_NO_PRED ? ((1u << E) - 1u) : pget<E>(pf, out.pred);
#pragma unroll
                for (int e = 0; e < E; ++e)
                    if (i + e < len && ((mask >> e) & 1u)) {
                        switch (out.kind) {
                            case OUT_SUM: cell_accum_value<T>(OUT_SUM, acc[o], x[e]); break;
                            case OUT_MAX: cell_accum_value<T>(OUT_MAX, acc[o], x[e]); break;
                            default: cell_accum_value<T>(OUT_MIN, acc[o], x[e]); break;
                        }
                    }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Pre-decoded micro-ops.  The program is the same for every tile, so it is decoded ONCE per block into shared
// memory: one 16-byte micro-op per instruction = {opcode, dst, a, b} where a value register is already the byte
// offset of its cell 0 in the register file (bit 31: a single broadcast cell) and a predicate register is already its
// shift in the predicate word.  Per instruction a tile then costs one broadcast 128-bit shared load, one dispatch and the
// operand accesses at `base + offset + cell * cell_stride` for C cells.
// ---------------------------------------------------------------------------------------------------------
// micro-op word x = opcode + forwarding variant (operand a / b is the previous value result) + VM_ST (write the result back)
constexpr uint32_t VM_FA = OP_COUNT_, VM_FB = 2 * OP_COUNT_, VM_ST = 0x100, VM_SINGLE = 0x80000000u;
struct VmTables {
    uint4 uop[SG_MAX_INSTR];    // {op, dst, a, b}
    uint4 vin[SG_MAX_IN];       // 128-bit loadable vector inputs: {ptr.lo, ptr.hi, register byte offset, input index}
    int n_vin, n_slow;          // inputs served by the list above / by the generic loader (shifted, strided, BOOL, converting, misaligned)
    uint8_t slow[SG_MAX_IN];
    uint32_t reg_off[SG_MAX_VREG];  // byte offset of cell 0 of program register k in the file | VM_SINGLE for a broadcast register
};

// register-file accessor of one cell of the micro-op kernel (ragged tiles, slow inputs): same interface as VmRegs
template <class T, int E> struct VmCellRef {
    uint32_t base;              // shared-window address of this thread's slot in cell 0 of the file
    uint32_t cell_off;          // this cell's byte offset inside a multi-cell register
    const uint32_t* reg_off;
    __device__ __forceinline__ uint32_t addr(uint8_t k) const {
        const uint32_t o = reg_off[k];
        return base + (o & ~VM_SINGLE) + ((o & VM_SINGLE) ? 0u : cell_off);
    }
    __device__ __forceinline__ void get(uint8_t k, T (&o)[E]) const {
        uint32_t w[4];
        asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w[0]), "=r"(w[1]), "=r"(w[2]), "=r"(w[3]) : "r"(addr(k)) : "memory");
        memcpy(o, w, 16);
    }
    __device__ __forceinline__ void put(uint8_t k, const T (&o)[E]) {
        uint32_t w[4];
        memcpy(w, o, 16);
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr(k)), "r"(w[0]), "r"(w[1]), "r"(w[2]), "r"(w[3]) : "memory");
    }
};

template <int E, int VB, int C> __device__ __forceinline__ void vm_decode(const SgProg& g, const SgArgs& a, VmTables& t) {
    constexpr uint32_t CS = (uint32_t)VB * 16u;
    const int n = g.shape.n_instr;
    // file layout: the C-cell registers first, then one broadcast cell per immediate / device scalar
    bool single[SG_MAX_VREG] = {};
    for (int k = 0; k < g.shape.n_in; ++k)
        if ((g.in[k].kind == IN_SCALAR || g.in[k].kind == IN_IMM) && g.in[k].reg < SG_MAX_VREG) single[g.in[k].reg] = true;
    uint32_t off = 0;
    for (int r = 0; r < g.shape.n_vreg && r < SG_MAX_VREG; ++r)
        if (!single[r]) { t.reg_off[r] = off; off += (uint32_t)C * CS; }
    for (int r = 0; r < g.shape.n_vreg && r < SG_MAX_VREG; ++r)
        if (single[r]) { t.reg_off[r] = off | VM_SINGLE; off += CS; }
    // fwd[i]: which operand slot of instruction i is the result of the most recent value instruction (kept in hardware registers)
    uint8_t fwd[SG_MAX_INSTR];
    int last_dst = -1;
    for (int i = 0; i < n; ++i) {
        const SgInstr ins = g.code[i];
        const bool reads_v = op_is_value(ins.op) || op_is_compare(ins.op);
        const bool unary = op_is_unary_value(ins.op);
        fwd[i] = 0;
        if (reads_v && last_dst >= 0) {
            if (ins.a == last_dst) fwd[i] = VM_FA;
            else if (!unary && ins.b == last_dst) fwd[i] = VM_FB;
        }
        if (op_is_value(ins.op)) last_dst = ins.dst;
    }
    for (int i = 0; i < n; ++i) {
        const SgInstr ins = g.code[i];
        uint4 u;
        bool store = false;
        if (op_is_value(ins.op)) {
            // the result must reach the shared-memory file unless every later read of it (before the register is
            // redefined) is a forwarded operand slot and no output reads it
            for (int o = 0; o < g.shape.n_out; ++o) {
                const uint8_t k = g.out[o].kind;
                if ((k == OUT_STORE || k == OUT_SUM || k == OUT_MAX || k == OUT_MIN || k == OUT_FILTER) && g.out[o].src == ins.dst) store = true;
            }
            for (int j = i + 1; j < n && !store; ++j) {
                const SgInstr nx = g.code[j];
                if (op_is_value(nx.op) || op_is_compare(nx.op)) {
                    const bool unary = op_is_unary_value(nx.op);
                    if (nx.a == ins.dst && fwd[j] != VM_FA) store = true;
                    if (!unary && nx.b == ins.dst && fwd[j] != VM_FB) store = true;
                }
                if (op_is_value(nx.op) && nx.dst == ins.dst) break;
            }
            u.y = t.reg_off[ins.dst] & ~VM_SINGLE; u.z = t.reg_off[ins.a]; u.w = t.reg_off[ins.b];
        } else if (op_is_compare(ins.op)) { u.y = ins.dst * E; u.z = t.reg_off[ins.a]; u.w = t.reg_off[ins.b]; }
        else { u.y = ins.dst * E; u.z = ins.a * E; u.w = ins.b * E; }
        u.x = (uint32_t)ins.op + fwd[i] + (store ? VM_ST : 0u);
        t.uop[i] = u;
    }
    int nv = 0, ns = 0;
    for (int k = 0; k < g.shape.n_in; ++k) {
        const SgIn in = g.in[k];
        if (in.kind == IN_SCALAR || in.kind == IN_IMM) continue;      // loaded once, before the tile loop
        if (in.kind == IN_VEC && ((a.vec_ok >> k) & 1)) {
            const unsigned long long p = (unsigned long long)a.in_ptr[k];
            t.vin[nv++] = make_uint4((uint32_t)p, (uint32_t)(p >> 32), t.reg_off[in.reg] & ~VM_SINGLE, (uint32_t)k);
        } else t.slow[ns++] = (uint8_t)k;
    }
    t.n_vin = nv; t.n_slow = ns;
}

__device__ __forceinline__ uint4 lds128(uint32_t addr) {
    uint4 w;
    asm volatile("ld.shared.v4.b32 {%0,%1,%2,%3}, [%4];" : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w) : "r"(addr) : "memory");
    return w;
}
__device__ __forceinline__ void sts128(uint32_t addr, const uint4& w) {
    asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(w.x), "r"(w.y), "r"(w.z), "r"(w.w) : "memory");
}
// operand `o` (a register byte offset, VM_SINGLE for a broadcast cell) of all C cells
template <class T, int E, int C, uint32_t CS> __device__ __forceinline__ void vm_get(uint32_t base, uint32_t o, T (&x)[C][E]) {
    if (o & VM_SINGLE) {        // one value for the whole pass: read once (uniform branch)
        const uint4 w = lds128(base + (o & ~VM_SINGLE));
#pragma unroll
        for (int c = 0; c < C; ++c) memcpy(x[c], &w, 16);
    } else {
#pragma unroll
        for (int c = 0; c < C; ++c) { const uint4 w = lds128(base + o + (uint32_t)c * CS); memcpy(x[c], &w, 16); }
    }
}
template <class T, int E, int C, uint32_t CS> __device__ __forceinline__ void vm_put(uint32_t addr, const T (&o)[C][E]) {
#pragma unroll
    for (int c = 0; c < C; ++c) { uint4 w; memcpy(&w, o[c], 16); sts128(addr + (uint32_t)c * CS, w); }
}

// `base` = shared-window address of this thread's slot in cell 0 of the file; `uops` = address of the micro-op table.
// `last` (the previous value result) stays in hardware registers: a forwarded operand is not re-read from shared memory and a
// result that only forwarded operands consume is never written there (shared-memory bandwidth bounds this kernel otherwise).
// The forwarding variants are separate cases of ONE switch: fetching operands in a common stage and dispatching on the opcode
// alone was measured slower (121 instead of 88 thread instructions per element: the selects between `last` and the fetched operands
// become predicated register moves over all C * E values).
template <class T, int E, int C, uint32_t CS>
__device__ __forceinline__ void vm_exec_uops(uint32_t uops, int n_instr, uint32_t base, unsigned int (&pf)[C]) {
    constexpr unsigned int EM = (1u << E) - 1u;
    T last[C][E];
#pragma unroll
    for (int c = 0; c < C; ++c)
#pragma unroll
        for (int e = 0; e < E; ++e) last[c][e] = T(0);
    for (int i = 0; i < n_instr; ++i) {
        const uint4 u = lds128(uops + (uint32_t)i * 16u);      // same address in every thread: a broadcast
        switch (u.x & 0xffu) {
#define SG_VM_EACH _Pragma("unroll") for (int c = 0; c < C; ++c) _Pragma("unroll") for (int e = 0; e < E; ++e)
#define SG_VM_BIN(OPC)                                                                                           \
    case OPC: {                                                                                                  \
        T x[C][E], y[C][E];                                                                                      \
        vm_get<T, E, C, CS>(base, u.z, x); vm_get<T, E, C, CS>(base, u.w, y);                                    \
        SG_VM_EACH last[c][e] = value_op<T>(OPC, x[c][e], y[c][e]);                                              \
    } break;                                                                                                     \
    case OPC + VM_FA: {                                                                                          \
        T y[C][E];                                                                                               \
        vm_get<T, E, C, CS>(base, u.w, y);                                                                       \
        SG_VM_EACH last[c][e] = value_op<T>(OPC, last[c][e], y[c][e]);                                           \
    } break;                                                                                                     \
    case OPC + VM_FB: {                                                                                          \
        T x[C][E];                                                                                               \
        vm_get<T, E, C, CS>(base, u.z, x);                                                                       \
        SG_VM_EACH last[c][e] = value_op<T>(OPC, x[c][e], last[c][e]);                                           \
    } break;
#define SG_VM_UN(OPC)                                                                                            \
    case OPC: {                                                                                                  \
        T x[C][E];                                                                                               \
        vm_get<T, E, C, CS>(base, u.z, x);                                                                       \
        SG_VM_EACH last[c][e] = value_op<T>(OPC, x[c][e], x[c][e]);                                              \
    } break;                                                                                                     \
    case OPC + VM_FA: {                                                                                          \
        SG_VM_EACH last[c][e] = value_op<T>(OPC, last[c][e], last[c][e]);                                        \
    } break;
#define SG_VM_CMP_BODY(OPC, X, Y)                                                                                \
        _Pragma("unroll") for (int c = 0; c < C; ++c) {                                                          \
            unsigned int bits = 0;                                                                               \
            _Pragma("unroll") for (int e = 0; e < E; ++e) bits |= (unsigned int)compare_op<T>(OPC, X[c][e], Y[c][e]) << e; \
            pf[c] = (pf[c] & ~(EM << u.y)) | (bits << u.y);                                                      \
        }
#define SG_VM_CMP(OPC)                                                                                           \
    case OPC: {                                                                                                  \
        T x[C][E], y[C][E];                                                                                      \
        vm_get<T, E, C, CS>(base, u.z, x); vm_get<T, E, C, CS>(base, u.w, y);                                    \
        SG_VM_CMP_BODY(OPC, x, y)                                                                                \
    } break;                                                                                                     \
    case OPC + VM_FA: {                                                                                          \
        T y[C][E];                                                                                               \
        vm_get<T, E, C, CS>(base, u.w, y);                                                                       \
        SG_VM_CMP_BODY(OPC, last, y)                                                                             \
    } break;                                                                                                     \
    case OPC + VM_FB: {                                                                                          \
        T x[C][E];                                                                                               \
        vm_get<T, E, C, CS>(base, u.z, x);                                                                       \
        SG_VM_CMP_BODY(OPC, x, last)                                                                             \
    } break;
            SG_VM_BIN(OP_ADD) SG_VM_BIN(OP_SUB) SG_VM_BIN(OP_MUL) SG_VM_BIN(OP_DIV) SG_VM_BIN(OP_MIN) SG_VM_BIN(OP_MAX) SG_VM_BIN(OP_MOD)
            SG_VM_UN(OP_NEG) SG_VM_UN(OP_ABS) SG_VM_UN(OP_MOV) SG_VM_UN(OP_SQRT)
            SG_VM_CMP(OP_EQ) SG_VM_CMP(OP_NE) SG_VM_CMP(OP_LT) SG_VM_CMP(OP_LE) SG_VM_CMP(OP_GT) SG_VM_CMP(OP_GE)
#undef SG_VM_BIN
#undef SG_VM_UN
#undef SG_VM_CMP
#undef SG_VM_CMP_BODY
#undef SG_VM_EACH
            case OP_AND:
#pragma unroll
                for (int c = 0; c < C; ++c) pf[c] = (pf[c] & ~(EM << u.y)) | ((((pf[c] >> u.z) & (pf[c] >> u.w)) & EM) << u.y);
                break;
            case OP_OR:
#pragma unroll
                for (int c = 0; c < C; ++c) pf[c] = (pf[c] & ~(EM << u.y)) | ((((pf[c] >> u.z) | (pf[c] >> u.w)) & EM) << u.y);
                break;
            default:    // OP_NOT
#pragma unroll
                for (int c = 0; c < C; ++c) pf[c] = (pf[c] & ~(EM << u.y)) | (((~(pf[c] >> u.z)) & EM) << u.y);
                break;
        }
        if (u.x & VM_ST) vm_put<T, E, C, CS>(base + u.y, last);
    }
}

// outputs of a FULL tile (inside every value's length, vector-aligned): no per-element guards
template <class T, int E, int VB, int C>
__device__ __forceinline__ void vm_emit_full(const SgProg& g, const SgArgs& a, int64_t i0, uint32_t base, const uint32_t* reg_off, const unsigned int (&pf)[C],
                                             Cell (&acc)[SG_MAX_OUT]) {
    constexpr unsigned int EM = (1u << E) - 1u;
    constexpr uint32_t CS = (uint32_t)VB * 16u;
#pragma unroll
    for (int o = 0; o < SG_MAX_OUT; ++o) {
        if (o >= g.shape.n_out) break;
        const SgOut out = g.out[o];
        switch (out.kind) {
            case OUT_STORE: {
                T x[C][E];
                vm_get<T, E, C, CS>(base, reg_off[out.src], x);
                if ((a.vec_ok >> (16 + o)) & 1) {
#pragma unroll
                    for (int c = 0; c < C; ++c)
                        st_stream(reinterpret_cast<int4*>(reinterpret_cast<T*>(a.out_ptr[o]) + i0 + (int64_t)c * (VB * E)), *reinterpret_cast<const int4*>(x[c]));
                } else {
#pragma unroll
                    for (int c = 0; c < C; ++c)
#pragma unroll
                        for (int e = 0; e < E; ++e) reinterpret_cast<T*>(a.out_ptr[o])[i0 + (int64_t)c * (VB * E) + e] = x[c][e];
                }
            } break;
            case OUT_STORE_BOOL:
#pragma unroll
                for (int c = 0; c < C; ++c)
#pragma unroll
                    for (int e = 0; e < E; ++e) reinterpret_cast<uint8_t*>(a.out_ptr[o])[i0 + (int64_t)c * (VB * E) + e] = (pf[c] >> (out.src * E + e)) & 1u;
                break;
            case OUT_ALL:
#pragma unroll
                for (int c = 0; c < C; ++c) acc[o].a &= (unsigned long long)(((pf[c] >> (out.src * E)) & EM) == EM);
                break;
            case OUT_ANY:
#pragma unroll
                for (int c = 0; c < C; ++c) acc[o].a |= (unsigned long long)(((pf[c] >> (out.src * E)) & EM) != 0u);
                break;
            case OUT_COUNT:
#pragma unroll
                for (int c = 0; c < C; ++c) acc[o].a += (unsigned long long)__popc((pf[c] >> (out.src * E)) & EM);
                break;
            case OUT_SUM: case OUT_MAX: case OUT_MIN: {
                T x[C][E];
                vm_get<T, E, C, CS>(base, reg_off[out.src], x);
                if (out.pred == SG_NO_PRED) {
                    if (out.kind == OUT_SUM) {
#pragma unroll
                        for (int c = 0; c < C; ++c)
#pragma unroll
                            for (int e = 0; e < E; ++e) cell_accum_value<T>(OUT_SUM, acc[o], x[c][e]);
                    } else if (out.kind == OUT_MAX) {
#pragma unroll
                        for (int c = 0; c < C; ++c)
#pragma unroll
                            for (int e = 0; e < E; ++e) cell_accum_value<T>(OUT_MAX, acc[o], x[c][e]);
                    } else {
#pragma unroll
                        for (int c = 0; c < C; ++c)
#pragma unroll
                            for (int e = 0; e < E; ++e) cell_accum_value<T>(OUT_MIN, acc[o], x[c][e]);
                    }
                } else {
#pragma unroll
                    for (int c = 0; c < C; ++c) {
                        const unsigned int mask = (pf[c] >> (out.pred * E)) & EM;
#pragma unroll
                        for (int e = 0; e < E; ++e)
                            if ((mask >> e) & 1u) {
                                if (out.kind == OUT_SUM) cell_accum_value<T>(OUT_SUM, acc[o], x[c][e]);
                                else if (out.kind == OUT_MAX) cell_accum_value<T>(OUT_MAX, acc[o], x[c][e]);
                                else cell_accum_value<T>(OUT_MIN, acc[o], x[c][e]);
                            }
                    }
                }
            } break;
            default: break;     // OUT_FILTER: handled by the compaction kernel
        }
    }
}

// VB threads per block, C cells per value register and thread (vm_config)
template <class T, int VB, int C>
__global__ void __launch_bounds__(VB, VB == 128 ? 4 : 3) pass1d_bytecode(const __grid_constant__ SgProg g, const __grid_constant__ SgArgs a) {
    extern __shared__ __align__(16) unsigned char vm_file[];
    __shared__ __align__(16) VmTables tab;
    constexpr int E = VmE<T>::value;
    constexpr uint32_t CS = (uint32_t)VB * 16u;
    constexpr int VM_TILE = VB * E * C;             // C cells of VB*E consecutive elements each
    pdl_wait();
    pdl_trigger();
    Cell acc[SG_MAX_OUT];
    uint8_t kind[SG_MAX_OUT];
    bool has_reduction = false;
    unsigned int need_mask = 0, flagged = 0;
#pragma unroll
    for (int o = 0; o < SG_MAX_OUT; ++o) {
        kind[o] = (o < g.shape.n_out) ? g.out[o].kind : (uint8_t)OUT_STORE;
        acc[o] = cell_identity<T>(kind[o]);
        has_reduction |= out_is_reduction(kind[o]);
        if (o < g.shape.n_out) need_mask |= 1u << o;
    }
    const bool early_exit = (g.shape.flags & PF_EARLY_EXIT) && !a.no_early_exit;

    if (threadIdx.x == 0) vm_decode<E, VB, C>(g, a, tab);
    const uint32_t file = (uint32_t)__cvta_generic_to_shared(vm_file);
    const uint32_t uops = (uint32_t)__cvta_generic_to_shared(tab.uop);
    const uint32_t base = file + threadIdx.x * 16u;
    __syncthreads();
    VmCellRef<T, E> rf[C];
#pragma unroll
    for (int c = 0; c < C; ++c) { rf[c].base = base; rf[c].cell_off = (uint32_t)c * CS; rf[c].reg_off = tab.reg_off; }
    unsigned int pf[C];
#pragma unroll
    for (int c = 0; c < C; ++c) pf[c] = 0;
    for (int k = 0; k < g.shape.n_in; ++k) {
        const SgIn in = g.in[k];
        if (in.kind == IN_SCALAR || in.kind == IN_IMM) {        // one broadcast cell
            T x[E];
            const T s = load_elem<T>(in.kind, in.ref, k, a, 0);
#pragma unroll
            for (int e = 0; e < E; ++e) x[e] = s;
            rf[0].put(in.reg, x);
        }
    }
    __syncthreads();
    const int n_instr = g.shape.n_instr, n_vin = tab.n_vin, n_slow = tab.n_slow;
    // tiles over the aligned body [head, n) — the last tile is guarded; then the head [0, head) one vector at a time
    const int64_t body = a.n - a.head;
    const int64_t n_tiles = (body + VM_TILE - 1) / VM_TILE;
    const int64_t head_tiles = (a.head + VM_TILE - 1) / VM_TILE;
    unsigned int it = 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles + head_tiles; tile += gridDim.x, ++it) {
        if (early_exit && (it & 1u) == 0) {
            const unsigned int w = ld_relaxed_u32(&a.ctrl[1]);
            if ((w & need_mask) == need_mask || (w & a.exit_any) != 0) break;
        }
        const bool in_body = tile < n_tiles;
        const int64_t hi = in_body ? a.n : a.head;
        const int64_t i0 = (in_body ? a.head + tile * VM_TILE : (tile - n_tiles) * VM_TILE) + (int64_t)threadIdx.x * E;
        // full: the whole tile lies inside every value's length and the body is 16-byte aligned
        const bool full = (tile < a.n_full_tiles);
        if (full) {
            const int64_t boff = i0 * (int64_t)sizeof(T);
            for (int j = 0; j < n_vin; ++j) {
                const uint4 v = tab.vin[j];
                const char* p = reinterpret_cast<const char*>(((unsigned long long)v.y << 32) | v.x) + boff;
                int4 w[C];
#pragma unroll
                for (int c = 0; c < C; ++c) w[c] = ld_stream_rw(reinterpret_cast<const int4*>(p + (size_t)c * CS));
#pragma unroll
                for (int c = 0; c < C; ++c) sts128(base + v.z + (uint32_t)c * CS, *reinterpret_cast<const uint4*>(&w[c]));
            }
            for (int j = 0; j < n_slow; ++j)
#pragma unroll
                for (int c = 0; c < C; ++c) vm_load<T, E>(g, a, tab.slow[j], i0 + (int64_t)c * (VB * E), false, rf[c], pf[c]);
            vm_exec_uops<T, E, C, CS>(uops, n_instr, base, pf);
            vm_emit_full<T, E, VB, C>(g, a, i0, base, tab.reg_off, pf, acc);
        } else if (i0 < hi) {
#pragma unroll
            for (int c = 0; c < C; ++c)
                for (int k = 0; k < g.shape.n_in; ++k) vm_load<T, E>(g, a, k, i0 + (int64_t)c * (VB * E), false, rf[c], pf[c]);      // guarded: reads past the end give zeros
            vm_exec_uops<T, E, C, CS>(uops, n_instr, base, pf);
#pragma unroll
            for (int c = 0; c < C; ++c)
                if (i0 + (int64_t)c * (VB * E) < hi) vm_emit<T, E>(g, a, i0 + (int64_t)c * (VB * E), hi, false, rf[c], pf[c], acc);
        }
        if (early_exit) {
#pragma unroll
            for (int o = 0; o < SG_MAX_OUT; ++o) {
                if (o >= g.shape.n_out) break;
                bool decided = (kind[o] == OUT_ALL) ? (acc[o].a == 0) : (acc[o].a != 0);
                if (!(flagged & (1u << o)) && __any_sync(0xffffffffu, decided)) {
                    flagged |= 1u << o;
                    if ((threadIdx.x & 31) == 0) atomicOr(&a.ctrl[1], 1u << o);
                }
            }
        }
    }
    epilogue_1d<T, SG_MAX_OUT>(acc, kind, a, has_reduction);
}

}  // namespace sgk
#endif  // SG_PASS1D_VM_CUH_
