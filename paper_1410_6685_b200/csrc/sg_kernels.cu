// sg_kernels.cu — kernel instantiation, the template registry and launch geometry (sm_100a).
#include "sg_kernels.h"

#include <cuda.h>

#include <stdio.h>
#include <string.h>

#include <algorithm>

#include "sg_filter.cuh"
#include "sg_pass1d_tmpl.cuh"
#include "sg_pass1d_vm.cuh"
#include "sg_pass2d.cuh"

namespace {

using namespace sgk;

typedef cudaError_t (*LaunchFn)(const SgArgs&, int grid, cudaStream_t);
template <class P> constexpr size_t smem_of() {
    if constexpr ((P::prog.shape.flags & PF_2D) != 0) return sgk::Meta2D<P>::SMEM;
    else if constexpr ((P::prog.shape.flags & PF_FILTER) != 0) return sgk::FilterTemplateEval<P>::SMEM;
    else return 0;
}
typedef int (*OccFn)();

struct Entry {
    const char* name;
    const SgProg* prog;
    LaunchFn launch;
    OccFn occupancy;
    int tile;       // elements per tile (1-D, filter) or strip width (2-D)
};

template <class P> constexpr int tile_of() {
    if (P::prog.shape.flags & PF_FILTER) return FilterTemplateEval<P>::TILE;
    return BLOCK * Meta1D<P>::E;
}

// TMA tensor map of one filter input: the vector seen as `rows` rows of 128 bytes, box = 256 rows (one tile), 128-byte
// swizzle (sg_filter.cuh).  The driver entry point is fetched once through the runtime (no link against libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
bool encode_filter_tmap(void* out128, const void* base, long rows) {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess) fn = (EncodeTiledFn)p;
        else cudaGetLastError();
    }
    if (!fn || rows <= 0 || rows > 0x7fffffffl) return false;
    static_assert(sizeof(CUtensorMap) == 128, "tensor map size");
    const cuuint64_t dims[2] = {32, (cuuint64_t)rows};
    const cuuint64_t strides[1] = {128};
    const cuuint32_t box[2] = {32, (cuuint32_t)F_ROWS};
    const cuuint32_t estr[2] = {1, 1};
    alignas(64) CUtensorMap m;
    if (fn(&m, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
           CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    memcpy(out128, &m, 128);
    return true;
}
template <class P> bool encode_filter_tmaps(SgArgs& a) {
    typedef FilterTemplateEval<P> EV;
    if (EV::NSTG == 0 || !((a.vec_ok >> 31) & 1) || a.n_full_tiles <= 0) return false;
    int slot = 0;       // index among the IN_VEC inputs
    for (int k = 0; k < P::prog.shape.n_in; ++k) {
        if (P::prog.in[k].kind != IN_VEC) continue;
        if (slot < EV::NSTG && !encode_filter_tmap(a.tmap[slot], a.in_ptr[k], (long)a.n_full_tiles * F_ROWS)) return false;
        ++slot;
    }
    return true;
}

template <class P> cudaError_t launch_template(const SgArgs& a, int grid, cudaStream_t s) {
    if constexpr ((P::prog.shape.flags & PF_2D) != 0) {
        static bool attr_set = false;
        if (!attr_set) { cudaFuncSetAttribute(pass2d_template<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<P>()); attr_set = true; }
        pass2d_template<P><<<grid, BLOCK, smem_of<P>(), s>>>(a);
    }
    else if constexpr ((P::prog.shape.flags & PF_FILTER) != 0) {
        static bool attr_set = false;
        if (!attr_set) { cudaFuncSetAttribute(filter1d_template<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<P>()); attr_set = true; }
        SgArgs a2 = a;
        a2.vec_ok &= ~(1 << 30);
        if (encode_filter_tmaps<P>(a2)) a2.vec_ok |= (1 << 30);
        filter1d_template<P><<<grid, FilterTemplateEval<P>::CT + 32, smem_of<P>(), s>>>(a2);
    }
    else pass1d_template<P><<<grid, BLOCK, 0, s>>>(a);
    return cudaGetLastError();
}
template <class P> int occupancy_template() {
    static int cached = 0;      // one query per instance per process (the query costs tens of microseconds)
    if (cached > 0) return cached;
    int occ = 0;
    cudaError_t e;
    if constexpr ((P::prog.shape.flags & PF_2D) != 0) {
        cudaFuncSetAttribute(pass2d_template<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<P>());
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pass2d_template<P>, BLOCK, smem_of<P>());
    }
    else if constexpr ((P::prog.shape.flags & PF_FILTER) != 0) {
        cudaFuncSetAttribute(filter1d_template<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<P>());
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, filter1d_template<P>, FilterTemplateEval<P>::CT + 32, smem_of<P>());
    }
    else e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pass1d_template<P>, BLOCK, 0);
    if (e != cudaSuccess || occ <= 0) return 1;
    cached = occ;
    return occ;
}

// Each SG_TEMPLATE(name, unroll, min_blocks, row_unroll, {program}) in the generated file defines a policy type
// and registers it.  The program initialisers are written by paper_1410_6685_b200/gen_templates.py from the plan
// builder's own canonical output, so a registered chain always matches its signature.
#define SG_TEMPLATE(NAME, UNROLL, MINB, ROWU, ...)                                   \
    struct T_##NAME {                                                                \
        static constexpr SgProg prog = __VA_ARGS__;                                  \
        static constexpr int unroll = UNROLL, min_blocks = MINB, row_unroll = ROWU, stages = 3;  \
    };
#include "sg_templates_gen.inc"
#undef SG_TEMPLATE

#define SG_TEMPLATE(NAME, UNROLL, MINB, ROWU, ...) \
    {#NAME, &T_##NAME::prog, &launch_template<T_##NAME>, &occupancy_template<T_##NAME>, tile_of<T_##NAME>()},
const Entry g_entries[] = {
    {"bytecode", nullptr, nullptr, nullptr, 0},
#include "sg_templates_gen.inc"
};
#undef SG_TEMPLATE
const int g_n_entries = (int)(sizeof(g_entries) / sizeof(g_entries[0]));

template <class T, int C> cudaError_t launch_pass1d_bytecode(const SgProg& g, const SgArgs& a, int grid, cudaStream_t s) {
    static bool attr_set = false;
    if (!attr_set) { cudaFuncSetAttribute(pass1d_bytecode<T, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vm_file_bytes(VM_VREG, 1)); attr_set = true; }
    pass1d_bytecode<T, C><<<grid, BLOCK, vm_file_bytes(g.shape.n_vreg, C), s>>>(g, a);
    return cudaGetLastError();
}
template <class T> cudaError_t launch_bytecode_t(const SgProg& g, const SgArgs& a, const SgGeom& geom, cudaStream_t s) {
    if (g.shape.flags & PF_FILTER) {
        static bool attr_set = false;
        if (!attr_set) { cudaFuncSetAttribute(filter1d_bytecode<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FilterBytecodeEval<T>::SMEM); attr_set = true; }
        filter1d_bytecode<T><<<geom.grid, BLOCK + 32, FilterBytecodeEval<T>::SMEM, s>>>(g, a);
        return cudaGetLastError();
    }
    return geom.vm_cells == 2 ? launch_pass1d_bytecode<T, 2>(g, a, geom.grid, s) : launch_pass1d_bytecode<T, 1>(g, a, geom.grid, s);
}
// blocks per SM of the bytecode kernels (the 1-D pass depends on the size of its register file: queried once per size)
template <class T> int occupancy_bytecode_t(bool filter, int n_vreg, int cells) {
    static int cached_filter = 0, cached[VM_VREG + 1][VM_MAX_CELLS + 1] = {};
    int occ = 0;
    cudaError_t e;
    if (filter) {
        if (cached_filter > 0) return cached_filter;
        cudaFuncSetAttribute(filter1d_bytecode<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FilterBytecodeEval<T>::SMEM);
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, filter1d_bytecode<T>, BLOCK + 32, FilterBytecodeEval<T>::SMEM);
        if (e != cudaSuccess || occ <= 0) return 1;
        return cached_filter = occ;
    }
    n_vreg = std::min(std::max(n_vreg, 1), VM_VREG);
    if (cached[n_vreg][cells] > 0) return cached[n_vreg][cells];
    const size_t smem = vm_file_bytes(n_vreg, cells);
    if (cells == 2) {
        cudaFuncSetAttribute(pass1d_bytecode<T, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vm_file_bytes(VM_VREG, 1));
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pass1d_bytecode<T, 2>, BLOCK, smem);
    } else {
        cudaFuncSetAttribute(pass1d_bytecode<T, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vm_file_bytes(VM_VREG, 1));
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pass1d_bytecode<T, 1>, BLOCK, smem);
    }
    if (e != cudaSuccess || occ <= 0) return 1;
    return cached[n_vreg][cells] = occ;
}
int occupancy_bytecode(int dtype, bool filter, int n_vreg = VM_VREG, int cells = 1) {
    switch (dtype) {
        case DT_F32: return occupancy_bytecode_t<float>(filter, n_vreg, cells);
        case DT_F64: return occupancy_bytecode_t<double>(filter, n_vreg, cells);
        case DT_I32: return occupancy_bytecode_t<int32_t>(filter, n_vreg, cells);
        default: return occupancy_bytecode_t<long long>(filter, n_vreg, cells);
    }
}

int elem_size(int dtype) { return (dtype == DT_F32 || dtype == DT_I32) ? 4 : 8; }

int fail(char* err, size_t cap, int code, const char* msg) {
    if (err && cap) snprintf(err, cap, "%s", msg);
    return code;
}

}  // namespace

int sgk_template_count() { return g_n_entries - 1; }
const char* sgk_template_name(int id) { return (id >= 1 && id < g_n_entries) ? g_entries[id].name : "bytecode"; }
const SgProg* sgk_template_prog(int id) { return (id >= 1 && id < g_n_entries) ? g_entries[id].prog : nullptr; }
int sgk_find_template(const SgProg& prog) {
    for (int i = 1; i < g_n_entries; ++i)
        if (memcmp(g_entries[i].prog, &prog, sizeof(SgProg)) == 0) return i;
    return 0;
}

int sgk_plan(const SgProg& prog, SgArgs& a, int force_bytecode, int sm_count, int has_device, SgGeom* geom, char* err, size_t errcap) {
    const int es = elem_size(prog.shape.dtype);
    const int V = 16 / es;
    const bool is2d = prog.shape.flags & PF_2D, isfilter = prog.shape.flags & PF_FILTER;
    memset(geom, 0, sizeof(*geom));
    int tid = force_bytecode ? 0 : sgk_find_template(prog);
    if (tid == 0 && !is2d && prog.shape.n_vreg > VM_VREG)
        return fail(err, errcap, -9, "fused chain needs more value registers than the bytecode evaluator has; flush earlier");

    // alignment of every vector-accessed operand relative to the pass origin
    long mis = -1;          // common misalignment in elements, -1 = not yet fixed
    bool congruent = true;
    int vec_ok = 0;
    auto misalign = [&](const void* p) { return (long)(((uintptr_t)p % 16) / es); };
    auto consider = [&](const void* p, int bit) {
        if (((uintptr_t)p % es) != 0) { congruent = false; return; }
        long m = misalign(p);
        if (mis < 0) mis = m;
        if (m == mis) vec_ok |= 1 << bit; else congruent = false;
    };
    for (int o = 0; o < prog.shape.n_out; ++o)
        if (prog.out[o].kind == OUT_STORE) consider(a.out_ptr[o], 16 + o);
    for (int k = 0; k < prog.shape.n_in; ++k)
        if (prog.in[k].kind == IN_VEC || (is2d && prog.in[k].kind == IN_ROWB)) consider(a.in_ptr[k], k);
    if (mis < 0) mis = 0;

    if (is2d) {
        if (tid == 0 && has_device) return fail(err, errcap, -10, "matrix pass has no precompiled template instance (2-D bytecode evaluator not built)");
        bool ok = congruent && mis == 0 && (a.cols % V) == 0;
        for (int k = 0; k < prog.shape.n_in; ++k)
            if (prog.in[k].kind == IN_VEC && (a.in_stride[k] % V) != 0) ok = false;
        for (int o = 0; o < prog.shape.n_out; ++o)
            if (prog.out[o].kind == OUT_STORE && (a.out_len[o] % V) != 0) ok = false;
        if (!ok) return fail(err, errcap, -10, "matrix pass needs 16-byte aligned rows (base, leading dimension and column count)");
        const int occ = (has_device && tid) ? g_entries[tid].occupancy() : 2;
        const int SW = tid ? g_entries[tid].tile : BLOCK * 2 * V;
        a.n_strips = (int)((a.cols + SW - 1) / SW);
        const long target = (long)sm_count * occ;
        long max_chunks = std::max<long>(1, (a.n + RB - 1) / RB);
        long n_chunks = std::min<long>(max_chunks, std::max<long>(1, target / std::max(1, a.n_strips)));
        long rpc = (a.n + n_chunks - 1) / n_chunks;
        rpc = std::max<long>(RB, (rpc + RB - 1) / RB * RB);
        n_chunks = std::max<long>(1, (a.n + rpc - 1) / rpc);
        a.rows_per_chunk = rpc;
        a.n_chunks = (int)n_chunks;
        geom->template_id = tid;
        geom->grid = (int)(a.n_strips * n_chunks);
        geom->tile = SW;
        size_t off = (size_t)geom->grid * SG_MAX_OUT * sizeof(Cell);
        for (int o = 0; o < prog.shape.n_out; ++o) {
            a.ws_off[o] = 0;
            if (!out_is_reduction(prog.out[o].kind)) continue;
            if (prog.out[o].axis == AXIS_COLS) { a.ws_off[o] = (int64_t)off; off += (size_t)n_chunks * a.cols * sizeof(Cell); }
            if (prog.out[o].axis == AXIS_ROWS) { a.ws_off[o] = (int64_t)off; off += (size_t)a.n_strips * a.n * sizeof(Cell); }
        }
        geom->ws_bytes = off;
        geom->ctrl_words = a.n_strips + (int)n_chunks;
        a.vec_ok = vec_ok;
        a.head = 0; a.n_full_tiles = 0;
        return 0;
    }

    if (isfilter) {
        const int tile = tid ? g_entries[tid].tile : F_TILE_BYTES / es;
        const int occ = has_device ? (tid ? g_entries[tid].occupancy() : occupancy_bytecode(prog.shape.dtype, true)) : 4;
        const long n_tiles = (a.n + tile - 1) / tile;
        if (a.n >= (1ll << 40) || n_tiles >= 0x3fffffffl) return fail(err, errcap, -9, "filter input too long for the tile-state word");
        a.n_tiles = (int)n_tiles;
        a.vec_ok = vec_ok | ((congruent && mis == 0) ? (1 << 31) : 0);
        // tiles that lie inside every vector operand's and every output's length take the unguarded (staged) path
        long lmin = a.n;
        for (int o = 0; o < prog.shape.n_out; ++o) lmin = std::min<long>(lmin, a.out_len[o]);
        for (int k = 0; k < prog.shape.n_in; ++k)
            if (prog.in[k].kind == IN_VEC) lmin = std::min<long>(lmin, a.in_len[k]);
        a.head = 0; a.n_full_tiles = std::max<long>(0, lmin) / tile;
        geom->template_id = tid;
        geom->tile = tile;
        geom->grid = (int)std::max<long>(1, std::min<long>(n_tiles, (long)sm_count * occ));
        geom->ws_bytes = (size_t)geom->grid * SG_MAX_OUT * sizeof(Cell);
        geom->state_words = (size_t)n_tiles;
        return 0;
    }

    // 1-D pass.  Template instances need every vector operand congruent (common head); otherwise the bytecode
    // kernel runs with per-operand 128-bit eligibility.
    if (tid && !congruent) tid = 0;
    const int cells = vm_cells(prog.shape.n_vreg);
    const int tile = tid ? g_entries[tid].tile : vm_tile(es, cells);
    geom->vm_cells = cells;
    long lmin = a.n;
    for (int o = 0; o < prog.shape.n_out; ++o) lmin = std::min<long>(lmin, a.out_len[o]);
    const long head = std::min<long>((V - mis) % V, a.n);
    const long body = std::max<long>(0, lmin - head);
    a.head = head;
    a.n_full_tiles = body / tile;
    a.vec_ok = vec_ok;
    const int occ = has_device ? (tid ? g_entries[tid].occupancy() : occupancy_bytecode(prog.shape.dtype, false, prog.shape.n_vreg, cells)) : 4;
    long want = tid ? a.n_full_tiles : ((a.n - head + tile - 1) / tile + (head + tile - 1) / tile);
    geom->template_id = tid;
    geom->tile = tile;
    geom->grid = (int)std::max<long>(1, std::min<long>(want, (long)sm_count * occ));
    geom->ws_bytes = (size_t)geom->grid * SG_MAX_OUT * sizeof(Cell);
    return 0;
}

cudaError_t sgk_launch(const SgProg& prog, const SgArgs& args, const SgGeom& geom, cudaStream_t stream) {
    if (geom.template_id > 0) return g_entries[geom.template_id].launch(args, geom.grid, stream);
    switch (prog.shape.dtype) {
        case DT_F32: return launch_bytecode_t<float>(prog, args, geom, stream);
        case DT_F64: return launch_bytecode_t<double>(prog, args, geom, stream);
        case DT_I32: return launch_bytecode_t<int32_t>(prog, args, geom, stream);
        case DT_I64: return launch_bytecode_t<long long>(prog, args, geom, stream);
        default: return cudaErrorInvalidValue;
    }
}
