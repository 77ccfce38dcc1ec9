// sg_tmpl_launch.cuh — launch / occupancy wrappers of the precompiled template instances (internal).
// The instances of sg_templates_gen.inc are compiled in SG_NSHARDS translation units (sg_tmpl_shard.cu, built once per
// shard with -DSG_SHARD=k) so that the library builds in parallel; every shard sees every program (plain constexpr data)
// but instantiates only the kernels of the instances it owns (index % SG_NSHARDS == SG_SHARD).
#ifndef SG_TMPL_LAUNCH_CUH_
#define SG_TMPL_LAUNCH_CUH_

#include <cuda.h>

#include <string.h>

#include "sg_filter.cuh"
#include "sg_kernels.h"
#include "sg_pass1d_tmpl.cuh"
#include "sg_pass2d.cuh"

#define SG_NSHARDS 8

namespace sgk {

typedef cudaError_t (*LaunchFn)(const SgArgs&, int grid, cudaStream_t);
template <class P> constexpr size_t smem_of() {
    if constexpr ((P::prog.shape.flags & PF_2D) != 0) return sgk::Meta2D<P>::SMEM;
    else if constexpr ((P::prog.shape.flags & PF_FILTER) != 0) return sgk::FilterTemplateEval<P>::SMEM;
    else return 0;
}
typedef int (*OccFn)();


template <class P> constexpr int tile_of() {
    if constexpr ((P::prog.shape.flags & PF_FILTER) != 0) return FilterTemplateEval<P>::TILE;
    else return BLOCK * Meta1D<P>::E;
}

// TMA tensor map of one filter input: the vector seen as `rows` rows of 128 bytes, box = 256 rows (one tile), 128-byte
// swizzle (sg_filter.cuh).  The driver entry point is fetched once through the runtime (no link against libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                  const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
inline bool encode_filter_tmap(void* out128, const void* base, long rows) {
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

// Function attributes and occupancy are per DEVICE: the caches below are indexed by the current device (the context makes
// its device current around every entry point), so several contexts on different GPUs in one process stay correct.
constexpr int SG_MAX_DEVICES = 64;
inline int current_device_slot() {
    int d = 0;
    if (cudaGetDevice(&d) != cudaSuccess) { cudaGetLastError(); d = 0; }
    return (d >= 0 && d < SG_MAX_DEVICES) ? d : 0;
}

// one launch with programmatic stream serialisation allowed (see pdl_wait in sg_device.cuh)
template <class... KArgs, class... Args>
inline cudaError_t sgk_launch_pdl(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t s, const Args&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)block); cfg.dynamicSmemBytes = smem; cfg.stream = s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

template <class P> cudaError_t launch_template(const SgArgs& a, int grid, cudaStream_t s) {
    if constexpr ((P::prog.shape.flags & PF_2D) != 0) {
        if constexpr (!Meta2D<P>::has_reduction) {
            if ((a.vec_ok >> 28) & 1) return sgk_launch_pdl(pass2d_tile_template<P>, grid, BLOCK, 0, s, a);     // bit 28 (sgk_plan): one tile per block
        }
        static bool attr_set[SG_MAX_DEVICES] = {};
        bool& set = attr_set[current_device_slot()];
        if (!set) { cudaFuncSetAttribute(pass2d_template<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<P>()); set = true; }
        return sgk_launch_pdl(pass2d_template<P>, grid, BLOCK, smem_of<P>(), s, a);
    }
    else if constexpr ((P::prog.shape.flags & PF_FILTER) != 0) {
        static bool attr_set[SG_MAX_DEVICES] = {};
        bool& set = attr_set[current_device_slot()];
        if (!set) { cudaFuncSetAttribute(filter1d_template<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_of<P>()); set = true; }
        SgArgs a2 = a;
        a2.vec_ok &= ~(1 << 30);
        if (encode_filter_tmaps<P>(a2)) a2.vec_ok |= (1 << 30);
        return sgk_launch_pdl(filter1d_template<P>, grid, FilterTemplateEval<P>::CT + 32, smem_of<P>(), s, a2);
    }
    else return sgk_launch_pdl(pass1d_template<P>, grid, BLOCK, 0, s, a);
}
template <class P> int occupancy_template() {
    static int cached_dev[SG_MAX_DEVICES] = {};     // one query per instance and device (the query costs tens of microseconds)
    int& cached = cached_dev[current_device_slot()];
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


struct Entry {
    const char* name;
    const SgProg* prog;
    LaunchFn launch;
    OccFn occupancy;
    int tile;       // elements per tile (1-D, filter) or strip width (2-D)
};
// only the owning shard names (and thereby instantiates) the kernel of an instance
template <class P, bool OWN> struct EntryOf { static Entry make(const char* name) { return {name, &P::prog, nullptr, nullptr, tile_of<P>()}; } };
template <class P> struct EntryOf<P, true> {
    static Entry make(const char* name) { return {name, &P::prog, &launch_template<P>, &occupancy_template<P>, tile_of<P>()}; }
};

}  // namespace sgk
#endif  // SG_TMPL_LAUNCH_CUH_
