// sg_vm_shard.cu — the bytecode kernels of ONE element type: compiled four times with -DSG_VM_DTYPE=0..3 (DT_F32, DT_F64,
// DT_I32, DT_I64; paper_1410_6685_b200/build.py) so that the interpreters build in parallel.  sg_kernels.cu dispatches on
// the pass dtype to sgk_launch_bytecode_<k> / sgk_occupancy_bytecode_<k>.
#include <algorithm>

#include "sg_filter.cuh"
#include "sg_kernels.h"
#include "sg_pass1d_vm.cuh"
#include "sg_pass2d_vm.cuh"
#include "sg_tmpl_launch.cuh"

#ifndef SG_VM_DTYPE
#error "compile with -DSG_VM_DTYPE=<0..3>"
#endif

namespace {

using namespace sgk;

template <class T, int CFG> cudaError_t launch_pass1d_bytecode(const SgProg& g, const SgArgs& a, int grid, cudaStream_t s) {
    constexpr int VB = vm_config(CFG).threads, C = vm_config(CFG).cells;
    static bool attr_dev[SG_MAX_DEVICES] = {};
    bool& attr_set = attr_dev[current_device_slot()];
    if (!attr_set) { cudaFuncSetAttribute(pass1d_bytecode<T, VB, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)VM_MAX_FILE_BYTES); attr_set = true; }
    int r, i;
    vm_count_regs(g, &r, &i);
    return sgk_launch_pdl(pass1d_bytecode<T, VB, C>, grid, VB, vm_file_bytes_cfg(r, i, CFG), s, g, a);
}
template <class T> cudaError_t launch_bytecode_t(const SgProg& g, const SgArgs& a, const SgGeom& geom, cudaStream_t s) {
    if (g.shape.flags & PF_2D) {
        static bool attr_dev[SG_MAX_DEVICES] = {};
        bool& attr_set = attr_dev[current_device_slot()];
        if (!attr_set) { cudaFuncSetAttribute(pass2d_bytecode<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)VM_FILE_BYTES); attr_set = true; }
        return sgk_launch_pdl(pass2d_bytecode<T>, geom.grid, BLOCK, VM_FILE_BYTES, s, g, a);
    }
    if (g.shape.flags & PF_FILTER) {
        static bool attr_dev[SG_MAX_DEVICES] = {};
        bool& attr_set = attr_dev[current_device_slot()];
        if (!attr_set) { cudaFuncSetAttribute(filter1d_bytecode<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FilterBytecodeEval<T>::SMEM); attr_set = true; }
        return sgk_launch_pdl(filter1d_bytecode<T>, geom.grid, BLOCK + 32, FilterBytecodeEval<T>::SMEM, s, g, a);
    }
    switch (geom.vm_cfg) {
        case 2: return launch_pass1d_bytecode<T, 2>(g, a, geom.grid, s);
        case 1: return launch_pass1d_bytecode<T, 1>(g, a, geom.grid, s);
        default: return launch_pass1d_bytecode<T, 0>(g, a, geom.grid, s);
    }
}
template <class T, int CFG> int occupancy_pass1d(size_t smem) {
    constexpr int VB = vm_config(CFG).threads, C = vm_config(CFG).cells;
    int occ = 0;
    cudaFuncSetAttribute(pass1d_bytecode<T, VB, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)VM_MAX_FILE_BYTES);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pass1d_bytecode<T, VB, C>, VB, smem) != cudaSuccess || occ <= 0) { cudaGetLastError(); return 1; }
    return occ;
}
// blocks per SM of the bytecode kernels (the 1-D pass depends on the size of its register file: one query per size and configuration)
template <class T> int occupancy_bytecode_t(bool filter, int file_kib, int cfg) {
    static int cached_filter_dev[SG_MAX_DEVICES] = {}, cached_dev[SG_MAX_DEVICES][VM_NCFG][128] = {};
    const int slot = current_device_slot();
    if (filter) {
        int& cached_filter = cached_filter_dev[slot];
        if (cached_filter > 0) return cached_filter;
        int occ = 0;
        cudaFuncSetAttribute(filter1d_bytecode<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FilterBytecodeEval<T>::SMEM);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, filter1d_bytecode<T>, BLOCK + 32, FilterBytecodeEval<T>::SMEM) != cudaSuccess || occ <= 0) { cudaGetLastError(); return 1; }
        return cached_filter = occ;
    }
    cfg = std::min(std::max(cfg, 0), VM_NCFG - 1);
    file_kib = std::min(std::max(file_kib, 1), 127);
    int& cached = cached_dev[slot][cfg][file_kib];
    if (cached > 0) return cached;
    const size_t smem = (size_t)file_kib * 1024;
    switch (cfg) {
        case 2: return cached = occupancy_pass1d<T, 2>(smem);
        case 1: return cached = occupancy_pass1d<T, 1>(smem);
        default: return cached = occupancy_pass1d<T, 0>(smem);
    }
}
}  // namespace

#define SG_CAT2(a, b) a##b
#define SG_CAT(a, b) SG_CAT2(a, b)
cudaError_t SG_CAT(sgk_launch_bytecode_, SG_VM_DTYPE)(const SgProg& g, const SgArgs& a, const SgGeom& geom, cudaStream_t s) {
    return launch_bytecode_t<sgk::TypeOf<SG_VM_DTYPE>::type>(g, a, geom, s);
}
int SG_CAT(sgk_occupancy_bytecode_, SG_VM_DTYPE)(bool filter, int file_kib, int cfg) {
    return occupancy_bytecode_t<sgk::TypeOf<SG_VM_DTYPE>::type>(filter, file_kib, cfg);
}
