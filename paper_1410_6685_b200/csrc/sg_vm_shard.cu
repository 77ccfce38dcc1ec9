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

template <class T, int C> cudaError_t launch_pass1d_bytecode(const SgProg& g, const SgArgs& a, int grid, cudaStream_t s) {
    static bool attr_dev[SG_MAX_DEVICES] = {};
    bool& attr_set = attr_dev[current_device_slot()];
    if (!attr_set) { cudaFuncSetAttribute(pass1d_bytecode<T, C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)vm_file_bytes(VM_VREG, 1)); attr_set = true; }
    return sgk_launch_pdl(pass1d_bytecode<T, C>, grid, BLOCK, vm_file_bytes(g.shape.n_vreg, C), s, g, a);
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
    return geom.vm_cells == 2 ? launch_pass1d_bytecode<T, 2>(g, a, geom.grid, s) : launch_pass1d_bytecode<T, 1>(g, a, geom.grid, s);
}
// blocks per SM of the bytecode kernels (the 1-D pass depends on the size of its register file: queried once per size)
template <class T> int occupancy_bytecode_t(bool filter, int n_vreg, int cells) {
    static int cached_filter_dev[SG_MAX_DEVICES] = {}, cached_dev[SG_MAX_DEVICES][VM_VREG + 1][VM_MAX_CELLS + 1] = {};
    const int slot = current_device_slot();
    int& cached_filter = cached_filter_dev[slot];
    int (&cached)[VM_VREG + 1][VM_MAX_CELLS + 1] = cached_dev[slot];
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
}  // namespace

#define SG_CAT2(a, b) a##b
#define SG_CAT(a, b) SG_CAT2(a, b)
cudaError_t SG_CAT(sgk_launch_bytecode_, SG_VM_DTYPE)(const SgProg& g, const SgArgs& a, const SgGeom& geom, cudaStream_t s) {
    return launch_bytecode_t<sgk::TypeOf<SG_VM_DTYPE>::type>(g, a, geom, s);
}
int SG_CAT(sgk_occupancy_bytecode_, SG_VM_DTYPE)(bool filter, int n_vreg, int cells) {
    return occupancy_bytecode_t<sgk::TypeOf<SG_VM_DTYPE>::type>(filter, n_vreg, cells);
}
