// sg_kernels.h — host-side interface between the plan builder (sg_runtime.cpp) and the kernels (sg_kernels.cu).
#ifndef SG_KERNELS_H_
#define SG_KERNELS_H_

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "sg_prog.h"

struct SgGeom {
    int template_id;        // 0 = bytecode kernel, k > 0 = template instance k
    int grid;               // blocks
    int tile;               // elements per tile of the chosen kernel (1-D / filter), strip width (2-D)
    size_t ws_bytes;        // workspace bytes this launch needs (partial cells)
    size_t state_words;     // filter: tile-state words needed
    int ctrl_words;         // control words needed beyond the first 8 (2-D tickets)
    int vm_cfg;             // bytecode 1-D pass: configuration index (threads per block, cells per register: vm_config in sg_pass1d_vm.cuh)
};

// Registry of precompiled template instances (sg_templates_gen.inc).
int sgk_template_count();
const char* sgk_template_name(int id);              // 1-based
const SgProg* sgk_template_prog(int id);
int sgk_find_template(const SgProg& prog);          // 0 if none

// Chooses the kernel (template instance unless force_bytecode / misaligned operands) and fills the geometry
// fields of `args` (head, n_full_tiles, vec_ok, strips/chunks, ws_off).  sm_count/has_device: plan-only contexts
// pass has_device = 0 and nothing touches CUDA.  Returns 0 or an sg_status error (message in err).
int sgk_plan(const SgProg& prog, SgArgs& args, int force_bytecode, int sm_count, int has_device, SgGeom* geom, char* err, size_t errcap);

cudaError_t sgk_launch(const SgProg& prog, const SgArgs& args, const SgGeom& geom, cudaStream_t stream);

// sg_transpose.cu: out[c][r] = in[r][c] for a rows x cols row-major matrix of 4- or 8-byte elements (device pointers).
cudaError_t sgk_transpose(const void* in, int64_t ld_in, int64_t rows, int64_t cols, void* out, int64_t ld_out, int elem_size, cudaStream_t stream);

// sg_ge.cu: steps [k0, k1) of Listing 5's determinant loop on the n x n row-major F64 matrix M as one persistent cooperative
// kernel (device pointers; det / minpiv: one double each; ready: one zeroed 32-bit word).  *launched_grid: the grid used.
cudaError_t sgk_ge_loop(double* M, int64_t n, int64_t ld, double* det, double* minpiv, double eps, int64_t k0, int64_t k1, unsigned int* ready, int sm_count,
                        cudaStream_t stream, int* launched_grid);

// sg_sort.cu: Listing 3's quicksort, one recursion level per launch over a device-side segment table (DT_* dtype; device pointers;
// workspace of sgk_quicksort_workspace_bytes; host_flag: 8 pinned 32-bit words).  *error bit 0: a key matched none of <, =, > (NaN).
size_t sgk_quicksort_workspace_bytes(int64_t n, int elem_size);
cudaError_t sgk_quicksort(int dtype, const void* in, void* out, int64_t n, void* workspace, int sm_count, unsigned int* host_flag, cudaStream_t stream,
                          int* launches, unsigned int* error);

#endif  // SG_KERNELS_H_
