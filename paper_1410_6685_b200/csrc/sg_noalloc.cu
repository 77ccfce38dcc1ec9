// sg_noalloc.cu — sg_vec_sum_noalloc: the `sum` reduction for callers that may not allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  No context, no cudaMalloc / cudaFree,
// no allocating library call: the scratch memory a reduction needs (partials + the last-block ticket) is a file-scope
// `static __device__` array of SG_NOALLOC_SCRATCH_BYTES, held by every GPU that loads the library until the process exits.
//
// The kernel is a variant of the 1-D pass's reduction (sg_pass1d.cuh): the same accumulator cells (fp64: double-double TwoSum,
// fp32: fp64 running sum), the same block reduction and last-block ticket, but ONE PARTIAL PER TILE instead of one per block, so
//   * the scratch bounds the input: n <= SG_NOALLOC_MAX_N elements (one 16-byte cell per NA_TILE elements);
//   * the result does not depend on the grid: partials are combined in tile order by the last block to finish.
//
// The array's name is a host-side stand-in in host code, not a device address: the address the kernel gets comes from
// cudaGetSymbolAddress, asked once per device with that device current (scratch_of below).
//
// Every call shares the array.  Partials are overwritten before they are read; the ticket word must start at zero and is
// cleared on the caller's stream before each launch (a call that was aborted cannot poison the next).  Calls that OVERLAP on the
// GPU (two streams, two host threads) race on it: serialise them on one stream or with events.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/sg.h"
#include "sg_pass1d.cuh"

namespace {

using namespace sgk;

constexpr int NA_THREADS = 256;
constexpr int NA_TILE = 8192;                                       // elements per tile = per partial cell
constexpr int64_t NA_MAX_TILES = SG_NOALLOC_MAX_N / NA_TILE;        // 16384
constexpr size_t NA_HEADER = 256;                                   // [0]: ticket
static_assert(SG_NOALLOC_MAX_N % NA_TILE == 0, "whole tiles");
static_assert(SG_NOALLOC_SCRATCH_BYTES == NA_HEADER + NA_MAX_TILES * sizeof(Cell), "sg.h states the size of the scratch array");
constexpr int NA_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char sg_noalloc_scratch[SG_NOALLOC_SCRATCH_BYTES];

template <class T>
__global__ void __launch_bounds__(NA_THREADS) sum_noalloc(const T* __restrict__ x, int64_t n, int64_t n_tiles, unsigned char* scratch, double* out) {
    __shared__ Cell s_red[32];
    __shared__ unsigned int s_last;
    typedef typename Traits<T>::vec VEC;
    constexpr int V = Traits<T>::V;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    Cell* partial = reinterpret_cast<Cell*>(scratch + NA_HEADER);
    const uint8_t kind[1] = {OUT_SUM};
    const bool vec = (reinterpret_cast<uintptr_t>(x) % 16) == 0;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        Cell acc[1] = {cell_identity<T>(OUT_SUM)};
        const int64_t base = tile * NA_TILE;
        if (vec && base + NA_TILE <= n) {
            const VEC* src = reinterpret_cast<const VEC*>(x + base);
#pragma unroll
            for (int u = 0; u < NA_TILE / (NA_THREADS * V); ++u) {
                VEC q = ld_stream(src + u * NA_THREADS + threadIdx.x);
                const T* qe = reinterpret_cast<const T*>(&q);
#pragma unroll
                for (int e = 0; e < V; ++e) cell_accum_value<T>(OUT_SUM, acc[0], qe[e]);
            }
        } else {
            const int64_t end = (base + NA_TILE < n) ? base + NA_TILE : n;
            for (int64_t i = base + threadIdx.x; i < end; i += NA_THREADS) cell_accum_value<T>(OUT_SUM, acc[0], x[i]);
        }
        block_reduce_cells<T, 1>(acc, kind, s_red);
        if (threadIdx.x == 0) partial[tile] = acc[0];
    }
    if (threadIdx.x == 0) {
        unsigned int t;     // release: this block's partials are visible to whoever observes the increment
        asm volatile("atom.add.release.gpu.global.u32 %0, [%1], 1;" : "=r"(t) : "l"(ticket) : "memory");
        s_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();        // acquire side: the other blocks' partials
    Cell acc[1] = {cell_identity<T>(OUT_SUM)};
    for (int64_t t = threadIdx.x; t < n_tiles; t += NA_THREADS) {
        Cell other;
        const unsigned long long* src = reinterpret_cast<const unsigned long long*>(&partial[t]);
        other.a = __ldcg(src); other.b = __ldcg(src + 1);
        cell_combine<T>(OUT_SUM, acc[0], other);
    }
    block_reduce_cells<T, 1>(acc, kind, s_red);
    if (threadIdx.x == 0) {
        *out = __longlong_as_double((long long)cell_final<T>(OUT_SUM, acc[0]));
        *ticket = 0;
    }
}

int na_fail(char* err, int64_t cap, int code, const char* msg) {
    if (err && cap > 0) snprintf(err, (size_t)cap, "%s", msg);
    return code;
}

// device address of this device's copy of the scratch array and its SM count; asked once per device, with that device current
struct NaDevice { unsigned char* scratch = nullptr; int sm_count = 0; };
cudaError_t scratch_of(int device, NaDevice* out) {
    static std::mutex mu;
    static NaDevice dev[NA_MAX_DEVICES];
    std::lock_guard<std::mutex> lock(mu);
    if (!dev[device].scratch) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, sg_noalloc_scratch);
        if (e != cudaSuccess) return e;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess) return e;
        dev[device].sm_count = sms;
        dev[device].scratch = static_cast<unsigned char*>(p);
    }
    *out = dev[device];
    return cudaSuccess;
}

}  // namespace

extern "C" sg_status sg_vec_sum_noalloc(int32_t device, void* stream, sg_dtype dtype, const void* dev_x, int64_t n, double* dev_out, char* err, int64_t errcap) {
    if (err && errcap > 0) err[0] = 0;
    if (device < 0 || device >= NA_MAX_DEVICES) return (sg_status)na_fail(err, errcap, SG_ERR_ARG, "sg_vec_sum_noalloc: device index out of range");
    if (n < 0 || !dev_out || (n > 0 && !dev_x)) return (sg_status)na_fail(err, errcap, SG_ERR_ARG, "sg_vec_sum_noalloc: null pointer or negative count");
    if (dtype != SG_F32 && dtype != SG_F64) return (sg_status)na_fail(err, errcap, SG_ERR_DTYPE, "sg_vec_sum_noalloc: SG_F32 or SG_F64 only");
    if (n > SG_NOALLOC_MAX_N) {
        char msg[192];
        snprintf(msg, sizeof msg, "sg_vec_sum_noalloc: %lld elements exceed SG_NOALLOC_MAX_N = %lld (the static scratch array holds one partial per %d elements)",
                 (long long)n, (long long)SG_NOALLOC_MAX_N, NA_TILE);
        return (sg_status)na_fail(err, errcap, SG_ERR_CAPACITY, msg);
    }
    const size_t es = dtype == SG_F32 ? 4 : 8;
    if (n > 0 && (reinterpret_cast<uintptr_t>(dev_x) % es) != 0) return (sg_status)na_fail(err, errcap, SG_ERR_ARG, "sg_vec_sum_noalloc: dev_x is not aligned to its element size");
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); return (sg_status)na_fail(err, errcap, SG_ERR_CUDA, "sg_vec_sum_noalloc: no usable CUDA device (there is no CPU fallback)"); }
    if (prev != device && cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return (sg_status)na_fail(err, errcap, SG_ERR_CUDA, "sg_vec_sum_noalloc: cudaSetDevice failed"); }
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    NaDevice d;
    cudaError_t e = scratch_of(device, &d);
    if (e == cudaSuccess) e = cudaMemsetAsync(d.scratch, 0, NA_HEADER, s);          // the ticket starts at zero
    if (e == cudaSuccess) {
        const int64_t n_tiles = (n + NA_TILE - 1) / NA_TILE;
        int64_t grid = (int64_t)d.sm_count * 8;
        if (grid > n_tiles) grid = n_tiles;
        if (grid < 1) grid = 1;                                                     // n = 0: one block writes the empty sum, +0.0
        if (dtype == SG_F32) sum_noalloc<float><<<(unsigned)grid, NA_THREADS, 0, s>>>(static_cast<const float*>(dev_x), n, n_tiles, d.scratch, dev_out);
        else sum_noalloc<double><<<(unsigned)grid, NA_THREADS, 0, s>>>(static_cast<const double*>(dev_x), n, n_tiles, d.scratch, dev_out);
        e = cudaGetLastError();
    }
    if (prev != device) cudaSetDevice(prev);
    if (e != cudaSuccess) {
        char msg[192];
        snprintf(msg, sizeof msg, "sg_vec_sum_noalloc: %s", cudaGetErrorString(e));
        return (sg_status)na_fail(err, errcap, SG_ERR_CUDA, msg);
    }
    return SG_OK;
}
