// sg_bulk.cuh — bulk asynchronous copies (the TMA engine's 1-D form, cp.async.bulk) and mbarrier helpers.
// Streaming kernels whose loads cannot all be kept in flight from registers stage their tiles through a ring of
// shared-memory buffers: one elected thread issues the copies several stages ahead, completion is signalled by
// transaction bytes on an mbarrier, every thread then reads its elements from shared memory.
// Requirements of cp.async.bulk: source, destination and size are multiples of 16 bytes.
#ifndef SG_BULK_CUH_
#define SG_BULK_CUH_

#include <cuda_runtime.h>
#include <stdint.h>

namespace sgk {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}
// explicit shared-window accesses (32-bit shared address + byte offset): no generic-address translation per access
template <class T> __device__ __forceinline__ void sts_elem(uint32_t base, uint32_t idx, T v) {
    if constexpr (sizeof(T) == 4) {
        uint32_t w; memcpy(&w, &v, 4);
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(base + idx * 4u), "r"(w) : "memory");
    } else {
        unsigned long long w; memcpy(&w, &v, 8);
        asm volatile("st.shared.b64 [%0], %1;" ::"r"(base + idx * 8u), "l"(w) : "memory");
    }
}
template <class T> __device__ __forceinline__ T lds_elem(uint32_t base, uint32_t idx) {
    T v;
    if constexpr (sizeof(T) == 4) {
        uint32_t w;
        asm volatile("ld.shared.b32 %0, [%1];" : "=r"(w) : "r"(base + idx * 4u) : "memory");
        memcpy(&v, &w, 4);
    } else {
        unsigned long long w;
        asm volatile("ld.shared.b64 %0, [%1];" : "=l"(w) : "r"(base + idx * 8u) : "memory");
        memcpy(&v, &w, 8);
    }
    return v;
}
// compaction append: if bit BIT of `mask` is set, store v at shared-window byte address `addr` and advance it —
// a predicate-producing logic op, a predicated store and a predicated add (no branch)
template <class T, int BIT> __device__ __forceinline__ void sts_append_if(uint32_t& addr, unsigned int mask, T v) {
    if constexpr (sizeof(T) == 4) {
        uint32_t w; memcpy(&w, &v, 4);
        asm volatile("{\n.reg .pred p;\n.reg .b32 t;\nand.b32 t, %2, %3;\nsetp.ne.u32 p, t, 0;\n@p st.shared.b32 [%0], %1;\n@p add.u32 %0, %0, 4;\n}\n"
                     : "+r"(addr) : "r"(w), "r"(mask), "n"(1u << BIT) : "memory");
    } else {
        unsigned long long w; memcpy(&w, &v, 8);
        asm volatile("{\n.reg .pred p;\n.reg .b32 t;\nand.b32 t, %2, %3;\nsetp.ne.u32 p, t, 0;\n@p st.shared.b64 [%0], %1;\n@p add.u32 %0, %0, 8;\n}\n"
                     : "+r"(addr) : "l"(w), "r"(mask), "n"(1u << BIT) : "memory");
    }
}
// a value the compiler must keep in a register (it will not re-derive it at every use)
__device__ __forceinline__ uint32_t pin_reg(uint32_t x) {
    asm volatile("mov.b32 %0, %0;" : "+r"(x));
    return x;
}
// non-blocking: has the phase with this parity completed?
__device__ __forceinline__ bool mbar_test(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// named barrier over the first `nthreads` threads' warps (barrier 0 is __syncthreads)
template <int ID, int NTHREADS> __device__ __forceinline__ void named_bar_sync() {
    asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NTHREADS) : "memory");
}
// global -> shared bulk copy; completion adds `bytes` transaction bytes to `bar`
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)), "l"(gmem_src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// TMA tensor copy global -> shared of one box of a 2-D tensor map (128 bytes in parameter/constant/global memory,
// 64-byte aligned): coordinates (c0 = innermost, c1); completion adds the box's bytes to `bar`
__device__ __forceinline__ void tma_load_2d(uint32_t smem_dst, const void* tmap, int c0, int c1, uint64_t* bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_dst), "l"(tmap),
                 "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}
// generic-proxy accesses to shared memory are ordered before later async-proxy (bulk copy) accesses
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace sgk
#endif  // SG_BULK_CUH_
