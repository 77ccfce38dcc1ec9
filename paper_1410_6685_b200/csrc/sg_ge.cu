// sg_ge.cu — Listing 5's whole determinant loop as ONE persistent cooperative kernel.
//
// The paper issues one kernel per row and step and names exactly that as the reason for its one slow benchmark ("loops, which
// have the effect of additional kernel launches").  Here the host launches once; the n steps run on the device:
//
//   * Rows are owned cyclically: row j belongs to block j mod G for the whole loop, so the step-k update of a row always follows
//     its step-(k-1) update in program order of ONE block.  The only dependence between blocks is the pivot row: step k needs
//     row k in its final state (all updates of steps < k applied).
//   * That dependence is one monotonic counter `ready` (rows 0 .. ready-1 are final).  The owner of row k+1 updates it FIRST in
//     step k and publishes ready = k+2 (release) before it touches its other rows; every block acquires ready >= k+1 before
//     step k.  No grid-wide barrier: blocks drift apart by as much as the data dependences allow, and the chain
//     "update row k+1 -> publish -> next owner" costs one row, not one step.
//   * Per step a block reads the pivot row once into shared memory (L2 hit: it was written a moment ago), then streams its
//     own rows ONE AT A TIME, GE_CH 128-bit vectors per thread in flight along the row (16 bytes read + 16 written per vector).  The factors f_j = M[j,k] / M[k,k]
//     of all the block's rows are computed BEFORE any of those rows is modified (the row's own column k is overwritten by
//     the update).
//   * Arithmetic is BASELINE.json:configs[4]'s update, one rounding per primitive: t = f_j * M[k,c]; M[j,c] = M[j,c] - t over
//     ALL columns c (R11), so the result is bit-identical to n applications of the matrix pass and to the oracle.
//   * The listing's control flow is evaluated on the device: Result := Result * pivot BEFORE the approximately-zero test
//     (PAPER.md:338-339); a pivot with |pivot| <= eps ends the loop for every block at the same step (they all read the same final
//     M[k,k]); a row whose entry below the pivot is approximately zero is left as it is.
//
// Launched with cudaLaunchCooperativeKernel: every block must be resident, because blocks wait on one another's rows.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sg_kernels.h"

namespace {

constexpr int GE_THREADS = 512;
// Rows of a block in flight x vectors per row and thread in flight, measured (whole loop, ms at 2048^2 / 4096^2 / 8192^2):
//   4 x 2 (round 2's first version): 15.3 / 90.3 / 761      2 x 4: 15.6 / 85.2 / 740      1 x 8: 13.9 / 83.1 / 736      8 x 1: 16.3 / 95.2 / 776
//   1 x 4: 11.4 / 70.3 / 698      2 x 2: 11.5 / 71.5 / 701      1 x 2: 11.3 / 74.2 / 709      1 x 3: 11.4 / 77.1 / 688      1 x 6: 12.1 / 70.5 / 698
// Streaming several rows (addresses a leading dimension apart) at once and many bytes in flight per thread is what the memory system
// serves worse — the same finding as for the matrix passes (sg_pass2d_tile.cuh).
#ifndef SG_GE_RR
#define SG_GE_RR 1
#endif
#ifndef SG_GE_CH
#define SG_GE_CH 4
#endif
constexpr int GE_RR = SG_GE_RR;     // rows of one block in flight
constexpr int GE_CH = SG_GE_CH;     // 128-bit vectors per row and thread in flight

struct GeArgs {
    double* M;
    int64_t n, ld;
    double* det;                    // one element: Result
    double* minpiv;                 // one element: smallest |pivot| met so far (<= eps: the loop has ended)
    double eps;
    int64_t k0, k1;
    unsigned int* ready;            // zeroed; rows 0 .. k0 + *ready are final
    int max_rows;                   // rows one block can own in one step (size of the factor arrays)
    int panel;                      // columns of the pivot row held in shared memory at a time (a multiple of 2)
};

__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ double2 ldcg2(const double* p) {
    double2 r;
    asm volatile("ld.global.cg.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ void stcg2(double* p, double2 v) { asm volatile("st.global.cg.v2.f64 [%0], {%1,%2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory"); }
__device__ __forceinline__ double ldcg1(const double* p) {
    double r;
    asm volatile("ld.global.cg.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ void stcg1(double* p, double v) { asm volatile("st.global.cg.f64 [%0], %1;" ::"l"(p), "d"(v) : "memory"); }

// rows [first, first + cnt*G) step G of this block, columns [c0, c0 + pc) of the panel in shared memory
template <bool ALIGNED>
__device__ __forceinline__ void update_rows(const GeArgs& a, const double* s_piv, const double* s_f, const unsigned char* s_skip, int64_t first, int cnt, int G,
                                            int idx0, int64_t c0, int pc) {
    for (int r0 = 0; r0 < cnt; r0 += GE_RR) {
        double f[GE_RR];
        bool act[GE_RR];
        double* row[GE_RR];
#pragma unroll
        for (int r = 0; r < GE_RR; ++r) {
            const bool in = r0 + r < cnt;
            act[r] = in && !s_skip[idx0 + r0 + r];
            f[r] = in ? s_f[idx0 + r0 + r] : 0.0;
            row[r] = a.M + (first + (int64_t)(r0 + r) * G) * a.ld + c0;
        }
        if (ALIGNED) {
            const int nv = pc >> 1;         // vectors in the panel
            for (int vb = threadIdx.x; vb < nv; vb += GE_THREADS * GE_CH) {
                double2 m[GE_RR][GE_CH];
#pragma unroll
                for (int r = 0; r < GE_RR; ++r)
#pragma unroll
                    for (int i = 0; i < GE_CH; ++i) {
                        const int v = vb + i * GE_THREADS;
                        if (act[r] && v < nv) m[r][i] = ldcg2(row[r] + 2 * v);
                    }
#pragma unroll
                for (int i = 0; i < GE_CH; ++i) {
                    const int v = vb + i * GE_THREADS;
                    if (v >= nv) continue;
                    const double2 p = *reinterpret_cast<const double2*>(s_piv + 2 * v);
#pragma unroll
                    for (int r = 0; r < GE_RR; ++r) {
                        if (!act[r]) continue;
                        double2 o;
                        o.x = __dsub_rn(m[r][i].x, __dmul_rn(f[r], p.x));
                        o.y = __dsub_rn(m[r][i].y, __dmul_rn(f[r], p.y));
                        stcg2(row[r] + 2 * v, o);
                    }
                }
            }
        } else {
            for (int cb = threadIdx.x; cb < pc; cb += GE_THREADS * GE_CH) {
                double m[GE_RR][GE_CH];
#pragma unroll
                for (int r = 0; r < GE_RR; ++r)
#pragma unroll
                    for (int i = 0; i < GE_CH; ++i) {
                        const int c = cb + i * GE_THREADS;
                        if (act[r] && c < pc) m[r][i] = ldcg1(row[r] + c);
                    }
#pragma unroll
                for (int i = 0; i < GE_CH; ++i) {
                    const int c = cb + i * GE_THREADS;
                    if (c >= pc) continue;
                    const double p = s_piv[c];
#pragma unroll
                    for (int r = 0; r < GE_RR; ++r)
                        if (act[r]) stcg1(row[r] + c, __dsub_rn(m[r][i], __dmul_rn(f[r], p)));
                }
            }
        }
    }
}

template <bool ALIGNED>
__global__ void __launch_bounds__(GE_THREADS, 2) ge_loop(const GeArgs a) {
    extern __shared__ __align__(16) unsigned char ge_smem[];
    double* const s_piv = reinterpret_cast<double*>(ge_smem);                       // [panel]
    double* const s_f = s_piv + a.panel;                                              // [max_rows] factors of this block's rows
    unsigned char* const s_skip = reinterpret_cast<unsigned char*>(s_f + a.max_rows); // [max_rows] row left as it is
    const int G = (int)gridDim.x, b = (int)blockIdx.x;
    const int64_t n = a.n;
    double det = 0.0, minp = 0.0;
    {
        const double m0 = ldcg1(a.minpiv);
        if (m0 <= a.eps) return;            // an approximately-zero pivot was met by an earlier call: the loop has ended (uniform)
        if (b == 0 && threadIdx.x == 0) { det = ldcg1(a.det); minp = m0; }
    }
    for (int64_t k = a.k0; k < a.k1; ++k) {
        // row k is final once `ready` says so (row k0 is final on entry)
        if (threadIdx.x == 0) {
            const unsigned int need = (unsigned int)(k - a.k0);
            while (ld_acquire_u32(a.ready) < need) __nanosleep(64);
        }
        __syncthreads();                    // also: everybody is done with the shared arrays of the previous step
        const double* prow = a.M + k * a.ld;
        const double pivot = ldcg1(prow + k);
        if (b == 0 && threadIdx.x == 0) {
            det = __dmul_rn(det, pivot);                                // Result := Result * pivot
            const double ap = fabs(pivot);
            minp = (ap < minp) ? ap : minp;                             // MIN(minpiv, |pivot|) = (b < a) ? b : a
        }
        if (fabs(pivot) <= a.eps) break;                                // approximately zero: the loop ends, uniform
        if (k + 1 >= n) continue;
        // this block's rows of the step: j = first, first + G, ... < n with j > k and j mod G == b
        const int64_t lo = k + 1;
        const int64_t first = lo + (((int64_t)b - lo) % G + G) % G;
        const int cnt = first < n ? (int)((n - first + G - 1) / G) : 0;
        const bool owns_next = cnt > 0 && first == lo;                  // row k+1 is mine: it is the next pivot row
        // factors of ALL my rows, read before any of them changes
        for (int r = threadIdx.x; r < cnt; r += GE_THREADS) {
            const double pj = ldcg1(a.M + (first + (int64_t)r * G) * a.ld + k);
            s_skip[r] = fabs(pj) <= a.eps;
            s_f[r] = __ddiv_rn(pj, pivot);
        }
        const int n_panels = (int)((n + a.panel - 1) / a.panel);
        // phase 0: the next pivot row alone (all panels), then publish; phase 1: the rest of my rows
        for (int phase = 0; phase < 2; ++phase) {
            const int idx0 = (phase == 0) ? 0 : (owns_next ? 1 : 0);
            const int pcnt = (phase == 0) ? (owns_next ? 1 : 0) : cnt - idx0;
            if (phase == 0 && !owns_next) continue;
            if (pcnt > 0 || (phase == 0))
                for (int p = 0; p < n_panels; ++p) {
                    const int64_t c0 = (int64_t)p * a.panel;
                    const int pc = (int)((n - c0) < a.panel ? (n - c0) : a.panel);
                    // with one panel the pivot row loaded in phase 0 is still there in phase 1
                    if (!(n_panels == 1 && phase == 1 && owns_next)) {
                        __syncthreads();        // nobody reads the previous panel (or writes s_f) any more
                        if (ALIGNED) {
                            for (int v = threadIdx.x; v < (pc >> 1); v += GE_THREADS) *reinterpret_cast<double2*>(s_piv + 2 * v) = ldcg2(prow + c0 + 2 * v);
                        } else {
                            for (int c = threadIdx.x; c < pc; c += GE_THREADS) s_piv[c] = ldcg1(prow + c0 + c);
                        }
                        __syncthreads();
                    }
                    if (pcnt > 0) update_rows<ALIGNED>(a, s_piv, s_f, s_skip, first + (int64_t)idx0 * G, pcnt, G, idx0, c0, pc);
                }
            if (phase == 0) {
                __syncthreads();                // every thread has stored its part of row k+1
                if (threadIdx.x == 0) {
                    __threadfence();
                    st_release_u32(a.ready, (unsigned int)(k + 1 - a.k0));          // rows 0 .. k+1 are final
                }
            }
        }
    }
    if (b == 0 && threadIdx.x == 0) { stcg1(a.det, det); stcg1(a.minpiv, minp); }
}

size_t ge_smem_bytes(int panel, int max_rows) { return (size_t)panel * 8 + (size_t)max_rows * 8 + (((size_t)max_rows + 15) & ~(size_t)15); }

}  // namespace

// Steps [k0, k1) of Listing 5 on the n x n row-major F64 matrix M (device pointers; det / minpiv: one double each; ready: one
// zeroed 32-bit word).  Returns the launch status; *launched_grid receives the grid size (reports).
cudaError_t sgk_ge_loop(double* M, int64_t n, int64_t ld, double* det, double* minpiv, double eps, int64_t k0, int64_t k1, unsigned int* ready, int sm_count,
                        cudaStream_t stream, int* launched_grid) {
    if (k1 <= k0) return cudaSuccess;
    const bool aligned = (((uintptr_t)M) % 16 == 0) && (ld % 2 == 0) && (n % 2 == 0);
    GeArgs a{};
    a.M = M; a.n = n; a.ld = ld; a.det = det; a.minpiv = minpiv; a.eps = eps; a.k0 = k0; a.k1 = k1; a.ready = ready;
    int max_smem = 0, dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    // whole pivot row in shared memory when two blocks per SM still fit, else panels of 8192 columns (64 KiB)
    const int64_t want_cols = (n + 1) & ~(int64_t)1;
    a.panel = (int)((want_cols * 8 <= 96 * 1024) ? want_cols : 8192);
    if (a.panel < 2) a.panel = 2;
    const void* fn = aligned ? (const void*)ge_loop<true> : (const void*)ge_loop<false>;
    // grid: every block must be resident (blocks wait on one another); rows per block follow from the grid
    int occ = 0, grid = sm_count;
    for (int iter = 0; iter < 3; ++iter) {
        a.max_rows = (int)((n + grid - 1) / grid) + 1;
        const size_t smem = ge_smem_bytes(a.panel, a.max_rows);
        if ((int)smem > max_smem) return cudaErrorInvalidValue;
        cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, GE_THREADS, smem);
        if (e != cudaSuccess) return e;
        if (occ < 1) return cudaErrorLaunchOutOfResources;
        const int g2 = sm_count * (occ > 2 ? 2 : occ);
        if (g2 == grid) break;
        grid = g2;
    }
    a.max_rows = (int)((n + grid - 1) / grid) + 1;
    const size_t smem = ge_smem_bytes(a.panel, a.max_rows);
    cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (launched_grid) *launched_grid = grid;
    void* params[] = {&a};
    return cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(GE_THREADS), params, smem, stream);
}
