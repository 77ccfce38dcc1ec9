// sg_sort.cu — Listing 3's quicksort on the device, one recursion LEVEL per launch.
//
// The listing's body is: pivot := a[a.count // 2]; left / mid / right := the three stable filters `item < / = / > pivot`;
// Result := quicksort(left) ++ mid ++ quicksort(right).  All partitions of one recursion depth are disjoint segments of one
// buffer, so a level is ONE launch over a device-side segment table; counts never visit the host.
//
// The multi-output partition: a tile of a segment is read ONCE, the three predicates are evaluated against the segment's
// device-resident pivot, and the three stable compactions are written in the same pass:
//     left   -> next-level buffer at  start + rank_<            (forward, stable)
//     right  -> next-level buffer at  start + count - 1 - rank_>  (from the END of the segment's span, i.e. stored in REVERSE
//               logical order: `>` needs no count of its own — rank_> = index - rank_< - rank_=; the child segment carries a
//               `reversed` flag and is read back to front, so its logical order is the stable one)
//     mid    -> staging buffer at      start + rank_=            (its final place start + |left| + rank_= needs |left|, known only
//               when the segment's last tile has resolved; one copy job per segment moves it at the next launch)
// Ranks across the tiles of a segment come from ONE decoupled look-back chain over packed (count_<, count_=) tile states.
// left and right occupy the parent's own span [start, start + count): offsets in the scratch buffers ARE final offsets in the
// result, `concatenate` costs nothing.
//
// A segment of at most QS_SMALL elements is finished by one block in shared memory with the same level-wise algorithm (the
// listing's recursion down to a.count = 1, every sub-segment of a level partitioned at once by a segmented scan) and written
// to its final place in the result.
//
// An element that is neither <, = nor > the pivot (a NaN key, or any key against a NaN pivot) belongs to none of the listing's
// three filters: the listing would drop it and violate its own postcondition Result.count = a.count.  The kernels flag that
// case; the entry point reports SG_ERR_CONTRACT.
#include <cuda_runtime.h>
#include <stdint.h>

#include "sg_kernels.h"

namespace {

constexpr int QS_THREADS = 256, QS_EPT = 8, QS_TILE = QS_THREADS * QS_EPT;      // 2048 elements per tile
constexpr int QS_SMALL = QS_TILE;                                               // segments up to this size are sorted by one block
constexpr unsigned long long QS_AGG = 1ull << 62, QS_INC = 2ull << 62, QS_FLAGS = 3ull << 62, QS_CNT = (1ull << 31) - 1;

enum : unsigned int { QS_KIND_SEG = 0, QS_KIND_MIDCOPY = 1 };

struct QsSeg {
    long long start;            // offset of the segment's span (source buffer, next-level buffer and result alike); MIDCOPY: offset in the staging buffer
    long long count;
    long long aux;              // MIDCOPY: destination offset in the result
    unsigned int kind_rev;      // bit 0: stored in reverse logical order; bits 1..: kind
    unsigned int tile_base;     // first work id of the segment's tiles
};
struct QsLevel { unsigned int ticket, n_work, n_segs, pad; };

struct QsCtl {                  // device-resident control block
    QsLevel lvl[3];             // rotating: level L uses lvl[L % 3], appends to lvl[(L+1) % 3], clears lvl[(L+2) % 3]
    unsigned int error;         // bit 0: an element matched none of <, =, > (NaN)
    unsigned int pad[3];
};

template <class T> struct QsArgs {
    const T* src;               // this level's keys (level 0: the caller's input)
    T* dst;                     // next level's keys
    T* out;                     // the result
    T* mid;                     // staging of this level's `=` runs
    const T* mid_prev;          // staging written by the previous level (read by this level's copy jobs; the two alternate, so a
                                // child's `=` run never lands on its parent's before that has been copied)
    const QsSeg* segs;          // this level's table
    const unsigned int* work;   // work id -> segment index
    QsSeg* next_segs;
    unsigned int* next_work;
    unsigned long long* state;      // tile states of this level (zeroed)
    unsigned long long* state_next; // cleared for the next level
    QsCtl* ctl;
    int level;
    unsigned int cap_segs, cap_work;
};

__device__ __forceinline__ unsigned long long qs_ld_state(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ void qs_st_state(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long qs_pack(unsigned long long flag, unsigned long long lt, unsigned long long eq) { return flag | (lt << 31) | eq; }

// exclusive block scan of a packed pair of small counts (each total < 2^16); returns the exclusive prefix, *total = block total
__device__ __forceinline__ unsigned int qs_block_scan(unsigned int x, unsigned int* s_warp, unsigned int* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    unsigned int incl = x;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned int wex = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < QS_THREADS / 32; ++w) {
        const unsigned int t = s_warp[w];
        if (w < warp) wex += t;
        tot += t;
    }
    __syncthreads();            // s_warp may be reused by the caller
    *total = tot;
    return wex + incl - x;
}

// append a segment (or a copy job) to the next level and give it its work ids; called by every thread of the block
template <class T>
__device__ __forceinline__ void qs_append(const QsArgs<T>& a, QsLevel* nxt, long long start, long long count, long long aux, unsigned int kind, unsigned int rev,
                                          unsigned int* s_tmp) {
    if (count <= 0) return;
    const unsigned int ntiles = (kind == QS_KIND_SEG && count <= QS_SMALL) ? 1u : (unsigned int)((count + QS_TILE - 1) / QS_TILE);
    if (threadIdx.x == 0) {
        const unsigned int idx = atomicAdd(&nxt->n_segs, 1u);
        const unsigned int base = atomicAdd(&nxt->n_work, ntiles);
        if (idx < a.cap_segs && base + ntiles <= a.cap_work) {
            QsSeg s;
            s.start = start; s.count = count; s.aux = aux; s.kind_rev = (kind << 1) | rev; s.tile_base = base;
            a.next_segs[idx] = s;
        } else atomicOr(&a.ctl->error, 2u);     // cannot happen with the capacities of sgk_quicksort (kept as a guard)
        s_tmp[0] = idx; s_tmp[1] = base;
    }
    __syncthreads();
    const unsigned int idx = s_tmp[0], base = s_tmp[1];
    if (idx < a.cap_segs && base + ntiles <= a.cap_work)
        for (unsigned int i = threadIdx.x; i < ntiles; i += QS_THREADS) a.next_work[base + i] = idx;
    __syncthreads();
}

template <class T> __device__ __forceinline__ long long qs_phys(const QsSeg& s, long long i) { return (s.kind_rev & 1u) ? s.start + s.count - 1 - i : s.start + i; }

// ---- a segment of at most QS_SMALL elements: the listing's recursion level by level in shared memory ---------------------------
template <class T>
__device__ __forceinline__ void qs_sort_small(const QsArgs<T>& a, const QsSeg& seg, unsigned char* smem, unsigned int* s_warp) {
    T* val[2] = {reinterpret_cast<T*>(smem), reinterpret_cast<T*>(smem) + QS_SMALL};
    unsigned short* head[2] = {reinterpret_cast<unsigned short*>(val[1] + QS_SMALL), reinterpret_cast<unsigned short*>(val[1] + QS_SMALL) + QS_SMALL};
    unsigned short* len[2] = {head[1] + QS_SMALL, head[1] + 2 * QS_SMALL};
    unsigned int* scan = reinterpret_cast<unsigned int*>(len[1] + QS_SMALL);        // inclusive packed (lt | eq << 16) counts
    const int cnt = (int)seg.count;
    for (int i = threadIdx.x; i < QS_SMALL; i += QS_THREADS) {
        if (i < cnt) val[0][i] = a.src[qs_phys<T>(seg, i)];
        head[0][i] = 0;
        len[0][i] = (unsigned short)(i < cnt ? cnt : 1);
    }
    __syncthreads();
    int cur = 0;
    bool bad = false;
    for (;;) {
        // classify this thread's QS_EPT consecutive elements against the pivot of their sub-segment
        const int i0 = threadIdx.x * QS_EPT;
        unsigned int cls[QS_EPT];       // 0 inactive, 1 lt, 2 eq, 3 gt, 4 none
        unsigned int mine = 0;
#pragma unroll
        for (int e = 0; e < QS_EPT; ++e) {
            const int i = i0 + e;
            const int h = head[cur][i], l = len[cur][i];
            cls[e] = 0;
            if (i < cnt && l > 1) {
                const T x = val[cur][i], p = val[cur][h + l / 2];          // pivot := a[a.count // 2]
                cls[e] = (x < p) ? 1u : (x == p) ? 2u : (x > p) ? 3u : 4u;
            }
            mine += (cls[e] == 1u) + ((cls[e] == 2u) << 16);
        }
        unsigned int tot;
        unsigned int run = qs_block_scan(mine, s_warp, &tot);
#pragma unroll
        for (int e = 0; e < QS_EPT; ++e) {
            run += (cls[e] == 1u) + ((cls[e] == 2u) << 16);
            scan[i0 + e] = run;
        }
        __syncthreads();
        bool more = false;
        const int nxt = cur ^ 1;
#pragma unroll
        for (int e = 0; e < QS_EPT; ++e) {
            const int i = i0 + e;
            if (i >= cnt) continue;
            const int h = head[cur][i], l = len[cur][i];
            int pos = i, nh = h, nl_ = l;
            if (cls[e] != 0) {
                const unsigned int base = h > 0 ? scan[h - 1] : 0u, incl = scan[i], segtot = scan[h + l - 1] - base;
                const int n_lt = (int)(segtot & 0xffffu), n_eq = (int)(segtot >> 16);
                const unsigned int own = (cls[e] == 1u) + ((cls[e] == 2u) << 16);
                const unsigned int ex = incl - own - base;
                const int r_lt = (int)(ex & 0xffffu), r_eq = (int)(ex >> 16);
                if (cls[e] == 1u) { pos = h + r_lt; nh = h; nl_ = n_lt; }
                else if (cls[e] == 2u) { pos = h + n_lt + r_eq; nh = pos; nl_ = 1; }
                else {
                    pos = h + n_lt + n_eq + ((i - h) - r_lt - r_eq);
                    nh = h + n_lt + n_eq; nl_ = l - n_lt - n_eq;
                    if (cls[e] == 4u) { bad = true; nl_ = 1; nh = pos; }
                }
            }
            val[nxt][pos] = val[cur][i];
            head[nxt][pos] = (unsigned short)nh;
            len[nxt][pos] = (unsigned short)nl_;
            more |= nl_ > 1;
        }
        cur = nxt;
        const int any_bad = __syncthreads_or(bad);
        if (any_bad) {
            if (threadIdx.x == 0) atomicOr(&a.ctl->error, 1u);
            break;
        }
        if (!__syncthreads_or(more)) break;
    }
    for (int i = threadIdx.x; i < cnt; i += QS_THREADS) a.out[seg.start + i] = val[cur][i];
    __syncthreads();
}

// ---- one tile of a big segment: three stable compactions in one read -----------------------------------------------------------
template <class T>
__device__ __forceinline__ void qs_partition_tile(const QsArgs<T>& a, const QsSeg& seg, unsigned int id, QsLevel* nxt, unsigned int* s_warp, unsigned long long* s_excl) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned int t = id - seg.tile_base;
    const long long n_tiles = (seg.count + QS_TILE - 1) / QS_TILE;
    const T pivot = a.src[qs_phys<T>(seg, seg.count / 2)];             // pivot := a[a.count // 2], device-resident
    const long long i0 = (long long)t * QS_TILE + (long long)threadIdx.x * QS_EPT;      // logical index of this thread's first element
    T x[QS_EPT];
    unsigned int cls[QS_EPT];
    unsigned int mine = 0;
    bool bad = false;
#pragma unroll
    for (int e = 0; e < QS_EPT; ++e) {
        const long long i = i0 + e;
        cls[e] = 0;
        if (i < seg.count) {
            x[e] = a.src[qs_phys<T>(seg, i)];
            cls[e] = (x[e] < pivot) ? 1u : (x[e] == pivot) ? 2u : (x[e] > pivot) ? 3u : 4u;
            bad |= cls[e] == 4u;
        }
        mine += (cls[e] == 1u) + ((cls[e] == 2u) << 16);
    }
    unsigned int tot;
    const unsigned int ex = qs_block_scan(mine, s_warp, &tot);
    const unsigned long long t_lt = tot & 0xffffu, t_eq = tot >> 16;
    // decoupled look-back over the earlier tiles of THIS segment (work ids tile_base .. id-1)
    if (warp == 0) {
        unsigned long long e_lt = 0, e_eq = 0;
        if (t == 0) {
            if (lane == 0) qs_st_state(&a.state[id], qs_pack(QS_INC, t_lt, t_eq));
        } else {
            if (lane == 0) qs_st_state(&a.state[id], qs_pack(QS_AGG, t_lt, t_eq));
            long long look = (long long)id - 1;
            for (;;) {
                const long long idx = look - lane;
                unsigned long long w;
                for (;;) {
                    w = (idx >= (long long)seg.tile_base) ? qs_ld_state(&a.state[idx]) : qs_pack(QS_INC, 0, 0);     // before the first tile: prefix 0
                    const bool valid = (w & QS_FLAGS) != 0;
                    const bool inc = (w & QS_FLAGS) == QS_INC;
                    const unsigned int vmask = __ballot_sync(0xffffffffu, valid), imask = __ballot_sync(0xffffffffu, inc);
                    const unsigned int before_inc = imask ? ((imask & (0u - imask)) - 1u) : 0xffffffffu;
                    if ((~vmask & before_inc) == 0u) break;
                    __nanosleep(100);
                }
                const unsigned int imask = __ballot_sync(0xffffffffu, (w & QS_FLAGS) == QS_INC);
                const int upto = imask ? __ffs(imask) : 32;             // lanes 0 .. upto-1 contribute
                unsigned long long c_lt = (lane < upto) ? ((w >> 31) & QS_CNT) : 0ull, c_eq = (lane < upto) ? (w & QS_CNT) : 0ull;
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1) {
                    c_lt += __shfl_xor_sync(0xffffffffu, c_lt, d);
                    c_eq += __shfl_xor_sync(0xffffffffu, c_eq, d);
                }
                e_lt += c_lt; e_eq += c_eq;
                if (imask) break;
                look -= 32;
            }
            if (lane == 0) qs_st_state(&a.state[id], qs_pack(QS_INC, e_lt + t_lt, e_eq + t_eq));
        }
        if (lane == 0) { s_excl[0] = e_lt; s_excl[1] = e_eq; }
    }
    __syncthreads();
    const long long e_lt = (long long)s_excl[0], e_eq = (long long)s_excl[1];
    long long r_lt = e_lt + (ex & 0xffffu), r_eq = e_eq + (ex >> 16);
#pragma unroll
    for (int e = 0; e < QS_EPT; ++e) {
        const long long i = i0 + e;
        if (cls[e] == 1u) a.dst[seg.start + r_lt++] = x[e];
        else if (cls[e] == 2u) a.mid[seg.start + r_eq++] = x[e];
        else if (cls[e] == 3u) a.dst[seg.start + seg.count - 1 - (i - r_lt - r_eq)] = x[e];
    }
    if (__any_sync(0xffffffffu, bad) && lane == 0) atomicOr(&a.ctl->error, 1u);
    __syncthreads();        // s_excl is read; the scratch words below are free again
    if ((long long)t == n_tiles - 1) {
        // the segment's totals are known: its `=` run is copied to the result at the next launch, its children join the next level
        const long long n_lt = e_lt + (long long)t_lt, n_eq = e_eq + (long long)t_eq, n_gt = seg.count - n_lt - n_eq;
        qs_append<T>(a, nxt, seg.start, n_eq, seg.start + n_lt, QS_KIND_MIDCOPY, 0u, s_warp);
        qs_append<T>(a, nxt, seg.start, n_lt, 0, QS_KIND_SEG, 0u, s_warp);
        qs_append<T>(a, nxt, seg.start + n_lt + n_eq, n_gt, 0, QS_KIND_SEG, 1u, s_warp);
    }
}

template <class T> constexpr size_t qs_smem_bytes() { return (size_t)2 * QS_SMALL * sizeof(T) + (size_t)4 * QS_SMALL * sizeof(unsigned short) + (size_t)QS_SMALL * sizeof(unsigned int); }

template <class T>
__global__ void __launch_bounds__(QS_THREADS) qs_level(const QsArgs<T> a) {
    extern __shared__ __align__(16) unsigned char qs_smem[];
    __shared__ unsigned int s_warp[QS_THREADS / 32];
    __shared__ unsigned long long s_excl[2];
    __shared__ unsigned int s_id;
    QsLevel* const cur = &a.ctl->lvl[a.level % 3];
    QsLevel* const nxt = &a.ctl->lvl[(a.level + 1) % 3];
    // housekeeping for the launches to come: the level after next starts from zero counters, the next level from cleared tile states
    if (blockIdx.x == 0 && threadIdx.x == 0) { QsLevel* z = &a.ctl->lvl[(a.level + 2) % 3]; z->ticket = 0; z->n_work = 0; z->n_segs = 0; }
    for (unsigned int i = blockIdx.x * QS_THREADS + threadIdx.x; i < a.cap_work; i += gridDim.x * QS_THREADS) a.state_next[i] = 0ull;
    const unsigned int n_work = cur->n_work < a.cap_work ? cur->n_work : a.cap_work;
    for (;;) {
        if (threadIdx.x == 0) s_id = atomicAdd(&cur->ticket, 1u);       // work ids in increasing order: a tile's predecessors are running or done
        __syncthreads();
        const unsigned int id = s_id;
        __syncthreads();
        if (id >= n_work) break;
        const QsSeg seg = a.segs[a.work[id]];
        if ((seg.kind_rev >> 1) == QS_KIND_MIDCOPY) {
            const long long off = (long long)(id - seg.tile_base) * QS_TILE;
            for (long long i = off + threadIdx.x; i < seg.count && i < off + QS_TILE; i += QS_THREADS) a.out[seg.aux + i] = a.mid_prev[seg.start + i];
        } else if (seg.count <= QS_SMALL) qs_sort_small<T>(a, seg, qs_smem, s_warp);
        else qs_partition_tile<T>(a, seg, id, nxt, s_warp, s_excl);
    }
}

__global__ void qs_init(QsCtl* ctl, QsSeg* segs, unsigned int* work, unsigned long long* state, long long n, unsigned int cap_work) {
    const unsigned int ntiles = n <= QS_SMALL ? 1u : (unsigned int)((n + QS_TILE - 1) / QS_TILE);
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        for (int l = 0; l < 3; ++l) { ctl->lvl[l].ticket = 0; ctl->lvl[l].n_work = 0; ctl->lvl[l].n_segs = 0; ctl->lvl[l].pad = 0; }
        ctl->lvl[0].n_work = ntiles; ctl->lvl[0].n_segs = 1;
        ctl->error = 0;
        QsSeg s; s.start = 0; s.count = n; s.aux = 0; s.kind_rev = 0; s.tile_base = 0;
        segs[0] = s;
    }
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < cap_work; i += gridDim.x * blockDim.x) {
        state[i] = 0ull;
        if (i < ntiles) work[i] = 0u;
    }
}

struct QsLayout { size_t keys0, keys1, mid0, mid1, segs0, segs1, work0, work1, state0, state1, ctl, total; unsigned int cap_segs, cap_work; };
QsLayout qs_layout(long long n, int es) {
    QsLayout L{};
    auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
    const size_t parents = (size_t)(n / (QS_SMALL + 1)) + 1;            // big segments of one level are disjoint and longer than QS_SMALL
    L.cap_segs = (unsigned int)(3 * parents + 2);                       // per parent: two children and one copy job
    L.cap_work = (unsigned int)((size_t)n / QS_TILE + 3 * parents + 4);
    size_t off = 0;
    L.keys0 = off; off += up((size_t)n * es);
    L.keys1 = off; off += up((size_t)n * es);
    L.mid0 = off; off += up((size_t)n * es);
    L.mid1 = off; off += up((size_t)n * es);
    L.segs0 = off; off += up((size_t)L.cap_segs * sizeof(QsSeg));
    L.segs1 = off; off += up((size_t)L.cap_segs * sizeof(QsSeg));
    L.work0 = off; off += up((size_t)L.cap_work * 4);
    L.work1 = off; off += up((size_t)L.cap_work * 4);
    L.state0 = off; off += up((size_t)L.cap_work * 8);
    L.state1 = off; off += up((size_t)L.cap_work * 8);
    L.ctl = off; off += up(sizeof(QsCtl));
    L.total = off;
    return L;
}

template <class T>
cudaError_t qs_run(const T* in, T* out, long long n, char* ws, int sm_count, unsigned int* host_flag, cudaStream_t stream, int* launches, unsigned int* error) {
    const QsLayout L = qs_layout(n, (int)sizeof(T));
    T* keys[2] = {reinterpret_cast<T*>(ws + L.keys0), reinterpret_cast<T*>(ws + L.keys1)};
    QsSeg* segs[2] = {reinterpret_cast<QsSeg*>(ws + L.segs0), reinterpret_cast<QsSeg*>(ws + L.segs1)};
    unsigned int* work[2] = {reinterpret_cast<unsigned int*>(ws + L.work0), reinterpret_cast<unsigned int*>(ws + L.work1)};
    unsigned long long* state[2] = {reinterpret_cast<unsigned long long*>(ws + L.state0), reinterpret_cast<unsigned long long*>(ws + L.state1)};
    QsCtl* ctl = reinterpret_cast<QsCtl*>(ws + L.ctl);
    static bool attr_set[64] = {};
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev >= 0 && dev < 64 && !attr_set[dev]) {
        cudaError_t e = cudaFuncSetAttribute(qs_level<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)qs_smem_bytes<T>());
        if (e != cudaSuccess) return e;
        attr_set[dev] = true;
    }
    qs_init<<<32, 256, 0, stream>>>(ctl, segs[0], work[0], state[0], n, L.cap_work);
    *launches = 1;
    const int grid = sm_count * 3;
    // a first batch sized for the expected depth of random keys, then batches of 8 levels; ONE 16-byte read-back per batch tells
    // whether work is left (counts and segment tables never visit the host)
    int depth = 6;
    for (long long m = n; m > QS_SMALL; m >>= 1) depth += 2;
    int level = 0;
    for (int batch = 0;; ++batch) {
        const int todo = batch == 0 ? depth : 8;
        for (int i = 0; i < todo; ++i, ++level) {
            QsArgs<T> a{};
            a.src = level == 0 ? in : keys[(level + 1) & 1];            // level L writes keys[L & 1]
            a.dst = keys[level & 1];
            a.out = out;
            a.mid = reinterpret_cast<T*>(ws + ((level & 1) ? L.mid1 : L.mid0));
            a.mid_prev = reinterpret_cast<const T*>(ws + ((level & 1) ? L.mid0 : L.mid1));
            a.segs = segs[level & 1]; a.work = work[level & 1];
            a.next_segs = segs[(level + 1) & 1]; a.next_work = work[(level + 1) & 1];
            a.state = state[level & 1]; a.state_next = state[(level + 1) & 1];
            a.ctl = ctl; a.level = level; a.cap_segs = L.cap_segs; a.cap_work = L.cap_work;
            qs_level<T><<<grid, QS_THREADS, qs_smem_bytes<T>(), stream>>>(a);
            ++*launches;
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        // lvl[level % 3] is the table the NEXT launch would consume
        e = cudaMemcpyAsync(host_flag, &ctl->lvl[level % 3], 16, cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaMemcpyAsync(host_flag + 4, &ctl->error, 4, cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) return e;
        *error = host_flag[4];
        if (host_flag[1] == 0 || *error) break;     // n_work of the next level
    }
    return cudaSuccess;
}

}  // namespace

size_t sgk_quicksort_workspace_bytes(int64_t n, int elem_size) { return qs_layout(n, elem_size).total; }

// dtype: DT_F32 / DT_F64 / DT_I32 / DT_I64.  host_flag: 8 pinned 32-bit words.  *error: bit 0 = a key matched none of <, =, > (NaN).
cudaError_t sgk_quicksort(int dtype, const void* in, void* out, int64_t n, void* workspace, int sm_count, unsigned int* host_flag, cudaStream_t stream,
                          int* launches, unsigned int* error) {
    *launches = 0; *error = 0;
    if (n <= 0) return cudaSuccess;
    char* ws = reinterpret_cast<char*>(workspace);
    switch (dtype) {
        case DT_F32: return qs_run<float>((const float*)in, (float*)out, n, ws, sm_count, host_flag, stream, launches, error);
        case DT_F64: return qs_run<double>((const double*)in, (double*)out, n, ws, sm_count, host_flag, stream, launches, error);
        case DT_I32: return qs_run<int32_t>((const int32_t*)in, (int32_t*)out, n, ws, sm_count, host_flag, stream, launches, error);
        case DT_I64: return qs_run<long long>((const long long*)in, (long long*)out, n, ws, sm_count, host_flag, stream, launches, error);
        default: return cudaErrorInvalidValue;
    }
}
