// sg_pass2d_tile.cuh — pass2d_body_tile<P>: the fused matrix pass (sg_pass2d.cuh) for passes that only STORE (no reductions: the
// Gaussian-elimination row update of Listing 5, scaling, elementwise matrix chains) on aligned rows, as
// SHORT-LIVED blocks in row-major tile order.
//
// A block owns one tile: rows_per_chunk (2) rows x one strip of SW columns (8 KiB of fp64 with two 128-bit accesses per thread),
// tile t = row-block * n_strips + strip, so the grid sweeps the matrix linearly, row after row.  Every operand is loaded straight
// into registers: the matrix elements (streaming), the ROW-broadcast segment of the strip (the same 8 KiB for every row: it stays
// in L2) and the row's COL-broadcast scalar.  Measured on the row update at 16384^2 fp64, in place (standalone probe, then this
// kernel; profiles/r02_grid_shape.md):
//     staged persistent blocks of (strip, 928 rows), sg_pass2d.cuh ......... 0.749 ms   5.7 TB/s  (0.88 of the measured copy peak)
//     the same with rows handed out by tickets (units of 8 .. 256 rows) .... 0.748 - 0.753 ms: the static shares were not the limit
//     one tile per block, 1 / 2 / 4 / 8 / 64 rows per block (probe) ........ 0.622 / 0.640 / 0.696 / 0.718 / 0.787 ms
//     this kernel through the library (two passes: factors + update), staged / 1 / 2 / 4 rows per block: 0.704 / 0.630 / 0.623 / 0.638 ms
// What costs is a block that streams SEVERAL rows (addresses one leading dimension apart) at once, and many bytes in flight per
// block; the linear sweep of small tiles is what the memory system serves at its copy rate.  The block scheduler hands the tiles
// out, which also evens out the SMs' different write throughput (sg_kernels.cu).
#ifndef SG_PASS2D_TILE_CUH_
#define SG_PASS2D_TILE_CUH_

namespace sgk {

template <class P>
__device__ __forceinline__ void pass2d_body_tile(const SgArgs& a) {
    typedef Meta2D<P> M;
    typedef typename M::T T;
    typedef typename M::VEC VEC;
    constexpr int U = M::U, V = M::V, E = M::E;
    constexpr auto IS = std::make_integer_sequence<int, M::S.n_instr>{};
    constexpr SgProg g = P::prog;

    const int64_t strip = blockIdx.x % (unsigned int)a.n_strips, rb = blockIdx.x / (unsigned int)a.n_strips;
    const int64_t r_begin = rb * a.rows_per_chunk;
    const int64_t r_end = (r_begin + a.rows_per_chunk < a.n) ? r_begin + a.rows_per_chunk : a.n;
    int64_t col[U];
    bool cvalid[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
        col[u] = strip * M::SW + (int64_t)(u * BLOCK + threadIdx.x) * V;
        cvalid[u] = (a.cols - col[u]) >= V;
    }
    T v[M::NV][E];
    bool p[M::NP][E];
#pragma unroll
    for (int k = 0; k < M::S.n_in; ++k) {
        const SgIn in = g.in[k];
        if (in.kind == IN_SCALAR || in.kind == IN_IMM) {
            const T s = load_elem<T>(in.kind, in.ref, k, a, 0);
#pragma unroll
            for (int e = 0; e < E; ++e) v[in.reg][e] = s;
        } else if (in.kind == IN_ROWB) {
#pragma unroll
            for (int u = 0; u < U; ++u) {
                VEC x = VEC();
                if (cvalid[u]) x = *reinterpret_cast<const VEC*>(reinterpret_cast<const T*>(a.in_ptr[k]) + col[u]);
                const T* xe = reinterpret_cast<const T*>(&x);
#pragma unroll
                for (int e = 0; e < V; ++e) v[in.reg][u * V + e] = xe[e];
            }
        }
    }
    for (int64_t r = r_begin; r < r_end; ++r) {
#pragma unroll
        for (int k = 0; k < M::S.n_in; ++k) {
            const SgIn in = g.in[k];
            if (in.kind == IN_VEC) {
                const T* rowp = reinterpret_cast<const T*>(a.in_ptr[k]) + r * a.in_stride[k];
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    VEC x = VEC();
                    if (cvalid[u]) x = ld_stream_rw(reinterpret_cast<const VEC*>(rowp + col[u]));      // the pass may write the same matrix in place: no .nc
                    const T* xe = reinterpret_cast<const T*>(&x);
#pragma unroll
                    for (int e = 0; e < V; ++e) v[in.reg][u * V + e] = xe[e];
                }
            } else if (in.kind == IN_COLB) {
                const T sc = reinterpret_cast<const T*>(a.in_ptr[k])[r];
#pragma unroll
                for (int e = 0; e < E; ++e) v[in.reg][e] = sc;
            }
        }
        exec_body<P, T, M::NV, M::NP, E>(v, p, a, IS);
#pragma unroll
        for (int o = 0; o < M::S.n_out; ++o) {
            const SgOut out = g.out[o];
            if (out.kind != OUT_STORE) continue;
            T* rowp = reinterpret_cast<T*>(a.out_ptr[o]) + r * a.out_len[o];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                if (!cvalid[u]) continue;
                VEC x;
                T* xe = reinterpret_cast<T*>(&x);
#pragma unroll
                for (int e = 0; e < V; ++e) xe[e] = v[out.src][u * V + e];
                st_stream(reinterpret_cast<VEC*>(rowp + col[u]), x);
            }
        }
    }
}

// its own kernel: no staging buffers, few registers — six to eight blocks per SM instead of the staged kernel's two
template <class P>
__global__ void __launch_bounds__(BLOCK, 6) pass2d_tile_template(const __grid_constant__ SgArgs a) {
    pdl_wait();
    pdl_trigger();
    if constexpr (!Meta2D<P>::has_reduction) pass2d_body_tile<P>(a);
}

}  // namespace sgk
#endif  // SG_PASS2D_TILE_CUH_
