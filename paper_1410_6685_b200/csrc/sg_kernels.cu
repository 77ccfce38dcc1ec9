// sg_kernels.cu — kernel instantiation, the template registry and launch geometry (sm_100a).
#include "sg_kernels.h"

#include <cuda.h>

#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>

#include "sg_pass1d_vm.cuh"
#include "sg_tmpl_launch.cuh"

static_assert(SG_NSHARDS == 8, "the shard list below names eight tables");
const sgk::Entry* sgk_shard_entries_0(int*); const sgk::Entry* sgk_shard_entries_1(int*); const sgk::Entry* sgk_shard_entries_2(int*);
const sgk::Entry* sgk_shard_entries_3(int*); const sgk::Entry* sgk_shard_entries_4(int*); const sgk::Entry* sgk_shard_entries_5(int*);
const sgk::Entry* sgk_shard_entries_6(int*); const sgk::Entry* sgk_shard_entries_7(int*);

// sg_vm_shard.cu, one per element type (index = DT_*)
cudaError_t sgk_launch_bytecode_0(const SgProg&, const SgArgs&, const SgGeom&, cudaStream_t); int sgk_occupancy_bytecode_0(bool, int, int);
cudaError_t sgk_launch_bytecode_1(const SgProg&, const SgArgs&, const SgGeom&, cudaStream_t); int sgk_occupancy_bytecode_1(bool, int, int);
cudaError_t sgk_launch_bytecode_2(const SgProg&, const SgArgs&, const SgGeom&, cudaStream_t); int sgk_occupancy_bytecode_2(bool, int, int);
cudaError_t sgk_launch_bytecode_3(const SgProg&, const SgArgs&, const SgGeom&, cudaStream_t); int sgk_occupancy_bytecode_3(bool, int, int);

namespace {

using namespace sgk;

// registry: the shards' tables merged (entry i is owned by shard i % SG_NSHARDS); entry 0 is the bytecode kernel
struct Registry {
    Entry e[512];
    int n = 1;
    Registry() {
        e[0] = {"bytecode", nullptr, nullptr, nullptr, 0};
        typedef const Entry* (*ShardFn)(int*);
        const ShardFn shards[SG_NSHARDS] = {sgk_shard_entries_0, sgk_shard_entries_1, sgk_shard_entries_2, sgk_shard_entries_3,
                                            sgk_shard_entries_4, sgk_shard_entries_5, sgk_shard_entries_6, sgk_shard_entries_7};
        int cnt = 0;
        const Entry* tabs[SG_NSHARDS];
        for (int s = 0; s < SG_NSHARDS; ++s) tabs[s] = shards[s](&cnt);
        for (int i = 0; i < cnt && n < 512; ++i) e[n++] = tabs[i % SG_NSHARDS][i];
    }
};
const Registry& registry() { static const Registry r; return r; }
#define g_entries (registry().e)
#define g_n_entries (registry().n)

int occupancy_bytecode(int dtype, bool filter, int n_vreg = 64 /* file KiB */, int cells = 0 /* vm config */) {
    switch (dtype) {
        case DT_F32: return sgk_occupancy_bytecode_0(filter, n_vreg, cells);
        case DT_F64: return sgk_occupancy_bytecode_1(filter, n_vreg, cells);
        case DT_I32: return sgk_occupancy_bytecode_2(filter, n_vreg, cells);
        default: return sgk_occupancy_bytecode_3(filter, n_vreg, cells);
    }
}

int elem_size(int dtype) { return (dtype == DT_F32 || dtype == DT_I32) ? 4 : 8; }

long env_long(const char* name, long dflt) {
    const char* s = getenv(name);
    return (s && *s) ? atol(s) : dflt;
}

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
    if (tid == 0 && prog.shape.n_vreg > VM_VREG)
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
    // a converting input is read as vectors of V SOURCE elements: the same element misalignment, measured against V * its element size
    for (int k = 0; k < prog.shape.n_in; ++k) {
        if (prog.in[k].kind != IN_VEC_CVT) continue;
        const int ss = elem_size(prog.in[k].ref);
        const uintptr_t p = (uintptr_t)a.in_ptr[k];
        if (p % ss != 0) { congruent = false; continue; }
        const long m = (long)((p % (uintptr_t)(V * ss)) / ss);
        if (mis < 0) mis = m;
        if (m == mis) vec_ok |= 1 << k; else congruent = false;
    }
    if (mis < 0) mis = 0;

    if (is2d) {
        for (int k = 0; k < prog.shape.n_in; ++k)
            if (prog.in[k].kind == IN_VEC_CVT) return fail(err, errcap, -10, "dtype conversion inside a matrix pass");
        if (tid == 0) {
            // no precompiled instance: the 2-D bytecode evaluator (sg_pass2d_vm.cuh) — blocks own whole rows, every access guarded
            bool has_cols = false;
            for (int o = 0; o < prog.shape.n_out; ++o) {
                has_cols |= out_is_reduction(prog.out[o].kind) && prog.out[o].axis == AXIS_COLS;
            }
            const long blocks = std::max<long>(1, std::min<long>(a.n, (long)sm_count * (has_cols ? 1 : 2)));
            geom->template_id = 0;
            geom->grid = (int)blocks;
            geom->tile = BLOCK * V;
            geom->vm_cfg = 0;
            size_t off = (size_t)geom->grid * SG_MAX_OUT * sizeof(Cell);
            for (int o = 0; o < prog.shape.n_out; ++o) {
                a.ws_off[o] = 0;
                if (out_is_reduction(prog.out[o].kind) && prog.out[o].axis == AXIS_COLS) { a.ws_off[o] = (int64_t)off; off += (size_t)blocks * a.cols * sizeof(Cell); }
            }
            geom->ws_bytes = off;
            geom->ctrl_words = 1;
            a.vec_ok = 0; a.head = 0; a.n_full_tiles = 0; a.n_strips = 0; a.n_chunks = 0; a.rows_per_chunk = 0;
            return 0;
        }
        bool ok = congruent && mis == 0 && (a.cols % V) == 0;
        for (int k = 0; k < prog.shape.n_in; ++k)
            if (prog.in[k].kind == IN_VEC && (a.in_stride[k] % V) != 0) ok = false;
        for (int o = 0; o < prog.shape.n_out; ++o)
            if (prog.out[o].kind == OUT_STORE && (a.out_len[o] % V) != 0) ok = false;
        // rows that are not 16-byte aligned (odd column counts / leading dimensions): the same kernel's guarded form (bit 29)
        const int unaligned_rows = ok ? 0 : (1 << 29);
        const int occ = (has_device && tid) ? g_entries[tid].occupancy() : 2;
        const int SW = tid ? g_entries[tid].tile : BLOCK * 2 * V;
        a.n_strips = (int)((a.cols + SW - 1) / SW);
        static const long mult2d = env_long("SG_GRID_MULT_2D", 1), tile2d = env_long("SG_2D_TILE", 1), tile_rows = env_long("SG_2D_TILE_ROWS", 2);
        const long target = (long)sm_count * occ * mult2d;
        bool any_reduction = false, any_bool_store = false;
        for (int o = 0; o < prog.shape.n_out; ++o) {
            any_reduction |= out_is_reduction(prog.out[o].kind);
            any_bool_store |= prog.out[o].kind == OUT_STORE_BOOL;
        }
        const long rpb = std::max<long>(1, tile_rows);
        if (tid && ok && !any_reduction && !any_bool_store && tile2d && a.n > 0 && a.n_strips > 0 && (a.n_strips * ((a.n + rpb - 1) / rpb)) < 0x7fffffffl) {
            // store-only pass on aligned rows: short-lived blocks, one tile of tile_rows x SW per block in row-major order (sg_pass2d_tile.cuh)
            a.rows_per_chunk = rpb;
            a.n_chunks = 0;
            geom->template_id = tid;
            geom->grid = (int)(a.n_strips * ((a.n + rpb - 1) / rpb));
            geom->tile = SW;
            geom->ws_bytes = 0;
            geom->ctrl_words = 0;
            for (int o = 0; o < prog.shape.n_out; ++o) a.ws_off[o] = 0;
            a.vec_ok = (vec_ok & ~(3 << 28)) | (1 << 28);
            a.head = 0; a.n_full_tiles = 0;
            return 0;
        }
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
        a.vec_ok = (vec_ok & ~(3 << 28)) | unaligned_rows;
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
    const int vcfg = vm_pick_config(prog);
    const int tile = tid ? g_entries[tid].tile : vm_tile_cfg(es, vcfg);
    geom->vm_cfg = vcfg;
    int vm_r = 0, vm_i = 0;
    vm_count_regs(prog, &vm_r, &vm_i);
    const int file_kib = (int)((vm_file_bytes_cfg(vm_r, vm_i, vcfg) + 1023) / 1024);
    long lmin = a.n;
    for (int o = 0; o < prog.shape.n_out; ++o) lmin = std::min<long>(lmin, a.out_len[o]);
    const long head = std::min<long>((V - mis) % V, a.n);
    const long body = std::max<long>(0, lmin - head);
    a.head = head;
    a.n_full_tiles = body / tile;
    a.vec_ok = vec_ok;
    const int occ = has_device ? (tid ? g_entries[tid].occupancy() : occupancy_bytecode(prog.shape.dtype, false, file_kib, vcfg)) : 4;
    long want = tid ? a.n_full_tiles : ((a.n - head + tile - 1) / tile + (head + tile - 1) / tile);
    geom->template_id = tid;
    geom->tile = tile;
    {
        // Launch shape (measured on B200, profiles/r02_grid_shape.md).  Equal static shares of a persistent grid finish at very
        // different times on this part: SM pairs differ up to 2x in WRITE throughput (1R+1W over 592 blocks: the median block is
        // done 100 us before the last of 372 us), read-only streams by 6 % (10 us of 156 us).  So
        //   * a pass that only stores (no epilogue) runs as many short-lived blocks of K_STORE strided tiles, the hardware block
        //     scheduler balances them:      x := x * a, 2^27 fp64: 0.360 -> 0.313 ms (0.92 -> 1.06 of the measured copy peak);
        //     K = 1 / 2 / 3 / 4 / 8: 0.310 / 0.313 / 0.315 / 0.316 / 0.322 ms in place, 0.354 / 0.312 / 0.313 / 0.315 / 0.320 to a second buffer;
        //   * a pass with reductions keeps the persistent grid (one epilogue per block: 4096 blocks cost +9 %, 131072 blocks 3x).
        //     Taking only the first PCT % of its share strided and the rest through tile tickets (sg_pass1d_tmpl.cuh) evens the
        //     blocks out — read-only, PCT = 100 / 92 / 85 / 75 / 60: config 1 at 2^28 0.338 / 0.327 / 0.324 / 0.325 / 0.327 ms; with
        //     stores (divide + contracts, 2^26), PCT = 100 / 50 / 30 / 0: 0.258 / 0.249 / 0.250 / 0.250 ms — but which block adds which
        //     tile then differs from run to run, and a FLOATING-POINT SUM accumulated that way is no longer the same bits on every
        //     run.  Making it order-independent (one partial cell per ticket, added in ticket order by the epilogue) costs what the
        //     tickets gain: a cell per tile 0.365 ms, a cell per 4 tiles 0.340 - 0.342 ms against 0.345 ms static (config 1 at 2^28),
        //     sum(x) 0.159 - 0.163 against 0.157 ms.  So tickets are used only where every reduction of the pass is exact in any order
        //     (integer sums, max/min, counts, quantifiers); passes with a floating-point sum keep the static shares;
        //   * early-exit passes stay static.  Their exit is taken per thread; a ticket loop needs a block-uniform one (thread 0 reads
        //     the decided word with every ticket and hands out "no more tiles") — built and measured on config 3 (2^28 fp32, both
        //     quantifiers), static share 100 / 92 / 85 / 75 / 60 %: clean pass 0.183 / 0.180 / 0.183 / 0.186 / 0.193 ms, time to answer
        //     for a violation at n - n/64 0.170 / 0.179 / 0.182 / 0.185 / 0.191 ms: the barrier per ticketed tile costs this
        //     shuffle-heavy pass what the balance gains, so it was not kept.
        // The environment variables override the defaults for such sweeps; they are read once.
        bool has_red = false, has_store = false;
        for (int o = 0; o < prog.shape.n_out; ++o) {
            has_red |= out_is_reduction(prog.out[o].kind);
            has_store |= prog.out[o].kind == OUT_STORE || prog.out[o].kind == OUT_STORE_BOOL;
        }
        const bool ee = (prog.shape.flags & PF_EARLY_EXIT) != 0;
        static const long k_store = env_long("SG_GRID_K_STORE", 2), k_red = env_long("SG_GRID_K_RED", 0), k_ee = env_long("SG_GRID_K_EE", 0);
        static const long pct_ro = env_long("SG_STATIC_PCT_RO", 85), pct_rw = env_long("SG_STATIC_PCT_RW", 50), dyn_min = env_long("SG_DYN_MIN_ITERS", 8);
        const long K = !tid ? 0 : ee ? k_ee : has_red ? k_red : k_store;     // the bytecode kernel decodes its program per block: persistent
        long blocks = std::min<long>(want, (long)sm_count * occ);
        if (K > 0) blocks = std::max<long>(blocks, (want + K - 1) / K);
        // short reduction passes: fewer, longer-lived blocks (SG_SMALL_OCC per SM while a full grid would get < SG_SMALL_TILES tiles per block)
        static const long small_occ = env_long("SG_SMALL_OCC", 0), small_tiles = env_long("SG_SMALL_TILES", 4);
        if (tid && has_red && K == 0 && small_occ > 0 && want < (long)sm_count * occ * small_tiles) blocks = std::min<long>(want, (long)sm_count * std::min<long>(occ, small_occ));
        geom->grid = (int)std::max<long>(1, blocks);
        const long pct = has_store ? pct_rw : pct_ro;
        const long per_block = a.n_full_tiles / geom->grid;
        a.static_tiles = a.n_full_tiles;
        const bool is_float = prog.shape.dtype == DT_F32 || prog.shape.dtype == DT_F64;
        bool float_sum = false;
        for (int o = 0; o < prog.shape.n_out; ++o) float_sum |= is_float && prog.out[o].kind == OUT_SUM;
        if (tid && has_red && !ee && !float_sum && pct >= 0 && pct < 100 && per_block >= dyn_min) a.static_tiles = per_block * pct / 100 * geom->grid;
    }
    geom->ws_bytes = (size_t)geom->grid * SG_MAX_OUT * sizeof(Cell);
    return 0;
}

cudaError_t sgk_launch(const SgProg& prog, const SgArgs& args, const SgGeom& geom, cudaStream_t stream) {
    if (geom.template_id > 0) return g_entries[geom.template_id].launch(args, geom.grid, stream);
    switch (prog.shape.dtype) {
        case DT_F32: return sgk_launch_bytecode_0(prog, args, geom, stream);
        case DT_F64: return sgk_launch_bytecode_1(prog, args, geom, stream);
        case DT_I32: return sgk_launch_bytecode_2(prog, args, geom, stream);
        case DT_I64: return sgk_launch_bytecode_3(prog, args, geom, stream);
        default: return cudaErrorInvalidValue;
    }
}
