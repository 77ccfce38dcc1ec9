// sg_ctx.h — host runtime data structures (internal): context, handle table, pending-action list, plan.
// PAPER.md:284 "a method call is not executed, but rather added to a list of pending actions"
// "the optimizer constructs an execution plan from the pending operations ... a DAG, representing data and
// kernels as two different types of nodes".  Here: Value = data node, Node = kernel node, Pass = merged kernel.
#ifndef SG_CTX_H_
#define SG_CTX_H_

#include <cuda_runtime.h>
#include <stdint.h>

#include <string>
#include <utility>
#include <vector>

#include "../../include/sg.h"
#include "sg_kernels.h"
#include "sg_prog.h"

enum ValueKind { VK_VEC = 0, VK_MAT = 1, VK_SCALAR = 2 };
enum NodeKind { NK_MAP = 0, NK_REDUCE = 1, NK_FILTER = 2 };
// node-level opcode of the dtype conversion (sg_cast): never part of a program — the plan builder lowers it to an IN_VEC_CVT
// input (conversion at load) followed by OP_MOV
constexpr uint8_t NODE_OP_CAST = 0x40;
enum OperandKind { OPD_VALUE = 0, OPD_IMM = 1, OPD_SHIFT = 2 /* value shifted by +1 element */ };

struct Value {
    int kind = VK_VEC;
    int dtype = SG_F32;
    int64_t rows = 1, cols = 0;     // vector: rows = 1, cols = n
    int64_t ld = 0;                 // matrix: leading dimension in elements
    int64_t stride = 1;             // vector: element stride (ld for a column view)
    char* ptr = nullptr;            // element 0 when materialised
    bool materialised = false;
    bool owned = false;             // ptr allocated by the context
    int node = -1;                  // producing pending node, -1 if none
    int user_refs = 0;
    int64_t count_slot = -1;        // filter output: scalar slot holding the kept count; cols is the capacity until resolved
    bool count_known = true;
    int64_t slot = -1;              // VK_SCALAR produced by a reduction: slot in the scalar slab
    bool alive = true;
    bool fresh_alloc = false;       // storage allocated by the flush in progress (given back if that flush fails before it runs)
    uint32_t gen = 0;               // generation of the table slot (upper half of the handle): a recycled slot does not answer to its old handle
    bool undecided = false;         // quantifier whose pass ended early at a violated contract before it was decided: reading it is an error
};

struct Operand {
    int kind = OPD_VALUE;
    int value = -1;
    int bcast = SG_BCAST_NONE;
    uint64_t imm = 0;               // raw bits, already converted to the node's operand dtype
};

struct Node {
    int kind = NK_MAP;
    uint8_t op = 0;                 // NK_MAP: OP_*; NK_REDUCE: OUT_SUM..OUT_COUNT
    int n_opd = 0;
    Operand opd[2];
    int out = -1;                   // result value
    int out2 = -1;                  // NK_FILTER: the count scalar
    int axis = AXIS_ALL;
    int dtype = SG_F32;             // operand dtype (V file) — SG_BOOL for pure logic nodes
    int src_dtype = -1;             // OP_CAST: element type of the operand in memory (converted to `dtype` as it is loaded)
    bool is2d = false;
    int64_t rows = 1, cols = 0;     // iteration domain
    bool inplace = false;           // out's storage was given by the caller (dst_or_0)
    // plan state
    bool needed = false, post = false, done = false;
    int pass = -1;
};

struct Contract { int value; int kind; std::string tag; };

// `exact`: the pass reads element i of the range for element i of its domain (an index-for-index read).  Shifted (neighbour),
// broadcast and scalar reads are not: an in-place writer of the same storage can never share their pass.
struct MemRange { const char* lo; const char* hi; const char* ptr; int64_t stride, ld, rows, cols; bool exact; };

struct PassInput { uint8_t kind; const char* ptr; int64_t stride; uint64_t imm; int reg; int value; bool boolvec; int64_t len; uint8_t src_dtype; };

struct Pass {
    bool is2d = false, has_filter = false, has_store = false;
    int dtype = -1;                 // V-file dtype, -1 = not fixed yet (only BOOL nodes so far)
    int64_t rows = 1, cols = 0;     // domain (1-D: cols = max length)
    std::vector<int> nodes;
    std::vector<MemRange> reads, writes;
    // built program
    SgProg prog;
    SgArgs args;
    SgGeom geom;
    int n_mem_in = 0, n_scalar_in = 0;
    int64_t bytes = 0;
};

struct Launch { SgProg prog; SgArgs args; SgGeom geom; };

// Plan cache (SURVEY.md §8 a2 "plan cache keyed by DAG signature"): the pass assignment of a pending list — the part of planning that
// compares every operation with every pass and may repeat itself under tighter limits — remembered under the SIGNATURE of that list:
// every operation, the identity pattern and the storage (address, shape, liveness) of every value it names, the contracts and the
// context flags, as bytes.  A step that enqueues the same program over the same buffers again (any immediates) re-uses the
// assignment; programs are still built and bound to their pointers by every flush.
struct PlanMemo {
    std::string key;
    int attempt = 0;                // which limits the assignment succeeded under (sg_plan.cpp)
    std::vector<int> node_pass;     // per pending operation: its pass (-1: not needed)
    std::vector<char> node_spill;   // per pending operation: its result is stored for a later pass
    std::vector<Pass> passes;       // skeletons: domain, dtype, flags, operations (no programs, no memory ranges)
};

struct sg_ctx {
    int device = -1;
    bool plan_only = true;
    cudaStream_t stream = nullptr;
    sg_alloc alloc{};
    bool has_alloc = false;
    uint32_t flags = 0;
    int sm_count = 148;
    std::string err;

    std::vector<Value> values;      // handle h <-> values[h-1]
    std::vector<int> free_values;   // slots of dead values no pending operation names any more: reused by new handles
    std::vector<int> live;          // indices of values that may still be alive (compacted at every flush: a flush costs O(live), not O(history))
    std::vector<Node> nodes;        // pending actions, in call order
    std::vector<Contract> contracts;

    // device resources
    char* workspace = nullptr; size_t workspace_bytes = 0;
    unsigned long long* tile_state = nullptr; size_t tile_state_words = 0;
    unsigned int* ctrl = nullptr; int ctrl_words = 0;
    uint32_t epoch = 0;
    char* slab = nullptr;           // device scalar slots, 8 bytes each
    char* slab_host = nullptr;      // pinned mirror
    int64_t slab_slots = 0, slab_next = 0;
    std::vector<int64_t> slab_free;
    cudaEvent_t ev_done = nullptr, ev_t0 = nullptr, ev_t1 = nullptr;
    bool mirror_pending = false;
    // sg_timing_begin/end: one event pair per flush, resolved at the end (no host sync inside the timed region)
    bool timing = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> timing_events;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> timing_pool;
    uintptr_t fake_next = 0x10000000;   // plan-only contexts: distinct fake addresses

    // last flush
    std::vector<Launch> last;
    sg_stats stats{};
    std::vector<SgProg> dumps;      // canonical programs of the last flush; sg_plan_dump renders them as text on demand
    std::vector<char*> deferred_free;
    std::vector<PlanMemo> plan_cache;   // a few entries, replaced round robin
    size_t plan_cache_next = 0;
    int64_t plan_cache_hits = 0, plan_cache_misses = 0;
    int plan_cache_miss_streak = 0, plan_cache_pause = 0;   // a loop whose lists never repeat (other buffers every step) stops paying for signatures
};

// Makes the context's device current for the duration of one entry point and restores the caller's device afterwards
// (a process may hold contexts on several GPUs; no entry point changes the caller's current device).
struct SgDeviceScope {
    int prev = -1;
    bool switched = false;
    explicit SgDeviceScope(const sg_ctx* c) {
        if (!c || c->plan_only) return;
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; return; }
        if (prev != c->device) switched = cudaSetDevice(c->device) == cudaSuccess;
    }
    ~SgDeviceScope() { if (switched && prev >= 0) cudaSetDevice(prev); }
    SgDeviceScope(const SgDeviceScope&) = delete;
    SgDeviceScope& operator=(const SgDeviceScope&) = delete;
};

// sg_plan.cpp
sg_status sg_flush_impl(sg_ctx* c);
std::string sg_dump_prog(const SgProg& g);   // sg_build.cpp
// helpers shared by sg_api.cpp / sg_plan.cpp
inline int dtype_size(int dt) { return dt == SG_BOOL ? 1 : (dt == SG_F32 || dt == SG_I32) ? 4 : 8; }
sg_status sg_fail(sg_ctx* c, sg_status code, const std::string& msg);
void* sg_dev_alloc(sg_ctx* c, size_t bytes);
void sg_dev_free(sg_ctx* c, void* p);
int64_t sg_slot_alloc(sg_ctx* c);

#endif  // SG_CTX_H_
