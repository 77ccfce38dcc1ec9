/* sg.h — C ABI of the B200-native fused deferred-collection library (SafeGPU hot path, arXiv 1410.6685).
 *
 * What it is: device collections (vectors, row-major matrices) "equipped with primitive data-parallel
 * operations" (Table 2; vectors PAPER.md:199-207; matrices PAPER.md:209-219).
 * A call to an operation is NOT executed: it is appended to the context's list of pending actions
 * (PAPER.md:284).  Execution is triggered by (1) reading a scalar result (sg_scalar_get), (2) asking for a
 * collection's data or count (sg_vec_data / sg_vec_count on a pending filter output), or (3) sg_flush, the
 * paper's `update`.  At that point the plan builder turns the pending list into an
 * execution-plan DAG, merges kernel vertices and collapses anonymous intermediates and
 * launches one fused sm_100a kernel per pass over HBM.
 *
 * Conventions
 *  - All pointers named dev_* are DEVICE pointers; everything else is a HOST pointer.  No torch types.
 *  - Device buffers handed in are BORROWED: the caller keeps them alive until the handle is released and the
 *    context's stream has drained.  Buffers the library allocates (materialised results, filter outputs when
 *    no buffer is given, scalars, workspaces) are owned by the context and freed on sg_release/sg_ctx_destroy.
 *  - Every function returns sg_status: 0 = SG_OK, negative = error; sg_last_error(ctx) has the text.
 *    Shape / dtype / alias errors are raised at enqueue (they are the paper's scalar contracts);
 *    device-evaluated contracts and CUDA errors surface at sg_flush / sg_scalar_get.  A failed enqueue leaves
 *    the pending list unchanged.
 *  - One context per host thread; all GPU work is issued on the context's stream, on the context's device: every entry point
 *    makes that device current for its own duration and restores the caller's current device before it returns.
 *  - Indices are 0-based; ranges are half-open [start, finish).
 *  - Arithmetic semantics (identical in the CPU oracle): one IEEE-754 rounding per primitive
 *    (no FMA contraction); immediates are converted to the collection's dtype at enqueue; integers wrap;
 *    integer DIV/MOD truncate toward zero, divisor 0 gives 0; MIN(a,b) = (b<a)?b:a, MAX(a,b) = (a<b)?b:a;
 *    SUM of floats returns f64 (double-double / f64 accumulation), SUM of ints returns wrapping i64;
 *    MAX/MIN reductions use the IEEE total order on bit patterns; empty: ALL=1, ANY=0, SUM=0, COUNT=0.
 */
#ifndef SG_H_
#define SG_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sg_ctx sg_ctx;   /* opaque */
typedef int64_t sg_handle;      /* > 0 valid, opaque; vectors, matrices and scalars share one table.  A handle is a table slot tagged
                                 * with the slot's generation: slots of released values are reused, so a loop that releases what it
                                 * makes keeps the table at its high-water mark; a handle used after its last release is
                                 * SG_ERR_ARG (unknown handle), never an alias of the slot's next value */
typedef int32_t sg_status;

enum {
    SG_OK = 0,
    SG_ERR_ARG = -1,        /* null / unknown handle / bad enum / out-of-range index */
    SG_ERR_SHAPE = -2,      /* operand counts differ (the API's built-in dimension contract) */
    SG_ERR_DTYPE = -3,      /* operand dtypes differ or op undefined for the dtype */
    SG_ERR_EMPTY = -4,      /* MAX/MIN of an empty collection */
    SG_ERR_ALIAS = -5,      /* a pass would read a shifted/overlapping view of memory it writes in place */
    SG_ERR_OOM = -6,
    SG_ERR_CUDA = -7,       /* CUDA runtime error, or no usable device (the library has NO CPU fallback) */
    SG_ERR_CONTRACT = -8,   /* a registered contract evaluated false at flush; sg_last_error names its tag */
    SG_ERR_CAPACITY = -9,   /* filter output exceeded the caller's buffer, or a pass exceeds the plan limits */
    SG_ERR_UNSUPPORTED = -10
};

typedef enum { SG_F32 = 0, SG_F64 = 1, SG_I32 = 2, SG_I64 = 3, SG_BOOL = 4 /* 1 byte, 0/1 */ } sg_dtype;

/* Elementwise operations (PAPER.md:205 plus/minus/multiplied_by/divided_by + component-wise variants;
 * predicates of filter/for_all/exists agents PAPER.md:177-191).  Binary ops take two operands, each a
 * collection handle, an immediate or a device scalar; at least one must be a handle.  When no operand is a vector or
 * matrix (device scalars and immediates only) the result is a ONE-element vector: this is how avg = sum / count
 * stays on the device. */
typedef enum {
    SG_ADD = 0, SG_SUB = 1, SG_MUL = 2, SG_DIV = 3, SG_MIN = 4, SG_MAX = 5, SG_MOD = 6,   /* T,T -> T   */
    SG_NEG = 7, SG_ABS = 8,                                                              /* T   -> T   */
    SG_EQ = 9, SG_NE = 10, SG_LT = 11, SG_LE = 12, SG_GT = 13, SG_GE = 14,               /* T,T -> BOOL */
    SG_AND = 15, SG_OR = 16, SG_NOT = 17,                                                /* BOOL -> BOOL */
    SG_SQRT = 19    /* correctly rounded IEEE square root, the `project (agent sqrt)` of PAPER.md:171-175 (sqrt(-0) = -0,
                       sqrt(x < 0) = NaN).  F32/F64 -> same dtype.  I32/I64 VECTOR -> F64, the paper's own example
                       `agent (a: INT): DOUBLE do Result := sqrt (a) end`: the integers are converted (sg_cast) as they are loaded,
                       in the same pass.  SG_ERR_DTYPE on BOOL.  18 is reserved. */
} sg_op;

typedef enum { SG_SUM = 0, SG_RMAX = 1, SG_RMIN = 2, SG_COUNT = 3 /* number of true in a BOOL collection */ } sg_red;
typedef enum { SG_AXIS_ALL = 0, SG_AXIS_ROWS = 1 /* one result per row */, SG_AXIS_COLS = 2 /* one per column */ } sg_axis;
typedef enum { SG_OPERAND_HANDLE = 0, SG_OPERAND_IMM_F64 = 1, SG_OPERAND_IMM_I64 = 2 } sg_operand_kind;
typedef enum {
    SG_BCAST_NONE = 0,
    SG_BCAST_ROW = 1,   /* a vector of length cols, the same for every row of a matrix domain    */
    SG_BCAST_COL = 2    /* a vector of length rows, the same for every column of a matrix domain */
} sg_bcast;
typedef enum { SG_CONTRACT_PRE = 0, SG_CONTRACT_POST = 1 } sg_contract_kind;

typedef struct {
    int32_t kind;       /* sg_operand_kind */
    int32_t bcast;      /* sg_bcast (handles only) */
    sg_handle h;        /* vector / matrix / scalar handle (a scalar handle broadcasts to every element) */
    double f;           /* SG_OPERAND_IMM_F64 */
    int64_t i;          /* SG_OPERAND_IMM_I64 */
} sg_operand;

/* Optional device allocator (e.g. torch's caching allocator).  NULL => cudaMallocAsync/cudaFreeAsync on the stream. */
typedef struct {
    void* (*alloc)(void* user, size_t bytes);   /* returns a DEVICE pointer or NULL */
    void (*free)(void* user, void* dev_ptr);
    void* user;
} sg_alloc;

/* Context flags (sg_ctx_set_flags). */
enum {
    SG_FLAG_UNFUSED = 1,        /* lower every pending op to its own launch with materialised temporaries:
                                   the "one kernel per method call" plan of PAPER.md:282 (measurement baseline) */
    SG_FLAG_FORCE_BYTECODE = 2, /* never pick a precompiled template instance; always run the bytecode kernel */
    SG_FLAG_NO_EARLY_EXIT = 4,  /* quantifier passes read the whole collection even after a witness is found */
    SG_FLAG_NO_PLAN_CACHE = 8   /* plan every flush from scratch (the plan cache below is on by default) */
};

/* Plan statistics of the last flush (tests, reports). */
typedef struct {
    int32_t n_passes;           /* fused passes == kernel launches of the last flush */
    int32_t n_nodes;            /* pending operations consumed */
    int32_t n_template;         /* passes that ran a precompiled template instance */
    int32_t n_bytecode;         /* passes that ran the bytecode kernel */
    int64_t bytes_min;          /* algorithmic bytes of the plan: every distinct input read once + every materialised output written once */
    int64_t launches_total;     /* kernels launched by this context since creation */
    int32_t pass_n_in[16];      /* per pass (the first 16 passes of the flush; a flush may hold up to 256): distinct memory inputs */
    int32_t pass_n_instr[16];   /* per pass: elementwise instructions in the fused body */
    int32_t pass_n_out[16];     /* per pass: outputs (stores + reductions + quantifiers + compaction) */
    int32_t pass_n_args[16];    /* per pass: kernel data arguments = memory inputs + scalar/immediate operands + outputs */
    int32_t pass_kernel[16];    /* per pass: 0 = bytecode, k > 0 = template instance id k */
} sg_stats;

/* device >= 0: a CUDA device; cuda_stream: a cudaStream_t (NULL = default stream).
 * device == -1: PLAN-ONLY context — no CUDA calls are made, dev pointers may be NULL, sg_flush builds the
 * plan and updates sg_plan_stats but launches nothing (host-logic tests; the template generator). */
sg_status sg_ctx_create(sg_ctx** out, int device, void* cuda_stream, const sg_alloc* alloc_or_null);
sg_status sg_ctx_destroy(sg_ctx* ctx);
sg_status sg_ctx_set_flags(sg_ctx* ctx, uint32_t flags);
const char* sg_last_error(sg_ctx* ctx);

/* from_array's device half: wrap n elements at dev_ptr (borrowed).  dev_ptr NULL => the
 * context allocates (uninitialised) storage. */
sg_status sg_vec_create(sg_ctx* ctx, sg_dtype dtype, int64_t n, void* dev_ptr, sg_handle* out);
/* Row-major matrix, ld_elems >= cols is the distance between rows in elements. */
sg_status sg_mat_create(sg_ctx* ctx, sg_dtype dtype, int64_t rows, int64_t cols, int64_t ld_elems, void* dev_ptr, sg_handle* out);
/* subset(start, finish): a view sharing memory; of a pending vector it flushes first. */
sg_status sg_vec_subset(sg_ctx* ctx, sg_handle v, int64_t start, int64_t finish, sg_handle* out);
/* row(i): an index-adjusted vector view. */
sg_status sg_mat_row(sg_ctx* ctx, sg_handle m, int64_t i, sg_handle* out_vec);
/* rows [r0, r1) of a matrix as a matrix view (submatrix by rows). */
sg_status sg_mat_rows(sg_ctx* ctx, sg_handle m, int64_t r0, int64_t r1, sg_handle* out_mat);
/* column(j): a DEFERRED copy of the column into new storage; rows [r0, r1) of it. */
sg_status sg_mat_col(sg_ctx* ctx, sg_handle m, int64_t j, int64_t r0, int64_t r1, sg_handle* out_vec);
/* item(i,j) as a device scalar usable as an operand without a host round trip. */
sg_status sg_mat_elem(sg_ctx* ctx, sg_handle m, int64_t i, int64_t j, sg_handle* out_scalar);

/* Append one elementwise operation.  operands[0..n): 1 for unary ops, 2 for binary.
 * dst_or_0 != 0: the result replaces the contents of that vector/matrix (in-place variants) and
 * *out == dst_or_0; otherwise *out is a new pending collection that is materialised at flush only if the
 * caller still holds it (sg_release it first to keep an intermediate in registers, "anonymous
 * intermediate result").
 * Handles that share storage (a collection and its subset / row / row-block / element views): the pending list behaves like eager
 * execution in program order — an operation reads what the operations enqueued before it left in memory, whichever handle they went
 * through (R25).  An in-place operation may read its destination only index-for-index (the same view); an operand that
 * overlaps the destination any other way is SG_ERR_ALIAS at the flush.  A chain that exceeds what one pass holds (10 distinct
 * inputs, 8 outputs, 32 operations) is planned as several passes; a flush holds up to 256 passes (SG_ERR_CAPACITY beyond). */
sg_status sg_enqueue(sg_ctx* ctx, sg_op op, const sg_operand* operands, int32_t n, sg_handle dst_or_0, sg_handle* out);

/* project (transform: FUNCTION[T, U]): COLLECTION[U] with the value-preserving conversion as the transform:
 * a deferred vector of dtype `to` whose element i is element i of v converted.  Integer -> float: round to nearest even.
 * Float -> integer: truncation toward zero, saturating at the target's range, NaN -> 0 (R23).  F64 -> F32: round to
 * nearest even; F32 -> F64 and I32 -> I64: exact; I64 -> I32: the low 32 bits (wrap).  The conversion costs no pass of its own:
 * the operand is converted while it is loaded by the pass that consumes the result (a pending operand is stored first — a pass
 * has one value type).  dst_or_0 as in sg_enqueue (dtype `to`).  Errors: SG_ERR_DTYPE (BOOL), SG_ERR_UNSUPPORTED (matrix,
 * scalar or strided view). */
sg_status sg_cast(sg_ctx* ctx, sg_handle v, sg_dtype to, sg_handle dst_or_0, sg_handle* out);

/* Terminal reductions sum/max/min and COUNT, deferred: *out is a scalar handle; reading it is
 * the trigger, so several reductions and contracts of one chain share one pass (R7).
 * SG_AXIS_ROWS / SG_AXIS_COLS on a matrix give a vector handle of per-row / per-column results.
 * acc: the accumulator = result dtype.  SG_ACC_DEFAULT, or exactly the dtype the semantics fix: SUM -> SG_F64 for float inputs
 * (double-double / f64 accumulation), SG_I64 for int inputs (wrapping); RMAX/RMIN -> the input dtype; COUNT -> SG_I64.  Any other
 * value is SG_ERR_DTYPE: a narrower accumulator could not meet the stated sum tolerances and is not emulated. */
#define SG_ACC_DEFAULT (-1)
sg_status sg_reduce(sg_ctx* ctx, sg_handle h, sg_red kind, int32_t acc, sg_axis axis, sg_handle* out);
/* for_all / exists over a BOOL collection; *out is a BOOL scalar handle. */
sg_status sg_forall(sg_ctx* ctx, sg_handle h_bool, sg_handle* out_bool);
sg_status sg_exists(sg_ctx* ctx, sg_handle h_bool, sg_handle* out_bool);
/* for_all i in [0, n-2]: v[i] cmp v[i+1]; cmp in SG_EQ..SG_GE.  is_sorted == SG_LE.
 * n <= 1 => true. */
sg_status sg_forall_adjacent(sg_ctx* ctx, sg_handle v, sg_op cmp, sg_handle* out_bool);
/* filter: stable compaction of `values` where mask_bool is true, deferred.
 * dev_out_or_null: caller's output buffer of `capacity` elements (NULL => the context allocates n elements).
 * *out_vec is a vector whose count is known after the flush (sg_vec_count); *out_count an I64 scalar handle. */
sg_status sg_filter(sg_ctx* ctx, sg_handle values, sg_handle mask_bool, void* dev_out_or_null, int64_t capacity,
                    sg_handle* out_vec, sg_handle* out_count);
/* Register a BOOL scalar (from sg_forall/sg_exists) as a pre- or postcondition: the flush
 * that evaluates it returns SG_ERR_CONTRACT if it is false.  A POST contract reads the STORED values of
 * collections materialised by the same flush (R17). */
sg_status sg_contract(sg_ctx* ctx, sg_handle h_bool_scalar, int32_t kind, const char* tag);

/* update: plan + launch everything pending, asynchronously on the stream.  The flush's scalar results reach a
 * pinned host mirror without a host synchronisation: a reduction's last block writes its 8-byte results there itself, scalars
 * produced otherwise (filter counts, one-element passes) follow in one asynchronous copy.  Returns SG_ERR_CONTRACT (after a stream sync) only if
 * contracts are registered.  Transactional: when the plan cannot be built (SG_ERR_UNSUPPORTED, SG_ERR_CAPACITY, SG_ERR_ALIAS,
 * SG_ERR_OOM, ...) nothing has been launched, the error is returned and the pending list is DISCARDED — result handles of the
 * discarded operations name no data (release them), in-place destinations keep their previous contents, and the context is
 * ready for new work.  If a launch fails, the passes already queued count as executed and the rest is discarded. */
sg_status sg_flush(sg_ctx* ctx);
/* Trigger (1): flushes if s is pending, waits for the stream, copies the scalar (size of its dtype).
 * SG_ERR_CONTRACT if s is a quantifier that was NOT EVALUATED: its pass ended early at a violated registered contract before s was
 * decided (a for_all already false or an exists already true on the prefix read so far IS decided and readable). */
sg_status sg_scalar_get(sg_ctx* ctx, sg_handle s, void* host_out, size_t bytes);
sg_status sg_scalar_dtype(sg_ctx* ctx, sg_handle s, int32_t* dtype);
/* Trigger (2): count / device pointer of a collection; flushes (and syncs, for a filter output) if the collection is pending — or if
 * a pending in-place result lives in the same storage under ANOTHER handle (a subset / row view of it, the collection it is a view of):
 * handles that share storage behave like eager execution in program order. */
sg_status sg_vec_count(sg_ctx* ctx, sg_handle v, int64_t* n);
sg_status sg_vec_data(sg_ctx* ctx, sg_handle v, void** dev_ptr);
/* to_array (PAPER.md:153-155, 195, 284 trigger (2)): flushes if pending, waits, copies the collection's elements
 * (count * element size bytes, contiguous) to HOST memory in one action.  bytes must be >= that size. */
sg_status sg_vec_read(sg_ctx* ctx, sg_handle v, void* host_out, size_t bytes);
/* Drop the caller's reference.  An unreferenced pending intermediate is never materialised.  A collection or scalar that a
 * pending operation still reads may be released before the flush: its storage lives until that flush has consumed it.
 * After the last release the handle is invalid (SG_ERR_ARG); its table slot is reused by later handles. */
sg_status sg_release(sg_ctx* ctx, sg_handle h);

/* transpose: a NEW cols x rows matrix with out[j][i] = m[i][j] (F32/F64/I32/I64), written to dev_out_or_null
 * (borrowed, leading dimension ld_out elements; NULL => allocated by the context; ld_out 0 => rows of m).  A pure data mover with
 * no elementwise body to fuse into, so it is not deferred: operations pending on m are flushed first (trigger (2)),
 * then one tiled kernel is enqueued on the context stream (asynchronous; nothing is read back).  Errors: SG_ERR_ARG,
 * SG_ERR_DTYPE (BOOL), SG_ERR_ALIAS (dev_out overlaps m), SG_ERR_OOM, SG_ERR_CUDA. */
sg_status sg_mat_transpose(sg_ctx* ctx, sg_handle m, void* dev_out_or_null, int64_t ld_out, sg_handle* out_mat);

/* Listing 5's loop for steps k in [k0, k1) of the square F64 matrix m (any size and leading dimension), run by
 * ONE persistent kernel without the host in the loop (the paper's per-row launches are its slow case,
 * PAPER.md:389).  det and minpiv are one-element F64 vectors with storage; the caller initialises det to 1 (`Result := 1`) and
 * minpiv to +inf.  Step k, in the listing's statement order:
 *     pivot := M[k,k];  det <- det * pivot;  minpiv <- MIN(minpiv, ABS(pivot));
 *     if |pivot| <= eps (`double_approx_equals (pivot, 0.0)` with the explicit eps the paper leaves open): the loop
 *         ENDS — no row is touched by this or any later step, det keeps the product including this pivot (a signed zero for
 *         eps = 0), and a later call on the same det/minpiv does nothing (minpiv <= eps records the exit);
 *     else for ALL rows j > k whose entry M[j,k] is not approximately zero:
 *         M[j,:] <- M[j,:] - (M[j,k] / M[k,k]) * M[k,:]   (BASELINE.json:configs[4]'s update over all columns, one rounding per
 *         primitive; the factor is read before the row changes).
 * Not deferred: operations pending on the context are flushed first, then the kernel is enqueued on the stream (asynchronous,
 * nothing is read back: n steps run without a host synchronisation).  The zero-pivot decision is taken on the device; the
 * caller reads det and, if it wants the listing's `ok`, tests minpiv > eps.
 * Errors: SG_ERR_ARG (handles, range, eps < 0 or NaN), SG_ERR_SHAPE (not square, det/minpiv not one element), SG_ERR_DTYPE,
 * SG_ERR_CUDA. */
sg_status sg_mat_ge_steps(sg_ctx* ctx, sg_handle m, sg_handle det, sg_handle minpiv, double eps, int64_t k0, int64_t k1);

/* Listing 3's quicksort as a library composite: Result = quicksort(left) ++ mid ++
 * quicksort(right) with pivot a[a.count // 2] and the three STABLE filters item < / = / > pivot, so the result is the stable sort
 * of v (equal keys, -0 and +0 included, keep their order).  One launch per recursion LEVEL: every partition of a level is a
 * segment of one buffer, a tile is read once and its three compactions are written in the same pass (multi-output partition,
 * ranks by one decoupled look-back chain per segment), `concatenate` is free (left and right are written at their final
 * offsets); segments that fit one block are finished in shared memory.  Counts and segment tables stay on the device; the host
 * reads 20 bytes per batch of levels to learn whether work is left.  *out is a NEW vector (dev_out_or_null: caller's buffer of
 * v.count elements, else allocated by the context); v is not modified.  Not deferred: pending operations are flushed first.
 * Errors: SG_ERR_EMPTY (the listing's precondition a.count > 0), SG_ERR_DTYPE (BOOL), SG_ERR_ARG (not a unit-stride vector),
 * SG_ERR_ALIAS (dev_out overlaps v), SG_ERR_OOM, SG_ERR_CUDA, and SG_ERR_CONTRACT when a key is neither <, = nor > its pivot (a
 * NaN): the listing's three filters would drop it and violate its own postcondition Result.count = a.count. */
sg_status sg_vec_quicksort(sg_ctx* ctx, sg_handle v, void* dev_out_or_null, sg_handle* out);

/* The `sum` reduction for callers that MAY NOT ALLOCATE: code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc.  Takes no context and calls no cudaMalloc, cudaFree or allocating library
 * routine: the scratch memory of the reduction (one 16-byte partial per 8192 elements + the last-block ticket) is a file-scope
 * static __device__ array of SG_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.
 *   device    CUDA device ordinal (0 .. 63); made current for the call and restored
 *   stream    cudaStream_t of that device (NULL: the default stream); the call enqueues one 256-byte memset (the ticket must
 *             start at zero) and one kernel on it and returns without synchronising
 *   dtype     SG_F32 or SG_F64 (else SG_ERR_DTYPE)
 *   dev_x     DEVICE pointer, n elements, unit stride, aligned to the element size (16-byte alignment takes the 128-bit path);
 *             owned by the caller, read only
 *   n         0 <= n <= SG_NOALLOC_MAX_N; more is rejected with SG_ERR_CAPACITY and a message, nothing is launched
 *   dev_out   DEVICE pointer to one double, owned by the caller: receives the sum (n = 0: +0.0), valid when the stream reaches it
 *   err/errcap  optional HOST buffer for the error text (there is no context to ask)
 * Arithmetic = sg_reduce(SG_SUM): fp64 input in double-double TwoSum cells, fp32 input in fp64, partials combined in tile
 * order by the last block to finish (deterministic, independent of the grid); the same tolerances hold.
 * SHARED STATE: every call on a device uses the same array, which keeps the last call's contents.  Calls that OVERLAP on the GPU
 * (different streams, or host threads that do not order their calls) race on it; order them on one stream or with events.
 * Errors: SG_ERR_ARG, SG_ERR_DTYPE, SG_ERR_CAPACITY, SG_ERR_CUDA (no usable device: there is no CPU fallback). */
#define SG_NOALLOC_MAX_N ((int64_t)1 << 27)
#define SG_NOALLOC_SCRATCH_BYTES (256 + 16 * 16384)
sg_status sg_vec_sum_noalloc(int32_t device, void* stream, sg_dtype dtype, const void* dev_x, int64_t n, double* dev_out, char* err, int64_t errcap);

sg_status sg_plan_stats(sg_ctx* ctx, sg_stats* out);
/* Canonical program of pass `pass` of the last flush as text (template generator, tests). Returns bytes needed. */
int64_t sg_plan_dump(sg_ctx* ctx, int32_t pass, char* buf, int64_t cap);
/* Device time of the last flush's launches in milliseconds (CUDA events on the context's stream). */
/* Plan cache (the optimizer runs at every trigger; a loop triggers the same pending list again and again): the pass
 * assignment of a pending list is remembered under the list's signature — operations, the identity pattern, storage and liveness of
 * the values they name, contracts, flags; immediates excluded — and re-used when the same list over the same buffers is flushed
 * again.  Programs are built and bound to their pointers by every flush.  Counts since the context was created. */
sg_status sg_plan_cache_stats(sg_ctx* ctx, int64_t* hits, int64_t* misses);
sg_status sg_last_flush_ms(sg_ctx* ctx, float* ms);
/* Device time of every flush between begin and end, without a host synchronisation inside the region: each flush records
 * its own CUDA event pair on the context's stream; sg_timing_end waits for the last one and returns the sum in
 * milliseconds and the number of flushes (the measurement of a pipelined sequence of steps). */
sg_status sg_timing_begin(sg_ctx* ctx);
sg_status sg_timing_end(sg_ctx* ctx, float* total_ms, int32_t* n_flushes);
/* Replays the last flush's launch sequence `reps` times on the stream (same buffers, same plan, no host plan
 * build) and returns the mean device time per replay in ms: the measurement entry point. */
sg_status sg_replay_last(sg_ctx* ctx, int32_t reps, float* ms_per_rep);
/* The same launch sequence captured `reps` times in a row into ONE CUDA graph (programmatic dependent launches included), so the
 * device runs the repetitions back to back without the host in between; the graph is launched three times:
 * device time (CUDA events) and launch-inclusive wall time (host clock, first graph launch to stream completion), both per repetition
 * — the measurement of passes that take a few microseconds (SURVEY.md §8(d) note iii).  SG_ERR_UNSUPPORTED if the plan contains a
 * filter pass (its tile states are tagged with a per-launch epoch). */
sg_status sg_replay_last_graph(sg_ctx* ctx, int32_t reps, float* device_ms_per_rep, float* wall_ms_per_rep);
/* Number of precompiled template instances in the registry and the name of instance id k (1-based). */
int32_t sg_template_count(void);
const char* sg_template_name(int32_t k);
const char* sg_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SG_H_ */
