// sg_prog.h — the canonical program of one fused pass (internal; shared by the host plan builder and the kernels).
//
// A pass is what the optimizer of PAPER.md:301-309 leaves of a group of pending operations after merging
// kernel vertices and collapsing intermediates: distinct memory inputs, a straight-line elementwise body over
// registers, and outputs (stores of materialised collections, terminal reductions PAPER.md:203, quantifiers
// PAPER.md:145-151, stream compaction PAPER.md:141-143).  `SgProg` is plain data: its bytes are the pass
// SIGNATURE.  A precompiled template instance is selected when the bytes match (sg_templates_gen.inc); any
// other program runs on the bytecode kernel, which interprets the same bytes.
#ifndef SG_PROG_H_
#define SG_PROG_H_

#include <stdint.h>

enum : uint8_t {
    // value ops: V,V -> V
    OP_ADD = 0, OP_SUB = 1, OP_MUL = 2, OP_DIV = 3, OP_MIN = 4, OP_MAX = 5, OP_MOD = 6,
    // V -> V
    OP_NEG = 7, OP_ABS = 8,
    // V,V -> P
    OP_EQ = 9, OP_NE = 10, OP_LT = 11, OP_LE = 12, OP_GT = 13, OP_GE = 14,
    // P,P -> P ; P -> P
    OP_AND = 15, OP_OR = 16, OP_NOT = 17,
    // V -> V copy (materialising an input into another buffer)
    OP_MOV = 18,
    // V -> V, float dtypes only: correctly rounded square root (`project(agent sqrt)`)
    OP_SQRT = 19,
    OP_COUNT_
};

enum : uint8_t {
    IN_VEC = 0,     // unit-stride collection, element i of the pass domain at ptr[i]
    IN_SHIFT = 1,   // element i is element i+1 of input `ref` (neighbour predicates)
    IN_STRIDED = 2, // element i at ptr[i*stride] (column(j) of a row-major matrix)
    IN_SCALAR = 3,  // one device scalar broadcast to every element (closed agent argument)
    IN_IMM = 4,     // host immediate, passed as a kernel argument (the `a` of aX+Y)
    IN_ROWB = 5,    // 2-D: vector indexed by the column, same for every row
    IN_COLB = 6,    // 2-D: vector indexed by the row, same for every column
    IN_BOOLVEC = 7, // unit-stride BOOL collection (1 byte per element) loaded into a predicate register
    IN_VEC_CVT = 8  // unit-stride collection of ANOTHER element type (`ref` = its DT_*), converted to the pass dtype as it is loaded:
                    // the dtype-changing `project (transform: FUNCTION[T, U]): COLLECTION[U]` of PAPER.md:137-139, 171-175
};

enum : uint8_t {
    OUT_STORE = 0,      // materialise V reg `src`
    OUT_STORE_BOOL = 1, // materialise P reg `src` as bytes
    OUT_SUM = 2, OUT_MAX = 3, OUT_MIN = 4,   // reductions of V reg `src` (masked by P reg `pred` unless 0xFF)
    OUT_ALL = 5, OUT_ANY = 6, OUT_COUNT = 7, // quantifiers / count of P reg `src`
    OUT_FILTER = 8      // stable compaction of V reg `src` where P reg `pred`
};

enum : uint8_t { AXIS_ALL = 0, AXIS_ROWS = 1, AXIS_COLS = 2 };
enum : uint8_t { DT_F32 = 0, DT_F64 = 1, DT_I32 = 2, DT_I64 = 3, DT_BOOL = 4 };

enum : uint8_t {
    PF_2D = 1,          // matrix domain (rows x cols with leading dimension)
    PF_FILTER = 2,      // has an OUT_FILTER (decoupled look-back kernel)
    PF_EARLY_EXIT = 4   // only quantifier outputs: blocks poll the decided word once per tile
};

#define SG_MAX_IN 10
#define SG_MAX_INSTR 32
#define SG_MAX_OUT 8
#define SG_MAX_VREG 24
#define SG_MAX_PREG 8
#define SG_NO_PRED 0xFF
#define SG_MAX_TMAP 2

struct SgInstr { uint8_t op, dst, a, b; };
struct SgIn { uint8_t kind, ref, reg, pad; };      // ref: IN_SHIFT: the shifted input; IN_VEC_CVT: source DT_*.  reg: V (or P for IN_BOOLVEC) register the input is loaded into
struct SgOut { uint8_t kind, src, pred, axis; };

struct SgShape {
    uint8_t dtype;      // element type of the V file
    uint8_t flags;      // PF_*
    uint8_t n_in, n_instr, n_out, n_vreg, n_preg, pad;
};

struct SgProg {
    SgShape shape;
    SgIn in[SG_MAX_IN];
    SgInstr code[SG_MAX_INSTR];
    SgOut out[SG_MAX_OUT];
};

// Truncating int32 division by a pass constant d, |d| >= 2: q = (mulhi(x, M) + x*addsel) >> s, plus one if negative.
struct SgDiv { int32_t M, addsel, s, neg_d; uint32_t valid, pad[3]; };

// Runtime arguments of one pass (never part of the signature).
struct SgArgs {
    int64_t n;                      // 1-D: domain length; 2-D: rows
    int64_t cols;                   // 2-D: columns
    const void* in_ptr[SG_MAX_IN];  // element 0 of the pass domain (IN_SHIFT: unused)
    int64_t in_len[SG_MAX_IN];      // elements readable through the input (guards the ragged path)
    int64_t in_stride[SG_MAX_IN];   // IN_STRIDED: element stride; 2-D IN_VEC: leading dimension
    uint64_t imm[SG_MAX_IN];        // IN_IMM: raw bits of the immediate in the pass dtype
    SgDiv imm_div[SG_MAX_IN];       // IN_IMM, i32 passes: signed magic number for division/modulo by the immediate (valid == 0 if |d| <= 1), see magic_div_i32
    void* out_ptr[SG_MAX_OUT];      // STORE: buffer; reductions/quantifiers: 8-byte device scalar slot (AXIS_ALL) or vector
    void* out_host[SG_MAX_OUT];     // AXIS_ALL reductions/quantifiers: the slot's place in the PINNED HOST mirror, written by the last block
                                    // together with the device slot (no copy engine between two passes of a stream), or null
    int64_t out_len[SG_MAX_OUT];    // valid length of the output's source value (<= n); 2-D STORE: leading dimension
    int64_t out_cap[SG_MAX_OUT];    // FILTER: capacity in elements
    void* out_aux[SG_MAX_OUT];      // FILTER: device int64 slot that receives the kept count
    void* workspace;                // per-block partials: [grid][SG_MAX_OUT] 16-byte cells (+ tile states for filter)
    unsigned long long* tile_state; // FILTER: one state word per tile (dedicated buffer, see sg_filter.cuh)
    unsigned int* ctrl;             // zeroed control words: [0] ticket, [1] decided mask, [2] dynamic tile counter, [3] overflow
    int64_t head;                   // leading elements handled by the ragged path so that the body is 16-byte aligned
    int64_t n_full_tiles;           // full tiles of the aligned body
    int64_t static_tiles;           // 1-D template passes: tiles [0, static_tiles) are taken strided (block + it * grid); the tiles after them are
                                    // handed out by tickets on ctrl[2] (passes with reductions only; = n_full_tiles: no tickets), see sg_kernels.cu
    int32_t vec_ok;                 // bit i: input i may use 128-bit loads; bit (16+o): output o may use 128-bit stores
    int32_t no_early_exit;
    uint32_t exit_any;              // quantifier outputs that are registered for_all contracts: one violation ends the pass
    uint32_t epoch;                 // FILTER: tags the tile states of this launch (stale states of earlier launches are invalid)
    int32_t n_tiles;                // FILTER: tiles of the look-back scan
    // 2-D tiling
    int32_t n_strips, n_chunks;
    int64_t rows_per_chunk;
    int64_t ws_off[SG_MAX_OUT];     // 2-D: byte offset in workspace of the per-chunk (AXIS_COLS) / per-strip (AXIS_ROWS) partial cells
    // FILTER: TMA tensor maps (CUtensorMap, 128 bytes each) of the staged inputs, encoded by the launcher: the input seen as
    // rows of 128 bytes, box = 256 rows, 128-byte swizzle (sg_filter.cuh); vec_ok bit 30 says they are valid
    alignas(64) unsigned char tmap[SG_MAX_TMAP][128];
};

#endif  // SG_PROG_H_
