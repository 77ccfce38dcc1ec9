// CPU ORACLE — TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, single-threaded evaluator of the SafeGPU collection primitives
// (arXiv 1410.6685).  Every primitive is its own full loop that reads fully
// materialised inputs and writes a fully materialised output: this is literally
// the "one kernel per method call, launched one after the other" plan that the
// paper names as the naive design.  The fused GPU plan must reach
// exactly these values (fusion only merges kernels / collapses intermediates,
// PAPER.md:301-309), so the oracle is the plain definition written out.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may load this library.  It shares no code with the CUDA path.
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py).
// -ffp-contract=off is mandatory: every elementwise op rounds once (R1).
//
// Parity pins: every function below is pinned by tests/test_oracle_*.py
// (closed forms, exact rational re-evaluation, library routines, brute force).
//
// dtype codes: 0 = f32, 1 = f64, 2 = i32, 3 = i64.   Booleans are 1 byte, 0/1.
// All functions return 0 on success, a negative code on a bad argument.

#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>

namespace {

enum { F32 = 0, F64 = 1, I32 = 2, I64 = 3 };
enum { ADD = 0, SUB = 1, MUL = 2, DIV = 3, MIN = 4, MAX = 5, MOD = 6 };      // binary arithmetic
enum { NEG = 0, ABS = 1, SQRT = 2 };                                          // unary
enum { EQ = 0, NE = 1, LT = 2, LE = 3, GT = 4, GE = 5 };                      // comparisons
enum { AND = 0, OR = 1, NOT = 2 };                                            // logical

// ---------------------------------------------------------------------------
// Elementwise arithmetic (PAPER.md:205 plus/minus/multiplied_by/divided_by and
// component-wise variants; PAPER.md:133-139 for_each/project).
// Floats: one IEEE-754 round-to-nearest operation per primitive.
// Integers: two's-complement wrap-around; DIV/MOD truncate toward zero;
// divisor 0 -> result 0 (the built-in non-zero contract reports it);
// INT_MIN / -1 -> INT_MIN, INT_MIN % -1 -> 0   (R14).
// MIN(a,b) = (b<a)?b:a ; MAX(a,b) = (a<b)?b:a  (DESIGN.md R-minmax).
// ---------------------------------------------------------------------------
template <class T> struct UnsignedOf;
template <> struct UnsignedOf<int32_t> { typedef uint32_t type; };
template <> struct UnsignedOf<int64_t> { typedef uint64_t type; };

template <class T> bool float_bin(int op, T a, T b, T* r) {
    switch (op) {
        case ADD: *r = a + b; return true;
        case SUB: *r = a - b; return true;
        case MUL: *r = a * b; return true;
        case DIV: *r = a / b; return true;
        case MIN: *r = (b < a) ? b : a; return true;
        case MAX: *r = (a < b) ? b : a; return true;
        default: return false;
    }
}

template <class T> bool int_bin(int op, T a, T b, T* r) {
    typedef typename UnsignedOf<T>::type U;
    const T lowest = std::numeric_limits<T>::min();
    switch (op) {
        case ADD: *r = (T)((U)a + (U)b); return true;
        case SUB: *r = (T)((U)a - (U)b); return true;
        case MUL: *r = (T)((U)a * (U)b); return true;
        case DIV:
            if (b == 0) *r = 0;
            else if (a == lowest && b == (T)-1) *r = lowest;
            else *r = a / b;
            return true;
        case MOD:
            if (b == 0) *r = 0;
            else if (b == (T)-1) *r = 0;
            else *r = a % b;
            return true;
        case MIN: *r = (b < a) ? b : a; return true;
        case MAX: *r = (a < b) ? b : a; return true;
        default: return false;
    }
}

inline bool bin(int op, float a, float b, float* r) { return float_bin(op, a, b, r); }
inline bool bin(int op, double a, double b, double* r) { return float_bin(op, a, b, r); }
inline bool bin(int op, int32_t a, int32_t b, int32_t* r) { return int_bin(op, a, b, r); }
inline bool bin(int op, int64_t a, int64_t b, int64_t* r) { return int_bin(op, a, b, r); }

// zip: out[i] = a[i] op b[i]
template <class T> int zip_t(int op, int64_t n, const T* a, const T* b, T* out) {
    for (int64_t i = 0; i < n; ++i)
        if (!bin(op, a[i], b[i], &out[i])) return -2;
    return 0;
}
// scalar: out[i] = a[i] op s   (reversed: s op a[i])
template <class T> int scalar_t(int op, int64_t n, const T* a, T s, int reversed, T* out) {
    for (int64_t i = 0; i < n; ++i) {
        bool ok = reversed ? bin(op, s, a[i], &out[i]) : bin(op, a[i], s, &out[i]);
        if (!ok) return -2;
    }
    return 0;
}

// unary NEG / ABS: sign-bit operations for floats (abs(-0) = +0), wrap for ints.
// SQRT (the agent of Listing `project`: `a.project(agent sqrt)`): the IEEE-754 correctly rounded
// square root in the collection's own dtype (sqrt(-0) = -0, sqrt(x<0) = NaN); floats only (R20).
inline float un(int op, float a) {
    if (op == SQRT) return std::sqrt(a);
    uint32_t u; std::memcpy(&u, &a, 4);
    u = (op == NEG) ? (u ^ 0x80000000u) : (u & 0x7fffffffu);
    std::memcpy(&a, &u, 4); return a;
}
inline double un(int op, double a) {
    if (op == SQRT) return std::sqrt(a);
    uint64_t u; std::memcpy(&u, &a, 8);
    u = (op == NEG) ? (u ^ 0x8000000000000000ull) : (u & 0x7fffffffffffffffull);
    std::memcpy(&a, &u, 8); return a;
}
inline int32_t un(int op, int32_t a) {
    uint32_t u = (uint32_t)a;
    if (op == NEG || a < 0) u = 0u - u;
    return (int32_t)u;
}
inline int64_t un(int op, int64_t a) {
    uint64_t u = (uint64_t)a;
    if (op == NEG || a < 0) u = 0ull - u;
    return (int64_t)u;
}
template <class T> int unary_t(int op, int64_t n, const T* a, T* out) {
    if (op == SQRT && std::numeric_limits<T>::is_integer) return -3;
    if (op != NEG && op != ABS && op != SQRT) return -2;
    for (int64_t i = 0; i < n; ++i) out[i] = un(op, a[i]);
    return 0;
}

// comparisons -> BOOL (IEEE: NaN compares false except NE; -0 == +0)
template <class T> bool cmp1(int c, T a, T b, uint8_t* r) {
    switch (c) {
        case EQ: *r = (a == b); return true;
        case NE: *r = (a != b); return true;
        case LT: *r = (a < b); return true;
        case LE: *r = (a <= b); return true;
        case GT: *r = (a > b); return true;
        case GE: *r = (a >= b); return true;
        default: return false;
    }
}
template <class T> int cmp_t(int c, int64_t n, const T* a, const T* b, uint8_t* out) {
    for (int64_t i = 0; i < n; ++i)
        if (!cmp1(c, a[i], b[i], &out[i])) return -2;
    return 0;
}
template <class T> int cmp_scalar_t(int c, int64_t n, const T* a, T s, uint8_t* out) {
    for (int64_t i = 0; i < n; ++i)
        if (!cmp1(c, a[i], s, &out[i])) return -2;
    return 0;
}
// neighbour predicate b_i = x_i cmp x_{i+1}, i in [0, n-2]: the zip of subset(0,n-1)
// with subset(1,n) (is_sorted PAPER.md:203, 261).
template <class T> int adj_t(int c, int64_t n, const T* a, uint8_t* out) {
    for (int64_t i = 0; i + 1 < n; ++i)
        if (!cmp1(c, a[i], a[i + 1], &out[i])) return -2;
    return 0;
}

// ---------------------------------------------------------------------------
// Reductions (PAPER.md:203 sum/min/max "by multiple reductions on the device").
// SUM of floats: long double accumulator, ascending index order, Neumaier
// compensation, rounded once to double (R1/S).  Ints: wrap-around int64.
// ---------------------------------------------------------------------------
template <class T> double sum_float(int64_t n, const T* a) {
    long double s = 0.0L, c = 0.0L;
    for (int64_t i = 0; i < n; ++i) {
        long double x = (long double)a[i];
        long double t = s + x;
        long double as = s < 0 ? -s : s, ax = x < 0 ? -x : x;
        if (as >= ax) c += (s - t) + x; else c += (x - t) + s;
        s = t;
    }
    return (double)(s + c);
}
template <class T> int64_t sum_int(int64_t n, const T* a) {
    uint64_t s = 0;
    for (int64_t i = 0; i < n; ++i) s += (uint64_t)(int64_t)a[i];
    return (int64_t)s;
}

// MAX / MIN under the IEEE total order on bit patterns (-0 < +0; NaNs outside +-inf):
// map sign-magnitude bits to a monotone unsigned key (R15).
inline uint32_t key(float a) {
    uint32_t u; std::memcpy(&u, &a, 4);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
inline uint64_t key(double a) {
    uint64_t u; std::memcpy(&u, &a, 8);
    return (u & 0x8000000000000000ull) ? ~u : (u | 0x8000000000000000ull);
}
inline uint32_t key(int32_t a) { return (uint32_t)a ^ 0x80000000u; }
inline uint64_t key(int64_t a) { return (uint64_t)a ^ 0x8000000000000000ull; }

template <class T> int extremum_t(int is_max, int64_t n, const T* a, T* out) {
    if (n <= 0) return -4;                      // empty: error (R4)
    T best = a[0];
    for (int64_t i = 1; i < n; ++i) {
        bool better = is_max ? (key(a[i]) > key(best)) : (key(a[i]) < key(best));
        if (better) best = a[i];
    }
    *out = best;
    return 0;
}

// filter: stable compaction, ascending index order.
template <class T> int64_t filter_t(int64_t n, const T* a, const uint8_t* mask, T* out) {
    int64_t m = 0;
    for (int64_t i = 0; i < n; ++i)
        if (mask[i]) out[m++] = a[i];
    return m;
}

// ---------------------------------------------------------------------------
// project (transform: FUNCTION[T, U]): COLLECTION[U] with the value-preserving conversion as the
// transform — the INT -> DOUBLE half of the paper's example `agent (a: INT): DOUBLE do Result := sqrt (a) end`
// (PAPER.md:171-175).  The paper does not define conversions; the reading (R23):
//   integer -> float : the nearest representable value, ties to even (an int32 is always exact in a double);
//   float -> integer : truncation toward zero; values beyond the target's range saturate at its ends; NaN -> 0;
//   double -> float  : round to nearest even;  float -> double, int32 -> int64 : exact;
//   int64 -> int32   : the low 32 bits (two's-complement wrap, like every integer operation here, R14).
// Written out case by case; the range tests are done in the floating type, where 2^31 and 2^63 are exact.
// ---------------------------------------------------------------------------
// float -> integer, F in {float, double}, I in {int32_t, int64_t}; two_p = 2^31 or 2^63 is exact in both floating types
template <class I, class F> I float_to_int(F x, F two_p) {
    if (x != x) return 0;                                                  // NaN
    if (x >= two_p) return std::numeric_limits<I>::max();                  // saturate
    if (x <= -two_p) return std::numeric_limits<I>::min();                 // -2^31 / -2^63 themselves are the minimum
    return (I)std::trunc(x);                                               // |x| < 2^(bits-1): the truncated value is representable
}
inline void cv(float x, float* r) { *r = x; }
inline void cv(float x, double* r) { *r = (double)x; }                                     // exact
inline void cv(float x, int32_t* r) { *r = float_to_int<int32_t, float>(x, 2147483648.0f); }
inline void cv(float x, int64_t* r) { *r = float_to_int<int64_t, float>(x, 9223372036854775808.0f); }
inline void cv(double x, float* r) { *r = (float)x; }                                      // IEEE round to nearest even
inline void cv(double x, double* r) { *r = x; }
inline void cv(double x, int32_t* r) { *r = float_to_int<int32_t, double>(x, 2147483648.0); }
inline void cv(double x, int64_t* r) { *r = float_to_int<int64_t, double>(x, 9223372036854775808.0); }
inline void cv(int32_t x, float* r) { *r = (float)x; }                                     // IEEE round to nearest even
inline void cv(int32_t x, double* r) { *r = (double)x; }                                   // exact
inline void cv(int32_t x, int32_t* r) { *r = x; }
inline void cv(int32_t x, int64_t* r) { *r = (int64_t)x; }                                 // sign extension
inline void cv(int64_t x, float* r) { *r = (float)x; }                                     // IEEE round to nearest even
inline void cv(int64_t x, double* r) { *r = (double)x; }                                   // IEEE round to nearest even
inline void cv(int64_t x, int32_t* r) { *r = (int32_t)(uint32_t)(uint64_t)x; }             // low 32 bits
inline void cv(int64_t x, int64_t* r) { *r = x; }
template <class T, class S> void cast_loop(int64_t n, const S* a, T* out) {
    for (int64_t i = 0; i < n; ++i) cv(a[i], &out[i]);
}
template <class S> int cast_from(int to, int64_t n, const S* a, void* out) {
    switch (to) {
        case F32: cast_loop(n, a, (float*)out); return 0;
        case F64: cast_loop(n, a, (double*)out); return 0;
        case I32: cast_loop(n, a, (int32_t*)out); return 0;
        case I64: cast_loop(n, a, (int64_t*)out); return 0;
        default: return -1;
    }
}

}  // namespace

#define DISPATCH(dtype, CALL)                                  \
    switch (dtype) {                                           \
        case F32: { typedef float T; return CALL; }            \
        case F64: { typedef double T; return CALL; }           \
        case I32: { typedef int32_t T; return CALL; }          \
        case I64: { typedef int64_t T; return CALL; }          \
        default: return -1;                                    \
    }

extern "C" {

int orc_zip(int op, int dtype, int64_t n, const void* a, const void* b, void* out) {
    DISPATCH(dtype, zip_t<T>(op, n, (const T*)a, (const T*)b, (T*)out));
}

// s points to ONE scalar already converted to the vector dtype at enqueue (DESIGN.md R-imm).
int orc_scalar(int op, int dtype, int64_t n, const void* a, const void* s, int reversed, void* out) {
    DISPATCH(dtype, scalar_t<T>(op, n, (const T*)a, *(const T*)s, reversed, (T*)out));
}

int orc_unary(int op, int dtype, int64_t n, const void* a, void* out) {
    DISPATCH(dtype, unary_t<T>(op, n, (const T*)a, (T*)out));
}

int orc_cmp(int c, int dtype, int64_t n, const void* a, const void* b, uint8_t* out) {
    DISPATCH(dtype, cmp_t<T>(c, n, (const T*)a, (const T*)b, out));
}

int orc_cmp_scalar(int c, int dtype, int64_t n, const void* a, const void* s, uint8_t* out) {
    DISPATCH(dtype, cmp_scalar_t<T>(c, n, (const T*)a, *(const T*)s, out));
}

int orc_adj(int c, int dtype, int64_t n, const void* a, uint8_t* out) {
    DISPATCH(dtype, adj_t<T>(c, n, (const T*)a, out));
}

int orc_logic(int op, int64_t n, const uint8_t* a, const uint8_t* b, uint8_t* out) {
    for (int64_t i = 0; i < n; ++i) {
        bool x = a[i] != 0, y = (op == NOT) ? false : (b[i] != 0);
        switch (op) {
            case AND: out[i] = x && y; break;
            case OR: out[i] = x || y; break;
            case NOT: out[i] = !x; break;
            default: return -2;
        }
    }
    return 0;
}

// out: double for f32/f64 inputs, int64 for i32/i64 inputs.  Empty -> 0.
int orc_sum(int dtype, int64_t n, const void* a, void* out) {
    switch (dtype) {
        case F32: *(double*)out = sum_float(n, (const float*)a); return 0;
        case F64: *(double*)out = sum_float(n, (const double*)a); return 0;
        case I32: *(int64_t*)out = sum_int(n, (const int32_t*)a); return 0;
        case I64: *(int64_t*)out = sum_int(n, (const int64_t*)a); return 0;
        default: return -1;
    }
}

int orc_extremum(int is_max, int dtype, int64_t n, const void* a, void* out) {
    DISPATCH(dtype, extremum_t<T>(is_max, n, (const T*)a, (T*)out));
}

// for_all / exists / count of a BOOL vector.  Empty: ALL = 1, ANY = 0.
int orc_all(int64_t n, const uint8_t* m, uint8_t* out) {
    uint8_t r = 1;
    for (int64_t i = 0; i < n; ++i) r = r && (m[i] != 0);
    *out = r; return 0;
}
int orc_any(int64_t n, const uint8_t* m, uint8_t* out) {
    uint8_t r = 0;
    for (int64_t i = 0; i < n; ++i) r = r || (m[i] != 0);
    *out = r; return 0;
}
int orc_count(int64_t n, const uint8_t* m, int64_t* out) {
    int64_t c = 0;
    for (int64_t i = 0; i < n; ++i) c += (m[i] != 0);
    *out = c; return 0;
}

// returns the number of kept items in *count; out must have room for n items.
int orc_filter(int dtype, int64_t n, const void* a, const uint8_t* mask, void* out, int64_t* count) {
    switch (dtype) {
        case F32: *count = filter_t(n, (const float*)a, mask, (float*)out); return 0;
        case F64: *count = filter_t(n, (const double*)a, mask, (double*)out); return 0;
        case I32: *count = filter_t(n, (const int32_t*)a, mask, (int32_t*)out); return 0;
        case I64: *count = filter_t(n, (const int64_t*)a, mask, (int64_t*)out); return 0;
        default: return -1;
    }
}

// ---------------------------------------------------------------------------
// Matrix primitives (row-major storage).
// ---------------------------------------------------------------------------

// column(j): copy of the corresponding elements into new storage.
int orc_mat_col(int64_t rows, int64_t ld, const double* M, int64_t j, double* out) {
    for (int64_t r = 0; r < rows; ++r) out[r] = M[r * ld + j];
    return 0;
}

// out[r][c] = f[r] * p[c]: the product of a COL-broadcast vector and a ROW-broadcast vector.
int orc_outer_mul(int64_t rows, int64_t cols, const double* f, const double* p, double* out) {
    for (int64_t r = 0; r < rows; ++r)
        for (int64_t c = 0; c < cols; ++c) out[r * cols + c] = f[r] * p[c];
    return 0;
}

// per-row extremum (total order) of a rows x cols block with leading dimension ld.
int orc_row_extremum(int is_max, int64_t rows, int64_t cols, int64_t ld, const double* M, double* out) {
    if (cols <= 0) return -4;
    for (int64_t r = 0; r < rows; ++r) {
        int e = extremum_t<double>(is_max, cols, M + r * ld, &out[r]);
        if (e) return e;
    }
    return 0;
}

// per-column sum over the rows of a block: long double, ascending row order, compensated.
int orc_col_sum(int64_t rows, int64_t cols, int64_t ld, const double* M, double* out) {
    for (int64_t c = 0; c < cols; ++c) {
        long double s = 0.0L, comp = 0.0L;
        for (int64_t r = 0; r < rows; ++r) {
            long double x = (long double)M[r * ld + c];
            long double t = s + x;
            long double as = s < 0 ? -s : s, ax = x < 0 ? -x : x;
            if (as >= ax) comp += (s - t) + x; else comp += (x - t) + s;
            s = t;
        }
        out[c] = (double)(s + comp);
    }
    return 0;
}

// The Gaussian-elimination row-update step of BASELINE.json:configs[4] as one plain
// definition (SURVEY.md §8(c) "matrix"; PAPER.md:315-322, 337-356 for the fused row
// operation it comes from): for every row j > kr and every column c,
//     f_j = M[j][kc] / M[kr][kc]      (read before row j is modified)
//     t   = f_j * M[kr][c]            (rounded)
//     M[j][c] = M[j][c] - t           (rounded)
// then rowmax[j-kr-1] = max_c |M'[j][c]| (total order) and
//      colsum[c] = sum_{j>kr} M'[j][c] (long double, ascending j, compensated).
// kr = pivot row, kc = pivot column (kr == kc == k in the config; they are separate
// so that a test can run the definition on a column-sampled copy of a large matrix).
int orc_mat_step(int64_t rows, int64_t cols, int64_t ld, double* M, int64_t kr, int64_t kc,
                 double* rowmax, double* colsum) {
    if (kr < 0 || kr >= rows || kc < 0 || kc >= cols) return -3;
    const double pivot = M[kr * ld + kc];
    for (int64_t j = kr + 1; j < rows; ++j) {
        const double f = M[j * ld + kc] / pivot;
        for (int64_t c = 0; c < cols; ++c) {
            double t = f * M[kr * ld + c];
            M[j * ld + c] = M[j * ld + c] - t;
        }
    }
    const int64_t m = rows - kr - 1;
    for (int64_t j = 0; j < m; ++j) {
        const double* row = M + (kr + 1 + j) * ld;
        double best = un(ABS, row[0]);
        for (int64_t c = 1; c < cols; ++c) {
            double v = un(ABS, row[c]);
            if (key(v) > key(best)) best = v;
        }
        rowmax[j] = best;
    }
    if (m > 0) return orc_col_sum(m, cols, ld, M + (kr + 1) * ld, colsum);
    for (int64_t c = 0; c < cols; ++c) colsum[c] = 0.0;
    return 0;
}

// Determinant by Gaussian elimination, Listing 5, step by step in the paper's order:
//     Result := 1
//     for step = 0 .. n-1:
//         pivot := M[step][step]
//         Result := Result * pivot                                  (PAPER.md:338 — BEFORE the test below)
//         if pivot is approximately 0 -> the loop ends              (PAPER.md:339 double_approx_equals(pivot, 0.0) and the
//                                                                    else-branch PAPER.md:341-343 `step := matrix.rows`; the
//                                                                    paper leaves eps open: |pivot| <= eps, R5)
//         for every row j > step:
//             p_j := M[j][step]
//             if p_j is approximately 0 -> row j is left as it is   (PAPER.md:351 `if not double_approx_equals (pivot, 0.0)`)
//             else the row operation
// So a matrix with an approximately-zero pivot returns Result * pivot: a signed zero when eps = 0, a small non-zero
// number when eps > 0 — never a hard-wired 0.0 (R11a).
// The listing's row operation itself is garbled and rescales row j; the reading taken is
// BASELINE.json:configs[4]'s textbook update, the same orc_mat_step defines: f_j = p_j / pivot (read before the row
// changes), t = f_j * M[step][c], M[j][c] = M[j][c] - t, one rounding per primitive (R11).  M is overwritten by
// the eliminated matrix; *zero_step = the step whose pivot was ~0, or -1.
int orc_ge_determinant(int64_t n, int64_t ld, double* M, double eps, double* det, int64_t* zero_step) {
    if (n < 0 || ld < n) return -3;
    double result = 1.0;
    *zero_step = -1;
    for (int64_t step = 0; step < n; ++step) {
        const double pivot = M[step * ld + step];
        result = result * pivot;
        if (un(ABS, pivot) <= eps) { *zero_step = step; break; }
        for (int64_t j = step + 1; j < n; ++j) {
            const double pj = M[j * ld + step];
            if (un(ABS, pj) <= eps) continue;
            const double f = pj / pivot;
            for (int64_t c = 0; c < n; ++c) {
                double t = f * M[step * ld + c];
                M[j * ld + c] = M[j * ld + c] - t;
            }
        }
    }
    *det = result;
    return 0;
}

// dtype-changing projection: see cv() above (R23)
int orc_cast(int from, int to, int64_t n, const void* a, void* out) {
    switch (from) {
        case F32: return cast_from(to, n, (const float*)a, out);
        case F64: return cast_from(to, n, (const double*)a, out);
        case I32: return cast_from(to, n, (const int32_t*)a, out);
        case I64: return cast_from(to, n, (const int64_t*)a, out);
        default: return -1;
    }
}

}  // extern "C"
