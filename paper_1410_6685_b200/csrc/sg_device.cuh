// sg_device.cuh — device-side building blocks shared by every pass kernel (internal).
//   * elementwise primitives with exactly one IEEE rounding each (no FMA contraction: explicit _rn intrinsics,
//     and the library is compiled with -fmad=false),
//   * accumulator cells for the terminal reductions of PAPER.md:203 (double-double sums, total-order keys),
//   * warp-shuffle + shared-memory block reduction and the last-block-done cross-block combine.
#ifndef SG_DEVICE_CUH_
#define SG_DEVICE_CUH_

#include <cuda_runtime.h>
#include <stdint.h>

#include "sg_prog.h"

namespace sgk {

constexpr int BLOCK = 256;
constexpr int WARPS = BLOCK / 32;

template <int DT> struct TypeOf;
template <> struct TypeOf<DT_F32> { typedef float type; };
template <> struct TypeOf<DT_F64> { typedef double type; };
template <> struct TypeOf<DT_I32> { typedef int32_t type; };
template <> struct TypeOf<DT_I64> { typedef long long type; };

template <class T> struct Traits;
template <> struct Traits<float> { static constexpr int V = 4; typedef float4 vec; static constexpr bool is_float = true; };
template <> struct Traits<double> { static constexpr int V = 2; typedef double2 vec; static constexpr bool is_float = true; };
template <> struct Traits<int32_t> { static constexpr int V = 4; typedef int4 vec; static constexpr bool is_float = false; };
template <> struct Traits<long long> { static constexpr int V = 2; typedef longlong2 vec; static constexpr bool is_float = false; };

// ---------------------------------------------------------------------------------------------------------
// elementwise primitives
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float p_add(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float p_sub(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float p_mul(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float p_div(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ double p_add(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double p_sub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double p_mul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double p_div(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ float p_mod(float a, float) { return a; }      // rejected at enqueue (SG_ERR_DTYPE)
__device__ __forceinline__ double p_mod(double a, double) { return a; }

__device__ __forceinline__ int32_t p_add(int32_t a, int32_t b) { return (int32_t)((uint32_t)a + (uint32_t)b); }
__device__ __forceinline__ int32_t p_sub(int32_t a, int32_t b) { return (int32_t)((uint32_t)a - (uint32_t)b); }
__device__ __forceinline__ int32_t p_mul(int32_t a, int32_t b) { return (int32_t)((uint32_t)a * (uint32_t)b); }
__device__ __forceinline__ int32_t p_div(int32_t a, int32_t b) {
    if (b == 0) return 0;
    if (b == -1) return (int32_t)(0u - (uint32_t)a);      // INT_MIN / -1 -> INT_MIN (wrap)
    return a / b;
}
__device__ __forceinline__ int32_t p_mod(int32_t a, int32_t b) {
    if (b == 0 || b == -1) return 0;
    return a % b;
}
__device__ __forceinline__ long long p_add(long long a, long long b) { return (long long)((unsigned long long)a + (unsigned long long)b); }
__device__ __forceinline__ long long p_sub(long long a, long long b) { return (long long)((unsigned long long)a - (unsigned long long)b); }
__device__ __forceinline__ long long p_mul(long long a, long long b) { return (long long)((unsigned long long)a * (unsigned long long)b); }
__device__ __forceinline__ long long p_div(long long a, long long b) {
    if (b == 0) return 0;
    if (b == -1) return (long long)(0ull - (unsigned long long)a);
    return a / b;
}
__device__ __forceinline__ long long p_mod(long long a, long long b) {
    if (b == 0 || b == -1) return 0;
    return a % b;
}

__device__ __forceinline__ float p_neg(float a) { return __int_as_float(__float_as_int(a) ^ 0x80000000); }
__device__ __forceinline__ float p_abs(float a) { return __int_as_float(__float_as_int(a) & 0x7fffffff); }
__device__ __forceinline__ double p_neg(double a) { return __longlong_as_double(__double_as_longlong(a) ^ 0x8000000000000000ll); }
__device__ __forceinline__ double p_abs(double a) { return __longlong_as_double(__double_as_longlong(a) & 0x7fffffffffffffffll); }
__device__ __forceinline__ int32_t p_neg(int32_t a) { return (int32_t)(0u - (uint32_t)a); }
__device__ __forceinline__ int32_t p_abs(int32_t a) { return a < 0 ? (int32_t)(0u - (uint32_t)a) : a; }
__device__ __forceinline__ long long p_neg(long long a) { return (long long)(0ull - (unsigned long long)a); }
__device__ __forceinline__ long long p_abs(long long a) { return a < 0 ? (long long)(0ull - (unsigned long long)a) : a; }

// correctly rounded IEEE square root in the pass dtype (sqrt.rn.f32 / sqrt.rn.f64: never the approximate MUFU path);
// the integer overloads only keep value_op<T> instantiable — sg_enqueue rejects SQRT on integer collections
__device__ __forceinline__ float p_sqrt(float a) { return __fsqrt_rn(a); }
__device__ __forceinline__ double p_sqrt(double a) { return __dsqrt_rn(a); }
__device__ __forceinline__ int32_t p_sqrt(int32_t a) { return a; }
__device__ __forceinline__ long long p_sqrt(long long a) { return a; }

// dtype conversion of the dtype-changing projection (sg_cast; R23): integer -> float rounds to
// nearest even; float -> integer truncates toward zero, saturates at the target's range and maps NaN to 0 (the NaN case is
// written out: the 64-bit hardware conversion returns INT64_MIN for it); F64 -> F32 rounds to nearest even; I64 -> I32 keeps
// the low 32 bits.
template <class T, class S> __device__ __forceinline__ T cvt_elem(S x);
template <> __device__ __forceinline__ float cvt_elem<float, float>(float x) { return x; }
template <> __device__ __forceinline__ double cvt_elem<double, double>(double x) { return x; }
template <> __device__ __forceinline__ int32_t cvt_elem<int32_t, int32_t>(int32_t x) { return x; }
template <> __device__ __forceinline__ long long cvt_elem<long long, long long>(long long x) { return x; }
template <> __device__ __forceinline__ float cvt_elem<float, double>(double x) { return __double2float_rn(x); }
template <> __device__ __forceinline__ float cvt_elem<float, int32_t>(int32_t x) { return __int2float_rn(x); }
template <> __device__ __forceinline__ float cvt_elem<float, long long>(long long x) { return __ll2float_rn(x); }
template <> __device__ __forceinline__ double cvt_elem<double, float>(float x) { return (double)x; }
template <> __device__ __forceinline__ double cvt_elem<double, int32_t>(int32_t x) { return __int2double_rn(x); }
template <> __device__ __forceinline__ double cvt_elem<double, long long>(long long x) { return __ll2double_rn(x); }
template <> __device__ __forceinline__ int32_t cvt_elem<int32_t, float>(float x) { return (x != x) ? 0 : __float2int_rz(x); }
template <> __device__ __forceinline__ int32_t cvt_elem<int32_t, double>(double x) { return (x != x) ? 0 : __double2int_rz(x); }
template <> __device__ __forceinline__ int32_t cvt_elem<int32_t, long long>(long long x) { return (int32_t)(uint32_t)(unsigned long long)x; }
template <> __device__ __forceinline__ long long cvt_elem<long long, float>(float x) { return (x != x) ? 0ll : __float2ll_rz(x); }
template <> __device__ __forceinline__ long long cvt_elem<long long, double>(double x) { return (x != x) ? 0ll : __double2ll_rz(x); }
template <> __device__ __forceinline__ long long cvt_elem<long long, int32_t>(int32_t x) { return (long long)x; }
// one element of type DT_* `src_dt` at p[i], converted to T (run-time source type: ragged paths and the bytecode evaluator)
template <class T> __device__ __forceinline__ T load_cvt(const void* p, int64_t i, uint8_t src_dt) {
    switch (src_dt) {
        case DT_F32: return cvt_elem<T, float>(reinterpret_cast<const volatile float*>(p)[i]);
        case DT_F64: return cvt_elem<T, double>(reinterpret_cast<const volatile double*>(p)[i]);
        case DT_I32: return cvt_elem<T, int32_t>(reinterpret_cast<const volatile int32_t*>(p)[i]);
        default: return cvt_elem<T, long long>(reinterpret_cast<const volatile long long*>(p)[i]);
    }
}

// int32 division / modulo by a pass-constant divisor d (|d| >= 2) with a host-computed signed magic number
// (the classic multiply-high scheme for truncating signed division): q = mulhi(x, M) (+x or -x when the sign of
// M differs from that of d), arithmetic shift by s, plus one if negative.  Exact for every int32 x; the
// remainder x - q*d has the sign of the dividend (C semantics).  The fields are kernel-parameter constants.
__device__ __forceinline__ int32_t magic_div_i32(int32_t x, const SgDiv& m) {
    int32_t q = __mulhi(x, m.M);
    q = (int32_t)((uint32_t)q + (uint32_t)x * (uint32_t)m.addsel);
    q >>= m.s;
    q += (int32_t)((uint32_t)q >> 31);
    return q;
}
__device__ __forceinline__ int32_t magic_mod_i32(int32_t x, const SgDiv& m) {
    return (int32_t)((uint32_t)magic_div_i32(x, m) * (uint32_t)m.neg_d + (uint32_t)x);      // one multiply-add: x - q*d
}

// one value op; `op` is a compile-time constant in template instances and a warp-uniform value in the bytecode kernel
template <class T> __device__ __forceinline__ T value_op(uint8_t op, T a, T b) {
    switch (op) {
        case OP_ADD: return p_add(a, b);
        case OP_SUB: return p_sub(a, b);
        case OP_MUL: return p_mul(a, b);
        case OP_DIV: return p_div(a, b);
        case OP_MIN: return (b < a) ? b : a;
        case OP_MAX: return (a < b) ? b : a;
        case OP_MOD: return p_mod(a, b);
        case OP_NEG: return p_neg(a);
        case OP_ABS: return p_abs(a);
        case OP_SQRT: return p_sqrt(a);
        default: return a;      // OP_MOV
    }
}
template <class T> __device__ __forceinline__ bool compare_op(uint8_t op, T a, T b) {
    switch (op) {
        case OP_EQ: return a == b;
        case OP_NE: return a != b;
        case OP_LT: return a < b;
        case OP_LE: return a <= b;
        case OP_GT: return a > b;
        default: return a >= b;
    }
}
__device__ __forceinline__ bool logic_op(uint8_t op, bool a, bool b) {
    switch (op) {
        case OP_AND: return a && b;
        case OP_OR: return a || b;
        default: return !a;
    }
}
__host__ __device__ constexpr bool op_is_value(uint8_t op) { return op <= OP_ABS || op == OP_MOV || op == OP_SQRT; }
__host__ __device__ constexpr bool op_is_unary_value(uint8_t op) { return op == OP_NEG || op == OP_ABS || op == OP_MOV || op == OP_SQRT; }
__host__ __device__ constexpr bool op_is_compare(uint8_t op) { return op >= OP_EQ && op <= OP_GE; }

// ---------------------------------------------------------------------------------------------------------
// total-order keys (signed integers whose order is the IEEE total order on bit patterns; involutions)
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ long long to_key(float a) { int k = __float_as_int(a); return (long long)(k ^ ((k >> 31) & 0x7fffffff)); }
__device__ __forceinline__ long long to_key(double a) { long long k = __double_as_longlong(a); return k ^ ((k >> 63) & 0x7fffffffffffffffll); }
__device__ __forceinline__ long long to_key(int32_t a) { return (long long)a; }
__device__ __forceinline__ long long to_key(long long a) { return a; }
template <class T> __device__ __forceinline__ T from_key(long long k);
template <> __device__ __forceinline__ float from_key<float>(long long k) { int i = (int)k; return __int_as_float(i ^ ((i >> 31) & 0x7fffffff)); }
template <> __device__ __forceinline__ double from_key<double>(long long k) { return __longlong_as_double(k ^ ((k >> 63) & 0x7fffffffffffffffll)); }
template <> __device__ __forceinline__ int32_t from_key<int32_t>(long long k) { return (int32_t)k; }
template <> __device__ __forceinline__ long long from_key<long long>(long long k) { return k; }

// ---------------------------------------------------------------------------------------------------------
// accumulator cell: 16 bytes per output.
//   SUM f64 : (hi, lo) double-double, TwoSum accumulation       SUM f32 : hi = f64 running sum
//   SUM ints: a = wrapping int64                                 MAX/MIN : a = total-order key (f32: 32-bit key widened)
//   ALL/ANY : a = 0/1                                            COUNT   : a = int64
// ---------------------------------------------------------------------------------------------------------
struct Cell { unsigned long long a, b; };

__device__ __forceinline__ void dd_add_double(double& hi, double& lo, double x) {
    double s = __dadd_rn(hi, x);
    double bb = __dsub_rn(s, hi);
    double err = __dadd_rn(__dsub_rn(hi, __dsub_rn(s, bb)), __dsub_rn(x, bb));
    lo = __dadd_rn(lo, err);
    hi = s;
}
__device__ __forceinline__ void dd_add_dd(double& hi, double& lo, double h2, double l2) {
    double s = __dadd_rn(hi, h2);
    double bb = __dsub_rn(s, hi);
    double err = __dadd_rn(__dsub_rn(hi, __dsub_rn(s, bb)), __dsub_rn(h2, bb));
    err = __dadd_rn(err, __dadd_rn(lo, l2));
    double t = __dadd_rn(s, err);                 // FastTwoSum renormalisation
    lo = __dsub_rn(err, __dsub_rn(t, s));
    hi = t;
}

template <class T> __device__ __forceinline__ Cell cell_identity(uint8_t kind) {
    Cell c; c.a = 0; c.b = 0;
    if (kind == OUT_MAX) c.a = (unsigned long long)(sizeof(T) == 4 ? (long long)INT32_MIN : INT64_MIN);
    if (kind == OUT_MIN) c.a = (unsigned long long)(sizeof(T) == 4 ? (long long)INT32_MAX : INT64_MAX);
    if (kind == OUT_ALL) c.a = 1;
    return c;       // sums: +0.0 bits / 0
}

// accumulate one value (reductions of V registers)
template <class T> __device__ __forceinline__ void cell_accum_value(uint8_t kind, Cell& c, T x) {
    if (kind == OUT_SUM) {
        if (Traits<T>::is_float) {
            if (sizeof(T) == 8) {
                double hi = __longlong_as_double((long long)c.a), lo = __longlong_as_double((long long)c.b);
                dd_add_double(hi, lo, (double)x);
                c.a = (unsigned long long)__double_as_longlong(hi); c.b = (unsigned long long)__double_as_longlong(lo);
            } else {
                double hi = __longlong_as_double((long long)c.a);
                hi = __dadd_rn(hi, (double)x);
                c.a = (unsigned long long)__double_as_longlong(hi);
            }
        } else {
            c.a += (unsigned long long)(long long)x;
        }
    } else if (sizeof(T) == 4) {    // 32-bit keys: compare on the low word only
        int k = (int)to_key(x), cur = (int)(long long)c.a;
        if (kind == OUT_MAX ? (k > cur) : (k < cur)) c.a = (unsigned long long)(long long)k;
    } else {
        long long k = to_key(x);
        if (kind == OUT_MAX ? (k > (long long)c.a) : (k < (long long)c.a)) c.a = (unsigned long long)k;
    }
}
// accumulate one predicate (quantifiers / count)
__device__ __forceinline__ void cell_accum_pred(uint8_t kind, Cell& c, bool p) {
    if (kind == OUT_ALL) c.a &= (unsigned long long)p;
    else if (kind == OUT_ANY) c.a |= (unsigned long long)p;
    else c.a += (unsigned long long)p;
}
// combine two cells of the same output (fixed order: `c` is the left operand)
template <class T> __device__ __forceinline__ void cell_combine(uint8_t kind, Cell& c, const Cell& o) {
    switch (kind) {
        case OUT_SUM:
            if (Traits<T>::is_float) {
                double hi = __longlong_as_double((long long)c.a), lo = __longlong_as_double((long long)c.b);
                dd_add_dd(hi, lo, __longlong_as_double((long long)o.a), __longlong_as_double((long long)o.b));
                c.a = (unsigned long long)__double_as_longlong(hi); c.b = (unsigned long long)__double_as_longlong(lo);
            } else c.a += o.a;
            break;
        case OUT_MAX: if ((long long)o.a > (long long)c.a) c.a = o.a; break;
        case OUT_MIN: if ((long long)o.a < (long long)c.a) c.a = o.a; break;
        case OUT_ALL: c.a &= o.a; break;
        case OUT_ANY: c.a |= o.a; break;
        default: c.a += o.a; break;     // COUNT
    }
}
// final 8-byte value of an AXIS_ALL output
template <class T> __device__ __forceinline__ unsigned long long cell_final(uint8_t kind, const Cell& c) {
    if (kind == OUT_SUM && Traits<T>::is_float) {
        double r = __dadd_rn(__longlong_as_double((long long)c.a), __longlong_as_double((long long)c.b));
        return (unsigned long long)__double_as_longlong(r);
    }
    if (kind == OUT_MAX || kind == OUT_MIN) {
        T v = from_key<T>((long long)c.a);
        unsigned long long r = 0;
        if (sizeof(T) == 4) { uint32_t u; memcpy(&u, &v, 4); r = u; } else memcpy(&r, &v, 8);
        return r;
    }
    return c.a;
}

__device__ __forceinline__ Cell cell_shfl_down(const Cell& c, int delta) {
    Cell r;
    r.a = __shfl_down_sync(0xffffffffu, c.a, delta);
    r.b = __shfl_down_sync(0xffffffffu, c.b, delta);
    return r;
}
__device__ __forceinline__ Cell cell_shfl_xor(const Cell& c, int m) {
    Cell r;
    r.a = __shfl_xor_sync(0xffffffffu, c.a, m);
    r.b = __shfl_xor_sync(0xffffffffu, c.b, m);
    return r;
}

// shuffle only the words the output kind uses (a double-double sum needs both, everything else only `a`)
template <class T> __device__ __forceinline__ Cell cell_shfl_xor_kind(uint8_t kind, const Cell& c, int m) {
    Cell r;
    r.a = __shfl_xor_sync(0xffffffffu, c.a, m);
    r.b = (kind == OUT_SUM && Traits<T>::is_float && sizeof(T) == 8) ? __shfl_xor_sync(0xffffffffu, c.b, m) : 0ull;
    return r;
}

// Programmatic dependent launch: every pass kernel is launched with programmatic stream serialisation (sgk_launch_pdl), so its
// blocks may be scheduled while the previous kernel of the stream is still draining — the launch latency of a multi-pass flush
// (config 0: two 5 us passes) hides behind the predecessor's tail.  pdl_wait() returns once every prerequisite grid has completed
// and its memory is visible: it precedes the first access to global memory (inputs, control words, workspace).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// streaming 128-bit accesses: bypass L1 allocation, data is touched once
template <class VEC> __device__ __forceinline__ VEC ld_stream(const VEC* p) {
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return *reinterpret_cast<VEC*>(&r);
}
// same, for buffers the same pass also writes in place (no .nc)
template <class VEC> __device__ __forceinline__ VEC ld_stream_rw(const VEC* p) {
    int4 r;
    asm volatile("ld.global.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return *reinterpret_cast<VEC*>(&r);
}
template <class VEC> __device__ __forceinline__ void st_stream(VEC* p, const VEC& v) {
    const int4& r = *reinterpret_cast<const int4*>(&v);
    asm volatile("st.global.L1::no_allocate.v4.s32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(r.x), "r"(r.y), "r"(r.z), "r"(r.w) : "memory");
}
// N = 8, 16 or 32 streamed bytes (the converting loads read V source elements per 128-bit vector of the pass dtype)
template <int N> __device__ __forceinline__ void ld_stream_bytes(const void* p, void* out) {
    static_assert(N == 8 || N == 16 || N == 32, "8, 16 or 32 bytes");
    int* o = reinterpret_cast<int*>(out);
    if constexpr (N == 8) asm volatile("ld.global.nc.L1::no_allocate.v2.s32 {%0,%1}, [%2];" : "=r"(o[0]), "=r"(o[1]) : "l"(p));
    else {
        asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(o[0]), "=r"(o[1]), "=r"(o[2]), "=r"(o[3]) : "l"(p));
        if constexpr (N == 32)
            asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(o[4]), "=r"(o[5]), "=r"(o[6]), "=r"(o[7]) : "l"(reinterpret_cast<const char*>(p) + 16));
    }
}
__device__ __forceinline__ unsigned int ld_relaxed_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ unsigned int ld_volatile_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}

}  // namespace sgk
#endif  // SG_DEVICE_CUH_
