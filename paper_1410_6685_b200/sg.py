"""ctypes binding of the C-ABI library (include/sg.h).  Same names, argument marshalling only.

Every step of the hot path runs inside libsafegpu.so; this module converts python ints/floats to C arguments,
turns non-zero sg_status codes into SgError, and nothing else.  There is no CPU fallback: if the library cannot
be loaded, or a context cannot get its CUDA device, the call raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, create_string_buffer, c_char_p, c_double, c_float, c_int32, c_int64, c_size_t, c_uint32, c_void_p

# enums of include/sg.h
SG_F32, SG_F64, SG_I32, SG_I64, SG_BOOL = 0, 1, 2, 3, 4
(SG_ADD, SG_SUB, SG_MUL, SG_DIV, SG_MIN, SG_MAX, SG_MOD, SG_NEG, SG_ABS, SG_EQ, SG_NE, SG_LT, SG_LE, SG_GT, SG_GE, SG_AND, SG_OR,
 SG_NOT) = range(18)
SG_SQRT = 19    # 18 is reserved (include/sg.h)
SG_SUM, SG_RMAX, SG_RMIN, SG_COUNT = 0, 1, 2, 3
SG_AXIS_ALL, SG_AXIS_ROWS, SG_AXIS_COLS = 0, 1, 2
SG_OPERAND_HANDLE, SG_OPERAND_IMM_F64, SG_OPERAND_IMM_I64 = 0, 1, 2
SG_BCAST_NONE, SG_BCAST_ROW, SG_BCAST_COL = 0, 1, 2
SG_CONTRACT_PRE, SG_CONTRACT_POST = 0, 1
SG_FLAG_UNFUSED, SG_FLAG_FORCE_BYTECODE, SG_FLAG_NO_EARLY_EXIT, SG_FLAG_NO_PLAN_CACHE = 1, 2, 4, 8
SG_OK = 0
SG_ACC_DEFAULT = -1
SG_ERR = {-1: "SG_ERR_ARG", -2: "SG_ERR_SHAPE", -3: "SG_ERR_DTYPE", -4: "SG_ERR_EMPTY", -5: "SG_ERR_ALIAS", -6: "SG_ERR_OOM",
          -7: "SG_ERR_CUDA", -8: "SG_ERR_CONTRACT", -9: "SG_ERR_CAPACITY", -10: "SG_ERR_UNSUPPORTED"}
SG_ERR_ARG, SG_ERR_SHAPE, SG_ERR_DTYPE, SG_ERR_EMPTY, SG_ERR_ALIAS, SG_ERR_OOM, SG_ERR_CUDA, SG_ERR_CONTRACT, SG_ERR_CAPACITY, \
    SG_ERR_UNSUPPORTED = range(-1, -11, -1)

EXPORTS = [
    "sg_ctx_create", "sg_ctx_destroy", "sg_ctx_set_flags", "sg_last_error", "sg_vec_create", "sg_mat_create", "sg_vec_subset",
    "sg_mat_row", "sg_mat_rows", "sg_mat_col", "sg_mat_elem", "sg_mat_ge_steps", "sg_mat_transpose", "sg_vec_quicksort", "sg_vec_sum_noalloc", "sg_enqueue", "sg_cast", "sg_reduce", "sg_forall", "sg_exists",
    "sg_forall_adjacent", "sg_filter", "sg_contract", "sg_flush", "sg_scalar_get", "sg_scalar_dtype", "sg_vec_count", "sg_vec_data", "sg_vec_read",
    "sg_release", "sg_plan_stats", "sg_plan_dump", "sg_plan_cache_stats", "sg_last_flush_ms", "sg_timing_begin", "sg_timing_end", "sg_replay_last", "sg_replay_last_graph", "sg_template_count", "sg_template_name",
    "sg_version",
]


class sg_operand(Structure):
    _fields_ = [("kind", c_int32), ("bcast", c_int32), ("h", c_int64), ("f", c_double), ("i", c_int64)]


class sg_stats(Structure):
    _fields_ = [("n_passes", c_int32), ("n_nodes", c_int32), ("n_template", c_int32), ("n_bytecode", c_int32), ("bytes_min", c_int64),
                ("launches_total", c_int64), ("pass_n_in", c_int32 * 16), ("pass_n_instr", c_int32 * 16), ("pass_n_out", c_int32 * 16),
                ("pass_n_args", c_int32 * 16), ("pass_kernel", c_int32 * 16)]


class SgError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{SG_ERR.get(status, status)}: {message}")
        self.status = status


_LIB = None


def lib_path() -> str:
    """The in-tree library; SAFEGPU_LIB names another build of the same sources (kernel tuning experiments)."""
    return os.environ.get("SAFEGPU_LIB") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "libsafegpu.so")


def lib() -> ctypes.CDLL:
    """Loads libsafegpu.so (built in-tree by paper_1410_6685_b200.build).  Raises if it is missing."""
    global _LIB
    if _LIB is None:
        path = lib_path()
        if not os.path.exists(path):
            raise ImportError(f"{path} not found: build it with `python -m paper_1410_6685_b200.build` (no fallback exists)")
        L = ctypes.CDLL(path)
        L.sg_last_error.restype = c_char_p
        L.sg_template_name.restype = c_char_p
        L.sg_version.restype = c_char_p
        L.sg_plan_dump.restype = c_int64
        L.sg_ctx_create.argtypes = [POINTER(c_void_p), c_int32, c_void_p, c_void_p]
        L.sg_vec_create.argtypes = [c_void_p, c_int32, c_int64, c_void_p, POINTER(c_int64)]
        L.sg_mat_create.argtypes = [c_void_p, c_int32, c_int64, c_int64, c_int64, c_void_p, POINTER(c_int64)]
        L.sg_vec_subset.argtypes = [c_void_p, c_int64, c_int64, c_int64, POINTER(c_int64)]
        L.sg_mat_row.argtypes = [c_void_p, c_int64, c_int64, POINTER(c_int64)]
        L.sg_mat_rows.argtypes = [c_void_p, c_int64, c_int64, c_int64, POINTER(c_int64)]
        L.sg_mat_col.argtypes = [c_void_p, c_int64, c_int64, c_int64, c_int64, POINTER(c_int64)]
        L.sg_mat_elem.argtypes = [c_void_p, c_int64, c_int64, c_int64, POINTER(c_int64)]
        L.sg_enqueue.argtypes = [c_void_p, c_int32, POINTER(sg_operand), c_int32, c_int64, POINTER(c_int64)]
        L.sg_cast.argtypes = [c_void_p, c_int64, c_int32, c_int64, POINTER(c_int64)]
        L.sg_reduce.argtypes = [c_void_p, c_int64, c_int32, c_int32, c_int32, POINTER(c_int64)]
        L.sg_forall.argtypes = [c_void_p, c_int64, POINTER(c_int64)]
        L.sg_exists.argtypes = [c_void_p, c_int64, POINTER(c_int64)]
        L.sg_forall_adjacent.argtypes = [c_void_p, c_int64, c_int32, POINTER(c_int64)]
        L.sg_filter.argtypes = [c_void_p, c_int64, c_int64, c_void_p, c_int64, POINTER(c_int64), POINTER(c_int64)]
        L.sg_contract.argtypes = [c_void_p, c_int64, c_int32, c_char_p]
        L.sg_flush.argtypes = [c_void_p]
        L.sg_scalar_get.argtypes = [c_void_p, c_int64, c_void_p, c_size_t]
        L.sg_scalar_dtype.argtypes = [c_void_p, c_int64, POINTER(c_int32)]
        L.sg_vec_count.argtypes = [c_void_p, c_int64, POINTER(c_int64)]
        L.sg_vec_data.argtypes = [c_void_p, c_int64, POINTER(c_void_p)]
        L.sg_release.argtypes = [c_void_p, c_int64]
        L.sg_vec_read.argtypes = [c_void_p, c_int64, c_void_p, c_size_t]
        L.sg_plan_stats.argtypes = [c_void_p, POINTER(sg_stats)]
        L.sg_plan_dump.argtypes = [c_void_p, c_int32, c_char_p, c_int64]
        L.sg_plan_cache_stats.argtypes = [c_void_p, POINTER(c_int64), POINTER(c_int64)]
        L.sg_last_flush_ms.argtypes = [c_void_p, POINTER(c_float)]
        L.sg_replay_last.argtypes = [c_void_p, c_int32, POINTER(c_float)]
        L.sg_replay_last_graph.argtypes = [c_void_p, c_int32, POINTER(c_float), POINTER(c_float)]
        L.sg_mat_ge_steps.argtypes = [c_void_p, c_int64, c_int64, c_int64, c_double, c_int64, c_int64]
        L.sg_vec_quicksort.argtypes = [c_void_p, c_int64, c_void_p, POINTER(c_int64)]
        L.sg_vec_sum_noalloc.argtypes = [c_int32, c_void_p, c_int32, c_void_p, c_int64, c_void_p, c_char_p, c_int64]
        L.sg_mat_transpose.argtypes = [c_void_p, c_int64, c_void_p, c_int64, POINTER(c_int64)]
        L.sg_timing_begin.argtypes = [c_void_p]
        L.sg_timing_end.argtypes = [c_void_p, POINTER(c_float), POINTER(c_int32)]
        L.sg_ctx_set_flags.argtypes = [c_void_p, c_uint32]
        L.sg_ctx_destroy.argtypes = [c_void_p]
        L.sg_last_error.argtypes = [c_void_p]
        L.sg_template_name.argtypes = [c_int32]
        _LIB = L
    return _LIB


def _ck(ctx, status: int) -> None:
    if status != SG_OK:
        msg = lib().sg_last_error(ctx) if ctx else b""
        raise SgError(status, (msg or b"").decode())


# operand constructors (marshalling helpers)
def H(handle: int, bcast: int = SG_BCAST_NONE) -> sg_operand:
    return sg_operand(SG_OPERAND_HANDLE, bcast, handle, 0.0, 0)


def F(x: float) -> sg_operand:
    return sg_operand(SG_OPERAND_IMM_F64, 0, 0, float(x), 0)


def I(x: int) -> sg_operand:
    return sg_operand(SG_OPERAND_IMM_I64, 0, 0, 0.0, int(x))


def _opd(x) -> sg_operand:
    if isinstance(x, sg_operand):
        return x
    if isinstance(x, bool):
        raise TypeError("bool operand")
    if isinstance(x, int):
        return H(x)         # bare ints are handles; immediates are written F(..) / I(..)
    raise TypeError(f"operand {x!r}: use a handle, H(h, bcast), F(float) or I(int)")


def sg_version() -> str:
    return lib().sg_version().decode()


def sg_template_count() -> int:
    return lib().sg_template_count()


def sg_template_name(k: int) -> str:
    return lib().sg_template_name(k).decode()


def sg_ctx_create(device: int, cuda_stream: int | None = None):
    ctx = c_void_p()
    st = lib().sg_ctx_create(byref(ctx), device, c_void_p(cuda_stream or 0), None)
    if st != SG_OK:
        raise SgError(st, "sg_ctx_create failed (no usable CUDA device? the library has no CPU fallback)")
    return ctx


def sg_ctx_destroy(ctx) -> None:
    _ck(None, lib().sg_ctx_destroy(ctx))


def sg_ctx_set_flags(ctx, flags: int) -> None:
    _ck(ctx, lib().sg_ctx_set_flags(ctx, flags))


def sg_last_error(ctx) -> str:
    return lib().sg_last_error(ctx).decode()


def _h(fn, ctx, *args) -> int:
    out = c_int64(0)
    _ck(ctx, fn(ctx, *args, byref(out)))
    return out.value


def sg_vec_create(ctx, dtype: int, n: int, dev_ptr: int | None) -> int:
    return _h(lib().sg_vec_create, ctx, dtype, n, c_void_p(dev_ptr or 0))


def sg_mat_create(ctx, dtype: int, rows: int, cols: int, ld_elems: int, dev_ptr: int | None) -> int:
    return _h(lib().sg_mat_create, ctx, dtype, rows, cols, ld_elems, c_void_p(dev_ptr or 0))


def sg_vec_subset(ctx, v: int, start: int, finish: int) -> int:
    return _h(lib().sg_vec_subset, ctx, v, start, finish)


def sg_mat_row(ctx, m: int, i: int) -> int:
    return _h(lib().sg_mat_row, ctx, m, i)


def sg_mat_rows(ctx, m: int, r0: int, r1: int) -> int:
    return _h(lib().sg_mat_rows, ctx, m, r0, r1)


def sg_mat_col(ctx, m: int, j: int, r0: int, r1: int) -> int:
    return _h(lib().sg_mat_col, ctx, m, j, r0, r1)


def sg_mat_elem(ctx, m: int, i: int, j: int) -> int:
    return _h(lib().sg_mat_elem, ctx, m, i, j)


def sg_mat_transpose(ctx, m: int, dev_out: int | None = None, ld_out: int = 0) -> int:
    return _h(lib().sg_mat_transpose, ctx, m, c_void_p(dev_out or 0), ld_out)


def sg_vec_quicksort(ctx, v: int, dev_out: int | None = None) -> int:
    return _h(lib().sg_vec_quicksort, ctx, v, dev_out)


SG_NOALLOC_MAX_N = 1 << 27
SG_NOALLOC_SCRATCH_BYTES = 256 + 16 * 16384


def sg_vec_sum_noalloc(device: int, stream: int, dtype: int, dev_x: int, n: int, dev_out: int) -> None:
    """Sum of a device vector into a device double without any allocation (include/sg.h); asynchronous on `stream`."""
    err = create_string_buffer(256)
    st = lib().sg_vec_sum_noalloc(device, c_void_p(stream or 0), dtype, c_void_p(dev_x or 0), n, c_void_p(dev_out or 0), err, 256)
    if st != SG_OK:
        raise SgError(st, err.value.decode())


def sg_mat_ge_steps(ctx, m: int, det: int, minpiv: int, eps: float, k0: int, k1: int) -> None:
    _ck(ctx, lib().sg_mat_ge_steps(ctx, m, det, minpiv, float(eps), k0, k1))


def sg_enqueue(ctx, op: int, operands, dst_or_0: int = 0) -> int:
    ops = [_opd(x) for x in operands]
    arr = (sg_operand * len(ops))(*ops)
    return _h(lib().sg_enqueue, ctx, op, arr, len(ops), dst_or_0)


def sg_cast(ctx, v: int, to: int, dst_or_0: int = 0) -> int:
    return _h(lib().sg_cast, ctx, v, to, dst_or_0)


def sg_reduce(ctx, h: int, kind: int, axis: int = SG_AXIS_ALL, acc: int = SG_ACC_DEFAULT) -> int:
    return _h(lib().sg_reduce, ctx, h, kind, acc, axis)


def sg_forall(ctx, h_bool: int) -> int:
    return _h(lib().sg_forall, ctx, h_bool)


def sg_exists(ctx, h_bool: int) -> int:
    return _h(lib().sg_exists, ctx, h_bool)


def sg_forall_adjacent(ctx, v: int, cmp: int) -> int:
    return _h(lib().sg_forall_adjacent, ctx, v, cmp)


def sg_filter(ctx, values: int, mask_bool: int, dev_out: int | None = None, capacity: int = 0):
    out_vec, out_count = c_int64(0), c_int64(0)
    _ck(ctx, lib().sg_filter(ctx, values, mask_bool, c_void_p(dev_out or 0), capacity, byref(out_vec), byref(out_count)))
    return out_vec.value, out_count.value


def sg_contract(ctx, h_bool_scalar: int, kind: int, tag: str = "") -> None:
    _ck(ctx, lib().sg_contract(ctx, h_bool_scalar, kind, tag.encode()))


def sg_flush(ctx) -> None:
    _ck(ctx, lib().sg_flush(ctx))


_SCALAR_C = {SG_F32: c_float, SG_F64: c_double, SG_I32: c_int32, SG_I64: c_int64, SG_BOOL: ctypes.c_uint8}


def sg_scalar_dtype(ctx, s: int) -> int:
    dt = c_int32(0)
    _ck(ctx, lib().sg_scalar_dtype(ctx, s, byref(dt)))
    return dt.value


def sg_scalar_get(ctx, s: int):
    """Reads a scalar result (the trigger of PAPER.md:284): python float / int / bool according to its dtype."""
    dt = sg_scalar_dtype(ctx, s)
    buf = _SCALAR_C[dt]()
    _ck(ctx, lib().sg_scalar_get(ctx, s, byref(buf), ctypes.sizeof(buf)))
    return bool(buf.value) if dt == SG_BOOL else buf.value


def sg_vec_count(ctx, v: int) -> int:
    n = c_int64(0)
    _ck(ctx, lib().sg_vec_count(ctx, v, byref(n)))
    return n.value


def sg_vec_data(ctx, v: int) -> int:
    p = c_void_p()
    _ck(ctx, lib().sg_vec_data(ctx, v, byref(p)))
    return p.value or 0


def sg_vec_read(ctx, v: int, host_ptr: int, nbytes: int) -> None:
    """to_array: copies the collection to host memory at host_ptr (e.g. numpy_array.ctypes.data)."""
    _ck(ctx, lib().sg_vec_read(ctx, v, c_void_p(host_ptr), nbytes))


def sg_release(ctx, h: int) -> None:
    _ck(ctx, lib().sg_release(ctx, h))


def sg_plan_stats(ctx) -> sg_stats:
    st = sg_stats()
    _ck(ctx, lib().sg_plan_stats(ctx, byref(st)))
    return st


def sg_plan_dump(ctx, pass_index: int) -> str:
    need = lib().sg_plan_dump(ctx, pass_index, None, 0)
    if need < 0:
        raise IndexError(pass_index)
    buf = ctypes.create_string_buffer(need)
    lib().sg_plan_dump(ctx, pass_index, buf, need)
    return buf.value.decode()


def sg_plan_cache_stats(ctx):
    """(hits, misses) of the plan cache since the context was created."""
    h, m = c_int64(0), c_int64(0)
    _ck(ctx, lib().sg_plan_cache_stats(ctx, byref(h), byref(m)))
    return h.value, m.value


def sg_last_flush_ms(ctx) -> float:
    ms = c_float(0)
    _ck(ctx, lib().sg_last_flush_ms(ctx, byref(ms)))
    return ms.value


def sg_timing_begin(ctx) -> None:
    _ck(ctx, lib().sg_timing_begin(ctx))


def sg_timing_end(ctx) -> tuple[float, int]:
    """(sum of the device times of the flushes since sg_timing_begin in ms, number of flushes)."""
    ms, n = c_float(0), c_int32(0)
    _ck(ctx, lib().sg_timing_end(ctx, byref(ms), byref(n)))
    return ms.value, n.value


def sg_replay_last(ctx, reps: int) -> float:
    ms = c_float(0)
    _ck(ctx, lib().sg_replay_last(ctx, reps, byref(ms)))
    return ms.value


def sg_replay_last_graph(ctx, reps: int) -> tuple[float, float]:
    """(device ms, launch-inclusive wall ms) per replay of the last flush's launches from a CUDA graph."""
    dev, wall = c_float(0.0), c_float(0.0)
    _ck(ctx, lib().sg_replay_last_graph(ctx, reps, byref(dev), byref(wall)))
    return dev.value, wall.value
