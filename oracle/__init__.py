"""CPU ORACLE — test infrastructure only (ctypes wrapper over oracle/oracle.cpp).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It never imports the product package
(paper_1410_6685_b200) and shares no code with the CUDA path.

Every function executes ONE primitive of the SafeGPU collection API, unfused, over
fully materialised numpy arrays (the naive one-kernel-per-call plan),
single-threaded.  dtype follows the input array (float32/float64/int32/int64);
scalars are converted to that dtype before the loop (DESIGN.md R-imm).
"""
from __future__ import annotations

import builtins
import ctypes

import numpy as np

from . import build as _build

_DT = {np.dtype(np.float32): 0, np.dtype(np.float64): 1, np.dtype(np.int32): 2, np.dtype(np.int64): 3}
_BIN = {"add": 0, "sub": 1, "mul": 2, "div": 3, "min": 4, "max": 5, "mod": 6}
_UN = {"neg": 0, "abs": 1, "sqrt": 2}
_CMP = {"eq": 0, "ne": 1, "lt": 2, "le": 3, "gt": 4, "ge": 5}
_LOG = {"and": 0, "or": 1, "not": 2}

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
    return _lib


def _p(a: np.ndarray) -> ctypes.c_void_p:
    return ctypes.c_void_p(a.ctypes.data)


def _chk(rc: int, what: str) -> None:
    if rc == -4:
        raise ValueError(f"{what}: empty collection")
    if rc != 0:
        raise RuntimeError(f"{what}: oracle error {rc}")


def _c(a) -> np.ndarray:
    a = np.ascontiguousarray(a)
    if a.dtype not in _DT and a.dtype != np.uint8:
        raise TypeError(f"unsupported dtype {a.dtype}")
    return a


def _n(a: np.ndarray) -> ctypes.c_int64:
    return ctypes.c_int64(a.size)


def zip(op: str, a, b) -> np.ndarray:
    """out[i] = a[i] op b[i]   (plus/minus/compwise_multiply/compwise_divide)."""
    a, b = _c(a), _c(b)
    assert a.dtype == b.dtype and a.shape == b.shape
    out = np.empty_like(a)
    _chk(lib().orc_zip(_BIN[op], _DT[a.dtype], _n(a), _p(a), _p(b), _p(out)), "zip")
    return out


def scalar(op: str, a, s, reversed: bool = False) -> np.ndarray:
    """out[i] = a[i] op s  (or s op a[i])   (multiplied_by / divided_by)."""
    a = _c(a)
    sv = np.array([s], dtype=a.dtype)
    out = np.empty_like(a)
    _chk(lib().orc_scalar(_BIN[op], _DT[a.dtype], _n(a), _p(a), _p(sv), int(reversed), _p(out)), "scalar")
    return out


def unary(op: str, a) -> np.ndarray:
    """neg / abs (sign-bit operations) and sqrt (correctly rounded, floats only: the `project(agent sqrt)` of PAPER.md:171-175)."""
    a = _c(a)
    if op == "sqrt" and a.dtype.kind != "f":
        raise TypeError("sqrt needs a float collection")
    out = np.empty_like(a)
    _chk(lib().orc_unary(_UN[op], _DT[a.dtype], _n(a), _p(a), _p(out)), "unary")
    return out


def cast(a, to) -> np.ndarray:
    """project with the value-preserving conversion as the transform (R23): int -> float rounds to
    nearest even, float -> int truncates toward zero with saturation and NaN -> 0, int64 -> int32 keeps the low 32 bits."""
    a = _c(a)
    to = np.dtype(to)
    if a.dtype not in _DT or to not in _DT:
        raise TypeError("cast converts between float32, float64, int32 and int64")
    out = np.empty(a.shape, dtype=to)
    _chk(lib().orc_cast(_DT[a.dtype], _DT[to], _n(a), _p(a), _p(out)), "cast")
    return out


def project_sqrt(a) -> np.ndarray:
    """`c.project (agent (a: INT): DOUBLE do Result := sqrt (a) end)`: an integer collection gives a collection
    of doubles — the conversion, then the correctly rounded square root, two primitives; a float collection keeps its dtype."""
    a = _c(a)
    return unary("sqrt", cast(a, np.float64) if a.dtype.kind == "i" else a)


def cmp(op: str, a, b) -> np.ndarray:
    """BOOL[i] = a[i] cmp b[i]  (predicate agents)."""
    a, b = _c(a), _c(b)
    assert a.dtype == b.dtype and a.shape == b.shape
    out = np.empty(a.shape, dtype=np.uint8)
    _chk(lib().orc_cmp(_CMP[op], _DT[a.dtype], _n(a), _p(a), _p(b), _p(out)), "cmp")
    return out


def cmp_scalar(op: str, a, s) -> np.ndarray:
    a = _c(a)
    sv = np.array([s], dtype=a.dtype)
    out = np.empty(a.shape, dtype=np.uint8)
    _chk(lib().orc_cmp_scalar(_CMP[op], _DT[a.dtype], _n(a), _p(a), _p(sv), _p(out)), "cmp_scalar")
    return out


def adj(op: str, a) -> np.ndarray:
    """BOOL[i] = a[i] cmp a[i+1], i in [0, n-2]  (is_sorted == all(adj('le')))."""
    a = _c(a)
    out = np.empty(builtins.max(a.size - 1, 0), dtype=np.uint8)
    _chk(lib().orc_adj(_CMP[op], _DT[a.dtype], _n(a), _p(a), _p(out)), "adj")
    return out


def logic(op: str, a, b=None) -> np.ndarray:
    a = _c(a).astype(np.uint8, copy=False)
    b = a if b is None else _c(b).astype(np.uint8, copy=False)
    out = np.empty(a.shape, dtype=np.uint8)
    _chk(lib().orc_logic(_LOG[op], _n(a), _p(a), _p(b), _p(out)), "logic")
    return out


def sum(a):
    """float inputs -> python float (f64, long double accumulation rounded once); ints -> python int (wrapping int64)."""
    a = _c(a)
    if a.dtype.kind == "f":
        out = np.zeros(1, dtype=np.float64)
    else:
        out = np.zeros(1, dtype=np.int64)
    _chk(lib().orc_sum(_DT[a.dtype], _n(a), _p(a), _p(out)), "sum")
    return out[0].item()


def avg(a) -> float:
    """avg = sum(a) / count, one fp64 division of the once-rounded fp64 sum (int collections: the wrapping int64
    sum converted to fp64 first).  Empty collection: ValueError (R4)."""
    a = _c(a)
    if a.size == 0:
        raise ValueError("avg: empty collection")
    num = np.array([sum(a)], dtype=np.float64)
    den = np.array([a.size], dtype=np.float64)
    return zip("div", num, den)[0].item()


def _extremum(is_max: int, a):
    a = _c(a)
    out = np.zeros(1, dtype=a.dtype)
    _chk(lib().orc_extremum(is_max, _DT[a.dtype], _n(a), _p(a), _p(out)), "max/min")
    return out[0]


def max(a):
    return _extremum(1, a)


def min(a):
    return _extremum(0, a)


def all(m) -> bool:
    m = _c(m).astype(np.uint8, copy=False)
    out = np.zeros(1, dtype=np.uint8)
    _chk(lib().orc_all(_n(m), _p(m), _p(out)), "all")
    return bool(out[0])


def any(m) -> bool:
    m = _c(m).astype(np.uint8, copy=False)
    out = np.zeros(1, dtype=np.uint8)
    _chk(lib().orc_any(_n(m), _p(m), _p(out)), "any")
    return bool(out[0])


def count(m) -> int:
    m = _c(m).astype(np.uint8, copy=False)
    out = np.zeros(1, dtype=np.int64)
    _chk(lib().orc_count(_n(m), _p(m), _p(out)), "count")
    return int(out[0])


def filter(a, mask) -> np.ndarray:
    """Stable compaction of a where mask is true."""
    a = _c(a)
    mask = _c(mask).astype(np.uint8, copy=False)
    assert a.shape == mask.shape
    out = np.empty_like(a)
    cnt = ctypes.c_int64(0)
    _chk(lib().orc_filter(_DT[a.dtype], _n(a), _p(a), _p(mask), _p(out), ctypes.byref(cnt)), "filter")
    return out[: cnt.value].copy()


# --- matrices (float64, row-major) -------------------------------------------------

def mat_col(M, j: int) -> np.ndarray:
    M = _c(M)
    assert M.dtype == np.float64 and M.ndim == 2
    out = np.empty(M.shape[0], dtype=np.float64)
    _chk(lib().orc_mat_col(ctypes.c_int64(M.shape[0]), ctypes.c_int64(M.shape[1]), _p(M), ctypes.c_int64(j), _p(out)), "mat_col")
    return out


def outer_mul(f, p) -> np.ndarray:
    f, p = _c(f), _c(p)
    out = np.empty((f.size, p.size), dtype=np.float64)
    _chk(lib().orc_outer_mul(_n(f), _n(p), _p(f), _p(p), _p(out)), "outer_mul")
    return out


def row_max(M) -> np.ndarray:
    M = _c(M)
    out = np.empty(M.shape[0], dtype=np.float64)
    _chk(lib().orc_row_extremum(1, ctypes.c_int64(M.shape[0]), ctypes.c_int64(M.shape[1]), ctypes.c_int64(M.shape[1]), _p(M), _p(out)), "row_max")
    return out


def col_sum(M) -> np.ndarray:
    M = _c(M)
    out = np.empty(M.shape[1], dtype=np.float64)
    _chk(lib().orc_col_sum(ctypes.c_int64(M.shape[0]), ctypes.c_int64(M.shape[1]), ctypes.c_int64(M.shape[1]), _p(M), _p(out)), "col_sum")
    return out


def mat_step(M, kr: int, kc: int | None = None):
    """Row-update step of BASELINE.json:configs[4], in place on a copy. Returns (M', rowmax[rows-kr-1], colsum[cols])."""
    M = np.array(M, dtype=np.float64, order="C", copy=True)
    kc = kr if kc is None else kc
    rows, cols = M.shape
    rowmax = np.empty(rows - kr - 1, dtype=np.float64)
    colsum = np.empty(cols, dtype=np.float64)
    _chk(lib().orc_mat_step(ctypes.c_int64(rows), ctypes.c_int64(cols), ctypes.c_int64(cols), _p(M), ctypes.c_int64(kr), ctypes.c_int64(kc), _p(rowmax), _p(colsum)), "mat_step")
    return M, rowmax, colsum


def ge_determinant(M, eps: float = 0.0):
    """Listing 5: determinant by Gaussian elimination without pivoting, on a copy.

    Returns (det, eliminated matrix, zero_step) — zero_step is the step whose |pivot| <= eps, where the loop ended (det is then
    Result * pivot: the multiplication precedes the test), else -1."""
    M = np.array(M, dtype=np.float64, order="C", copy=True)
    if M.ndim != 2 or M.shape[0] != M.shape[1]:
        raise ValueError("square matrix expected")
    det = ctypes.c_double(0.0)
    zs = ctypes.c_int64(-1)
    _chk(lib().orc_ge_determinant(ctypes.c_int64(M.shape[0]), ctypes.c_int64(M.shape[1]), _p(M), ctypes.c_double(eps),
                                  ctypes.byref(det), ctypes.byref(zs)), "ge_determinant")
    return det.value, M, int(zs.value)
