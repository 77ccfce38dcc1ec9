"""CPU ORACLE — test infrastructure only.

The five workloads of BASELINE.json:configs evaluated primitive by primitive with the
unfused oracle (one full loop and one materialised temporary per operation, in the
order and parenthesisation fixed in DESIGN.md §3 / SURVEY.md §8(c)).
"""
from __future__ import annotations

import numpy as np

import oracle as orc


def dot_product(a, b) -> float:
    """Listing 4: a.compwise_multiply(b).sum."""
    return orc.sum(orc.zip("mul", a, b))


def axpy(alpha, x, y) -> np.ndarray:
    """aX+Y: X.multiplied_by(a).plus(Y)."""
    return orc.zip("add", orc.scalar("mul", x, alpha), y)


def cfg0_chain(a, b, c) -> np.ndarray:
    """z = (a+b)*2.5 - c  (BASELINE.json:configs[0])."""
    t1 = orc.zip("add", a, b)
    t2 = orc.scalar("mul", t1, 2.5)
    return orc.zip("sub", t2, c)


def cfg0(a, b, c) -> dict:
    z = cfg0_chain(a, b, c)
    return {
        "z": z,
        "sum": orc.sum(z),
        "max": orc.max(z),
        "min": orc.min(z),
        "pre": orc.any(orc.cmp_scalar("gt", a, 0.99)),                   # exists(a_i > 0.99)
        "post": orc.all(orc.cmp("eq", z, cfg0_chain(a, b, c))),          # for_all(z_i == recomputed)
    }


def cfg1_chain(x, y) -> np.ndarray:
    """w = abs(x*y + 0.5) - min(x,y)*3 + x/(1+y*y), left to right  (BASELINE.json:configs[1])."""
    t1 = orc.zip("mul", x, y)
    t2 = orc.scalar("add", t1, 0.5)
    t3 = orc.unary("abs", t2)
    t4 = orc.zip("min", x, y)
    t5 = orc.scalar("mul", t4, 3.0)
    t6 = orc.zip("sub", t3, t5)
    t7 = orc.zip("mul", y, y)
    t8 = orc.scalar("add", t7, 1.0, reversed=True)
    t9 = orc.zip("div", x, t8)
    return orc.zip("add", t6, t9)


def cfg1(x, y) -> dict:
    w = cfg1_chain(x, y)
    return {"w": w, "sum": orc.sum(w), "max": orc.max(w)}


def cfg2(x, modulus: int = 7, residue: int = 3) -> dict:
    """stable filter keeping x where x mod 7 == 3, count, int64 sum of kept (BASELINE.json:configs[2])."""
    m = orc.cmp_scalar("eq", orc.scalar("mod", x, modulus), residue)
    kept = orc.filter(x, m)
    return {"kept": kept, "count": int(kept.size), "count_mask": orc.count(m), "sum": orc.sum(kept)}


def cfg3(x) -> dict:
    """pre = for_all(x_i >= 0), post = is-sorted for_all(x_i <= x_{i+1})  (BASELINE.json:configs[3])."""
    return {"pre": orc.all(orc.cmp_scalar("ge", x, 0.0)), "post": orc.all(orc.adj("le", x))}


def cfg4_unfused(M, k: int) -> dict:
    """Row-update step for all j>k, primitive by primitive (BASELINE.json:configs[4])."""
    M = np.array(M, dtype=np.float64, order="C", copy=True)
    n_rows = M.shape[0]
    col = orc.mat_col(M, k)                                  # column(k): copy
    f = orc.scalar("div", col[k + 1:], M[k, k])              # f_j = M[j,k] / M[k,k]
    t = orc.outer_mul(f, M[k, :])                            # t = f_j * M[k,c]
    sub = orc.zip("sub", M[k + 1:, :], t)                    # M[j,c] - t
    M[k + 1:, :] = sub
    if n_rows - k - 1 > 0:
        rowmax = orc.row_max(orc.unary("abs", sub))
        colsum = orc.col_sum(sub)
    else:
        rowmax = np.empty(0)
        colsum = np.zeros(M.shape[1])
    return {"M": M, "rowmax": rowmax, "colsum": colsum}


def cfg4(M, k: int) -> dict:
    """Same step through the single plain-definition loop (orc_mat_step)."""
    Mo, rowmax, colsum = orc.mat_step(M, k)
    return {"M": Mo, "rowmax": rowmax, "colsum": colsum}


def concatenate(a, b) -> np.ndarray:
    """concatenate: a new container of the elements of a followed by those of b."""
    a, b = np.ascontiguousarray(a), np.ascontiguousarray(b)
    assert a.dtype == b.dtype
    out = np.empty(a.size + b.size, dtype=a.dtype)
    out[: a.size] = a
    out[a.size:] = b
    return out


def quicksort(a) -> np.ndarray:
    """Listing 3, step by step: pivot := a[a.count // 2] (0-based, R10); left/right/mid := the three
    stable filters with item < / > / = pivot; Result := quicksort(left).concatenate(mid).concatenate(quicksort(right)).
    Precondition a.count > 0.  The recursion of the listing is written with an explicit stack (same calls, same order of
    results); an empty left or right part is skipped, as its quicksort would violate the precondition."""
    a = np.ascontiguousarray(a)
    if a.size == 0:
        raise ValueError("quicksort: require a.count > 0")
    pieces = []                     # sorted runs in final order
    stack = [a]                     # sub-collections still to sort, leftmost on top
    while stack:
        v = stack.pop()
        if isinstance(v, tuple):    # an already final run (a `mid`)
            pieces.append(v[0])
            continue
        if v.size == 1:
            pieces.append(v)
            continue
        pivot = v[v.size // 2]
        left = orc.filter(v, orc.cmp_scalar("lt", v, pivot))
        right = orc.filter(v, orc.cmp_scalar("gt", v, pivot))
        mid = orc.filter(v, orc.cmp_scalar("eq", v, pivot))
        if right.size:
            stack.append(right)
        stack.append((mid,))
        if left.size:
            stack.append(left)
    out = pieces[0]
    for p in pieces[1:]:
        out = concatenate(out, p)
    return out


def right_multiply(M, v) -> np.ndarray:
    """`right_multiply` (matrix x column vector; Listing 1's `multiply` contract shape): result_i =
    (row(i) compwise_multiply v).sum — Listing 4's dot product per row, with the built-in dimension contract columns = v.count."""
    M, v = np.ascontiguousarray(M), np.ascontiguousarray(v)
    assert M.ndim == 2 and M.shape[1] == v.size and M.dtype == v.dtype
    return np.array([orc.sum(orc.zip("mul", M[i], v)) for i in range(M.shape[0])], dtype=np.float64)


def left_multiply(v, M) -> np.ndarray:
    """`left_multiply` (row vector x matrix): result_c = sum_i v_i * M[i,c] — every row scaled by its v_i (one
    rounding per product), then the column sums; dimension contract rows = v.count."""
    M, v = np.ascontiguousarray(M), np.ascontiguousarray(v)
    assert M.ndim == 2 and M.shape[0] == v.size and M.dtype == v.dtype == np.float64
    T = np.empty_like(M)
    for i in range(M.shape[0]):
        T[i] = orc.scalar("mul", M[i], v[i])
    return orc.col_sum(T) if M.shape[0] else np.zeros(M.shape[1])


def transpose(M) -> np.ndarray:
    """`transpose`: a new rows x cols -> cols x rows matrix with out[j][i] = M[i][j], written out element by element."""
    M = np.ascontiguousarray(M)
    assert M.ndim == 2
    out = np.empty((M.shape[1], M.shape[0]), dtype=M.dtype)
    for i in range(M.shape[0]):
        out[:, i] = M[i, :]
    return out
