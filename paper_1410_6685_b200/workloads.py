"""The paper's example programs and the five BASELINE.json workloads written against the C ABI (sg.py).

These are USER programs in the sense of the paper's listings: they only call collection primitives; every
arithmetic step runs inside libsafegpu.so.  Device pointers are plain ints (``tensor.data_ptr()``); with a
plan-only context (device -1) they may be None.  Each function returns a dict of handles; nothing executes
until a scalar is read or sg_flush is called.
"""
from __future__ import annotations

from . import sg
from .sg import F, H, I


def dot_product(ctx, dtype, n, pa, pb):
    """Listing 4: a.compwise_multiply(b).sum — the product is an anonymous intermediate."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    b = sg.sg_vec_create(ctx, dtype, n, pb)
    prod = sg.sg_enqueue(ctx, sg.SG_MUL, [a, b])
    s = sg.sg_reduce(ctx, prod, sg.SG_SUM)
    sg.sg_release(ctx, prod)
    return {"a": a, "b": b, "sum": s}


def axpy(ctx, dtype, n, alpha, px, py, pout=None):
    """aX+Y: X.multiplied_by(a).plus(Y) — one elementwise kernel with one extra scalar argument."""
    x = sg.sg_vec_create(ctx, dtype, n, px)
    y = sg.sg_vec_create(ctx, dtype, n, py)
    ax = sg.sg_enqueue(ctx, sg.SG_MUL, [x, F(alpha)])
    if pout is not None:
        out = sg.sg_vec_create(ctx, dtype, n, pout)
        r = sg.sg_enqueue(ctx, sg.SG_ADD, [ax, y], dst_or_0=out)
    else:
        r = sg.sg_enqueue(ctx, sg.SG_ADD, [ax, y])
    sg.sg_release(ctx, ax)
    return {"x": x, "y": y, "out": r}


def ge_row_op(ctx, n, prow_i, prow_step, pivot):
    """row(i).divided_by(pivot); row(i).in_place_minus(row(step)) -> (A[i]/pivot) - A[step]."""
    ri = sg.sg_vec_create(ctx, sg.SG_F64, n, prow_i)
    rs = sg.sg_vec_create(ctx, sg.SG_F64, n, prow_step)
    sg.sg_enqueue(ctx, sg.SG_DIV, [ri, F(pivot)], dst_or_0=ri)
    sg.sg_enqueue(ctx, sg.SG_SUB, [ri, rs], dst_or_0=ri)
    return {"row_i": ri, "row_step": rs}


def _cfg0_chain(ctx, a, b, c, dst=0):
    t1 = sg.sg_enqueue(ctx, sg.SG_ADD, [a, b])
    t2 = sg.sg_enqueue(ctx, sg.SG_MUL, [t1, F(2.5)])
    z = sg.sg_enqueue(ctx, sg.SG_SUB, [t2, c], dst_or_0=dst)
    sg.sg_release(ctx, t1)
    sg.sg_release(ctx, t2)
    return z


def cfg0(ctx, n, pa, pb, pc, pz=None, keep_z=True, contracts=True):
    """BASELINE.json:configs[0]: z = (a+b)*2.5 - c; sum/max/min(z); pre exists(a>0.99); post for_all(z == recomputed).

    keep_z=True  (plan P2): z is a named result -> stored by pass A; the postcondition re-reads it in pass B.
    keep_z=False (plan P1): z is released -> everything is one pass over a, b, c.
    """
    a = sg.sg_vec_create(ctx, sg.SG_F64, n, pa)
    b = sg.sg_vec_create(ctx, sg.SG_F64, n, pb)
    c = sg.sg_vec_create(ctx, sg.SG_F64, n, pc)
    res = {"a": a, "b": b, "c": c}
    if contracts:
        m = sg.sg_enqueue(ctx, sg.SG_GT, [a, F(0.99)])
        res["pre"] = sg.sg_exists(ctx, m)
        sg.sg_release(ctx, m)
        sg.sg_contract(ctx, res["pre"], sg.SG_CONTRACT_PRE, "exists(a_i > 0.99)")
    dst = sg.sg_vec_create(ctx, sg.SG_F64, n, pz) if (keep_z and pz is not None) else 0
    z = _cfg0_chain(ctx, a, b, c, dst)
    res["z"] = z
    res["sum"] = sg.sg_reduce(ctx, z, sg.SG_SUM)
    res["max"] = sg.sg_reduce(ctx, z, sg.SG_RMAX)
    res["min"] = sg.sg_reduce(ctx, z, sg.SG_RMIN)
    if contracts:
        z2 = _cfg0_chain(ctx, a, b, c)
        eq = sg.sg_enqueue(ctx, sg.SG_EQ, [z, z2])
        res["post"] = sg.sg_forall(ctx, eq)
        sg.sg_release(ctx, z2)
        sg.sg_release(ctx, eq)
        sg.sg_contract(ctx, res["post"], sg.SG_CONTRACT_POST, "for_all(z_i == (a_i+b_i)*2.5-c_i)")
    if not keep_z:
        sg.sg_release(ctx, z)
        res.pop("z")
    return res


def cfg1_chain(ctx, x, y):
    """w = abs(x*y + 0.5) - min(x,y)*3 + x/(1+y*y), ten primitives, left to right (BASELINE.json:configs[1])."""
    t1 = sg.sg_enqueue(ctx, sg.SG_MUL, [x, y])
    t2 = sg.sg_enqueue(ctx, sg.SG_ADD, [t1, F(0.5)])
    t3 = sg.sg_enqueue(ctx, sg.SG_ABS, [t2])
    t4 = sg.sg_enqueue(ctx, sg.SG_MIN, [x, y])
    t5 = sg.sg_enqueue(ctx, sg.SG_MUL, [t4, F(3.0)])
    t6 = sg.sg_enqueue(ctx, sg.SG_SUB, [t3, t5])
    t7 = sg.sg_enqueue(ctx, sg.SG_MUL, [y, y])
    t8 = sg.sg_enqueue(ctx, sg.SG_ADD, [F(1.0), t7])
    t9 = sg.sg_enqueue(ctx, sg.SG_DIV, [x, t8])
    w = sg.sg_enqueue(ctx, sg.SG_ADD, [t6, t9])
    for t in (t1, t2, t3, t4, t5, t6, t7, t8, t9):
        sg.sg_release(ctx, t)
    return w


def cfg1(ctx, n, px, py, keep_w=False):
    x = sg.sg_vec_create(ctx, sg.SG_F32, n, px)
    y = sg.sg_vec_create(ctx, sg.SG_F32, n, py)
    w = cfg1_chain(ctx, x, y)
    res = {"x": x, "y": y, "sum": sg.sg_reduce(ctx, w, sg.SG_SUM), "max": sg.sg_reduce(ctx, w, sg.SG_RMAX)}
    if keep_w:
        res["w"] = w
    else:
        sg.sg_release(ctx, w)
    return res


def cfg1_sharded(ctx, n_local, px, py, p_part_sum, p_part_max, gather):
    """config 1 on ONE collection sharded over the ranks.  Each rank runs the fused chain on its contiguous range (px,
    py: the shard's n_local elements) and leaves its partial sum (f64) and partial max (f32) in the one-element device buffers
    p_part_sum / p_part_max — device-resident, nothing visits the host.  `gather(kind)` is the exchange step: it returns (device
    pointer, count) of ALL ranks' partials of that kind in rank order (ranks.all_gather_1d over NCCL: 8 + 4 bytes per rank).  The
    combine is a pass of the library over those W-element vectors: a sum of W partial sums (double-double accumulation, fixed rank
    order: deterministic) and the max of W partial maxima under the total order.  Returns the handles of the two global scalars."""
    x = sg.sg_vec_create(ctx, sg.SG_F32, n_local, px)
    y = sg.sg_vec_create(ctx, sg.SG_F32, n_local, py)
    wv = cfg1_chain(ctx, x, y)
    s, m = sg.sg_reduce(ctx, wv, sg.SG_SUM), sg.sg_reduce(ctx, wv, sg.SG_RMAX)
    sg.sg_release(ctx, wv)
    ps = sg.sg_vec_create(ctx, sg.SG_F64, 1, p_part_sum)
    pm = sg.sg_vec_create(ctx, sg.SG_F32, 1, p_part_max)
    sg.sg_enqueue(ctx, sg.SG_ADD, [s, F(0.0)], dst_or_0=ps)            # the deferred scalars land in caller-visible device memory ...
    sg.sg_enqueue(ctx, sg.SG_MAX, [m, m], dst_or_0=pm)
    sg.sg_flush(ctx)                                                   # ... asynchronously: the collective is stream-ordered after it
    all_s, w_s = gather("sum")
    all_m, w_m = gather("max")
    gs = sg.sg_reduce(ctx, sg.sg_vec_create(ctx, sg.SG_F64, w_s, all_s), sg.SG_SUM)
    gm = sg.sg_reduce(ctx, sg.sg_vec_create(ctx, sg.SG_F32, w_m, all_m), sg.SG_RMAX)
    return {"x": x, "y": y, "sum": gs, "max": gm, "part_sum": s, "part_max": m, "ps": ps, "pm": pm}


def cfg2(ctx, n, px, pout=None, capacity=0, modulus=7, residue=3):
    """BASELINE.json:configs[2]: stable filter keeping x where x mod 7 == 3, count, int64 sum of the kept values."""
    x = sg.sg_vec_create(ctx, sg.SG_I32, n, px)
    r = sg.sg_enqueue(ctx, sg.SG_MOD, [x, I(modulus)])
    m = sg.sg_enqueue(ctx, sg.SG_EQ, [r, I(residue)])
    kept, count = sg.sg_filter(ctx, x, m, pout, capacity)
    s = sg.sg_reduce(ctx, kept, sg.SG_SUM)
    sg.sg_release(ctx, r)
    sg.sg_release(ctx, m)
    return {"x": x, "kept": kept, "count": count, "sum": s}


def cfg3(ctx, n, px, contracts=False):
    """BASELINE.json:configs[3]: pre for_all(x_i >= 0), post is-sorted for_all(x_i <= x_{i+1})."""
    x = sg.sg_vec_create(ctx, sg.SG_F32, n, px)
    ge = sg.sg_enqueue(ctx, sg.SG_GE, [x, F(0.0)])
    pre = sg.sg_forall(ctx, ge)
    sg.sg_release(ctx, ge)
    post = sg.sg_forall_adjacent(ctx, x, sg.SG_LE)
    if contracts:
        sg.sg_contract(ctx, pre, sg.SG_CONTRACT_PRE, "for_all(x_i >= 0)")
        sg.sg_contract(ctx, post, sg.SG_CONTRACT_PRE, "is_sorted")
    return {"x": x, "pre": pre, "post": post}


def cfg4(ctx, n, pM, k, ld=None):
    """BASELINE.json:configs[4]: M[j,:] -= (M[j,k]/M[k,k]) * M[k,:] for all j>k, fused with row-wise max|.| and column sums.

    Pass 1 (vector): f = column(k)[k+1:] / M[k,k]  — read BEFORE the rows are modified.
    Pass 2 (matrix): t = f (COL-broadcast) * row(k) (ROW-broadcast); rows(k+1..) -= t in place; rowmax, colsum.
    """
    ld = n if ld is None else ld
    M = sg.sg_mat_create(ctx, sg.SG_F64, n, n, ld, pM)
    res = {"M": M}
    if k + 1 >= n:
        return res
    piv = sg.sg_mat_elem(ctx, M, k, k)
    col = sg.sg_mat_col(ctx, M, k, k + 1, n)
    f = sg.sg_enqueue(ctx, sg.SG_DIV, [col, piv])
    rowk = sg.sg_mat_row(ctx, M, k)
    sub = sg.sg_mat_rows(ctx, M, k + 1, n)
    t = sg.sg_enqueue(ctx, sg.SG_MUL, [H(f, sg.SG_BCAST_COL), H(rowk, sg.SG_BCAST_ROW)])
    sg.sg_enqueue(ctx, sg.SG_SUB, [sub, t], dst_or_0=sub)
    ab = sg.sg_enqueue(ctx, sg.SG_ABS, [sub])
    res["rowmax"] = sg.sg_reduce(ctx, ab, sg.SG_RMAX, sg.SG_AXIS_ROWS)
    res["colsum"] = sg.sg_reduce(ctx, sub, sg.SG_SUM, sg.SG_AXIS_COLS)
    for h in (col, t, ab, piv, f):
        sg.sg_release(ctx, h)
    res["sub"] = sub
    return res


def ge_row_update(ctx, n, pM, k, ld=None):
    """Listing 5's row update alone: M[j,:] -= (M[j,k]/M[k,k]) * M[k,:] for all rows j > k in ONE matrix pass that
    only stores (config 4 without its two reductions).  Pass 1: the factors, read before the rows change; pass 2: the update."""
    ld = n if ld is None else ld
    M = sg.sg_mat_create(ctx, sg.SG_F64, n, n, ld, pM)
    res = {"M": M}
    if k + 1 >= n:
        return res
    piv = sg.sg_mat_elem(ctx, M, k, k)
    col = sg.sg_mat_col(ctx, M, k, k + 1, n)
    f = sg.sg_enqueue(ctx, sg.SG_DIV, [col, piv])
    rowk = sg.sg_mat_row(ctx, M, k)
    sub = sg.sg_mat_rows(ctx, M, k + 1, n)
    t = sg.sg_enqueue(ctx, sg.SG_MUL, [H(f, sg.SG_BCAST_COL), H(rowk, sg.SG_BCAST_ROW)])
    sg.sg_enqueue(ctx, sg.SG_SUB, [sub, t], dst_or_0=sub)
    for h in (col, t, piv, f, rowk):
        sg.sg_release(ctx, h)
    res["sub"] = sub
    return res


def ge_step(ctx, M, n, k, det, minpiv):
    """One step of Listing 5 enqueued without a trigger: Result := Result * pivot and the
    smallest |pivot| so far on a one-element domain, then, for all rows j > k in ONE matrix pass, the row update of
    BASELINE.json:configs[4] (the paper launches one kernel per row, its slow case PAPER.md:389).  The pivot stays on the
    device (sg_mat_elem), nothing is read back."""
    rowk = sg.sg_mat_row(ctx, M, k)
    d = sg.sg_vec_subset(ctx, rowk, k, k + 1)                   # M[k,k] as a one-element collection
    sg.sg_enqueue(ctx, sg.SG_MUL, [det, d], dst_or_0=det)
    ad = sg.sg_enqueue(ctx, sg.SG_ABS, [d])
    sg.sg_enqueue(ctx, sg.SG_MIN, [minpiv, ad], dst_or_0=minpiv)
    tmp = [ad, d]
    if k + 1 < n:
        piv = sg.sg_mat_elem(ctx, M, k, k)
        col = sg.sg_mat_col(ctx, M, k, k + 1, n)
        f = sg.sg_enqueue(ctx, sg.SG_DIV, [col, piv])          # read BEFORE the rows change: its own small pass
        sub = sg.sg_mat_rows(ctx, M, k + 1, n)
        t = sg.sg_enqueue(ctx, sg.SG_MUL, [H(f, sg.SG_BCAST_COL), H(rowk, sg.SG_BCAST_ROW)])
        sg.sg_enqueue(ctx, sg.SG_SUB, [sub, t], dst_or_0=sub)
        tmp += [piv, col, f, t, sub]
    return tmp + [rowk]


def ge_determinant(ctx, n, pM, pdet, pminpiv, ld=None, eps=0.0, native=True):
    """Listing 5: the whole determinant loop with no host synchronisation between steps.

    pdet / pminpiv: device float64[1] initialised by the caller to 1.0 / +inf.
    native=True: sg_mat_ge_steps — ONE persistent kernel runs all n steps, incl. the listing's control flow: Result := Result *
    pivot before the approximately-zero test, the loop ends at a pivot with |pivot| <= eps, rows whose entry
    below the pivot is ~0 are skipped.  Every decision of the method is taken on the device; this function
    only reads the two results back.
    native=False: the same steps as host-issued primitives (ge_step + one asynchronous flush per step = 3 launches per step):
    the measurement baseline for the paper's slow case.  It has no device-side loop exit, so it is the listing only
    for matrices without an approximately-zero pivot or sub-pivot entry.
    Returns (det, ok): det = Result as the device computed it; ok = no pivot was approximately zero."""
    ld = n if ld is None else ld
    M = sg.sg_mat_create(ctx, sg.SG_F64, n, n, ld, pM)
    det = sg.sg_vec_create(ctx, sg.SG_F64, 1, pdet)
    minpiv = sg.sg_vec_create(ctx, sg.SG_F64, 1, pminpiv)
    if native:
        sg.sg_mat_ge_steps(ctx, M, det, minpiv, eps, 0, n)
    else:
        for k in range(n):
            for h in ge_step(ctx, M, n, k, det, minpiv):
                sg.sg_release(ctx, h)
            sg.sg_flush(ctx)                                    # asynchronous: plan + launches of step k, no read-back
    gt = sg.sg_enqueue(ctx, sg.SG_GT, [minpiv, F(eps)])
    ok = sg.sg_forall(ctx, gt)
    value = sg.sg_reduce(ctx, det, sg.SG_RMAX)                  # max of one element = the element, bit for bit (a sum would turn -0 into +0): hands the scalar back (trigger (1))
    okv = bool(sg.sg_scalar_get(ctx, ok))
    detv = float(sg.sg_scalar_get(ctx, value))
    for h in (gt, ok, value, det, minpiv, M):
        sg.sg_release(ctx, h)
    return detv, okv


# ------------------------------------------------------------------------------------------------------------------
# the rest of the vector API
# ------------------------------------------------------------------------------------------------------------------
def project_sqrt(ctx, dtype, n, pa, pout=None):
    """`a.project (agent sqrt)`: a new collection of the correctly rounded square roots.  An INTEGER collection
    gives a collection of DOUBLEs (the paper's own example): the integers are converted as they are loaded, one pass, 4 or 8 bytes
    read and 8 written per element."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    out_dtype = dtype if dtype in (sg.SG_F32, sg.SG_F64) else sg.SG_F64
    dst = sg.sg_vec_create(ctx, out_dtype, n, pout) if pout is not None else 0
    r = sg.sg_enqueue(ctx, sg.SG_SQRT, [a], dst_or_0=dst)
    return {"a": a, "out": r}


def norm2(ctx, dtype, n, pa):
    """Euclidean norm sqrt(sum(a*a)): Listing 4's dot product followed by the sqrt agent applied to the
    device-resident sum (a one-element result; fp64 like every float sum).  Two passes: the vector pass and a 1-element pass."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    sq = sg.sg_enqueue(ctx, sg.SG_MUL, [a, a])
    s = sg.sg_reduce(ctx, sq, sg.SG_SUM)
    sg.sg_release(ctx, sq)
    r = sg.sg_enqueue(ctx, sg.SG_SQRT, [s])
    return {"a": a, "sum": s, "norm": r}


def avg(ctx, dtype, n, pa):
    """`avg` of a float collection = sum / count, divided on the device: the deferred fp64 sum is a device scalar
    operand of a one-element pass, nothing is read back in between."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    s = sg.sg_reduce(ctx, a, sg.SG_SUM)
    r = sg.sg_enqueue(ctx, sg.SG_DIV, [s, F(float(n))])
    return {"a": a, "sum": s, "avg": r}


def compwise_divide(ctx, dtype, n, pa, pb, pout=None, eps=None):
    """Listing 2: `require not other.exists (is_zero)`, `Result := a / b`, `ensure Result * other = Current`.

    The precondition is a registered device-evaluated contract fused into the pass that divides (the body writes only a fresh
    output, R17).  eps given: the postcondition is |Result*other - Current| <= eps (the approximate equality of
    PAPER.md:339), registered as a POST contract, so it re-reads the STORED quotient in a second pass (R17).  eps=None: exact
    equality as printed in the listing (false in general: a/b*b rounds twice) — evaluated as a plain quantifier, not
    registered, in the same pass.  A violated registered contract makes the flush fail with SG_ERR_CONTRACT and its tag."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    b = sg.sg_vec_create(ctx, dtype, n, pb)
    z = sg.sg_enqueue(ctx, sg.SG_EQ, [b, F(0.0) if dtype in (sg.SG_F32, sg.SG_F64) else I(0)])
    has_zero = sg.sg_exists(ctx, z)
    nz = sg.sg_enqueue(ctx, sg.SG_NOT, [z])
    pre = sg.sg_forall(ctx, nz)
    sg.sg_contract(ctx, pre, sg.SG_CONTRACT_PRE, "not other.exists (is_zero)")
    dst = sg.sg_vec_create(ctx, dtype, n, pout) if pout is not None else 0
    q = sg.sg_enqueue(ctx, sg.SG_DIV, [a, b], dst_or_0=dst)
    back = sg.sg_enqueue(ctx, sg.SG_MUL, [q, b])
    if eps is None:
        ok = sg.sg_enqueue(ctx, sg.SG_EQ, [back, a])
        tmp = [back]
    else:
        d = sg.sg_enqueue(ctx, sg.SG_SUB, [back, a])
        ad = sg.sg_enqueue(ctx, sg.SG_ABS, [d])
        ok = sg.sg_enqueue(ctx, sg.SG_LE, [ad, F(eps)])
        tmp = [back, d, ad]
    post = sg.sg_forall(ctx, ok)
    if eps is not None:
        sg.sg_contract(ctx, post, sg.SG_CONTRACT_POST, "Result * other = Current (approx)")
    for h in tmp + [z, nz, ok]:
        sg.sg_release(ctx, h)
    return {"a": a, "b": b, "out": q, "pre": pre, "has_zero": has_zero, "post": post}


def approx_equal(ctx, dtype, n, pa, pb, eps):
    """`double_approx_equals` lifted to collections: for_all(|a_i - b_i| <= eps), plus the largest deviation."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    b = sg.sg_vec_create(ctx, dtype, n, pb)
    d = sg.sg_enqueue(ctx, sg.SG_SUB, [a, b])
    ad = sg.sg_enqueue(ctx, sg.SG_ABS, [d])
    le = sg.sg_enqueue(ctx, sg.SG_LE, [ad, F(eps)])
    res = {"a": a, "b": b, "all": sg.sg_forall(ctx, le), "maxdev": sg.sg_reduce(ctx, ad, sg.SG_RMAX)}
    for h in (d, ad, le):
        sg.sg_release(ctx, h)
    return res


# ------------------------------------------------------------------------------------------------------------------
# quicksort (Listing 3)
# ------------------------------------------------------------------------------------------------------------------
_ES = {sg.SG_F32: 4, sg.SG_F64: 8, sg.SG_I32: 4, sg.SG_I64: 8}


def quicksort(ctx, dtype, n, pa, pout, pscratch0, pscratch1, contracts=True):
    """Listing 3 written over the C ABI.  pa: the input (left untouched); pout: the result; pscratch0/1: two device buffers of n
    elements each (caller-owned, like every buffer here).

    Each call of the listing's body becomes: the pivot a[a.count // 2] as a DEVICE scalar (it never visits the host: a
    one-element max), the three predicate agents `item < / = / > pivot` closed over it, their counts in one fused
    pass (the only values read back: they are the `count`s of left, mid and right, scalar contracts in the paper's sense,
    PAPER.md:270), then the three stable filters.  `concatenate` costs nothing: since the counts are known,
    each filter writes straight to its final place — left to [o, o+nl) and right to [o+nl+nm, o+n) of the scratch buffer of
    the next depth, mid to [o+nl, o+nl+nm) of the result — so quicksort(left) ++ mid ++ quicksort(right) is already contiguous.
    The recursion runs on an explicit stack (sub-ranges are disjoint, buffers alternate with the depth).
    Postconditions (contracts=True): Result.is_sorted as a registered device contract, Result.count = a.count on the host.
    Returns {"out": handle, "partitions": number of listing-body executions}."""
    if n <= 0:
        raise ValueError("quicksort: require a.count > 0")
    es = _ES[dtype]
    scratch = (pscratch0, pscratch1)
    stack = [(pa, 0, 0, n, 0)]              # (buffer base, element offset in that buffer, offset o in the result, count, depth)
    partitions = 0
    placed = 0
    while stack:
        base, off, o, m, depth = stack.pop()
        partitions += 1
        a = sg.sg_vec_create(ctx, dtype, m, base + off * es)
        mid1 = sg.sg_vec_subset(ctx, a, m // 2, m // 2 + 1)
        pivot = sg.sg_reduce(ctx, mid1, sg.SG_RMAX)                   # the element itself, device-resident
        lt = sg.sg_enqueue(ctx, sg.SG_LT, [a, H(pivot)])
        eq = sg.sg_enqueue(ctx, sg.SG_EQ, [a, H(pivot)])
        gt = sg.sg_enqueue(ctx, sg.SG_GT, [a, H(pivot)])
        if m == 1:                                                     # `if a.count = 1 then Result := a`: nothing to count
            hl = hm = None
            nl, nm = 0, 1
        else:
            hl, hm = sg.sg_reduce(ctx, lt, sg.SG_COUNT), sg.sg_reduce(ctx, eq, sg.SG_COUNT)
            nl, nm = sg.sg_scalar_get(ctx, hl), sg.sg_scalar_get(ctx, hm)  # trigger: one flush, two small passes
        nr = m - nl - nm
        nxt = scratch[depth % 2]
        outs = []
        if nl:
            outs.append(sg.sg_filter(ctx, a, lt, nxt + o * es, nl))
        outs.append(sg.sg_filter(ctx, a, eq, pout + (o + nl) * es, nm))
        if nr:
            outs.append(sg.sg_filter(ctx, a, gt, nxt + (o + nl + nm) * es, nr))
        sg.sg_flush(ctx)                                               # asynchronous: nothing is read back
        placed += nm
        for h in [hl, hm, lt, eq, gt, pivot, mid1, a] + [x for pair in outs for x in pair]:
            if h is not None:
                sg.sg_release(ctx, h)
        if nr > 0:
            stack.append((nxt, o + nl + nm, o + nl + nm, nr, depth + 1))
        if nl > 0:
            stack.append((nxt, o, o, nl, depth + 1))
    out = sg.sg_vec_create(ctx, dtype, n, pout)
    res = {"out": out, "partitions": partitions}
    if contracts:
        if placed != n:
            raise AssertionError(f"quicksort postcondition Result.count = a.count violated: {placed} != {n}")
        res["sorted"] = sg.sg_forall_adjacent(ctx, out, sg.SG_LE)
        sg.sg_contract(ctx, res["sorted"], sg.SG_CONTRACT_POST, "Result.is_sorted")
    return res


def quicksort_levels(ctx, dtype, n, pa, pout=None, contracts=True):
    """Listing 3 through the library composite sg_vec_quicksort: one segmented three-way partition launch per recursion level (the
    multi-output partition kernel), counts and segment tables stay on the device.  The listing's postconditions: Result.is_sorted
    as a registered device contract; Result.count = a.count is a scalar contract (O(1))."""
    a = sg.sg_vec_create(ctx, dtype, n, pa)
    out = sg.sg_vec_quicksort(ctx, a, pout)
    res = {"a": a, "out": out}
    if contracts:
        if sg.sg_vec_count(ctx, out) != n:
            raise AssertionError("quicksort postcondition Result.count = a.count violated")
        res["sorted"] = sg.sg_forall_adjacent(ctx, out, sg.SG_LE)
        sg.sg_contract(ctx, res["sorted"], sg.SG_CONTRACT_POST, "Result.is_sorted")
    return res


# ------------------------------------------------------------------------------------------------------------------
# memory-bound matrix-vector products
# ------------------------------------------------------------------------------------------------------------------
def right_multiply(ctx, rows, cols, pM, pv, ld=None):
    """matrix x column vector: result_i = sum_c M[i,c]*v[c] — the product is an anonymous intermediate of ONE matrix pass (v
    broadcast along the rows, per-row sums).  The dimension contract columns = v.count is checked at enqueue."""
    M = sg.sg_mat_create(ctx, sg.SG_F64, rows, cols, cols if ld is None else ld, pM)
    v = sg.sg_vec_create(ctx, sg.SG_F64, cols, pv)
    t = sg.sg_enqueue(ctx, sg.SG_MUL, [M, H(v, sg.SG_BCAST_ROW)])
    r = sg.sg_reduce(ctx, t, sg.SG_SUM, sg.SG_AXIS_ROWS)
    sg.sg_release(ctx, t)
    return {"M": M, "v": v, "out": r}


def left_multiply(ctx, rows, cols, pv, pM, ld=None):
    """row vector x matrix: result_c = sum_i v[i]*M[i,c] — v broadcast along the columns, per-column sums, one matrix pass."""
    M = sg.sg_mat_create(ctx, sg.SG_F64, rows, cols, cols if ld is None else ld, pM)
    v = sg.sg_vec_create(ctx, sg.SG_F64, rows, pv)
    t = sg.sg_enqueue(ctx, sg.SG_MUL, [M, H(v, sg.SG_BCAST_COL)])
    r = sg.sg_reduce(ctx, t, sg.SG_SUM, sg.SG_AXIS_COLS)
    sg.sg_release(ctx, t)
    return {"M": M, "v": v, "out": r}


def transpose(ctx, dtype, rows, cols, pM, pout=None, ld=None, ld_out=0):
    """`transpose`: a new cols x rows matrix; one tiled data-mover kernel (sg_mat_transpose), asynchronous."""
    M = sg.sg_mat_create(ctx, dtype, rows, cols, cols if ld is None else ld, pM)
    T = sg.sg_mat_transpose(ctx, M, pout, ld_out)
    return {"M": M, "out": T}
