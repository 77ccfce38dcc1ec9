"""GPU-vs-oracle parity for SURVEY.md §8(f)(3), the rest of the vector API: sqrt projection, avg
(PAPER.md:203), compwise_divide with its contracts (Listing 2), approximate equality.
Elementwise results (sqrt is the correctly rounded IEEE operation on both sides) and quantifiers bit-exact; sums, avg and the
norm within 1e-12 (fp64) / 1e-5 (fp32) relative."""
import numpy as np
import pytest

import oracle as orc
from paper_1410_6685_b200 import sg
from paper_1410_6685_b200 import workloads as W
from gpu_util import Ctx, dev, empty_dev
from test_gpu_parity import MODES, SIZES, bits_equal

pytestmark = pytest.mark.gpu
RNG = np.random.default_rng(4242)


def _sqrt_inputs(n, dtype):
    a = np.abs(RNG.standard_normal(n)).astype(dtype)
    special = np.array([0.0, -0.0, np.inf, -1.0, np.nan, 2.0, 1e-40, 3e38, 4.0, 1.0000001], dtype=dtype)
    k = min(n, special.size)
    if k:
        a[RNG.choice(n, k, replace=False)] = special[:k]
    return a


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n", SIZES)
def test_project_sqrt(mode, dtype, n):
    a = _sqrt_inputs(n, dtype)
    with Ctx(MODES[mode]) as c:
        ta, tout = dev(a), empty_dev(max(n, 1), dtype)
        c.keep += [ta, tout]
        r = W.project_sqrt(c.ctx, sg.SG_F32 if dtype is np.float32 else sg.SG_F64, n, ta.data_ptr(), tout.data_ptr())
        sg.sg_flush(c.ctx)
        got = c.read_vec(r["out"], dtype, n)
        assert sg.sg_plan_stats(c.ctx).n_passes == 1
    want = orc.unary("sqrt", a)
    assert bits_equal(got, want)
    assert np.array_equal(np.signbit(got), np.signbit(want)) or np.isnan(want).any()


def test_sqrt_fused_in_a_chain():
    """sqrt(x*x + y*y) (hypot written with primitives): every op rounds once; one pass; the value also feeds max and sum."""
    n = (1 << 18) + 77
    x, y = RNG.standard_normal(n).astype(np.float32), RNG.standard_normal(n).astype(np.float32)
    with Ctx() as c:
        hx, hy = c.vec(x), c.vec(y)
        xx = sg.sg_enqueue(c.ctx, sg.SG_MUL, [hx, hx])
        yy = sg.sg_enqueue(c.ctx, sg.SG_MUL, [hy, hy])
        s = sg.sg_enqueue(c.ctx, sg.SG_ADD, [xx, yy])
        r = sg.sg_enqueue(c.ctx, sg.SG_SQRT, [s])
        mx, sm = sg.sg_reduce(c.ctx, r, sg.SG_RMAX), sg.sg_reduce(c.ctx, r, sg.SG_SUM)
        for h in (xx, yy, s):
            sg.sg_release(c.ctx, h)
        got_max, got_sum = c.get(mx), c.get(sm)
        assert sg.sg_plan_stats(c.ctx).n_passes == 1
        got = c.read_vec(r, np.float32, n)
    want = orc.unary("sqrt", orc.zip("add", orc.zip("mul", x, x), orc.zip("mul", y, y)))
    assert bits_equal(got, want)
    assert np.float32(got_max) == orc.max(want)
    assert abs(got_sum - orc.sum(want)) <= 1e-5 * abs(orc.sum(want))


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-12), (np.float32, 1e-5)])
@pytest.mark.parametrize("n", [1, 2, 33, 1025, 70001, (1 << 20) + 3])
def test_avg_and_norm_stay_on_the_device(dtype, tol, n):
    a = (RNG.standard_normal(n) + 3.0).astype(dtype)
    sgdt = sg.SG_F32 if dtype is np.float32 else sg.SG_F64
    with Ctx() as c:
        ta = dev(a); c.keep.append(ta)
        r = W.avg(c.ctx, sgdt, n, ta.data_ptr())
        q = W.norm2(c.ctx, sgdt, n, ta.data_ptr())
        sg.sg_flush(c.ctx)                                   # nothing is read back between the sum and the division / sqrt
        got_avg = c.read_vec(r["avg"], np.float64, 1)[0]
        got_norm = c.read_vec(q["norm"], np.float64, 1)[0]
        got_sum, got_ss = c.get(r["sum"]), c.get(q["sum"])
    want_avg = orc.avg(a)
    want_ss = orc.sum(orc.zip("mul", a, a))
    want_norm = orc.unary("sqrt", np.array([want_ss]))[0]
    assert abs(got_avg - want_avg) <= tol * abs(want_avg)
    assert abs(got_norm - want_norm) <= tol * abs(want_norm)
    # the one-element pass itself is exact: it divides / takes the root of the device's own sum with one rounding
    assert got_avg == orc.zip("div", np.array([got_sum]), np.array([float(n)]))[0]
    assert got_norm == orc.unary("sqrt", np.array([got_ss]))[0]


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", [1, 33, 4097, (1 << 18) + 5])
def test_compwise_divide_listing2(mode, dtype, n):
    a = RNG.uniform(-4, 4, n).astype(dtype)
    b = (RNG.uniform(0.5, 2, n) * RNG.choice([-1.0, 1.0], n)).astype(dtype)
    eps = 1e-12 if dtype is np.float64 else 1e-5
    sgdt = sg.SG_F32 if dtype is np.float32 else sg.SG_F64
    want_q = orc.zip("div", a, b)
    back = orc.zip("mul", want_q, b)
    want_exact = orc.all(orc.cmp("eq", back, a))
    want_approx = orc.all(orc.cmp_scalar("le", orc.unary("abs", orc.zip("sub", back, a)), eps))
    assert want_approx is True
    for use_eps, want_post in ((None, want_exact), (eps, want_approx)):
        with Ctx(MODES[mode]) as c:
            ta, tb, tq = dev(a), dev(b), empty_dev(n, dtype)
            c.keep += [ta, tb, tq]
            r = W.compwise_divide(c.ctx, sgdt, n, ta.data_ptr(), tb.data_ptr(), tq.data_ptr(), eps=use_eps)
            assert c.get(r["post"]) == want_post
            assert c.get(r["pre"]) is True or c.get(r["pre"]) == 1
            assert not c.get(r["has_zero"])
            assert bits_equal(c.read_vec(r["out"], dtype, n), want_q)


@pytest.mark.parametrize("zero", [0.0, -0.0])
@pytest.mark.parametrize("pos", ["first", "middle", "last"])
def test_compwise_divide_zero_divisor_violates_the_precondition(zero, pos):
    n = 100003
    a = RNG.uniform(-4, 4, n)
    b = RNG.uniform(0.5, 2, n)
    b[{"first": 0, "middle": n // 2, "last": n - 1}[pos]] = zero
    assert orc.any(orc.cmp_scalar("eq", b, 0.0)) is True
    with Ctx() as c:
        ta, tb = dev(a), dev(b)
        c.keep += [ta, tb]
        W.compwise_divide(c.ctx, sg.SG_F64, n, ta.data_ptr(), tb.data_ptr(), eps=1e-12)
        with pytest.raises(sg.SgError) as e:
            sg.sg_flush(c.ctx)
        assert e.value.status == sg.SG_ERR_CONTRACT and "is_zero" in str(e.value)


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_approx_equal(mode, dtype):
    n = (1 << 17) + 9
    a = RNG.standard_normal(n).astype(dtype)
    noise = (RNG.uniform(-1, 1, n) * 1e-4).astype(dtype)
    b = orc.zip("add", a, noise)
    ad = orc.unary("abs", orc.zip("sub", a, b))
    sgdt = sg.SG_F32 if dtype is np.float32 else sg.SG_F64
    for eps in (1e-3, 1e-4, 5e-5, 0.0):
        with Ctx(MODES[mode]) as c:
            ta, tb = dev(a), dev(b)
            c.keep += [ta, tb]
            r = W.approx_equal(c.ctx, sgdt, n, ta.data_ptr(), tb.data_ptr(), eps)
            got_all, got_max = bool(c.get(r["all"])), c.get(r["maxdev"])
        assert got_all == orc.all(orc.cmp_scalar("le", ad, eps))
        assert dtype(got_max) == orc.max(ad)


# ----------------------------------------------------------------------------------------------------------
# quicksort (Listing 3)
# ----------------------------------------------------------------------------------------------------------
from oracle import configs as ocfg  # noqa: E402


def _quicksort_on_device(a, flags=0):
    n = a.size
    with Ctx(flags) as c:
        ta = dev(a)
        tout, s0, s1 = (empty_dev(n, a.dtype) for _ in range(3))
        c.keep += [ta, tout, s0, s1]
        before = ta.clone()
        r = W.quicksort(c.ctx, sg.SG_F32 if a.dtype == np.float32 else sg.SG_F64, n, ta.data_ptr(), tout.data_ptr(), s0.data_ptr(), s1.data_ptr())
        ok = c.get(r["sorted"])
        got = c.read_vec(r["out"], a.dtype, n)
        assert bits_equal(before.cpu().numpy(), ta.cpu().numpy())          # the argument is not modified
    return got, ok, r["partitions"]


@pytest.mark.parametrize("n", [1, 2, 3, 17, 1000, 4099, 20011])
def test_quicksort_listing3(n):
    for a in (RNG.standard_normal(n).astype(np.float32), RNG.integers(-50, 51, n).astype(np.float32)):
        got, ok, parts = _quicksort_on_device(a)
        want = ocfg.quicksort(a)
        assert ok is True and bits_equal(got, want)                         # stable filters => the result is unique, bit for bit
        assert parts <= n


def test_quicksort_signed_zeros_sorted_input_fp64_and_bytecode():
    a = np.array([0.0, 3.0, -0.0, 1.0, 0.0, -0.0, 3.0, -2.5], dtype=np.float32)
    got, ok, _ = _quicksort_on_device(a)
    assert ok and bits_equal(got, ocfg.quicksort(a))
    for a in (np.arange(3000, dtype=np.float64), np.arange(3000, dtype=np.float64)[::-1].copy(), RNG.standard_normal(2500)):
        got, ok, _ = _quicksort_on_device(a, sg.SG_FLAG_FORCE_BYTECODE)
        assert ok and bits_equal(got, ocfg.quicksort(a))


def _quicksort_levels(a, pout=False):
    from gpu_util import NP2SG
    n = a.size
    with Ctx() as c:
        ta = dev(a); c.keep.append(ta)
        before = ta.clone()
        tout = empty_dev(max(n, 1), a.dtype) if pout else None
        if tout is not None:
            c.keep.append(tout)
        r = W.quicksort_levels(c.ctx, NP2SG[a.dtype], n, ta.data_ptr(), tout.data_ptr() if pout else None)
        ok = c.get(r["sorted"])
        got = c.read_vec(r["out"], a.dtype, n)
        launches = sg.sg_plan_stats(c.ctx).launches_total
        assert bits_equal(before.cpu().numpy(), ta.cpu().numpy())          # the argument is not modified
    return got, ok, launches


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
@pytest.mark.parametrize("n", [1, 2, 3, 17, 1000, 2047, 2048, 2049, 4099, 20011, 65536 + 3])
def test_quicksort_levels_against_the_listing(dtype, n):
    """sg_vec_quicksort (one segmented three-way partition launch per recursion level) against the oracle's Listing-3 recursion: random
    keys, few distinct keys (long `=` runs: the staged mid copies), bit for bit (stable filters make the result unique)."""
    for a in ((RNG.standard_normal(n) * 1000).astype(dtype), RNG.integers(-50, 51, n).astype(dtype)):
        got, ok, _ = _quicksort_levels(a, pout=(n % 2 == 0))
        assert ok is True and bits_equal(got, ocfg.quicksort(a))


def test_quicksort_levels_structured_inputs():
    n = 50000
    base = np.arange(n, dtype=np.float64)
    cases = [base, base[::-1].copy(), np.zeros(n), np.where(np.arange(n) % 2 == 0, 0.0, -0.0), np.concatenate([base[: n // 2], base[: n // 2]]),
             np.repeat(np.arange(5, dtype=np.float64), n // 5)[::-1].copy()]
    z = RNG.integers(-3, 4, n).astype(np.float32)
    z[z == 0] = np.where(RNG.random((z == 0).sum()) < 0.5, np.float32(0.0), np.float32(-0.0))      # +0 and -0 keep their order (equal keys)
    cases.append(z)
    for a in cases:
        got, ok, _ = _quicksort_levels(a)
        assert ok is True and bits_equal(got, ocfg.quicksort(a)) and bits_equal(got, np.sort(a, kind="stable"))


def test_quicksort_levels_large_and_contracts():
    """2^20 + 7 fp32 keys: the listing's result is the stable sort (pinned for the oracle in test_oracle_pins.py at sizes the recursion
    finishes; a property that holds at any size), compared element by element; a few dozen launches, not one per partition."""
    n = (1 << 20) + 7
    a = inputs_normal(n)
    got, ok, launches = _quicksort_levels(a)
    assert ok is True and bits_equal(got, np.sort(a, kind="stable"))
    assert launches < 120
    m = 1 << 16                                                             # the same kernels on a prefix the oracle's recursion finishes in seconds
    got, ok, _ = _quicksort_levels(a[:m].copy())
    assert ok and bits_equal(got, ocfg.quicksort(a[:m]))
    with Ctx() as c:
        with pytest.raises(sg.SgError) as e:                                # require a.count > 0
            sg.sg_vec_quicksort(c.ctx, sg.sg_vec_create(c.ctx, sg.SG_F32, 0, None))
        assert e.value.status == sg.SG_ERR_EMPTY
        for k in (5, 5000):                                                 # a NaN key is in none of the three filters: Result.count = a.count fails
            b = a[: 3 * k].copy()
            b[k] = np.nan
            with pytest.raises(sg.SgError) as e:
                sg.sg_vec_quicksort(c.ctx, c.vec(b))
            assert e.value.status == sg.SG_ERR_CONTRACT and "Result.count" in str(e.value)
            assert ocfg.quicksort(b).size < b.size                          # the oracle's listing drops it too
        one = c.vec(np.array([np.nan], dtype=np.float32))                   # a.count = 1: Result := a, nothing is compared
        assert np.isnan(c.read_vec(sg.sg_vec_quicksort(c.ctx, one), np.float32, 1)[0])
        t = dev(a[:1000]); c.keep.append(t)
        with pytest.raises(sg.SgError) as e:
            sg.sg_vec_quicksort(c.ctx, sg.sg_vec_create(c.ctx, sg.SG_F32, 1000, t.data_ptr()), t.data_ptr() + 400)
        assert e.value.status == sg.SG_ERR_ALIAS


def test_quicksort_levels_of_a_view_and_of_a_pending_collection():
    """The argument may be a subset view (any alignment) or a pending collection (flushed first)."""
    a = inputs_normal(50021)
    with Ctx() as c:
        h = c.vec(a)
        view = sg.sg_vec_subset(c.ctx, h, 3, 50021 - 2)
        got = c.read_vec(sg.sg_vec_quicksort(c.ctx, view), np.float32)
        assert bits_equal(got, ocfg.quicksort(a[3:-2]))
        neg = sg.sg_enqueue(c.ctx, sg.SG_NEG, [h])                          # pending when the sort is asked for
        got = c.read_vec(sg.sg_vec_quicksort(c.ctx, neg), np.float32)
        assert bits_equal(got, ocfg.quicksort(orc.unary("neg", a)))
        assert bits_equal(c.read_vec(h, np.float32), a)


def inputs_normal(n):
    from paper_1410_6685_b200 import inputs
    return inputs.normal_f32(2, 0, n)


# ----------------------------------------------------------------------------------------------------------
# matrix-vector products — fp64 sums within 1e-12 relative of the oracle
# ----------------------------------------------------------------------------------------------------------
# any shape: rows that are not 16-byte aligned (odd fp64 column counts or leading dimensions) take the matrix pass's
# guarded form — the shapes (1,1,1), (2,3,3), (33,17,20), (777,2051,2051) are the ones the aligned-only kernel of round 1 rejected
@pytest.mark.parametrize("rows,cols,ld", [(1, 2, 2), (2, 2, 2), (3, 4, 6), (33, 18, 20), (258, 1030, 1030), (1030, 258, 264), (777, 2050, 2052),
                                          (1, 1, 1), (2, 3, 3), (4, 3, 3), (33, 17, 20), (33, 18, 19), (777, 2051, 2051), (515, 1025, 1031), (1, 1025, 1025)])
def test_matvec_right_and_left(rows, cols, ld):
    M = RNG.uniform(0.0, 1.0, (rows, cols))
    v, w = RNG.uniform(0.5, 1.5, cols), RNG.uniform(0.5, 1.5, rows)
    Mp = np.zeros((rows, ld))
    Mp[:, :cols] = M
    with Ctx() as c:
        tM, tv, tw = dev(Mp), dev(v), dev(w)
        c.keep += [tM, tv, tw]
        r = W.right_multiply(c.ctx, rows, cols, tM.data_ptr(), tv.data_ptr(), ld)
        sg.sg_flush(c.ctx)
        st_r = sg.sg_plan_stats(c.ctx)
        l = W.left_multiply(c.ctx, rows, cols, tw.data_ptr(), tM.data_ptr(), ld)
        sg.sg_flush(c.ctx)
        st_l = sg.sg_plan_stats(c.ctx)
        got_r, got_l = c.read_vec(r["out"], np.float64, rows), c.read_vec(l["out"], np.float64, cols)
    assert (st_r.n_passes, st_r.n_template, st_l.n_passes, st_l.n_template) == (1, 1, 1, 1)      # one matrix pass each
    want_r, want_l = ocfg.right_multiply(M, v), ocfg.left_multiply(w, M)
    assert np.all(np.abs(got_r - want_r) <= 1e-12 * np.abs(want_r))
    assert np.all(np.abs(got_l - want_l) <= 1e-12 * np.abs(want_l))


def test_matvec_odd_shapes_exact_integer_regime():
    """Rows of 3, 5 and 1023 doubles (never 16-byte aligned beyond row 0): exact in the integer regime, so bit-for-bit."""
    for rows, cols in ((4, 3), (7, 5), (130, 1023), (1023, 129)):
        M = RNG.integers(-8, 9, (rows, cols)).astype(np.float64)
        v, w = RNG.integers(-8, 9, cols).astype(np.float64), RNG.integers(-8, 9, rows).astype(np.float64)
        with Ctx() as c:
            tM, tv, tw = dev(M), dev(v), dev(w)
            c.keep += [tM, tv, tw]
            r = W.right_multiply(c.ctx, rows, cols, tM.data_ptr(), tv.data_ptr())
            sg.sg_flush(c.ctx)
            l = W.left_multiply(c.ctx, rows, cols, tw.data_ptr(), tM.data_ptr())
            got_r, got_l = c.read_vec(r["out"], np.float64, rows), c.read_vec(l["out"], np.float64, cols)
        assert bits_equal(got_r, ocfg.right_multiply(M, v)) and bits_equal(got_l, ocfg.left_multiply(w, M))


def test_matvec_exact_integer_regime_and_dimension_contract():
    M = RNG.integers(-8, 9, (300, 500)).astype(np.float64)
    v, w = RNG.integers(-8, 9, 500).astype(np.float64), RNG.integers(-8, 9, 300).astype(np.float64)
    with Ctx() as c:
        tM, tv, tw = dev(M), dev(v), dev(w)
        c.keep += [tM, tv, tw]
        r = W.right_multiply(c.ctx, 300, 500, tM.data_ptr(), tv.data_ptr())
        sg.sg_flush(c.ctx)
        l = W.left_multiply(c.ctx, 300, 500, tw.data_ptr(), tM.data_ptr())
        got_r, got_l = c.read_vec(r["out"], np.float64, 300), c.read_vec(l["out"], np.float64, 500)
        with pytest.raises(sg.SgError) as e:                       # columns /= v.count
            sg.sg_enqueue(c.ctx, sg.SG_MUL, [r["M"], sg.H(l["v"], sg.SG_BCAST_ROW)])      # a 300-vector along 500 columns
        assert e.value.status == sg.SG_ERR_SHAPE
    assert bits_equal(got_r, ocfg.right_multiply(M, v)) and bits_equal(got_l, ocfg.left_multiply(w, M))


# ----------------------------------------------------------------------------------------------------------
# transpose — a data mover, bit-exact
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.float64, np.float32, np.int32, np.int64])
@pytest.mark.parametrize("rows,cols,ld,ld_out", [(1, 1, 1, 0), (1, 7, 7, 0), (7, 1, 3, 9), (64, 64, 64, 0), (65, 63, 70, 66), (130, 1000, 1000, 0),
                                                 (1000, 130, 136, 1001), (257, 513, 513, 0),
                                                 # 4-byte elements with 8-byte aligned rows take the pair kernel (128 x 64 tiles): full tiles, ragged edges, padding
                                                 (128, 64, 64, 0), (256, 192, 192, 0), (300, 200, 202, 302), (1000, 130, 136, 1002)])
def test_transpose(dtype, rows, cols, ld, ld_out):
    M = RNG.integers(-10**6, 10**6, (rows, cols)).astype(dtype)
    Mp = np.full((rows, ld), -7, dtype=dtype)
    Mp[:, :cols] = M
    ldo = ld_out or rows
    with Ctx() as c:
        tM = dev(Mp)
        tout = dev(np.full((cols, ldo), -9, dtype=dtype))
        c.keep += [tM, tout]
        r = W.transpose(c.ctx, gpu_util_dtype(dtype), rows, cols, tM.data_ptr(), tout.data_ptr(), ld, ld_out)
        c.torch.cuda.synchronize()
        got = tout.cpu().numpy()
        # library-allocated output, then transposed back: the involution
        r2 = W.transpose(c.ctx, gpu_util_dtype(dtype), rows, cols, tM.data_ptr(), None, ld)
        back = sg.sg_mat_transpose(c.ctx, r2["out"])
        flat = np.empty(rows * cols, dtype=dtype)
        sg.sg_vec_read(c.ctx, back, flat.ctypes.data, flat.nbytes)
    want = ocfg.transpose(M)
    assert bits_equal(np.ascontiguousarray(got[:, :rows]), want)
    assert np.all(got[:, rows:] == -9)                                  # padding of the destination is not touched
    assert bits_equal(flat.reshape(rows, cols), M)


def gpu_util_dtype(dtype):
    from gpu_util import NP2SG
    return NP2SG[np.dtype(dtype)]


def test_transpose_runs_after_pending_writers_and_rejects_overlap():
    n = 130
    M = RNG.standard_normal((n, n))
    with Ctx() as c:
        tM = dev(M); c.keep.append(tM)
        hM = sg.sg_mat_create(c.ctx, sg.SG_F64, n, n, n, tM.data_ptr())
        v = sg.sg_vec_create(c.ctx, sg.SG_F64, n * n, tM.data_ptr())
        sg.sg_enqueue(c.ctx, sg.SG_MUL, [v, sg.F(2.0)], dst_or_0=v)    # pending in-place writer of the same memory
        hT = sg.sg_mat_transpose(c.ctx, hM)                            # flushes it first (trigger (2))
        flat = np.empty(n * n)
        sg.sg_vec_read(c.ctx, hT, flat.ctypes.data, flat.nbytes)
        with pytest.raises(sg.SgError) as e:
            sg.sg_mat_transpose(c.ctx, hM, tM.data_ptr() + 64, 0)
        assert e.value.status == sg.SG_ERR_ALIAS
    assert bits_equal(flat.reshape(n, n), ocfg.transpose(orc.scalar("mul", M.reshape(-1), 2.0).reshape(n, n)))


# ----------------------------------------------------------------------------------------------------------
# the dtype-changing project (R23) — bit-exact
# ----------------------------------------------------------------------------------------------------------
def _cast_inputs(n, src):
    if np.dtype(src).kind == "f":
        a = (RNG.standard_normal(n) * 10.0 ** RNG.integers(-3, 12, n)).astype(src)
        special = np.array([0.0, -0.0, 0.5, -0.5, 1.5, -1.5, 2147483647.0, 2147483648.0, -2147483648.0, -2147483904.0, 9.3e18, -9.3e18, np.inf, -np.inf,
                            np.nan, 16777217.0, 1.0 + 2.0 ** -24, 1e39, -1e39, 1e-46], dtype=src)
    else:
        info = np.iinfo(src)
        a = RNG.integers(info.min, info.max, n, dtype=src, endpoint=True)
        special = np.array([0, 1, -1, info.max, info.min, 2 ** 24 + 1, 2 ** 24 + 3, -(2 ** 24 + 1), 123456789], dtype=src)
        if src is np.int64:
            special = np.concatenate([special, np.array([2 ** 53 + 1, 2 ** 53 + 3, 2 ** 31, 2 ** 32 + 5, -(2 ** 31) - 1, 2 ** 40 + 2 ** 16 + 1], dtype=np.int64)])
    k = min(n, special.size)
    if k:
        a[RNG.choice(n, k, replace=False)] = special[:k]
    return a


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("src,dst", [(s, d) for s in (np.float32, np.float64, np.int32, np.int64) for d in (np.float32, np.float64, np.int32, np.int64)])
def test_cast_every_pair_of_types(mode, src, dst):
    from gpu_util import NP2SG
    for n in (0, 1, 3, 33, 1025, (1 << 16) + 1, 300001):
        a = _cast_inputs(n, src)
        with Ctx(MODES[mode]) as c:
            h = c.vec(a)
            r = sg.sg_cast(c.ctx, h, NP2SG[np.dtype(dst)])
            sg.sg_flush(c.ctx)
            got = c.read_vec(r, dst, n)
        assert bits_equal(got, orc.cast(a, dst)), (src, dst, n)


def test_cast_of_misaligned_views_and_into_caller_storage():
    """subset views start at odd elements: the converting load's vector path needs its own alignment (V source elements)."""
    from gpu_util import NP2SG
    n = 70001
    for src, dst in ((np.int32, np.float64), (np.int64, np.float32), (np.float64, np.int32), (np.float32, np.int64), (np.int32, np.float32)):
        a = _cast_inputs(n, src)
        for start in (0, 1, 2, 3, 5):
            with Ctx() as c:
                h = c.vec(a)
                v = sg.sg_vec_subset(c.ctx, h, start, n - 2)
                out = empty_dev(n, dst); c.keep.append(out)
                hd = sg.sg_vec_create(c.ctx, NP2SG[np.dtype(dst)], n - 2 - start, out.data_ptr() + 3 * np.dtype(dst).itemsize)   # misaligned destination too
                sg.sg_cast(c.ctx, v, NP2SG[np.dtype(dst)], hd)
                sg.sg_flush(c.ctx)
                got = c.read_vec(hd, dst, n - 2 - start)
            assert bits_equal(got, orc.cast(a[start:n - 2], dst)), (src, dst, start)


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("src", [np.int32, np.int64])
def test_project_sqrt_of_an_integer_collection_gives_doubles(mode, src):
    """c.project (agent (a: INT): DOUBLE do Result := sqrt (a) end) — ONE pass: convert at load, sqrt, store 8 B."""
    for n in (1, 33, 4097, (1 << 18) + 5):
        a = RNG.integers(0, np.iinfo(src).max, n, dtype=src, endpoint=True)
        a[: min(n, 6)] = np.array([0, 1, 4, 2, 2 ** 31 - 1, 46340 ** 2], dtype=src)[: min(n, 6)]
        if n > 10:
            a[7] = -4                                                       # sqrt of a negative number: NaN
        with Ctx(MODES[mode]) as c:
            ta, tout = dev(a), empty_dev(n, np.float64)
            c.keep += [ta, tout]
            r = W.project_sqrt(c.ctx, sg.SG_I32 if src is np.int32 else sg.SG_I64, n, ta.data_ptr(), tout.data_ptr())
            sg.sg_flush(c.ctx)
            st = sg.sg_plan_stats(c.ctx)
            got = c.read_vec(r["out"], np.float64, n)
        assert st.n_passes == (2 if mode == "unfused" else 1)
        if mode == "template":
            assert st.n_template == 1 and st.bytes_min == n * (np.dtype(src).itemsize + 8)
        assert bits_equal(got, orc.project_sqrt(a))


def test_cast_feeds_a_fused_chain_and_a_pending_operand_is_stored_first():
    """avg of an INT collection the long way: (x + 1) is an int32 pass, its stored result is converted as the f64 pass loads it."""
    n = (1 << 17) + 9
    x = RNG.integers(-1000, 1000, n, dtype=np.int32)
    with Ctx() as c:
        hx = c.vec(x)
        y = sg.sg_enqueue(c.ctx, sg.SG_ADD, [hx, sg.I(1)])
        f = sg.sg_cast(c.ctx, y, sg.SG_F64)
        sg.sg_release(c.ctx, y)
        h = sg.sg_enqueue(c.ctx, sg.SG_MUL, [f, sg.F(0.5)])
        sg.sg_release(c.ctx, f)
        s, mx = sg.sg_reduce(c.ctx, h, sg.SG_SUM), sg.sg_reduce(c.ctx, h, sg.SG_RMAX)
        got_s, got_mx = c.get(s), c.get(mx)
        assert sg.sg_plan_stats(c.ctx).n_passes == 2
        got = c.read_vec(h, np.float64, n)
    want = orc.scalar("mul", orc.cast(orc.scalar("add", x, 1), np.float64), 0.5)
    assert bits_equal(got, want) and got_mx == orc.max(want)
    assert abs(got_s - orc.sum(want)) <= 1e-12 * np.abs(want).sum()
