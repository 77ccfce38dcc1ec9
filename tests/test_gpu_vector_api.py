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


def test_sqrt_fused_in_a_chain_and_rejected_on_ints():
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
        hi = c.vec(np.arange(8, dtype=np.int32))
        with pytest.raises(sg.SgError):
            sg.sg_enqueue(c.ctx, sg.SG_SQRT, [hi])
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


# ----------------------------------------------------------------------------------------------------------
# matrix-vector products — fp64 sums within 1e-12 relative of the oracle
# ----------------------------------------------------------------------------------------------------------
# matrix passes need 16-byte aligned rows (even fp64 column count and leading dimension): the same contract as config 4's pass
@pytest.mark.parametrize("rows,cols,ld", [(1, 2, 2), (2, 2, 2), (3, 4, 6), (33, 18, 20), (258, 1030, 1030), (1030, 258, 264), (777, 2050, 2052)])
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


def test_matvec_misaligned_rows_fail_loudly():
    with Ctx() as c:
        tM, tv = dev(np.ones((4, 3))), dev(np.ones(3))
        c.keep += [tM, tv]
        W.right_multiply(c.ctx, 4, 3, tM.data_ptr(), tv.data_ptr())
        with pytest.raises(sg.SgError) as e:
            sg.sg_flush(c.ctx)
        assert e.value.status == sg.SG_ERR_UNSUPPORTED                # an error, never a fallback


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
                                                 (1000, 130, 136, 1001), (257, 513, 513, 0)])
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
