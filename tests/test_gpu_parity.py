"""GPU-vs-oracle parity (run on the B200 box: pytest -m gpu).  Every comparison goes through the C ABI
(paper_1410_6685_b200.sg) on cuda:0 and the CPU oracle (oracle/) on the same seeded inputs.

Bars (BASELINE.json north_star): integer / index / comparison / max / min / filter / quantifier results and
elementwise float results bit-exact; fp64 sums within 1e-12 relative, fp32 sums within 1e-5 relative of the
oracle's long-double sum (relative to sum|x| when the oracle's sum is exactly zero)."""
import numpy as np
import pytest

import oracle as orc
from oracle import configs as ocfg
from paper_1410_6685_b200 import inputs, sg
from paper_1410_6685_b200 import workloads as W
from gpu_util import Ctx, dev, rel_err

pytestmark = pytest.mark.gpu

SIZES = [0, 1, 2, 3, 31, 32, 33, 1023, 1024, 1025, 4097, (1 << 16) + 1]
MODES = {"template": 0, "bytecode": sg.SG_FLAG_FORCE_BYTECODE, "unfused": sg.SG_FLAG_UNFUSED}
RNG = np.random.default_rng(777)


def bits_equal(a, b):
    """Bit-for-bit equality; NaN results match any NaN (payload/sign of a generated NaN is hardware-canonical, R15)."""
    a, b = np.ascontiguousarray(a), np.ascontiguousarray(b)
    if a.shape != b.shape or a.dtype != b.dtype:
        return False
    if a.dtype.kind == "f":
        na, nb = np.isnan(a), np.isnan(b)
        if not np.array_equal(na, nb):
            return False
        a, b = np.where(na, 0, a), np.where(nb, 0, b)
    return a.tobytes() == b.tobytes()


def sum_ok(got, want, data, tol):
    return rel_err(got, want, float(np.abs(np.asarray(data, dtype=np.float64)).sum())) <= tol


# ----------------------------------------------------------------------------------------------------------
# the paper's small programs
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-12), (np.float32, 1e-5)])
@pytest.mark.parametrize("n", SIZES)
def test_dot_product_listing4(mode, dtype, tol, n):
    a = RNG.standard_normal(n).astype(dtype)
    b = RNG.standard_normal(n).astype(dtype)
    with Ctx(MODES[mode]) as c:
        ha, hb = c.vec(a), c.vec(b)
        prod = sg.sg_enqueue(c.ctx, sg.SG_MUL, [ha, hb])
        s = sg.sg_reduce(c.ctx, prod, sg.SG_SUM)
        sg.sg_release(c.ctx, prod)
        got = c.get(s)
        st = sg.sg_plan_stats(c.ctx)
    want = ocfg.dot_product(a, b)
    assert sum_ok(got, want, orc.zip("mul", a, b), tol), (got, want)
    assert st.n_passes == (2 if mode == "unfused" else 1)           # two kernels become one


@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n", SIZES)
def test_axpy(mode, dtype, n):
    x = RNG.standard_normal(n).astype(dtype)
    y = RNG.standard_normal(n).astype(dtype)
    with Ctx(MODES[mode]) as c:
        hx, hy = c.vec(x), c.vec(y)
        ax = sg.sg_enqueue(c.ctx, sg.SG_MUL, [hx, sg.F(1.7)])
        r = sg.sg_enqueue(c.ctx, sg.SG_ADD, [ax, hy])
        sg.sg_release(c.ctx, ax)
        got = c.read_vec(r, dtype)
    assert bits_equal(got, ocfg.axpy(1.7, x, y))


@pytest.mark.parametrize("mode", ["template", "bytecode"])
def test_ge_row_op_in_place(mode):
    n = 5000
    ri, rs = RNG.standard_normal(n), RNG.standard_normal(n)
    with Ctx(MODES[mode]) as c:
        hi, hs = c.vec(ri), c.vec(rs)
        sg.sg_enqueue(c.ctx, sg.SG_DIV, [hi, sg.F(3.0)], dst_or_0=hi)
        sg.sg_enqueue(c.ctx, sg.SG_SUB, [hi, hs], dst_or_0=hi)
        got = c.read_vec(hi, np.float64)
        st = sg.sg_plan_stats(c.ctx)
    assert st.n_passes == 1                                          # (A[i]/pivot) - A[step] in one kernel
    assert bits_equal(got, orc.zip("sub", orc.scalar("div", ri, 3.0), rs))


def test_fma_canaries_on_device():
    x = np.full(1000, 1.0 + 2.0 ** -12, dtype=np.float32)
    cc = np.full(1000, -(1.0 + 2.0 ** -11), dtype=np.float32)
    xd = np.full(1000, 1.0 + 2.0 ** -27, dtype=np.float64)
    cd = np.full(1000, -(1.0 + 2.0 ** -26), dtype=np.float64)
    for mode in MODES.values():
        for a, b in ((x, cc), (xd, cd)):
            with Ctx(mode) as c:
                ha, hb = c.vec(a), c.vec(b)
                sq = sg.sg_enqueue(c.ctx, sg.SG_MUL, [ha, ha])
                r = sg.sg_enqueue(c.ctx, sg.SG_ADD, [sq, hb])
                sg.sg_release(c.ctx, sq)
                got = c.read_vec(r, a.dtype)
            assert not got.any()                                     # a contracted fma would give 2^-24 / 2^-54


# ----------------------------------------------------------------------------------------------------------
# every primitive, every dtype, odd sizes, misaligned views (bytecode kernel: no template matches these)
# ----------------------------------------------------------------------------------------------------------
BIN = {"add": sg.SG_ADD, "sub": sg.SG_SUB, "mul": sg.SG_MUL, "div": sg.SG_DIV, "min": sg.SG_MIN, "max": sg.SG_MAX, "mod": sg.SG_MOD}
CMP = {"eq": sg.SG_EQ, "ne": sg.SG_NE, "lt": sg.SG_LT, "le": sg.SG_LE, "gt": sg.SG_GT, "ge": sg.SG_GE}


def rand(dtype, n):
    if np.dtype(dtype).kind == "f":
        a = (RNG.standard_normal(n) * 10).astype(dtype)
        if n > 4:
            a[:4] = [0.0, -0.0, 1.0, -1.0]
        return a
    info = np.iinfo(dtype)
    a = RNG.integers(-50, 50, n).astype(dtype)
    if n > 6:
        a[:6] = [0, 1, -1, info.min, info.max, 7]
    return a


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
@pytest.mark.parametrize("n", [0, 1, 33, 1025, 4099])
def test_all_primitives(dtype, n):
    a, b = rand(dtype, n), rand(dtype, n)
    ops = ["add", "sub", "mul", "div", "min", "max"] + (["mod"] if np.dtype(dtype).kind == "i" else [])
    imm = sg.F(2.5) if np.dtype(dtype).kind == "f" else sg.I(7)
    immv = 2.5 if np.dtype(dtype).kind == "f" else 7
    with Ctx() as c:
        ha, hb = c.vec(a), c.vec(b)
        res = {}
        for op in ops:
            res[op] = sg.sg_enqueue(c.ctx, BIN[op], [ha, hb])
            res[op + "_s"] = sg.sg_enqueue(c.ctx, BIN[op], [ha, imm])
            res[op + "_r"] = sg.sg_enqueue(c.ctx, BIN[op], [imm, ha])
        res["neg"] = sg.sg_enqueue(c.ctx, sg.SG_NEG, [ha])
        res["abs"] = sg.sg_enqueue(c.ctx, sg.SG_ABS, [ha])
        sg.sg_flush(c.ctx)                                           # several passes: the output limit splits them
        for op in ops:
            assert bits_equal(c.read_vec(res[op], dtype), orc.zip(op, a, b)), op
            assert bits_equal(c.read_vec(res[op + "_s"], dtype), orc.scalar(op, a, immv)), op
            assert bits_equal(c.read_vec(res[op + "_r"], dtype), orc.scalar(op, a, immv, reversed=True)), op
        assert bits_equal(c.read_vec(res["neg"], dtype), orc.unary("neg", a))
        assert bits_equal(c.read_vec(res["abs"], dtype), orc.unary("abs", a))
    with Ctx() as c:
        ha, hb = c.vec(a), c.vec(b)
        res = {op: sg.sg_enqueue(c.ctx, CMP[op], [ha, hb]) for op in CMP}
        lg = sg.sg_enqueue(c.ctx, sg.SG_AND, [res["le"], res["ne"]])
        lo = sg.sg_enqueue(c.ctx, sg.SG_OR, [res["lt"], res["eq"]])
        ln = sg.sg_enqueue(c.ctx, sg.SG_NOT, [res["gt"]])
        cnt = sg.sg_reduce(c.ctx, res["lt"], sg.SG_COUNT)
        sg.sg_flush(c.ctx)
        for op in CMP:
            assert bits_equal(c.read_vec(res[op], np.uint8), orc.cmp(op, a, b)), op
        assert bits_equal(c.read_vec(lg, np.uint8), orc.logic("and", orc.cmp("le", a, b), orc.cmp("ne", a, b)))
        assert bits_equal(c.read_vec(lo, np.uint8), orc.logic("or", orc.cmp("lt", a, b), orc.cmp("eq", a, b)))
        assert bits_equal(c.read_vec(ln, np.uint8), orc.logic("not", orc.cmp("gt", a, b)))
        assert c.get(cnt) == orc.count(orc.cmp("lt", a, b))


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
@pytest.mark.parametrize("n", [3, 1025, 70001])
def test_input_first_named_after_two_temporaries_died(dtype, n):
    """`((a+b)*(c+d) + e) * 3`: the multiplication gives two registers back and e is first named afterwards.  Every input of a tile is
    loaded before the first instruction runs, so e must not live in the register c+d is computed in (the plan builder gave inputs
    recycled registers until round 2: e was overwritten, silently in a template instance, out of bounds in the bytecode file)."""
    v = [rand(dtype, n) for _ in range(5)]
    imm = sg.F(3.0) if np.dtype(dtype).kind == "f" else sg.I(3)
    with Ctx() as c:
        h = [c.vec(x) for x in v]
        t1 = sg.sg_enqueue(c.ctx, sg.SG_ADD, [h[0], h[1]])
        t2 = sg.sg_enqueue(c.ctx, sg.SG_ADD, [h[2], h[3]])
        t3 = sg.sg_enqueue(c.ctx, sg.SG_MUL, [t1, t2])
        t4 = sg.sg_enqueue(c.ctx, sg.SG_ADD, [t3, h[4]])
        t5 = sg.sg_enqueue(c.ctx, sg.SG_MUL, [t4, imm])
        for t in (t1, t2, t3, t4):
            sg.sg_release(c.ctx, t)
        m = sg.sg_reduce(c.ctx, t5, sg.SG_RMAX)
        got, got_m = c.read_vec(t5, dtype), c.get(m)
        assert sg.sg_plan_stats(c.ctx).n_passes == 1
    want = orc.scalar("mul", orc.zip("add", orc.zip("mul", orc.zip("add", v[0], v[1]), orc.zip("add", v[2], v[3])), v[4]), 3.0 if np.dtype(dtype).kind == "f" else 3)
    assert bits_equal(got, want)
    assert bits_equal(np.array([got_m], dtype=dtype), np.array([orc.max(want)], dtype=dtype))


@pytest.mark.parametrize("mode", ["template", "unfused"])
@pytest.mark.parametrize("n", [1, 1025, 70001])
def test_superseded_inplace_result_read_by_a_later_pass(mode, n):
    """x := a + b (in place), t = x + max(b) (a scalar edge: t lives in a later pass and reads the FIRST version of x), x := max(a, b)
    (in place again: supersedes the first version, which never reaches the buffer), u = t * x.  The first version is spilled to
    storage of its own — round 2 spilled it into x's buffer, where the second version overwrote it before the later pass read it."""
    a, b, x0 = rand(np.float64, n), rand(np.float64, n), rand(np.float64, n)
    with Ctx(MODES[mode]) as c:
        ha, hb, hx = c.vec(a), c.vec(b), c.vec(x0)
        sg.sg_enqueue(c.ctx, sg.SG_ADD, [ha, hb], dst_or_0=hx)
        s = sg.sg_reduce(c.ctx, hb, sg.SG_RMAX)
        t = sg.sg_enqueue(c.ctx, sg.SG_ADD, [hx, s])
        sg.sg_enqueue(c.ctx, sg.SG_MAX, [ha, hb], dst_or_0=hx)
        u = sg.sg_enqueue(c.ctx, sg.SG_MUL, [t, hx])
        sg.sg_release(c.ctx, t)
        got_u, got_x = c.read_vec(u, np.float64), c.read_vec(hx, np.float64)
    v1, v2 = orc.zip("add", a, b), orc.zip("max", a, b)
    want_u = orc.zip("mul", orc.scalar("add", v1, float(orc.max(b))), v2)
    assert bits_equal(got_x, v2) and bits_equal(got_u, want_u)


@pytest.mark.parametrize("mode", ["template", "unfused"])
@pytest.mark.parametrize("pattern", ["read_through_a_handle_after_an_alias_wrote", "alias_read_between_two_inplace_results", "alias_read_by_the_superseding_operation"])
def test_aliasing_handles_follow_program_order(mode, pattern):
    """Two handles of the SAME storage (subset views) with in-place updates through both: the pending list must behave
    like eager execution in program order.  (The randomised view programs of tests/test_gpu_random_chains.py found all three.)"""
    n, s, L = 5000, 1000, 3000
    x = RNG.standard_normal(n)
    mem = x.copy()
    with Ctx(MODES[mode]) as c:
        hx = c.vec(x)
        v0, v1 = sg.sg_vec_subset(c.ctx, hx, s, s + L), sg.sg_vec_subset(c.ctx, hx, s, s + L)
        cur = lambda: mem[s:s + L].copy()
        if pattern == "read_through_a_handle_after_an_alias_wrote":
            sg.sg_enqueue(c.ctx, sg.SG_ADD, [v0, v1], dst_or_0=v0)                  # v0 := v0 + v1
            mem[s:s + L] = orc.zip("add", cur(), cur())
            sg.sg_enqueue(c.ctx, sg.SG_MUL, [sg.F(0.25), v1], dst_or_0=v1)          # v1 := 0.25 * v1   (the same memory)
            mem[s:s + L] = orc.scalar("mul", cur(), 0.25, reversed=True)
            t = sg.sg_enqueue(c.ctx, sg.SG_SUB, [sg.F(-1.0), v0])                   # reads v0: what the memory holds NOW
            want_t = orc.scalar("sub", cur(), -1.0, reversed=True)
        elif pattern == "alias_read_between_two_inplace_results":
            sg.sg_enqueue(c.ctx, sg.SG_MUL, [v0, sg.F(3.0)], dst_or_0=v0)           # v0 := 3 v0
            mem[s:s + L] = orc.scalar("mul", cur(), 3.0)
            t = sg.sg_enqueue(c.ctx, sg.SG_ADD, [v1, v1])                           # reads the alias: must see 3 v0 in memory
            want_t = orc.zip("add", cur(), cur())
            sg.sg_enqueue(c.ctx, sg.SG_SUB, [t, sg.F(1.0)], dst_or_0=v0)            # v0 := t - 1: supersedes the first result
            mem[s:s + L] = orc.scalar("sub", want_t, 1.0)
        else:
            sg.sg_enqueue(c.ctx, sg.SG_MUL, [v1, v0], dst_or_0=v0)                  # v0 := v1 * v0
            mem[s:s + L] = orc.zip("mul", cur(), cur())
            sg.sg_enqueue(c.ctx, sg.SG_MIN, [v1, v0], dst_or_0=v0)                  # v0 := min(v1, v0): v1 is the squared memory
            mem[s:s + L] = orc.zip("min", cur(), cur())
            t = sg.sg_enqueue(c.ctx, sg.SG_NEG, [v1])
            want_t = orc.unary("neg", cur())
        got_t, got_x = c.read_vec(t, np.float64), c.read_vec(hx, np.float64)
    assert bits_equal(got_x, mem) and bits_equal(got_t, want_t)


def test_fourteen_vectors_in_one_expression():
    """More distinct inputs than one pass holds (10): the chain is split into passes, the result is the oracle's."""
    n = 70001
    v = [rand(np.float64, n) for _ in range(14)]
    with Ctx() as c:
        h = [c.vec(x) for x in v]
        acc = h[0]
        for x in h[1:]:
            nxt = sg.sg_enqueue(c.ctx, sg.SG_ADD, [acc, x])
            if acc != h[0]:
                sg.sg_release(c.ctx, acc)
            acc = nxt
        got = c.read_vec(acc, np.float64)
        assert sg.sg_plan_stats(c.ctx).n_passes >= 2
    want = v[0]
    for x in v[1:]:
        want = orc.zip("add", want, x)
    assert bits_equal(got, want)


@pytest.mark.parametrize("mode", ["template", "unfused"])
def test_inplace_result_read_by_a_later_pass_orders_overlapping_writers(mode):
    """a := 2a (in place, pass 0); u = a + max(c) (a scalar edge puts it in pass 1, where a's new contents are read from the caller's
    buffer); b := b + 1 with b an OVERLAPPING view of the same buffer.  The write to b must not share pass 1 with the read of a
    (another thread's element): the read of a pending in-place result by a later pass is a memory read like any other (WAR edge;
    found by the soak run of the randomised view programs, seed 1040)."""
    n, L, s = 200000, 120000, 50000
    x, y = RNG.standard_normal(n), RNG.standard_normal(L)
    mem = x.copy()
    with Ctx(MODES[mode]) as c:
        hx, hc = c.vec(x), c.vec(y)
        a, b = sg.sg_vec_subset(c.ctx, hx, 0, L), sg.sg_vec_subset(c.ctx, hx, s, s + L)
        sg.sg_enqueue(c.ctx, sg.SG_MUL, [a, sg.F(2.0)], dst_or_0=a)
        mem[0:L] = orc.scalar("mul", mem[0:L].copy(), 2.0)
        m = sg.sg_reduce(c.ctx, hc, sg.SG_RMAX)
        u = sg.sg_enqueue(c.ctx, sg.SG_ADD, [a, m])
        want_u = orc.scalar("add", mem[0:L].copy(), float(orc.max(y)))
        sg.sg_enqueue(c.ctx, sg.SG_ADD, [b, sg.F(1.0)], dst_or_0=b)
        mem[s:s + L] = orc.scalar("add", mem[s:s + L].copy(), 1.0)
        sg.sg_flush(c.ctx)
        if mode == "template":
            assert sg.sg_plan_stats(c.ctx).n_passes == 3
        got_u, got_x = c.read_vec(u, np.float64), c.read_vec(hx, np.float64)
    assert bits_equal(got_u, want_u) and bits_equal(got_x, mem)


@pytest.mark.parametrize("dtype,tol", [(np.float32, 1e-5), (np.float64, 1e-12), (np.int32, 0), (np.int64, 0)])
@pytest.mark.parametrize("n", [1, 2, 33, 1024, 1025, 70001])
def test_reductions_all_dtypes(dtype, tol, n):
    a = rand(dtype, n)
    with Ctx() as c:
        ha = c.vec(a)
        s, mx, mn = (sg.sg_reduce(c.ctx, ha, k) for k in (sg.SG_SUM, sg.SG_RMAX, sg.SG_RMIN))
        gs, gmx, gmn = c.get(s), c.get(mx), c.get(mn)
        assert sg.sg_plan_stats(c.ctx).n_passes == 1
    if np.dtype(dtype).kind == "f":
        assert sum_ok(gs, orc.sum(a), a, tol)
    else:
        assert gs == orc.sum(a)
    assert bits_equal(np.array([gmx], dtype=dtype), np.array([orc.max(a)], dtype=dtype))
    assert bits_equal(np.array([gmn], dtype=dtype), np.array([orc.min(a)], dtype=dtype))


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_extremum_total_order_on_device(dtype):
    for arr in ([0.0, -0.0], [-0.0, 0.0], [1.0, np.inf, -np.inf, np.nan, -2.0], [1.0, np.copysign(np.nan, -1.0), 3.0]):
        a = np.array(arr * 300, dtype=dtype)
        with Ctx() as c:
            ha = c.vec(a)
            mx, mn = sg.sg_reduce(c.ctx, ha, sg.SG_RMAX), sg.sg_reduce(c.ctx, ha, sg.SG_RMIN)
            gmx, gmn = c.get(mx), c.get(mn)
        assert bits_equal(np.array([gmx], dtype=dtype), np.array([orc.max(a)], dtype=dtype)), arr
        assert bits_equal(np.array([gmn], dtype=dtype), np.array([orc.min(a)], dtype=dtype)), arr


def test_empty_collections():
    with Ctx() as c:
        e = c.vec(np.empty(0, dtype=np.float64))
        s = sg.sg_reduce(c.ctx, e, sg.SG_SUM)
        m = sg.sg_enqueue(c.ctx, sg.SG_GT, [e, sg.F(0.0)])
        fa, ex, cn = sg.sg_forall(c.ctx, m), sg.sg_exists(c.ctx, m), sg.sg_reduce(c.ctx, m, sg.SG_COUNT)
        assert c.get(s) == 0.0 and c.get(fa) is True and c.get(ex) is False and c.get(cn) == 0
        with pytest.raises(sg.SgError) as ei:
            sg.sg_reduce(c.ctx, e, sg.SG_RMAX)
        assert ei.value.status == sg.SG_ERR_EMPTY


def test_misaligned_views():
    n = 10007
    a, b = rand(np.float32, n), rand(np.float32, n)
    with Ctx() as c:
        ha, hb = c.vec(a), c.vec(b)
        for (sa, sb, m) in [(1, 1, 5000), (3, 3, 4097), (1, 2, 3000), (0, 3, 1025), (5, 0, 7)]:
            va, vb = sg.sg_vec_subset(c.ctx, ha, sa, sa + m), sg.sg_vec_subset(c.ctx, hb, sb, sb + m)
            r = sg.sg_enqueue(c.ctx, sg.SG_ADD, [va, vb])
            s = sg.sg_reduce(c.ctx, r, sg.SG_SUM)
            want = orc.zip("add", a[sa:sa + m], b[sb:sb + m])
            assert bits_equal(c.read_vec(r, np.float32), want), (sa, sb, m)
            assert sum_ok(c.get(s), orc.sum(want), want, 1e-5)
        # neighbour predicate written with subsets: two views of one buffer, one element apart
        x = np.sort(rand(np.float32, n))
        hx = c.vec(x)
        le = sg.sg_enqueue(c.ctx, sg.SG_LE, [sg.sg_vec_subset(c.ctx, hx, 0, n - 1), sg.sg_vec_subset(c.ctx, hx, 1, n)])
        assert c.get(sg.sg_forall(c.ctx, le)) is True


def test_enqueue_contracts_are_checked_on_the_host():
    with Ctx() as c:
        a, b = c.vec(np.zeros(10, dtype=np.float32)), c.vec(np.zeros(11, dtype=np.float32))
        d = c.vec(np.zeros(10, dtype=np.float64))
        with pytest.raises(sg.SgError) as ei:
            sg.sg_enqueue(c.ctx, sg.SG_ADD, [a, b])
        assert ei.value.status == sg.SG_ERR_SHAPE                    # dimension contract
        with pytest.raises(sg.SgError) as ei:
            sg.sg_enqueue(c.ctx, sg.SG_ADD, [a, d])
        assert ei.value.status == sg.SG_ERR_DTYPE
        with pytest.raises(sg.SgError) as ei:
            sg.sg_enqueue(c.ctx, sg.SG_MOD, [a, sg.I(3)])
        assert ei.value.status == sg.SG_ERR_DTYPE
        assert sg.sg_vec_count(c.ctx, a) == 10                       # count: O(1) scalar contract


# ----------------------------------------------------------------------------------------------------------
# config 0
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("n", [1 << 20, (1 << 16) + 3, 1000])
def test_cfg0(mode, n):
    a, b, cc = (inputs.uniform_pm1_f64(1, s, n) for s in range(3))
    want = ocfg.cfg0(a, b, cc)
    for keep_z in (True, False):
        with Ctx(MODES[mode]) as c:
            ta, tb, tc = (c.torch.from_numpy(x).cuda() for x in (a, b, cc))
            r = W.cfg0(c.ctx, n, ta.data_ptr(), tb.data_ptr(), tc.data_ptr(), keep_z=keep_z)
            gs, gmx, gmn, pre, post = (c.get(r[k]) for k in ("sum", "max", "min", "pre", "post"))
            st = sg.sg_plan_stats(c.ctx)
            if keep_z:
                assert bits_equal(c.read_vec(r["z"], np.float64), want["z"])
        assert sum_ok(gs, want["sum"], want["z"], 1e-12), (gs, want["sum"])
        assert gmx == want["max"] and gmn == want["min"]
        assert pre == want["pre"] and post == want["post"] and post is True
        if mode != "unfused":
            assert st.n_passes == (2 if keep_z else 1) and st.n_bytecode == (st.n_passes if mode == "bytecode" else 0)


def test_cfg0_violated_contracts_are_reported():
    n = 5000
    a, b, cc = (inputs.uniform_pm1_f64(1, s, n) for s in range(3))
    a = np.minimum(a, 0.5)                                           # exists(a > 0.99) is now false
    with Ctx() as c:
        ta, tb, tc = (c.torch.from_numpy(x).cuda() for x in (a, b, cc))
        r = W.cfg0(c.ctx, n, ta.data_ptr(), tb.data_ptr(), tc.data_ptr())
        with pytest.raises(sg.SgError) as ei:
            sg.sg_flush(c.ctx)
        assert ei.value.status == sg.SG_ERR_CONTRACT and "exists" in str(ei.value)
        assert c.get(r["pre"]) is False and c.get(r["post"]) is True


# ----------------------------------------------------------------------------------------------------------
# config 1
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("n", [1 << 22, (1 << 20) + 5, 777])
def test_cfg1(mode, n):
    x, y = inputs.normal_f32(2, 0, n), inputs.normal_f32(2, 1, n)
    want = ocfg.cfg1(x, y)
    with Ctx(MODES[mode]) as c:
        tx, ty = c.torch.from_numpy(x).cuda(), c.torch.from_numpy(y).cuda()
        r = W.cfg1(c.ctx, n, tx.data_ptr(), ty.data_ptr(), keep_w=True)
        gs, gmx = c.get(r["sum"]), c.get(r["max"])
        st = sg.sg_plan_stats(c.ctx)
        assert bits_equal(c.read_vec(r["w"], np.float32), want["w"])
    assert sum_ok(gs, want["sum"], want["w"], 1e-5), (gs, want["sum"])
    assert np.float32(gmx) == want["max"]
    assert st.n_passes == (12 if mode == "unfused" else 1)


def test_cfg1_full_size():
    n = 1 << 26
    x, y = inputs.normal_f32(2, 0, n), inputs.normal_f32(2, 1, n)
    want = ocfg.cfg1(x, y)
    with Ctx() as c:
        tx, ty = c.torch.from_numpy(x).cuda(), c.torch.from_numpy(y).cuda()
        r = W.cfg1(c.ctx, n, tx.data_ptr(), ty.data_ptr())
        gs, gmx = c.get(r["sum"]), c.get(r["max"])
        st = sg.sg_plan_stats(c.ctx)
    assert st.n_passes == 1 and st.n_template == 1 and st.bytes_min == 8 * n
    assert sum_ok(gs, want["sum"], want["w"], 1e-5) and np.float32(gmx) == want["max"]


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_float_sums_are_the_same_bits_on_every_run(dtype):
    """A pass with a floating-point sum keeps the static tile order (tile tickets, under which the block that adds a tile differs from
    run to run, are used only where every reduction is exact in any order): 30 runs at a size that would take tickets, one bit
    pattern."""
    n = (1 << 25) + 4099
    x, y = inputs.normal_f32(3, 0, n).astype(dtype), inputs.normal_f32(3, 1, n).astype(dtype)
    seen = set()
    with Ctx() as c:
        hx, hy = c.vec(x), c.vec(y)
        for _ in range(30):
            prod = sg.sg_enqueue(c.ctx, sg.SG_MUL, [hx, hy])
            s = sg.sg_reduce(c.ctx, prod, sg.SG_SUM)
            sg.sg_release(c.ctx, prod)
            seen.add(np.float64(c.get(s)).tobytes())
            sg.sg_release(c.ctx, s)
        assert sg.sg_plan_stats(c.ctx).n_template == 1
    assert len(seen) == 1
    got = np.frombuffer(seen.pop(), dtype=np.float64)[0]
    assert sum_ok(got, ocfg.dot_product(x, y), orc.zip("mul", x, y), 1e-12 if dtype is np.float64 else 1e-5)


@pytest.mark.parametrize("mode", ["template", "bytecode"])
def test_recycled_handle_slots_keep_results_right(mode):
    """300 steps in one context, every intermediate released: the handle table stays a few slots long (the slots of dead values are
    reused under a new generation) and every step's stored vector, sum and maximum still match the oracle."""
    n = 5000
    x = RNG.standard_normal(n).astype(np.float32)
    slots = set()
    with Ctx(MODES[mode]) as c:
        hx = c.vec(x)
        for it in range(300):
            k = np.float32(0.25 * (it % 7) - 0.5)
            t = sg.sg_enqueue(c.ctx, sg.SG_MUL, [hx, sg.F(float(k))])
            u = sg.sg_enqueue(c.ctx, sg.SG_ADD, [t, hx])                   # stored: read back below
            s, m = sg.sg_reduce(c.ctx, u, sg.SG_SUM), sg.sg_reduce(c.ctx, u, sg.SG_RMAX)
            sg.sg_release(c.ctx, t)
            got_s, got_m = c.get(s), c.get(m)
            slots |= {h & 0xffffffff for h in (t, u, s, m)}
            if it % 50 == 0 or it == 299:
                want_u = orc.zip("add", orc.scalar("mul", x, k), x)
                assert bits_equal(c.read_vec(u, np.float32), want_u)
                assert sum_ok(got_s, orc.sum(want_u), want_u, 1e-5) and np.float32(got_m) == orc.max(want_u)
            for h in (u, s, m):
                sg.sg_release(c.ctx, h)
        with pytest.raises(sg.SgError):                                     # a released handle is unknown, whatever its slot holds now
            sg.sg_vec_count(c.ctx, u)
    assert len(slots) <= 12, sorted(slots)


@pytest.mark.parametrize("dtype", [np.int32, np.int64, np.float32])
def test_exact_reductions_through_tile_tickets(dtype):
    """Integer sum / max / min (float: max / min only) of a vector long enough that the last part of the tiles is handed out through
    tickets (sg_pass1d_tmpl.cuh): bit-exact against the oracle, on every one of 10 runs; the tail is ragged."""
    n = (1 << 25) + 4099
    a = rand(dtype, n)
    is_int = np.dtype(dtype).kind == "i"
    want = ((orc.sum(a),) if is_int else ()) + (orc.max(a), orc.min(a))
    with Ctx() as c:
        ha = c.vec(a)
        for _ in range(10):
            hs = [sg.sg_reduce(c.ctx, ha, k) for k in ((sg.SG_SUM,) if is_int else ()) + (sg.SG_RMAX, sg.SG_RMIN)]
            got = tuple(c.get(h) for h in hs)
            assert sg.sg_plan_stats(c.ctx).n_passes == 1
            for h in hs:
                sg.sg_release(c.ctx, h)
            assert bits_equal(np.array(got[-2:], dtype=dtype), np.array(want[-2:], dtype=dtype))
            if is_int:
                assert got[0] == want[0]


def test_cfg1_headline_size():
    """The configuration bench.py's headline line times (BASELINE.json metric: the fused chain at 2^28 elements): sum and max against
    the oracle on ALL 2^28 elements, then every element of w (the same chain with w kept)."""
    n = 1 << 28
    x, y = inputs.normal_f32(2, 0, n), inputs.normal_f32(2, 1, n)
    want = ocfg.cfg1(x, y)
    with Ctx() as c:
        tx, ty = c.torch.from_numpy(x).cuda(), c.torch.from_numpy(y).cuda()
        r = W.cfg1(c.ctx, n, tx.data_ptr(), ty.data_ptr())
        gs, gmx = c.get(r["sum"]), c.get(r["max"])
        st = sg.sg_plan_stats(c.ctx)
        assert st.n_passes == 1 and st.n_template == 1 and st.bytes_min == 8 * n
        assert sum_ok(gs, want["sum"], want["w"], 1e-5) and np.float32(gmx) == want["max"]
        r2 = W.cfg1(c.ctx, n, tx.data_ptr(), ty.data_ptr(), keep_w=True)
        gs2 = c.get(r2["sum"])
        w = c.read_vec(r2["w"], np.float32)
    assert gs2 == gs and bits_equal(w, want["w"])


# ----------------------------------------------------------------------------------------------------------
# config 2
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["template", "bytecode"])
@pytest.mark.parametrize("n", [0, 1, 5, 4095, 4096, 4097, 3 * 4096 + 17, (1 << 20) + 11])
def test_cfg2(mode, n):
    x = inputs.uniform_i31(3, 0, n)
    want = ocfg.cfg2(x)
    with Ctx(MODES[mode]) as c:
        tx = c.torch.from_numpy(x).cuda()
        r = W.cfg2(c.ctx, n, tx.data_ptr())
        cnt, s = c.get(r["count"]), c.get(r["sum"])
        kept = c.read_vec(r["kept"], np.int32)
        assert sg.sg_plan_stats(c.ctx).n_passes == 1
    assert cnt == want["count"] and s == want["sum"]
    assert bits_equal(kept, want["kept"])                            # stable: identical order


@pytest.mark.parametrize("mode", ["template", "bytecode"])
@pytest.mark.parametrize("modulus", [2, 3, 7, 10, 16, 641, 65536, 65537, 2**31 - 1, -2, -7, -641, -2**31, 1, -1])
def test_filter_mod_by_any_immediate_divisor(mode, modulus):
    """The template path divides by a pass-constant with a host-computed signed magic number: every divisor class
    (powers of two, negative, +-1, INT_MIN) and dividends incl. negatives and INT_MIN/INT_MAX, bit-exact vs C semantics."""
    n = 3 * 8192 + 77
    x = (inputs.bits(11, 0, 0, n) >> np.uint64(32)).astype(np.uint32).view(np.int32).copy()     # full int32 range
    x[:8] = [0, 1, -1, np.iinfo(np.int32).min, np.iinfo(np.int32).max, modulus if abs(modulus) < 2**31 else 0, 7, -7]
    residue = int(x[100]) % abs(modulus) if modulus not in (1, -1) else 0
    if x[100] < 0 and residue:
        residue -= abs(modulus)                                      # C remainder has the sign of the dividend
    want = ocfg.cfg2(x, modulus, residue)
    assert want["count"] > 0
    with Ctx(MODES[mode]) as c:
        tx = c.torch.from_numpy(x).cuda()
        r = W.cfg2(c.ctx, n, tx.data_ptr(), modulus=modulus, residue=residue)
        cnt, s = c.get(r["count"]), c.get(r["sum"])
        kept = c.read_vec(r["kept"], np.int32)
    assert cnt == want["count"] and s == want["sum"]
    assert bits_equal(kept, want["kept"])


@pytest.mark.parametrize("modulus", [1, 2, 3])
def test_filter_high_selectivity(modulus):
    """All / half / a third of the values kept over 128 tiles: the compaction ring fills up, tiles wait for their offsets
    (single-tile runs), the ring wraps around; order and count stay exact."""
    n = (1 << 20) + 11
    x = inputs.uniform_i31(3, 7, n)
    want = ocfg.cfg2(x, modulus, 0)
    with Ctx() as c:
        tx = c.torch.from_numpy(x).cuda()
        r = W.cfg2(c.ctx, n, tx.data_ptr(), modulus=modulus, residue=0)
        cnt, s = c.get(r["count"]), c.get(r["sum"])
        kept = c.read_vec(r["kept"], np.int32)
    assert cnt == want["count"] and s == want["sum"]
    assert bits_equal(kept, want["kept"])


def test_filter_repeated_launches_share_tile_states():
    """One context, many filter launches of different lengths and selectivities: the tile-state words of earlier launches
    stay in memory and are told apart by the launch epoch only; replays (sg_replay_last) re-run the same launch."""
    rng = np.random.default_rng(7)
    with Ctx() as c:
        for rep in range(24):
            n = int(rng.integers(1, 40)) * 8192 + int(rng.integers(0, 8192))
            modulus = int(rng.choice([1, 2, 3, 7, 50, 1000]))
            x = inputs.uniform_i31(3, 100 + rep, n)
            want = ocfg.cfg2(x, modulus, 0)
            tx = c.torch.from_numpy(x).cuda()
            r = W.cfg2(c.ctx, n, tx.data_ptr(), modulus=modulus, residue=0)
            cnt, s = c.get(r["count"]), c.get(r["sum"])
            kept = c.read_vec(r["kept"], np.int32)
            assert cnt == want["count"] and s == want["sum"], (rep, n, modulus)
            assert bits_equal(kept, want["kept"]), (rep, n, modulus)
            if rep % 6 == 0:
                sg.sg_replay_last(c.ctx, 3)
                kept2 = np.empty(cnt, dtype=np.int32)
                c.torch.cuda.synchronize()
                sg.sg_vec_read(c.ctx, r["kept"], kept2.ctypes.data, kept2.nbytes)
                assert bits_equal(kept2, want["kept"]) and c.get(r["count"]) == want["count"]
            for h in r.values():
                sg.sg_release(c.ctx, h)


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int64])
def test_filter_other_dtypes_and_edge_masks(dtype):
    n = 3 * 4096 + 5
    a = rand(dtype, n)
    for thr, name in ((-1e9, "all"), (1e9, "none"), (0, "half")):
        with Ctx() as c:
            ha = c.vec(a)
            m = sg.sg_enqueue(c.ctx, sg.SG_GT, [ha, sg.F(thr) if np.dtype(dtype).kind == "f" else sg.I(int(thr))])
            kept, cnt = sg.sg_filter(c.ctx, ha, m)
            got = c.read_vec(kept, dtype)
            want = orc.filter(a, orc.cmp_scalar("gt", a, thr))
            assert c.get(cnt) == want.size and bits_equal(got, want), name


def test_filter_capacity_error():
    a = np.arange(10000, dtype=np.int32)
    with Ctx() as c:
        ha = c.vec(a)
        out = c.torch.empty(10, dtype=c.torch.int32, device="cuda")
        m = sg.sg_enqueue(c.ctx, sg.SG_GE, [ha, sg.I(0)])
        kept, cnt = sg.sg_filter(c.ctx, ha, m, out.data_ptr(), 10)
        assert c.get(cnt) == 10000
        with pytest.raises(sg.SgError) as ei:
            sg.sg_vec_count(c.ctx, kept)
        assert ei.value.status == sg.SG_ERR_CAPACITY
        assert out.cpu().numpy().tolist() == list(range(10))


@pytest.mark.parametrize("dtype", [np.float64, np.int64, np.float32])
def test_kept_sum_with_a_tight_caller_buffer(dtype):
    """Filter into a caller buffer of exactly the kept count, with the sum and the maximum of the kept values in the same pass (a
    chain without a template instance: the bytecode filter kernel).  The reductions run over the SOURCE elements under the mask —
    round 2 bounded them by the output's capacity and cut the sum short (found by the bursty-mask filter test)."""
    n = 70001
    x = rand(dtype, n)
    zero = 0.0 if np.dtype(dtype).kind == "f" else 0
    want = orc.filter(x, orc.cmp_scalar("gt", x, zero))
    with Ctx() as c:
        hx = c.vec(x)
        out = dev(np.zeros(want.size, dtype=dtype))
        c.keep.append(out)
        m = sg.sg_enqueue(c.ctx, sg.SG_GT, [hx, sg.F(0.0) if np.dtype(dtype).kind == "f" else sg.I(0)])
        fv, fc = sg.sg_filter(c.ctx, hx, m, out.data_ptr(), want.size)
        sg.sg_release(c.ctx, m)
        s, mx = sg.sg_reduce(c.ctx, fv, sg.SG_SUM), sg.sg_reduce(c.ctx, fv, sg.SG_RMAX)
        assert c.get(fc) == want.size and bits_equal(c.read_vec(fv, dtype, want.size), want)
        assert sum_ok(c.get(s), orc.sum(want), want, {np.float64: 1e-12, np.float32: 1e-5}.get(dtype, 0)) and dtype(c.get(mx)) == orc.max(want)
        assert sg.sg_plan_stats(c.ctx).n_bytecode == 1


def test_cfg2_full_size():
    n = 1 << 27
    x = inputs.uniform_i31(3, 0, n)
    want = ocfg.cfg2(x)
    with Ctx() as c:
        tx = c.torch.from_numpy(x).cuda()
        r = W.cfg2(c.ctx, n, tx.data_ptr())
        assert c.get(r["count"]) == want["count"] and c.get(r["sum"]) == want["sum"]
        assert bits_equal(c.read_vec(r["kept"], np.int32), want["kept"])


# ----------------------------------------------------------------------------------------------------------
# config 3
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", list(MODES))
@pytest.mark.parametrize("n", [2, 3, 1025, 8192, 8193, (1 << 20) + 1])
def test_cfg3(mode, n):
    x = inputs.sorted_cumsum_f32(4, 0, n)
    for flags in (0, sg.SG_FLAG_NO_EARLY_EXIT):
        cases = [("clean", x)]
        if n > 3:
            for j in sorted({1, n // 2, n - 2, inputs.violation_index(4, n)}):
                y = x.copy()
                inputs.inject_unsorted(y, j)
                cases.append((f"viol@{j}", y))
            z = x.copy()
            z[n // 3] = -1.0
            cases.append(("negative", z))
        for name, data in cases:
            want = ocfg.cfg3(data)
            with Ctx(MODES[mode] | flags) as c:
                t = c.torch.from_numpy(data).cuda()
                r = W.cfg3(c.ctx, n, t.data_ptr())
                assert (c.get(r["pre"]), c.get(r["post"])) == (want["pre"], want["post"]), (name, n)
                if mode != "unfused":
                    assert sg.sg_plan_stats(c.ctx).n_passes == 1


def test_cfg3_trivial_lengths():
    for n in (0, 1):
        with Ctx() as c:
            hx = c.vec(np.ones(n, dtype=np.float32))
            assert c.get(sg.sg_forall_adjacent(c.ctx, hx, sg.SG_LE)) is True     # n <= 1 => sorted


def test_cfg3_full_size():
    n = 1 << 28
    x = inputs.sorted_cumsum_f32(4, 0, n)
    j = inputs.violation_index(4, n)
    with Ctx() as c:
        t = c.torch.from_numpy(x).cuda()
        r = W.cfg3(c.ctx, n, t.data_ptr())
        assert (c.get(r["pre"]), c.get(r["post"])) == (True, True)
        st = sg.sg_plan_stats(c.ctx)
        assert st.n_passes == 1 and st.n_template == 1 and st.bytes_min == 4 * n
        t[j] = 0.5 * t[j - 1]
        r = W.cfg3(c.ctx, n, t.data_ptr())
        assert (c.get(r["pre"]), c.get(r["post"])) == (True, False)
    inputs.inject_unsorted(x, j)
    assert ocfg.cfg3(x) == {"pre": True, "post": False}


# ----------------------------------------------------------------------------------------------------------
# config 4
# ----------------------------------------------------------------------------------------------------------
def colsum_ok(got, want, col_abs_sum):
    return all(rel_err(g, w, s) <= 1e-12 for g, w, s in zip(got, want, col_abs_sum))


# odd n (and odd leading dimensions): rows that are not 16-byte aligned take the matrix pass's guarded form (PAPER.md:209-219 puts
# no condition on a matrix's shape)
@pytest.mark.parametrize("n,k,ld", [(2, 0, 2), (4, 1, 4), (34, 0, 34), (34, 33, 34), (258, 100, 258), (1030, 7, 1030), (2050, 2048, 2050), (1538, 0, 1538),
                                    (3, 0, 3), (3, 1, 3), (33, 5, 33), (33, 31, 37), (129, 0, 129), (1031, 7, 1031), (1031, 1000, 1040), (515, 3, 521), (64, 3, 67)])
def test_cfg4(n, k, ld):
    M = inputs.boosted_matrix_f64(5, 0, n)
    want = ocfg.cfg4(M, k)
    with Ctx() as c:
        buf = np.full((n, ld), 7.25)
        buf[:, :n] = M
        t = c.torch.from_numpy(buf).cuda()
        r = W.cfg4(c.ctx, n, t.data_ptr(), k, ld=ld)
        sg.sg_flush(c.ctx)
        c.torch.cuda.synchronize()
        full = t.cpu().numpy()
        got = np.ascontiguousarray(full[:, :n])
        assert bits_equal(got, want["M"])
        assert (full[:, n:] == 7.25).all()                              # the padding between rows is never written
        if k + 1 < n:
            rowmax = c.read_vec(r["rowmax"], np.float64)
            colsum = c.read_vec(r["colsum"], np.float64)
            assert bits_equal(rowmax, want["rowmax"])
            assert colsum_ok(colsum, want["colsum"], np.abs(want["M"][k + 1:]).sum(axis=0))
            assert sg.sg_plan_stats(c.ctx).n_passes == 2


@pytest.mark.parametrize("n,k,ld", [(2, 0, 2), (3, 1, 3), (34, 0, 34), (33, 5, 37), (258, 100, 258), (515, 3, 521), (1030, 7, 1030)])
def test_cfg4_through_the_matrix_bytecode_evaluator(n, k, ld):
    """SG_FLAG_FORCE_BYTECODE: the same step on pass2d_bytecode (the evaluator of matrix chains without a template instance)."""
    M = inputs.boosted_matrix_f64(5, 0, n)
    want = ocfg.cfg4(M, k)
    with Ctx(sg.SG_FLAG_FORCE_BYTECODE) as c:
        buf = np.full((n, ld), 7.25)
        buf[:, :n] = M
        t = c.torch.from_numpy(buf).cuda()
        r = W.cfg4(c.ctx, n, t.data_ptr(), k, ld=ld)
        sg.sg_flush(c.ctx)
        st = sg.sg_plan_stats(c.ctx)
        full = t.cpu().numpy()
        assert st.n_bytecode == st.n_passes == 2
        assert bits_equal(np.ascontiguousarray(full[:, :n]), want["M"]) and (full[:, n:] == 7.25).all()
        if k + 1 < n:
            assert bits_equal(c.read_vec(r["rowmax"], np.float64), want["rowmax"])
            assert colsum_ok(c.read_vec(r["colsum"], np.float64), want["colsum"], np.abs(want["M"][k + 1:]).sum(axis=0))


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32])
@pytest.mark.parametrize("rows,cols", [(1, 1), (5, 3), (33, 65), (130, 1027), (700, 260)])
def test_unregistered_matrix_chain_runs_on_the_bytecode_evaluator(dtype, rows, cols):
    """A matrix chain nobody registered a template for: B = (A + A) * v (ROW broadcast) - w (COL broadcast), kept; per-row max, per-column
    sum, whole-matrix min and a quantifier — one pass on pass2d_bytecode, compared with the oracle primitive by primitive."""
    from gpu_util import NP2SG
    if np.dtype(dtype).kind == "f":
        A = RNG.standard_normal((rows, cols)).astype(dtype)
        v, w = RNG.standard_normal(cols).astype(dtype), RNG.standard_normal(rows).astype(dtype)
    else:
        A = RNG.integers(-1000, 1000, (rows, cols)).astype(dtype)
        v, w = RNG.integers(-50, 50, cols).astype(dtype), RNG.integers(-50, 50, rows).astype(dtype)
    with Ctx() as c:
        tA, tv, tw = dev(A), dev(v), dev(w)
        c.keep += [tA, tv, tw]
        sgdt = NP2SG[np.dtype(dtype)]
        hA = sg.sg_mat_create(c.ctx, sgdt, rows, cols, cols, tA.data_ptr())
        hv, hw = sg.sg_vec_create(c.ctx, sgdt, cols, tv.data_ptr()), sg.sg_vec_create(c.ctx, sgdt, rows, tw.data_ptr())
        s2 = sg.sg_enqueue(c.ctx, sg.SG_ADD, [hA, hA])
        sv = sg.sg_enqueue(c.ctx, sg.SG_MUL, [s2, sg.H(hv, sg.SG_BCAST_ROW)])
        B = sg.sg_enqueue(c.ctx, sg.SG_SUB, [sv, sg.H(hw, sg.SG_BCAST_COL)])
        for h in (s2, sv):
            sg.sg_release(c.ctx, h)
        rmax = sg.sg_reduce(c.ctx, B, sg.SG_RMAX, sg.SG_AXIS_ROWS)
        csum = sg.sg_reduce(c.ctx, B, sg.SG_SUM, sg.SG_AXIS_COLS)
        mn = sg.sg_reduce(c.ctx, B, sg.SG_RMIN)
        pos = sg.sg_enqueue(c.ctx, sg.SG_GT, [B, sg.F(0.0) if np.dtype(dtype).kind == "f" else sg.I(0)])
        anyp, cnt = sg.sg_exists(c.ctx, pos), sg.sg_reduce(c.ctx, pos, sg.SG_COUNT)
        sg.sg_release(c.ctx, pos)
        got_min, got_any, got_cnt = c.get(mn), c.get(anyp), c.get(cnt)
        st = sg.sg_plan_stats(c.ctx)
        assert st.n_passes == 1 and st.n_bytecode == 1
        got_B = c.read_vec(B, dtype, rows * cols).reshape(rows, cols)
        got_rmax = c.read_vec(rmax, dtype, rows)
        got_csum = c.read_vec(csum, np.float64 if np.dtype(dtype).kind == "f" else np.int64, cols)
    want_B = np.empty_like(A)
    for r in range(rows):
        want_B[r] = orc.scalar("sub", orc.zip("mul", orc.zip("add", A[r], A[r]), v), w[r])
    assert bits_equal(got_B, want_B)
    assert bits_equal(got_rmax, np.array([orc.max(want_B[r]) for r in range(rows)], dtype=dtype))
    want_csum = [orc.sum(np.ascontiguousarray(want_B[:, cc])) for cc in range(cols)]
    if np.dtype(dtype).kind == "f":
        tol = 1e-12 if dtype is np.float64 else 1e-5
        assert all(abs(gv - wv) <= tol * max(np.abs(want_B[:, cc]).sum(), 1e-300) for cc, (gv, wv) in enumerate(zip(got_csum, want_csum)))
    else:
        assert got_csum.tolist() == want_csum
    assert dtype(got_min) == orc.min(want_B.reshape(-1)) and got_any == bool((want_B > 0).any()) and got_cnt == int((want_B > 0).sum())


def test_bool_matrix_kept_and_read_back_in_a_later_pass():
    """A BOOL matrix somebody keeps (a mask) is stored one byte per element and read back by a later matrix pass."""
    rows, cols = 37, 301
    A = RNG.standard_normal((rows, cols))
    B = RNG.standard_normal((rows, cols))
    with Ctx() as c:
        tA, tB = dev(A), dev(B)
        c.keep += [tA, tB]
        hA = sg.sg_mat_create(c.ctx, sg.SG_F64, rows, cols, cols, tA.data_ptr())
        hB = sg.sg_mat_create(c.ctx, sg.SG_F64, rows, cols, cols, tB.data_ptr())
        mask = sg.sg_enqueue(c.ctx, sg.SG_GT, [hA, sg.F(0.0)])          # kept: materialised as bytes
        sg.sg_flush(c.ctx)
        got_mask = c.read_vec(mask, np.uint8, rows * cols).reshape(rows, cols)
        other = sg.sg_enqueue(c.ctx, sg.SG_LT, [hB, sg.F(0.5)])
        both = sg.sg_enqueue(c.ctx, sg.SG_AND, [mask, other])
        sg.sg_release(c.ctx, other)
        per_row = sg.sg_reduce(c.ctx, both, sg.SG_COUNT, sg.SG_AXIS_ROWS)
        total = sg.sg_reduce(c.ctx, both, sg.SG_COUNT)
        sg.sg_release(c.ctx, both)
        got_total = c.get(total)
        got_rows = c.read_vec(per_row, np.int64, rows)
    want_mask = np.stack([orc.cmp_scalar("gt", A[r], 0.0) for r in range(rows)])
    want_both = np.stack([orc.logic("and", want_mask[r], orc.cmp_scalar("lt", B[r], 0.5)) for r in range(rows)])
    assert bits_equal(got_mask, want_mask)
    assert got_rows.tolist() == [orc.count(want_both[r]) for r in range(rows)] and got_total == orc.count(want_both.reshape(-1))


# the store-only row update (Listing 5 without config 4's reductions): aligned shapes run as one tile per block (sg_pass2d_tile.cuh),
# odd shapes through the staged kernel's guarded form; strips with a ragged right edge, one row, views with a leading dimension
@pytest.mark.parametrize("n,k,ld", [(2, 0, 2), (4, 1, 4), (34, 0, 34), (258, 100, 258), (1024, 0, 1024), (1030, 7, 1030), (2050, 2048, 2050), (2048, 5, 2048),
                                    (3100, 1, 3104), (1538, 0, 1540), (33, 5, 37), (1031, 7, 1031), (515, 3, 521)])
def test_ge_row_update_store_only(n, k, ld):
    M = inputs.boosted_matrix_f64(5, 0, n)
    want = ocfg.cfg4(M, k)["M"]
    with Ctx() as c:
        buf = np.full((n, ld), 7.25)
        buf[:, :n] = M
        t = c.torch.from_numpy(buf).cuda()
        W.ge_row_update(c.ctx, n, t.data_ptr(), k, ld=ld)
        sg.sg_flush(c.ctx)
        st = sg.sg_plan_stats(c.ctx)
        assert st.n_passes == 2 and st.n_template == 2
        c.torch.cuda.synchronize()
        full = t.cpu().numpy()
        assert bits_equal(np.ascontiguousarray(full[:, :n]), want)
        assert (full[:, n:] == 7.25).all()                              # the padding between rows is never written


def test_ge_row_update_full_size():
    n, k = 16384, 0
    M = inputs.boosted_matrix_f64(5, 0, n)
    want_M = orc.mat_step(M, k)[0]
    with Ctx() as c:
        t = c.torch.from_numpy(M).cuda()
        W.ge_row_update(c.ctx, n, t.data_ptr(), k)
        sg.sg_flush(c.ctx)
        got = t.cpu().numpy()
    assert bits_equal(got, want_M)


@pytest.mark.parametrize("k", [0, 8191])
def test_cfg4_full_size(k):
    """BASELINE.json:configs[4] at its full size, in bench.py's launch configuration: EVERY element of M', all n-k-1 row maxima
    and all n column sums against the oracle's definition (orc_mat_step on the whole matrix takes seconds)."""
    n = 16384
    M = inputs.boosted_matrix_f64(5, 0, n)
    want_M, want_rowmax, want_colsum = orc.mat_step(M, k)
    with Ctx() as c:
        t = c.torch.from_numpy(M).cuda()
        r = W.cfg4(c.ctx, n, t.data_ptr(), k)
        sg.sg_flush(c.ctx)
        st = sg.sg_plan_stats(c.ctx)
        assert st.n_passes == 2 and st.n_template == 2
        rowmax = c.read_vec(r["rowmax"], np.float64)
        colsum = c.read_vec(r["colsum"], np.float64)
        got = t.cpu().numpy()
    assert bits_equal(got, want_M)                                    # all 2^28 elements (rows <= k untouched included)
    assert rowmax.size == n - k - 1 and bits_equal(rowmax, want_rowmax)
    assert colsum.size == n and colsum_ok(colsum, want_colsum, np.abs(want_M[k + 1:]).sum(axis=0))


# ----------------------------------------------------------------------------------------------------------
# the whole Gaussian-elimination determinant loop (Listing 5)
# ----------------------------------------------------------------------------------------------------------
def ge_matrix(n, seed=5):
    """Config 4's matrix scaled by 1/n (diagonal ~ 1, off-diagonal ~ U[-1,1)/n) so that the determinant stays finite."""
    return inputs.boosted_matrix_f64(seed, 0, n) / float(n)


def run_ge(c, M, ld=None, eps=0.0, native=True):
    n = M.shape[0]
    ld = n if ld is None else ld
    buf = np.zeros((n, ld))
    buf[:, :n] = M
    t = c.torch.from_numpy(buf).cuda()
    det = c.torch.ones(1, dtype=c.torch.float64, device="cuda")
    minpiv = c.torch.full((1,), float("inf"), dtype=c.torch.float64, device="cuda")
    got, ok = W.ge_determinant(c.ctx, n, t.data_ptr(), det.data_ptr(), minpiv.data_ptr(), ld=ld, eps=eps, native=native)
    return got, ok, t.cpu().numpy()[:, :n], float(minpiv.item())


# any n and ld (odd ones included: rows that are not 16-byte aligned); sizes from one block's worth of rows to several rows per block
@pytest.mark.parametrize("n,ld", [(1, 1), (2, 2), (3, 3), (4, 6), (18, 18), (64, 64), (129, 129), (130, 136), (258, 258), (514, 520), (515, 515), (515, 522),
                                  (1200, 1200)])
def test_ge_determinant_loop(n, ld):
    M = ge_matrix(n)
    want_det, want_E, zs = orc.ge_determinant(M)
    assert zs == -1
    with Ctx() as c:
        got, ok, E, minpiv = run_ge(c, M, ld)
        assert ok
        assert bits_equal(np.array([got]), np.array([want_det]))        # same products in the same order: bit-exact
        assert bits_equal(np.ascontiguousarray(E), want_E)              # the eliminated matrix, every element
        assert minpiv == np.min(np.abs(np.diag(want_E)))
        assert sg.sg_plan_stats(c.ctx).n_passes <= 2                    # the loop itself is ONE kernel; the flush afterwards reads det / ok back
        if n <= 130:                                                    # the same steps as host-issued primitives (3 launches per step)
            got2, ok2, E2, _ = run_ge(c, M, ld, native=False)
            assert ok2 and got2 == got and bits_equal(np.ascontiguousarray(E2), want_E)


def test_ge_determinant_in_two_calls_and_large():
    """Steps [0, h) and [h, n) in two calls give the same bits as one call; 2200 x 2200: several rows per block and step."""
    n = 2200
    M = ge_matrix(n)
    want_det, want_E, zs = orc.ge_determinant(M)
    with Ctx() as c:
        t = c.torch.from_numpy(M).cuda()
        det = c.torch.ones(1, dtype=c.torch.float64, device="cuda")
        mp = c.torch.full((1,), float("inf"), dtype=c.torch.float64, device="cuda")
        hM = sg.sg_mat_create(c.ctx, sg.SG_F64, n, n, n, t.data_ptr())
        hd, hp = sg.sg_vec_create(c.ctx, sg.SG_F64, 1, det.data_ptr()), sg.sg_vec_create(c.ctx, sg.SG_F64, 1, mp.data_ptr())
        sg.sg_mat_ge_steps(c.ctx, hM, hd, hp, 0.0, 0, 777)
        sg.sg_mat_ge_steps(c.ctx, hM, hd, hp, 0.0, 777, n)
        c.torch.cuda.synchronize()
        assert bits_equal(np.array([det.item()]), np.array([want_det])) and bits_equal(t.cpu().numpy(), want_E)
        assert mp.item() == np.min(np.abs(np.diag(want_E)))


def test_ge_determinant_zero_pivot_is_decided_on_the_device():
    """Result := Result * pivot, THEN the approximately-zero test, whose else-branch ends the loop.  The library takes
    that decision (no arithmetic in the binding): det is Result * pivot and the matrix is eliminated exactly up to the zero step."""
    cases = [
        (np.array([[1.0, 2.0, 0.0, 0.0], [2.0, 4.0, 1.0, 0.0], [0.0, 1.0, 1.0, 0.0], [0.0, 0.0, 0.0, 1.0]]), 0.0),     # second pivot 4 - 2*2 = 0
        (np.array([[-1.0, 2.0], [3.0, -6.0]]), 0.0),                                                                    # Result = -1 * 0 = -0.0
        (np.array([[1e-9, 1.0], [1.0, 1.0]]), 1e-6),                                                                    # ~0 with an explicit eps: Result = 1e-9
        (np.array([[2.0, 1.0], [4.0, 2.0 + 2.0 ** -40]]), 1e-6),                                                        # Result = 2 * 2^-40
        (np.array([[2.0, 1.0], [1e-9, 3.0]]), 1e-6),                                                                    # the per-row guard: row 1 left as it is
    ]
    rng = np.random.default_rng(3)
    big = ge_matrix(300)
    big[200] = 0.5 * big[100] + 0.25 * big[150]                           # rank deficient: row 200 eliminates to (almost) nothing
    cases.append((big, 1e-9))
    sp = ge_matrix(96)
    sp[rng.integers(0, 96, 200), rng.integers(0, 96, 200)] = 0.0          # exact zeros below the pivots: skipped rows (eps = 0 guard)
    sp[np.arange(96), np.arange(96)] = 1.0 + np.arange(96) / 96.0
    cases.append((sp, 0.0))
    for M, eps in cases:
        want_det, want_E, zs = orc.ge_determinant(M, eps=eps)
        with Ctx() as c:
            got, ok, E, minpiv = run_ge(c, M, eps=eps)
            assert ok == (zs < 0), (M.shape, eps)
            assert bits_equal(np.array([got]), np.array([want_det])), (got, want_det)      # incl. the sign of a zero
            assert bits_equal(np.ascontiguousarray(E), want_E)                               # eliminated up to the zero step, untouched after it
            if zs >= 0:
                assert minpiv <= eps
    with Ctx() as c:
        M = np.array([[1e-9, 1.0], [1.0, 1.0]])
        got, ok, _, _ = run_ge(c, M, eps=0.0)                               # eps = 0: the tiny pivot is accepted
        assert ok and bits_equal(np.array([got]), np.array([orc.ge_determinant(M)[0]]))


# ----------------------------------------------------------------------------------------------------------
# plan hazards and context robustness on the device (round-1 review)
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["template", "bytecode"])
@pytest.mark.parametrize("n", [2, 33, 1025, (1 << 20) + 3, 1 << 22])
def test_neighbour_contract_then_inplace_update_reads_the_old_values(mode, n):
    """require x.is_sorted; x *= -1 in place.  x[i+1] is read by another thread / warp / block than the one that overwrites it: the
    update must run in a LATER pass.  With both in one pass the contract sees a mix of old and new values (sorted -> unsorted)."""
    x = inputs.sorted_cumsum_f32(4, 0, n)
    with Ctx(MODES[mode]) as c:
        t = dev(x); c.keep.append(t)
        hx = sg.sg_vec_create(c.ctx, sg.SG_F32, n, t.data_ptr())
        srt = sg.sg_forall_adjacent(c.ctx, hx, sg.SG_LE)
        ge0 = sg.sg_enqueue(c.ctx, sg.SG_GE, [hx, sg.F(0.0)])
        pre = sg.sg_forall(c.ctx, ge0)
        sg.sg_release(c.ctx, ge0)
        sg.sg_enqueue(c.ctx, sg.SG_MUL, [hx, sg.F(-1.0)], dst_or_0=hx)
        assert c.get(srt) is True and c.get(pre) is True
        assert sg.sg_plan_stats(c.ctx).n_passes == 2
        got = c.read_vec(hx, np.float32, n)
    assert bits_equal(got, orc.scalar("mul", x, -1.0))


def test_release_before_flush_on_the_device():
    n = (1 << 16) + 5
    a = RNG.standard_normal(n).astype(np.float32)
    with Ctx() as c:
        x = sg.sg_vec_create(c.ctx, sg.SG_F32, n, None)                 # context-owned storage, filled by a pass
        ha = c.vec(a)
        sg.sg_enqueue(c.ctx, sg.SG_ADD, [ha, sg.F(0.0)], dst_or_0=x)
        sg.sg_flush(c.ctx)
        y = sg.sg_enqueue(c.ctx, sg.SG_ADD, [x, sg.F(1.0)])
        sg.sg_release(c.ctx, x)                                         # released while y = x + 1 is pending
        s = sg.sg_reduce(c.ctx, y, sg.SG_SUM)
        got_s = c.get(s)
        q = sg.sg_enqueue(c.ctx, sg.SG_DIV, [s, sg.F(4.0)])             # a materialised scalar consumed by a new chain ...
        sg.sg_release(c.ctx, s)                                         # ... and released before the flush
        got_q = c.read_vec(q, np.float64, 1)[0]
        got_y = c.read_vec(y, np.float32, n)
    want_y = orc.scalar("add", orc.scalar("add", a, 0.0), 1.0)
    assert bits_equal(got_y, want_y)
    assert abs(got_s - orc.sum(want_y)) <= 1e-5 * np.abs(want_y).sum() and got_q == got_s / 4.0


def test_failed_flush_discards_and_the_context_goes_on():
    n = 4096
    a = RNG.standard_normal(n)
    with Ctx() as c:
        ha = c.vec(a)
        sg.sg_enqueue(c.ctx, sg.SG_ADD, [ha, sg.F(1.0)], dst_or_0=ha)   # an in-place update queued in the same (failing) flush
        many = [sg.sg_reduce(c.ctx, sg.sg_enqueue(c.ctx, sg.SG_MUL, [ha, sg.F(float(i))]), sg.SG_SUM) for i in range(2200)]     # > 256 passes
        with pytest.raises(sg.SgError) as e:
            sg.sg_flush(c.ctx)
        assert e.value.status == sg.SG_ERR_CAPACITY
        assert bits_equal(c.read_vec(ha, np.float64, n), a)             # nothing ran: the in-place destination keeps its contents
        r = sg.sg_enqueue(c.ctx, sg.SG_MUL, [ha, sg.F(3.0)])            # the context is usable
        assert bits_equal(c.read_vec(r, np.float64, n), orc.scalar("mul", a, 3.0))
        del many


def test_early_exit_leaves_no_half_evaluated_quantifier_readable():
    """A pass of quantifiers ends at the first violated registered contract.  A quantifier of the same pass that was not decided on
    the prefix read so far is NOT evaluated: reading it is an error; one that was decided (exists already true) is final."""
    n = 1 << 24
    x = inputs.sorted_cumsum_f32(4, 0, n)
    inputs.inject_unsorted(x, 1000)                                     # the violation sits at the very beginning
    with Ctx() as c:
        t = dev(x); c.keep.append(t)
        hx = sg.sg_vec_create(c.ctx, sg.SG_F32, n, t.data_ptr())
        srt = sg.sg_forall_adjacent(c.ctx, hx, sg.SG_LE)
        sg.sg_contract(c.ctx, srt, sg.SG_CONTRACT_PRE, "is_sorted")
        big = sg.sg_enqueue(c.ctx, sg.SG_GT, [hx, sg.F(float(x[n - 1]) * 0.999)])      # witnesses only at the far end
        ex_far = sg.sg_exists(c.ctx, big)
        small = sg.sg_enqueue(c.ctx, sg.SG_LT, [hx, sg.F(float(x[10]))])               # witnesses at the very beginning
        ex_near = sg.sg_exists(c.ctx, small)
        with pytest.raises(sg.SgError) as e:
            sg.sg_flush(c.ctx)
        assert e.value.status == sg.SG_ERR_CONTRACT and "is_sorted" in str(e.value)
        assert c.get(srt) is False
        # ex_far: true on the whole vector; after the early exit it is either decided (the pass got that far) or not evaluated — never a wrong False
        try:
            assert c.get(ex_far) is True
        except sg.SgError as err:
            assert err.status == sg.SG_ERR_CONTRACT and "not evaluated" in str(err)
        try:
            assert c.get(ex_near) is True
        except sg.SgError as err:
            assert err.status == sg.SG_ERR_CONTRACT
    with Ctx(sg.SG_FLAG_NO_EARLY_EXIT) as c:                            # without early exit everything is evaluated
        t = dev(x); c.keep.append(t)
        hx = sg.sg_vec_create(c.ctx, sg.SG_F32, n, t.data_ptr())
        srt = sg.sg_forall_adjacent(c.ctx, hx, sg.SG_LE)
        sg.sg_contract(c.ctx, srt, sg.SG_CONTRACT_PRE, "is_sorted")
        big = sg.sg_enqueue(c.ctx, sg.SG_GT, [hx, sg.F(float(x[n - 1]) * 0.999)])
        ex_far = sg.sg_exists(c.ctx, big)
        with pytest.raises(sg.SgError):
            sg.sg_flush(c.ctx)
        assert c.get(ex_far) is True and c.get(srt) is False


def test_cfg1_sharded_over_emulated_ranks():
    """ONE collection in W contiguous shards.  One GPU here, so the W ranks run one after the other (no kernel waits for
    another): each leaves its partial sum / max in device memory, the all-gather is emulated by a tensor that collects them in rank
    order, and the combine is the library's pass over the W partials — the same workload function bench.py --shard runs per rank."""
    from paper_1410_6685_b200 import ranks
    n, world = (1 << 22) + 5, 3
    x, y = inputs.normal_f32(2, 0, n), inputs.normal_f32(2, 1, n)
    want = ocfg.cfg1(x, y)
    with Ctx() as c:
        torch = c.torch
        all_sum = torch.zeros(world, dtype=torch.float64, device="cuda")
        all_max = torch.zeros(world, dtype=torch.float32, device="cuda")
        results = []
        for rank in range(world):
            lo, hi = ranks.shard_range(n, rank, world)
            xs, ys = inputs.normal_f32(2, 0, hi - lo, start=lo), inputs.normal_f32(2, 1, hi - lo, start=lo)   # a rank generates only its range
            assert bits_equal(xs, x[lo:hi])
            tx, ty = dev(xs), dev(ys)
            c.keep += [tx, ty]
            ps, pm = all_sum[rank:rank + 1], all_max[rank:rank + 1]          # this rank's slot of the gathered buffers

            def gather(kind):
                t = all_sum if kind == "sum" else all_max
                return t.data_ptr(), rank + 1                                  # the partials gathered so far, in rank order
            r = W.cfg1_sharded(c.ctx, hi - lo, tx.data_ptr(), ty.data_ptr(), ps.data_ptr(), pm.data_ptr(), gather)
            results.append((c.get(r["sum"]), c.get(r["max"])))
        gsum, gmax = results[-1]                                              # after the last rank every partial is there
    assert sum_ok(gsum, want["sum"], want["w"], 1e-5) and np.float32(gmax) == want["max"]


def test_vector_longer_than_2_31_elements():
    """Maximum sizes: 2^31 + 7 int32 elements (8 GiB): every index, tile and offset computation is 64-bit.  The oracle cannot hold this on
    every box, so the results are checked against closed forms that hold at any size (x_i = i mod 1000) and, for the compaction, against
    its exact periodic structure."""
    import torch
    n = (1 << 31) + 7
    free, _ = torch.cuda.mem_get_info()
    if free < 60 * (1 << 30):
        pytest.skip("needs 60 GiB of free device memory")
    idx = torch.arange(n, device="cuda", dtype=torch.int64)
    xi = (idx % 1000).to(torch.int32)
    del idx
    q, r = divmod(n, 1000)
    with Ctx() as c:
        hx = sg.sg_vec_create(c.ctx, sg.SG_I32, n, xi.data_ptr())
        s, mx, mn = (sg.sg_reduce(c.ctx, hx, k) for k in (sg.SG_SUM, sg.SG_RMAX, sg.SG_RMIN))
        eq7 = sg.sg_enqueue(c.ctx, sg.SG_EQ, [hx, sg.I(7)])
        cnt7 = sg.sg_reduce(c.ctx, eq7, sg.SG_COUNT)
        sg.sg_release(c.ctx, eq7)
        ge0 = sg.sg_enqueue(c.ctx, sg.SG_GE, [hx, sg.I(0)])
        all_ge0 = sg.sg_forall(c.ctx, ge0)
        sg.sg_release(c.ctx, ge0)
        srt = sg.sg_forall_adjacent(c.ctx, hx, sg.SG_LE)
        assert c.get(s) == q * 499500 + r * (r - 1) // 2 and c.get(mx) == 999 and c.get(mn) == 0
        assert c.get(cnt7) == q + (1 if r > 7 else 0) and c.get(all_ge0) is True and c.get(srt) is False
        # stable filter x mod 250 == 7: the kept values are 7, 257, 507, 757 repeated, in that order
        res = W.cfg2(c.ctx, n, xi.data_ptr(), modulus=250, residue=7)
        kept_n, kept_sum = c.get(res["count"]), c.get(res["sum"])
        tail = [v for v in (7, 257, 507, 757) if v < r]
        assert kept_n == 4 * q + len(tail) and kept_sum == q * (7 + 257 + 507 + 757) + sum(tail)
        assert sg.sg_plan_stats(c.ctx).n_template == 1
        ptr = sg.sg_vec_data(c.ctx, res["kept"])
        kept = c.read_vec(res["kept"], np.int32)
        assert kept.size == kept_n and ptr != 0
        pat = np.array([7, 257, 507, 757], dtype=np.int32)
        assert (kept[: 4 * q].reshape(q, 4) == pat).all() and kept[4 * q:].tolist() == tail
