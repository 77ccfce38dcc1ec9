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
from gpu_util import Ctx, rel_err

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


@pytest.mark.parametrize("n,k", [(2, 0), (4, 1), (34, 0), (34, 33), (258, 100), (1030, 7), (2050, 2048), (1538, 0)])
def test_cfg4(n, k):
    M = inputs.boosted_matrix_f64(5, 0, n)
    want = ocfg.cfg4(M, k)
    with Ctx() as c:
        t = c.torch.from_numpy(M).cuda()
        r = W.cfg4(c.ctx, n, t.data_ptr(), k)
        sg.sg_flush(c.ctx)
        c.torch.cuda.synchronize()
        got = t.cpu().numpy()
        assert bits_equal(got, want["M"])
        if k + 1 < n:
            rowmax = c.read_vec(r["rowmax"], np.float64)
            colsum = c.read_vec(r["colsum"], np.float64)
            assert bits_equal(rowmax, want["rowmax"])
            assert colsum_ok(colsum, want["colsum"], np.abs(want["M"][k + 1:]).sum(axis=0))
            assert sg.sg_plan_stats(c.ctx).n_passes == 2


@pytest.mark.parametrize("k", [0, 8191])
def test_cfg4_full_size_sampled(k):
    n = 16384
    M = inputs.boosted_matrix_f64(5, 0, n)
    S = sorted({0, 1, k, min(k + 1, n - 1), 4097, 8190, 8192, 12345, n - 1})
    Ms, _, colsum_s = orc.mat_step(M[:, [k] + S], k, 0)              # the definition on sampled columns (all rows)
    rows = sorted({k + 1, k + 2, (k + n) // 2, n - 1})
    with Ctx() as c:
        t = c.torch.from_numpy(M).cuda()
        r = W.cfg4(c.ctx, n, t.data_ptr(), k)
        sg.sg_flush(c.ctx)
        rowmax = c.read_vec(r["rowmax"], np.float64)
        colsum = c.read_vec(r["colsum"], np.float64)
        got_cols = t[:, S].cpu().numpy()
        got_rows = t[rows, :].cpu().numpy()
        head = t[: k + 1, :].cpu().numpy()
    assert bits_equal(np.ascontiguousarray(got_cols), np.ascontiguousarray(Ms[:, 1:]))
    assert bits_equal(head, M[: k + 1])                              # rows <= k untouched
    assert colsum_ok(colsum[S], colsum_s[1:], np.abs(Ms[k + 1:, 1:]).sum(axis=0))
    piv = M[k, k]
    for j, grow in zip(rows, got_rows):
        f = np.array([M[j, k]]) / piv                                # one row through the oracle primitives
        wrow = orc.zip("sub", M[j], orc.scalar("mul", M[k], f[0]))
        assert bits_equal(grow, wrow)
        assert rowmax[j - k - 1] == orc.max(orc.unary("abs", wrow))


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


# even n and ld: a matrix pass needs 16-byte aligned rows (SG_ERR_UNSUPPORTED otherwise, include/sg.h)
@pytest.mark.parametrize("n,ld", [(1, 1), (2, 2), (4, 6), (18, 18), (64, 64), (130, 136), (258, 258), (514, 520)])
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
        if n <= 130:                                                    # the same steps driven call by call from the binding
            got2, ok2, E2, _ = run_ge(c, M, ld, native=False)
            assert ok2 and got2 == got and bits_equal(np.ascontiguousarray(E2), want_E)


def test_ge_determinant_zero_pivot_contract():
    with Ctx() as c:
        M = np.array([[1.0, 2.0, 0.0, 0.0], [2.0, 4.0, 1.0, 0.0], [0.0, 1.0, 1.0, 0.0], [0.0, 0.0, 0.0, 1.0]])   # second pivot 4 - 2*2 = 0
        want, _, zs = orc.ge_determinant(M)
        got, ok, _, minpiv = run_ge(c, M)
        assert zs == 1 and want == 0.0 and got == 0.0 and not ok and minpiv == 0.0
    with Ctx() as c:
        M = np.array([[1e-9, 1.0], [1.0, 1.0]])                             # approximately zero with an explicit eps
        assert orc.ge_determinant(M, eps=1e-6)[0] == 0.0
        got, ok, _, _ = run_ge(c, M, eps=1e-6)
        assert got == 0.0 and not ok
        got, ok, _, _ = run_ge(c, M, eps=0.0)                               # eps = 0: the tiny pivot is accepted
        assert ok and bits_equal(np.array([got]), np.array([orc.ge_determinant(M)[0]]))
