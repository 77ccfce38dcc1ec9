"""Randomised differential test (SURVEY.md §8(c) pin table: "bytecode vs template ... and on random chains"): seeded random
operation DAGs over the C ABI against the CPU oracle, primitive by primitive.  A DAG mixes value operations, immediates, comparisons,
logic, stored and released intermediates, IN-PLACE results (dst_or_0), device scalars used as operands (an exact reduction of one
value broadcast into a later operation: a scalar edge, so the flush has several passes), reductions, quantifiers, the neighbour
predicate and a stable filter with its count and kept-sum — all pending in ONE flush.  No template instance matches such chains, so
what is exercised is the plan builder (pass assignment, spills, hazards, register allocation) and the bytecode evaluators; the same
DAG also runs unfused (one launch per operation) and must give the same bits.

Bars as everywhere: stored values, extrema, counts, filter outputs and quantifiers bit-exact; sums 1e-12 (fp64) / 1e-5 (fp32)."""
import os

import numpy as np
import pytest

import oracle as orc
from paper_1410_6685_b200 import sg
from gpu_util import Ctx, rel_err

pytestmark = pytest.mark.gpu

# SAFEGPU_FUZZ_SCALE=k runs k times as many seeds of every generator (a soak run; the default is what the suite runs)
FUZZ = max(1, int(os.environ.get("SAFEGPU_FUZZ_SCALE", "1")))

BIN = {"add": sg.SG_ADD, "sub": sg.SG_SUB, "mul": sg.SG_MUL, "div": sg.SG_DIV, "min": sg.SG_MIN, "max": sg.SG_MAX, "mod": sg.SG_MOD}
UN = {"neg": sg.SG_NEG, "abs": sg.SG_ABS, "sqrt": sg.SG_SQRT}
CMP = {"eq": sg.SG_EQ, "ne": sg.SG_NE, "lt": sg.SG_LT, "le": sg.SG_LE, "gt": sg.SG_GT, "ge": sg.SG_GE}
LOGIC = {"and": sg.SG_AND, "or": sg.SG_OR, "not": sg.SG_NOT}
RED = {"sum": sg.SG_SUM, "max": sg.SG_RMAX, "min": sg.SG_RMIN}
SIZES = [1, 2, 31, 257, 1024, 4097, 70001, 300007]
DTYPES = [np.float32, np.float64, np.int32, np.int64]


def bits_equal(a, b):
    a, b = np.ascontiguousarray(a), np.ascontiguousarray(b)
    if a.shape != b.shape or a.dtype != b.dtype:
        return False
    if a.dtype.kind == "f":
        na, nb = np.isnan(a), np.isnan(b)
        if not np.array_equal(na, nb):
            return False
        a, b = np.where(na, 0, a), np.where(nb, 0, b)
    return a.tobytes() == b.tobytes()


def make_input(rng, dtype, n):
    if np.dtype(dtype).kind == "f":
        a = (rng.standard_normal(n) * 4).astype(dtype)
        a[rng.integers(0, n, max(1, n // 50))] = rng.choice(np.array([0.0, -0.0, 1.0, -1.0, 0.5], dtype=dtype))
        return a
    a = rng.integers(-40, 40, n).astype(dtype)
    info = np.iinfo(dtype)
    a[rng.integers(0, n, max(1, n // 50))] = rng.choice(np.array([0, 1, -1, info.min, info.max, 7], dtype=dtype))
    return a


def build_dag(rng, dtype, inputs, rich=True):
    """Generates the steps AND evaluates them with the oracle as it goes (some choices depend on the data: a device scalar is only
    taken from a NaN-free value).  Value ids index `want`; ids [0, len(inputs)) are the inputs.  Returns (steps, keep, reds, want,
    storage, filt): keep = produced ids whose handle the caller holds on to (stored), reds = (kind, source id, step) scalar results,
    storage = ids that name caller-provided buffers at the end (an input, or the latest in-place result written into it), filt =
    (values id, mask id) of a final filter or None.  rich = False: value ops, comparisons, logic and reductions only."""
    is_f = np.dtype(dtype).kind == "f"
    n_inputs = len(inputs)
    want = dict(enumerate(inputs))
    vals, bools, steps = list(range(n_inputs)), [], []
    storage = set(range(n_inputs))
    reds = []
    nid = n_inputs
    for _ in range(int(rng.integers(4, 15))):
        r = rng.random()
        if r < 0.40 or (r < 0.72 and not bools and rng.random() < 0.5):
            op = str(rng.choice(list(BIN) if not is_f else [k for k in BIN if k != "mod"]))
            a = int(rng.choice(vals))
            q = rng.random()
            if q < 0.30:
                imm = float(rng.choice([0.5, 2.0, -3.25, 7.0])) if is_f else int(rng.choice([2, 3, 7, -5, 1]))
                rev = bool(rng.random() < 0.3)
                steps.append(("bin_imm", op, a, imm, rev, nid))
                want[nid] = orc.scalar(op, want[a], imm, reversed=rev)
            elif rich and q < 0.42:
                # a device scalar as operand: an EXACT reduction (max / min; an integer sum where the dtypes agree) of a NaN-free value
                src = int(rng.choice(vals))
                kinds = ["max", "min"] + (["sum"] if np.dtype(dtype) == np.dtype(np.int64) else [])
                kind = str(rng.choice(kinds))
                if is_f and np.isnan(want[src]).any():
                    continue
                sval = {"max": orc.max, "min": orc.min, "sum": orc.sum}[kind](want[src])
                sval = float(sval) if is_f else int(sval)
                steps.append(("bin_scalar", op, a, kind, src, nid))
                want[nid] = orc.scalar(op, want[a], sval)
                reds.append((kind, src, len(steps) - 1))          # the scalar itself is read too
            else:
                b = int(rng.choice(vals))
                if rich and q > 0.88:
                    # in place: the result replaces the contents of a caller-provided buffer; its handle names the new value from now on
                    k = int(rng.choice(sorted(storage)))
                    steps.append(("inplace", op, a, b, k, nid))
                    want[nid] = orc.zip(op, want[a], want[b])
                    vals.remove(k)
                    storage.discard(k)
                    storage.add(nid)
                else:
                    steps.append(("bin", op, a, b, nid))
                    want[nid] = orc.zip(op, want[a], want[b])
            vals.append(nid)
        elif r < 0.54:
            op = str(rng.choice(["neg", "abs"] + (["sqrt"] if is_f else [])))
            a = int(rng.choice(vals))
            steps.append(("un", op, a, nid))
            want[nid] = orc.unary(op, want[a])
            vals.append(nid)
        elif r < 0.80:
            op = str(rng.choice(list(CMP)))
            a = int(rng.choice(vals))
            if rng.random() < 0.4:
                imm = float(rng.choice([0.0, 1.0, -2.5])) if is_f else int(rng.choice([0, 3, -7]))
                steps.append(("cmp_imm", op, a, imm, nid))
                want[nid] = orc.cmp_scalar(op, want[a], imm)
            else:
                b = int(rng.choice(vals))
                steps.append(("cmp", op, a, b, nid))
                want[nid] = orc.cmp(op, want[a], want[b])
            bools.append(nid)
        elif bools:
            op = str(rng.choice(list(LOGIC)))
            a = int(rng.choice(bools))
            b = int(rng.choice(bools)) if op != "not" else -1
            steps.append(("logic", op, a, b, nid))
            want[nid] = orc.logic(op, want[a], want[b] if b >= 0 else None)
            bools.append(nid)
        else:
            continue
        nid += 1
    if not steps:                                          # every draw was a logic op without a BOOL to apply it to
        steps.append(("un", "neg", 0, nid))
        want[nid] = orc.unary("neg", want[0])
        vals.append(nid)
    produced_v = [v for v in vals if v >= n_inputs and v not in storage]
    produced_b = list(bools)
    keep = set(int(x) for x in rng.choice(produced_v, min(len(produced_v), int(rng.integers(0, 3))), replace=False)) if produced_v else set()
    if produced_b and rng.random() < 0.4:
        keep.add(int(rng.choice(produced_b)))
    for _ in range(int(rng.integers(1, 4))):
        if produced_v:
            reds.append((str(rng.choice(["sum", "max", "min"])), int(rng.choice(produced_v)), -1))
    for _ in range(int(rng.integers(0, 3))):
        if produced_b:
            reds.append((str(rng.choice(["all", "any", "count"])), int(rng.choice(produced_b)), -1))
    if rich and rng.random() < 0.3:
        reds.append(("adj_" + str(rng.choice(["le", "lt", "ge", "ne"])), int(rng.choice(vals)), -1))
    filt = None
    if rich and produced_b and rng.random() < 0.35:
        filt = (int(rng.choice(vals)), int(rng.choice(produced_b)))      # (values, mask): kept values, their count and their sum
    if not keep and not reds and filt is None and not (storage - set(range(n_inputs))):
        keep.add(produced_v[-1] if produced_v else produced_b[-1])
    return steps, keep, reds, want, storage, filt


def run_gpu(c, steps, keep, reds, inputs, dtype, filt=None):
    is_f = np.dtype(dtype).kind == "f"
    imm = (lambda x: sg.F(x)) if is_f else (lambda x: sg.I(x))
    h = {i: c.vec(a) for i, a in enumerate(inputs)}
    scalar_of_step, borrowed = {}, set(range(len(inputs)))
    for si, st in enumerate(steps):
        kind = st[0]
        if kind == "bin":
            h[st[4]] = sg.sg_enqueue(c.ctx, BIN[st[1]], [h[st[2]], h[st[3]]])
        elif kind == "bin_imm":
            ops = [imm(st[3]), h[st[2]]] if st[4] else [h[st[2]], imm(st[3])]
            h[st[5]] = sg.sg_enqueue(c.ctx, BIN[st[1]], ops)
        elif kind == "bin_scalar":
            s = sg.sg_reduce(c.ctx, h[st[4]], RED[st[3]])
            scalar_of_step[si] = s
            h[st[5]] = sg.sg_enqueue(c.ctx, BIN[st[1]], [h[st[2]], s])
        elif kind == "inplace":
            h[st[5]] = sg.sg_enqueue(c.ctx, BIN[st[1]], [h[st[2]], h[st[3]]], dst_or_0=h[st[4]])
            assert h[st[5]] == h[st[4]]
            borrowed.add(st[5])
        elif kind == "un":
            h[st[3]] = sg.sg_enqueue(c.ctx, UN[st[1]], [h[st[2]]])
        elif kind == "cmp":
            h[st[4]] = sg.sg_enqueue(c.ctx, CMP[st[1]], [h[st[2]], h[st[3]]])
        elif kind == "cmp_imm":
            h[st[4]] = sg.sg_enqueue(c.ctx, CMP[st[1]], [h[st[2]], imm(st[3])])
        else:
            h[st[4]] = sg.sg_enqueue(c.ctx, LOGIC[st[1]], [h[st[2]]] + ([h[st[3]]] if st[3] >= 0 else []))
    rh = []
    for kind, src, step in reds:
        if step >= 0:
            rh.append(scalar_of_step[step])
        elif kind in RED:
            rh.append(sg.sg_reduce(c.ctx, h[src], RED[kind]))
        elif kind == "count":
            rh.append(sg.sg_reduce(c.ctx, h[src], sg.SG_COUNT))
        elif kind.startswith("adj_"):
            rh.append(sg.sg_forall_adjacent(c.ctx, h[src], CMP[kind[4:]]))
        else:
            rh.append((sg.sg_forall if kind == "all" else sg.sg_exists)(c.ctx, h[src]))
    fres = None
    if filt is not None:
        fv, fc = sg.sg_filter(c.ctx, h[filt[0]], h[filt[1]])
        fres = (fv, fc, sg.sg_reduce(c.ctx, fv, sg.SG_SUM))
    for i, hv in h.items():                                 # anonymous intermediates: everything produced that is not kept
        if i not in borrowed and i not in keep:
            sg.sg_release(c.ctx, hv)
    sg.sg_flush(c.ctx)
    st = sg.sg_plan_stats(c.ctx)
    return h, [c.get(r) for r in rh], st, fres


def check_sum(got, w, tol, ctx):
    ws = orc.sum(w)
    if np.dtype(w.dtype).kind == "f":
        if not np.isfinite(ws):
            assert (np.isnan(ws) and np.isnan(got)) or ws == got, (ctx, got, ws)
        else:
            # the bar is relative to the RESULT (north_star).  A sum that cancels almost completely (x - x patterns over planted 1e19s:
            # condition 1e17) cannot meet it in any fixed precision: there the accumulator's resolution relative to sum|x| binds —
            # n * 2^-53 for fp32 data (fp64 accumulators), 2^-64 for fp64 data (double-double accumulators), R1
            sabs = float(np.abs(w.astype(np.float64)).sum())
            floor = sabs * (w.size * 2.0 ** -53 if w.dtype == np.float32 else 2.0 ** -64)
            assert rel_err(got, ws, sabs) <= tol or abs(got - ws) <= floor, (ctx, got, ws, sabs)
    else:
        assert got == ws, (ctx, got, ws)


@pytest.mark.parametrize("seed", range(400 * FUZZ))
def test_random_chains_match_the_oracle(seed):
    rng = np.random.default_rng(1000 + seed)
    dtype = DTYPES[seed % 4]
    n = int(SIZES[(seed // 4) % len(SIZES)])
    inputs = [make_input(rng, dtype, n) for _ in range(int(rng.integers(1, 4)))]
    steps, keep, reds, want, storage, filt = build_dag(rng, dtype, inputs, rich=seed >= 40)
    tol = {np.float32: 1e-5, np.float64: 1e-12}.get(dtype, 0)
    results = {}
    for mode, flags in (("fused", 0), ("unfused", sg.SG_FLAG_UNFUSED)):
        with Ctx(flags) as c:
            try:
                h, scal, st, fres = run_gpu(c, steps, keep, reds, inputs, dtype, filt)
            except sg.SgError as e:
                if mode == "unfused" and e.status == sg.SG_ERR_CAPACITY:    # one launch per operation: more than 256 passes in one flush (a plan limit)
                    continue
                raise
            assert st.n_passes >= 1
            for i in sorted(keep | storage):
                got = c.read_vec(h[i], want[i].dtype)
                assert bits_equal(got, want[i]), (mode, seed, "stored value", i, steps)
            for (kind, src, _), got in zip(reds, scal):
                w = want[src]
                ctx = (mode, seed, kind, steps)
                if kind == "sum":
                    check_sum(got, w, tol, ctx)
                elif kind in ("max", "min"):
                    ext = orc.max if kind == "max" else orc.min
                    # extrema follow the total order on bit patterns (R15: -NaN below -inf, +NaN above +inf); the SIGN of a
                    # generated NaN (sqrt of a negative) is the hardware's: x86 makes -NaN, the GPU +NaN — both readings are accepted
                    cands = [ext(w)]
                    if w.dtype.kind == "f" and np.isnan(w).any():
                        cands = [ext(np.where(np.isnan(w), np.copysign(np.nan, sgn), w).astype(w.dtype)) for sgn in (1.0, -1.0)]
                    assert any(bits_equal(np.array([got], dtype=dtype), np.array([wv], dtype=dtype)) for wv in cands), (ctx, got, cands)
                elif kind == "count":
                    assert got == orc.count(w), ctx
                elif kind.startswith("adj_"):
                    assert got == (orc.all(orc.adj(kind[4:], w)) if w.size > 1 else True), ctx
                else:
                    assert got == (orc.all(w) if kind == "all" else orc.any(w)), ctx
            if fres is not None:
                kept = orc.filter(want[filt[0]], want[filt[1]])
                cnt = c.get(fres[1])
                assert cnt == kept.size, (mode, seed, "filter count", cnt, kept.size)
                assert bits_equal(c.read_vec(fres[0], kept.dtype, cnt), kept), (mode, seed, "filter output", steps)
                check_sum(c.get(fres[2]), kept, tol, (mode, seed, "kept sum"))
            results[mode] = scal
    # fused and unfused plans of the same DAG: exact results are the same bits (sums only within the tolerance: another order)
    for (kind, _, _), a, b in zip(reds, results["fused"], results.get("unfused", results["fused"])):
        if kind != "sum" or np.dtype(dtype).kind != "f":
            assert a == b or (a != a and b != b), (seed, kind, a, b)


# ----------------------------------------------------------------------------------------------------------------------------------
# the same on the matrix domain: ROW-/COL-broadcast vector operands, per-row / per-column / whole-matrix
# reductions, in-place results, padded leading dimensions, odd shapes — the 2-D plan builder and pass2d_bytecode
# ----------------------------------------------------------------------------------------------------------------------------------
SHAPES = [(1, 1), (3, 5), (33, 65), (64, 130), (130, 257), (7, 1027), (257, 3)]
AXES = {"all": sg.SG_AXIS_ALL, "rows": sg.SG_AXIS_ROWS, "cols": sg.SG_AXIS_COLS}


def _ew(fn, *arrays):
    """An elementwise oracle primitive applied to matrices: the oracle sees the flattened elements, numpy only moves data."""
    shape = arrays[0].shape
    return fn(*[np.ascontiguousarray(a).reshape(-1) for a in arrays]).reshape(shape)


def _axis_reduce(fn, M, axis):
    if axis == "all":
        return fn(np.ascontiguousarray(M).reshape(-1))
    if axis == "rows":
        return [fn(np.ascontiguousarray(M[r])) for r in range(M.shape[0])]
    return [fn(np.ascontiguousarray(M[:, cc])) for cc in range(M.shape[1])]


def build_matrix_dag(rng, dtype, mats, v, w):
    """Like build_dag on rows x cols values.  Operands of a binary step: ("m", id) a matrix value, ("row",) the ROW-broadcast vector v,
    ("col",) the COL-broadcast vector w, ("imm", x), or ("axis", kind, axis, id): an exact per-row / per-column reduction of a matrix
    value, pending in the same flush, broadcast back along the other axis."""
    is_f = np.dtype(dtype).kind == "f"
    shape = mats[0].shape
    want = dict(enumerate(mats))
    n_in = len(mats)
    vals, bools, steps, reds = list(range(n_in)), [], [], []
    storage = set(range(n_in))
    nid = n_in

    def operand():
        q = rng.random()
        if q < 0.50:
            k = int(rng.choice(vals))
            return ("m", k), want[k]
        if q < 0.65:
            return ("row",), np.ascontiguousarray(np.broadcast_to(v, shape))
        if q < 0.80:
            return ("col",), np.ascontiguousarray(np.broadcast_to(w[:, None], shape))
        if q < 0.90:
            k = int(rng.choice(vals))
            if not (is_f and np.isnan(want[k]).any()):
                kind = str(rng.choice(["max", "min"] + (["sum"] if np.dtype(dtype) == np.dtype(np.int64) else [])))
                axis = str(rng.choice(["rows", "cols"]))
                vec = np.array(_axis_reduce({"max": orc.max, "min": orc.min, "sum": orc.sum}[kind], want[k], axis), dtype=dtype)
                full = np.broadcast_to(vec[:, None], shape) if axis == "rows" else np.broadcast_to(vec, shape)
                return ("axis", kind, axis, k), np.ascontiguousarray(full)
        imm = float(rng.choice([0.5, 2.0, -3.25, 7.0])) if is_f else int(rng.choice([2, 3, 7, -5, 1]))
        return ("imm", imm), imm

    for _ in range(int(rng.integers(3, 11))):
        r = rng.random()
        if r < 0.50 or not (bools or r < 0.85):
            op = str(rng.choice(list(BIN) if not is_f else [k for k in BIN if k != "mod"]))
            a = int(rng.choice(vals))
            (bk, bv), swap = operand(), bool(rng.random() < 0.3)
            if bk[0] == "imm":
                res = _ew(lambda x: orc.scalar(op, x, bv, reversed=swap), want[a])
            else:
                res = _ew(lambda x, y: orc.zip(op, y, x) if swap else orc.zip(op, x, y), want[a], bv)
            if rng.random() < 0.12:
                k = int(rng.choice(sorted(storage)))
                steps.append(("inplace", op, a, bk, swap, k, nid))
                vals.remove(k); storage.discard(k); storage.add(nid)
            else:
                steps.append(("bin", op, a, bk, swap, nid))
            want[nid] = res
            vals.append(nid)
        elif r < 0.62:
            op = str(rng.choice(["neg", "abs"] + (["sqrt"] if is_f else [])))
            a = int(rng.choice(vals))
            steps.append(("un", op, a, nid))
            want[nid] = _ew(lambda x: orc.unary(op, x), want[a])
            vals.append(nid)
        elif r < 0.85:
            op = str(rng.choice(list(CMP)))
            a = int(rng.choice(vals))
            bk, bv = operand()
            steps.append(("cmp", op, a, bk, nid))
            want[nid] = _ew(lambda x: orc.cmp_scalar(op, x, bv), want[a]) if bk[0] == "imm" else _ew(lambda x, y: orc.cmp(op, x, y), want[a], bv)
            bools.append(nid)
        else:
            op = str(rng.choice(list(LOGIC)))
            a = int(rng.choice(bools))
            b = int(rng.choice(bools)) if op != "not" else -1
            steps.append(("logic", op, a, b, nid))
            want[nid] = _ew(lambda x, y: orc.logic(op, x, y), want[a], want[b]) if b >= 0 else _ew(lambda x: orc.logic(op, x), want[a])
            bools.append(nid)
        nid += 1
    produced_v = [k for k in vals if k >= n_in and k not in storage]
    keep = set(int(x) for x in rng.choice(produced_v, min(len(produced_v), int(rng.integers(0, 3))), replace=False)) if produced_v else set()
    if bools and rng.random() < 0.3:
        keep.add(int(rng.choice(bools)))
    for _ in range(int(rng.integers(1, 4))):
        reds.append((str(rng.choice(["sum", "max", "min"])), str(rng.choice(list(AXES))), int(rng.choice(vals))))
    for _ in range(int(rng.integers(0, 3))):
        if bools:
            reds.append(("count", str(rng.choice(list(AXES))), int(rng.choice(bools))))
    return steps, keep, reds, want, storage


@pytest.mark.parametrize("seed", range(160 * FUZZ))
def test_random_matrix_chains_match_the_oracle(seed):
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(9000 + seed)
    dtype = DTYPES[seed % 4]
    rows, cols = SHAPES[(seed // 4) % len(SHAPES)]
    is_f = np.dtype(dtype).kind == "f"
    sgdt = NP2SG[np.dtype(dtype)]
    mats = [make_input(rng, dtype, rows * cols).reshape(rows, cols) for _ in range(int(rng.integers(1, 3)))]
    v, w = make_input(rng, dtype, cols), make_input(rng, dtype, rows)
    lds = [cols + int(rng.choice([0, 0, 1, 3])) for _ in mats]
    steps, keep, reds, want, storage = build_matrix_dag(rng, dtype, mats, v, w)
    tol = {np.float32: 1e-5, np.float64: 1e-12}.get(dtype, 0)
    pad_value = dtype(7)
    for mode, flags in (("fused", 0), ("unfused", sg.SG_FLAG_UNFUSED)):
        with Ctx(flags) as c:
            bufs = []
            for M, ld in zip(mats, lds):
                b = np.full((rows, ld), pad_value, dtype=dtype)
                b[:, :cols] = M
                bufs.append(dev(b))
            tv, tw = dev(v), dev(w)
            c.keep += bufs + [tv, tw]
            h = {i: sg.sg_mat_create(c.ctx, sgdt, rows, cols, lds[i], bufs[i].data_ptr()) for i in range(len(mats))}
            buf_of = {i: i for i in range(len(mats))}              # storage id -> caller buffer
            hv, hw = sg.sg_vec_create(c.ctx, sgdt, cols, tv.data_ptr()), sg.sg_vec_create(c.ctx, sgdt, rows, tw.data_ptr())
            imm = (lambda x: sg.F(x)) if is_f else (lambda x: sg.I(x))
            borrowed, extra = set(h), []

            def opd(bk):
                if bk[0] == "m":
                    return h[bk[1]]
                if bk[0] == "row":
                    return sg.H(hv, sg.SG_BCAST_ROW)
                if bk[0] == "col":
                    return sg.H(hw, sg.SG_BCAST_COL)
                if bk[0] == "axis":
                    red = sg.sg_reduce(c.ctx, h[bk[3]], RED[bk[1]], AXES[bk[2]])
                    extra.append(red)
                    return sg.H(red, sg.SG_BCAST_COL if bk[2] == "rows" else sg.SG_BCAST_ROW)
                return imm(bk[1])
            try:
                for st in steps:
                    if st[0] in ("bin", "inplace"):
                        ops = [h[st[2]], opd(st[3])]
                        if st[4]:
                            ops.reverse()
                        if st[0] == "bin":
                            h[st[5]] = sg.sg_enqueue(c.ctx, BIN[st[1]], ops)
                        else:
                            h[st[6]] = sg.sg_enqueue(c.ctx, BIN[st[1]], ops, dst_or_0=h[st[5]])
                            borrowed.add(st[6])
                            buf_of[st[6]] = buf_of[st[5]]
                    elif st[0] == "un":
                        h[st[3]] = sg.sg_enqueue(c.ctx, UN[st[1]], [h[st[2]]])
                    elif st[0] == "cmp":
                        h[st[4]] = sg.sg_enqueue(c.ctx, CMP[st[1]], [h[st[2]], opd(st[3])])
                    else:
                        h[st[4]] = sg.sg_enqueue(c.ctx, LOGIC[st[1]], [h[st[2]]] + ([h[st[3]]] if st[3] >= 0 else []))
                rh = [sg.sg_reduce(c.ctx, h[src], sg.SG_COUNT if kind == "count" else RED[kind], AXES[axis]) for kind, axis, src in reds]
                for i, hx in h.items():
                    if i not in borrowed and i not in keep:
                        sg.sg_release(c.ctx, hx)
                sg.sg_flush(c.ctx)
            except sg.SgError as e:
                if mode == "unfused" and e.status == sg.SG_ERR_CAPACITY:    # more than 256 passes in one flush
                    continue
                raise
            for i in sorted(keep):
                got = c.read_vec(h[i], want[i].dtype, rows * cols).reshape(rows, cols)
                assert bits_equal(got, want[i]), (mode, seed, "kept matrix", i, steps)
            c.torch.cuda.synchronize()
            for i in sorted(storage):
                full = bufs[buf_of[i]].cpu().numpy()
                assert bits_equal(np.ascontiguousarray(full[:, :cols]), want[i]), (mode, seed, "caller matrix", i, steps)
                assert (full[:, cols:] == pad_value).all(), (mode, seed, "padding touched", i)
            for (kind, axis, src), r in zip(reds, rh):
                M = want[src]
                ctx = (mode, seed, kind, axis, steps)
                out_dt = np.int64 if kind == "count" or (kind == "sum" and not is_f) else np.float64 if kind == "sum" else dtype
                got = np.array([c.get(r)], dtype=out_dt) if axis == "all" else c.read_vec(r, out_dt, rows if axis == "rows" else cols)
                if kind == "count":
                    assert got.tolist() == np.atleast_1d(_axis_reduce(orc.count, M, axis)).tolist(), ctx
                elif kind == "sum":
                    ws = np.atleast_1d(_axis_reduce(orc.sum, M, axis))
                    if not is_f:
                        assert got.tolist() == ws.tolist(), ctx
                    else:
                        sabs = np.atleast_1d(_axis_reduce(lambda x: float(np.abs(x.astype(np.float64)).sum()), M, axis))
                        for gvv, wv, sa in zip(got, ws, sabs):
                            if np.isfinite(wv):
                                assert rel_err(float(gvv), float(wv), sa) <= tol, (ctx, gvv, wv)
                            else:
                                assert (np.isnan(wv) and np.isnan(gvv)) or wv == gvv, (ctx, gvv, wv)
                else:
                    ext = orc.max if kind == "max" else orc.min
                    ok = bits_equal(got, np.atleast_1d(np.array(_axis_reduce(ext, M, axis), dtype=dtype)))
                    if not ok and is_f and np.isnan(M).any():          # the sign of a generated NaN is the hardware's (R15)
                        for sgn in (1.0, -1.0):
                            Ms = np.where(np.isnan(M), np.copysign(np.nan, sgn), M).astype(M.dtype)
                            ok = ok or bits_equal(got, np.atleast_1d(np.array(_axis_reduce(ext, Ms, axis), dtype=dtype)))
                    assert ok, (ctx, got[:8])


# ----------------------------------------------------------------------------------------------------------------------------------
# memory hazards: random programs over OVERLAPPING views (subset) of two buffers with in-place updates.  The
# deferred list must behave like eager execution in program order (a pending reader sees the contents as of its enqueue; RAW / WAR /
# WAW through overlapping storage order the passes, sg_plan.cpp) — the oracle IS eager execution on numpy views, one primitive at a time.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(200 * FUZZ))
def test_random_view_programs_match_eager_execution(seed):
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(20000 + seed)
    dtype = [np.float64, np.int32, np.float32, np.int64][seed % 4]
    is_f = np.dtype(dtype).kind == "f"
    n = int([40, 3000, 70001][(seed // 4) % 3])
    L = n // 3
    host = [make_input(rng, dtype, n) for _ in range(2)]
    views = []
    for _ in range(int(rng.integers(3, 7))):
        if views and rng.random() < 0.25:
            views.append(views[int(rng.integers(0, len(views)))])             # the very same view again
        else:
            s = int(rng.integers(0, n - L + 1))
            if rng.random() < 0.3:
                s = s // 4 * 4                                                # some 16-byte aligned starts
            views.append((int(rng.integers(0, 2)), s))
    overlap = lambda p, q: p[0] == q[0] and abs(p[1] - q[1]) < L
    imm = (lambda x: sg.F(x)) if is_f else (lambda x: sg.I(x))
    for mode, flags in (("fused", 0), ("unfused", sg.SG_FLAG_UNFUSED)):
        mem = [a.copy() for a in host]
        prog_rng = np.random.default_rng(30000 + seed)                        # the same program in both modes
        with Ctx(flags) as c:
            bufs = [dev(a) for a in host]
            c.keep += bufs
            hb = [sg.sg_vec_create(c.ctx, NP2SG[np.dtype(dtype)], n, t.data_ptr()) for t in bufs]
            hv = [sg.sg_vec_subset(c.ctx, hb[b], s, s + L) for b, s in views]
            cur = lambda k: mem[views[k][0]][views[k][1]:views[k][1] + L].copy()
            temps, kept, trace = [], [], []                                   # temps: (handle, eager value)
            try:
                for _ in range(int(prog_rng.integers(5, 13))):
                    op = str(prog_rng.choice(["add", "sub", "mul", "max", "min"]))
                    dst = int(prog_rng.integers(0, len(views))) if prog_rng.random() < 0.45 else -1

                    def pick():
                        q = prog_rng.random()
                        if q < 0.2:
                            x = float(prog_rng.choice([0.5, 2.0, -1.0])) if is_f else int(prog_rng.choice([2, 3, -1]))
                            return imm(x), x, None
                        if q < 0.45 and temps:
                            t = temps[int(prog_rng.integers(0, len(temps)))]
                            return t[0], t[1], None
                        for _ in range(20):
                            k = int(prog_rng.integers(0, len(views)))
                            # an in-place result may read its destination only index-for-index: the same view, or one that does not overlap
                            if dst < 0 or views[k] == views[dst] or not overlap(views[k], views[dst]):
                                return hv[k], cur(k), k
                        return hv[dst], cur(dst), dst
                    (ha, va, _), (hb2, vb, _) = pick(), pick()
                    if not isinstance(va, np.ndarray) and not isinstance(vb, np.ndarray):
                        ha, va = hv[dst if dst >= 0 else 0], cur(dst if dst >= 0 else 0)     # at least one collection operand
                    if isinstance(va, np.ndarray) and isinstance(vb, np.ndarray):
                        res = orc.zip(op, va, vb)
                    elif isinstance(va, np.ndarray):
                        res = orc.scalar(op, va, vb)
                    else:
                        res = orc.scalar(op, vb, va, reversed=True)
                    trace.append((op, dst))
                    if dst >= 0:
                        sg.sg_enqueue(c.ctx, BIN[op], [ha, hb2], dst_or_0=hv[dst])
                        b, s = views[dst]
                        mem[b][s:s + L] = res
                    else:
                        temps.append((sg.sg_enqueue(c.ctx, BIN[op], [ha, hb2]), res))
                for t in temps:
                    if prog_rng.random() < 0.5:
                        kept.append(t)
                    else:
                        sg.sg_release(c.ctx, t[0])
                red = [(sg.sg_reduce(c.ctx, hv[k], sg.SG_RMAX), sg.sg_reduce(c.ctx, hv[k], sg.SG_SUM), cur(k)) for k in range(min(2, len(views)))]
                sg.sg_flush(c.ctx)
            except sg.SgError as e:
                if mode == "unfused" and e.status == sg.SG_ERR_CAPACITY:      # more than 256 passes in one flush
                    continue
                raise
            for th, tv in kept:
                assert bits_equal(c.read_vec(th, dtype), tv), (mode, seed, "kept temporary", trace, views)
            for hm, hs, val in red:
                assert bits_equal(np.array([c.get(hm)], dtype=dtype), np.array([orc.max(val)], dtype=dtype)), (mode, seed, "max of a view", trace, views)
                check_sum(c.get(hs), val, 1e-12 if dtype is np.float64 else 1e-5, (mode, seed, "sum of a view"))
            c.torch.cuda.synchronize()
            for b in range(2):
                assert bits_equal(bufs[b].cpu().numpy(), mem[b]), (mode, seed, "buffer", b, trace, views)


# ----------------------------------------------------------------------------------------------------------------------------------
# Listing 5's way of working: ROW views of one matrix updated in place with other rows, immediates, element views
# (the pivot, sg_mat_elem) and pending scalars, mixed with whole-matrix and row-block updates through other handles of the same
# storage.  The oracle is eager execution on a numpy matrix, one primitive at a time.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(160 * FUZZ))
def test_random_row_programs_match_eager_execution(seed):
    from gpu_util import NP2SG, dev
    dtype = [np.float64, np.int64, np.float32, np.int32][seed % 4]
    is_f = np.dtype(dtype).kind == "f"
    rows, cols = [(6, 17), (9, 130), (5, 1027), (12, 64)][(seed // 4) % 4]
    rng = np.random.default_rng(40000 + seed)
    ld = cols + int(rng.choice([0, 0, 1, 2]))
    pad = dtype(9)
    host = np.full((rows, ld), pad, dtype=dtype)
    host[:, :cols] = make_input(rng, dtype, rows * cols).reshape(rows, cols)
    imm = (lambda x: sg.F(x)) if is_f else (lambda x: sg.I(x))
    pick_imm = lambda r: float(r.choice([0.5, 2.0, -1.0])) if is_f else int(r.choice([2, 3, -1]))
    for mode, flags in (("fused", 0), ("unfused", sg.SG_FLAG_UNFUSED)):
        mem = host.copy()
        pr = np.random.default_rng(50000 + seed)
        trace = []
        with Ctx(flags) as c:
            tM = dev(host)
            c.keep.append(tM)
            hM = sg.sg_mat_create(c.ctx, NP2SG[np.dtype(dtype)], rows, cols, ld, tM.data_ptr())
            rowh = {}

            def row(i):
                if i not in rowh:
                    rowh[i] = sg.sg_mat_row(c.ctx, hM, i)
                return rowh[i]
            cur = lambda i: mem[i, :cols].copy()
            temps, kept, ctemps = [], [], []
            try:
                for _ in range(int(pr.integers(6, 15))):
                    op = str(pr.choice(["add", "sub", "mul", "max", "min"]))
                    i, j = int(pr.integers(0, rows)), int(pr.integers(0, rows))
                    q = pr.random()
                    if q < 0.25:                                                    # r_i := r_i op r_j
                        sg.sg_enqueue(c.ctx, BIN[op], [row(i), row(j)], dst_or_0=row(i))
                        mem[i, :cols] = orc.zip(op, cur(i), cur(j))
                        trace.append(("row", op, i, j))
                    elif q < 0.35:                                                  # r_i := imm op r_i
                        x = pick_imm(pr)
                        sg.sg_enqueue(c.ctx, BIN[op], [imm(x), row(i)], dst_or_0=row(i))
                        mem[i, :cols] = orc.scalar(op, cur(i), x, reversed=True)
                        trace.append(("row_imm", op, i, x))
                    elif q < 0.50 and rows > 1:                                     # r_i := r_i op M[a, b], the element read where it lies NOW
                        a = int(pr.choice([k for k in range(rows) if k != i]))
                        b = int(pr.integers(0, cols))
                        e = sg.sg_mat_elem(c.ctx, hM, a, b)
                        sg.sg_enqueue(c.ctx, BIN[op], [row(i), e], dst_or_0=row(i))
                        mem[i, :cols] = orc.scalar(op, cur(i), mem[a, b].item())
                        sg.sg_release(c.ctx, e)
                        trace.append(("row_elem", op, i, a, b))
                    elif q < 0.62:                                                  # r_j := r_j op max(r_i): a pending scalar
                        s = sg.sg_reduce(c.ctx, row(i), sg.SG_RMAX)
                        sval = orc.max(cur(i))
                        sg.sg_enqueue(c.ctx, BIN[op], [row(j), s], dst_or_0=row(j))
                        mem[j, :cols] = orc.scalar(op, cur(j), float(sval) if is_f else int(sval))
                        sg.sg_release(c.ctx, s)
                        trace.append(("row_max", op, j, i))
                    elif q < 0.68:                                                  # t = r_i op r_j
                        temps.append((sg.sg_enqueue(c.ctx, BIN[op], [row(i), row(j)]), orc.zip(op, cur(i), cur(j))))
                        trace.append(("temp", op, i, j))
                    elif q < 0.74:                                                  # t = column(a)[r0:r1] op column(b)[r0:r1]: deferred strided copies
                        r0 = int(pr.integers(0, rows))
                        r1 = int(pr.integers(r0 + 1, rows + 1))
                        a, b = int(pr.integers(0, cols)), int(pr.integers(0, cols))
                        ca, cb = sg.sg_mat_col(c.ctx, hM, a, r0, r1), sg.sg_mat_col(c.ctx, hM, b, r0, r1)
                        ctemps.append((sg.sg_enqueue(c.ctx, BIN[op], [ca, cb]), orc.zip(op, np.ascontiguousarray(mem[r0:r1, a]), np.ascontiguousarray(mem[r0:r1, b]))))
                        if pr.random() < 0.5:
                            ctemps.append((ca, np.ascontiguousarray(mem[r0:r1, a]).copy()))
                        else:
                            sg.sg_release(c.ctx, ca)
                        sg.sg_release(c.ctx, cb)
                        trace.append(("cols", op, a, b, r0, r1))
                    elif q < 0.84 and temps:                                        # r_i := t op r_i
                        t = temps[int(pr.integers(0, len(temps)))]
                        sg.sg_enqueue(c.ctx, BIN[op], [t[0], row(i)], dst_or_0=row(i))
                        mem[i, :cols] = orc.zip(op, t[1], cur(i))
                        trace.append(("row_temp", op, i))
                    elif q < 0.92:                                                  # M := M op imm, through the matrix handle
                        x = pick_imm(pr)
                        sg.sg_enqueue(c.ctx, BIN[op], [hM, imm(x)], dst_or_0=hM)
                        mem[:, :cols] = orc.scalar(op, np.ascontiguousarray(mem[:, :cols]).reshape(-1), x).reshape(rows, cols)
                        trace.append(("mat_imm", op, x))
                    elif rows > 2:                                                  # B := B op r_k along the rows of a row block, k outside it
                        r0 = int(pr.integers(0, rows - 1))
                        r1 = int(pr.integers(r0 + 1, rows))
                        k = int(pr.choice([k for k in range(rows) if k < r0 or k >= r1]))
                        hB = sg.sg_mat_rows(c.ctx, hM, r0, r1)
                        sg.sg_enqueue(c.ctx, BIN[op], [hB, sg.H(row(k), sg.SG_BCAST_ROW)], dst_or_0=hB)
                        blk = np.ascontiguousarray(mem[r0:r1, :cols])
                        mem[r0:r1, :cols] = orc.zip(op, blk.reshape(-1), np.ascontiguousarray(np.broadcast_to(cur(k), blk.shape)).reshape(-1)).reshape(blk.shape)
                        sg.sg_release(c.ctx, hB)
                        trace.append(("block", op, r0, r1, k))
                for t in temps:
                    if pr.random() < 0.6:
                        kept.append(t)
                    else:
                        sg.sg_release(c.ctx, t[0])
                sg.sg_flush(c.ctx)
            except sg.SgError as e:
                if mode == "unfused" and e.status == sg.SG_ERR_CAPACITY:            # more than 256 passes in one flush
                    continue
                raise
            for th, tv in kept + ctemps:
                assert bits_equal(c.read_vec(th, dtype), tv), (mode, seed, "kept temporary", trace)
            c.torch.cuda.synchronize()
            assert bits_equal(tM.cpu().numpy(), mem), (mode, seed, "matrix", trace)


# ----------------------------------------------------------------------------------------------------------------------------------
# dtype-changing projections (R23): random programs that convert between the four element
# types (sg_cast, integer sqrt -> DOUBLE), compute in each type, and convert again — on misaligned subset views, into caller buffers,
# with reductions.  Every conversion is a pass boundary with a converting load (IN_VEC_CVT) of a stored operand.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(160 * FUZZ))
def test_random_cast_programs_match_the_oracle(seed):
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(60000 + seed)
    n = int([40, 3000, 70001][(seed // 4) % 3])
    L = n // 2
    base_dt = DTYPES[seed % 4]
    host = make_input(rng, base_dt, n)
    if np.dtype(base_dt).kind == "f":                        # values outside the integer ranges, halves, NaN and infinities: the conversion's edge cases
        host[rng.integers(0, n, max(1, n // 25))] = rng.choice(np.array([2.5, -2.5, 3e9, -3e9, 1e19, -1e19, 16777217.0, np.nan, np.inf, -np.inf], dtype=base_dt))
    else:
        host[rng.integers(0, n, max(1, n // 25))] = rng.choice(np.array([16777217, -16777217, 2147483647, -2147483648, 123456789], dtype=base_dt))
    starts = [int(rng.integers(0, n - L + 1)) for _ in range(2)]
    for mode, flags in (("fused", 0), ("unfused", sg.SG_FLAG_UNFUSED)):
        pr = np.random.default_rng(70000 + seed)
        with Ctx(flags) as c:
            tb = dev(host)
            c.keep.append(tb)
            hb = sg.sg_vec_create(c.ctx, NP2SG[np.dtype(base_dt)], n, tb.data_ptr())
            vals = [(sg.sg_vec_subset(c.ctx, hb, s, s + L), host[s:s + L].copy()) for s in starts]      # (handle, oracle value)
            borrowed = len(vals)
            outs, trace = [], []                                 # caller buffers written by converting in place: (tensor, want)
            try:
                for _ in range(int(pr.integers(4, 11))):
                    h, v = vals[int(pr.integers(0, len(vals)))]
                    q = pr.random()
                    if q < 0.45:                                 # convert to another element type (sometimes straight into a caller buffer)
                        to = DTYPES[int(pr.integers(0, 4))]
                        w = orc.cast(v, to)
                        if pr.random() < 0.25:
                            off = int(pr.integers(0, 4))
                            t = dev(np.zeros(L + 8, dtype=to))
                            c.keep.append(t)
                            hd = sg.sg_vec_subset(c.ctx, sg.sg_vec_create(c.ctx, NP2SG[np.dtype(to)], L + 8, t.data_ptr()), off, off + L)
                            vals.append((sg.sg_cast(c.ctx, h, NP2SG[np.dtype(to)], hd), w))
                            outs.append((t, off, w))
                        else:
                            vals.append((sg.sg_cast(c.ctx, h, NP2SG[np.dtype(to)]), w))
                        trace.append(("cast", v.dtype.name, np.dtype(to).name))
                    elif q < 0.60:                               # sqrt: an integer vector gives doubles (the paper's example)
                        vals.append((sg.sg_enqueue(c.ctx, sg.SG_SQRT, [h]), orc.project_sqrt(v)))
                        trace.append(("sqrt", v.dtype.name))
                    else:                                        # an operation inside one element type
                        same = [k for k, (_, x) in enumerate(vals) if x.dtype == v.dtype]
                        h2, v2 = vals[int(pr.choice(same))]
                        op = str(pr.choice(["add", "sub", "mul", "max", "min"]))
                        vals.append((sg.sg_enqueue(c.ctx, BIN[op], [h, h2]), orc.zip(op, v, v2)))
                        trace.append((op, v.dtype.name))
                keep = [k for k in range(borrowed, len(vals)) if pr.random() < 0.5]
                red = [(sg.sg_reduce(c.ctx, vals[k][0], sg.SG_RMAX), sg.sg_reduce(c.ctx, vals[k][0], sg.SG_SUM), vals[k][1])
                       for k in pr.choice(len(vals), min(2, len(vals)), replace=False)]
                for k in range(borrowed, len(vals)):
                    if k not in keep and not any(vals[k][1] is w for _, _, w in outs):
                        sg.sg_release(c.ctx, vals[k][0])
                sg.sg_flush(c.ctx)
            except sg.SgError as e:
                if mode == "unfused" and e.status == sg.SG_ERR_CAPACITY:        # more than 256 passes in one flush
                    continue
                raise
            for k in keep:
                assert bits_equal(c.read_vec(vals[k][0], vals[k][1].dtype), vals[k][1]), (mode, seed, "kept value", k, trace)
            for hm, hs, v in red:
                cands = [orc.max(v)]
                if v.dtype.kind == "f" and np.isnan(v).any():
                    cands = [orc.max(np.where(np.isnan(v), np.copysign(np.nan, sgn), v).astype(v.dtype)) for sgn in (1.0, -1.0)]
                got = np.array([c.get(hm)], dtype=v.dtype)
                assert any(bits_equal(got, np.array([w], dtype=v.dtype)) for w in cands), (mode, seed, "max", got, cands, trace)
                check_sum(c.get(hs), v, 1e-12 if v.dtype == np.float64 else 1e-5, (mode, seed, "sum", trace))
            c.torch.cuda.synchronize()
            for t, off, w in outs:
                full = t.cpu().numpy()
                assert bits_equal(full[off:off + L], w) and not full[:off].any() and not full[off + L:].any(), (mode, seed, "caller buffer", trace)
            assert bits_equal(tb.cpu().numpy(), host), (mode, seed, "source modified")


# ----------------------------------------------------------------------------------------------------------------------------------
# contracts and the early exit (R19a): random sets of quantifiers over one vector, some registered as
# PRE / POST contracts, with and without a violation and with and without SG_FLAG_NO_EARLY_EXIT, next to a reduction body.
# Rules checked: the flush reports SG_ERR_CONTRACT exactly when a registered contract is false; a value that is handed back is the
# oracle's; "not evaluated" is only ever the answer for a quantifier that was not yet decided when a violated contract ended its pass.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(200 * FUZZ))
def test_random_contract_sets_follow_the_rules(seed):
    from gpu_util import NP2SG
    rng = np.random.default_rng(80000 + seed)
    dtype = [np.float32, np.float64, np.int32][seed % 3]
    is_f = np.dtype(dtype).kind == "f"
    n = int([33, 5000, 300007, (1 << 21) + 3][(seed // 3) % 4])
    x = np.sort(rng.integers(0, 1000, n)).astype(dtype)                      # ascending, many ties, values 0 .. 999
    if rng.random() < 0.6:                                                   # one or two planted breaks of the order / of the range
        for _ in range(int(rng.integers(1, 3))):
            j = int(rng.integers(0, n))
            x[j] = dtype(rng.choice([-5, 2000, 0, 500]))
    flags = sg.SG_FLAG_NO_EARLY_EXIT if rng.random() < 0.3 else 0
    imm = (lambda v: sg.F(float(v))) if is_f else (lambda v: sg.I(int(v)))
    with Ctx(flags) as c:
        hx = c.vec(x)
        quants = []                                                          # (handle, truth, kind, registered)
        for _ in range(int(rng.integers(2, 6))):
            q = rng.random()
            if q < 0.3:
                op = str(rng.choice(["le", "lt", "ge"]))
                h = sg.sg_forall_adjacent(c.ctx, hx, CMP[op])
                truth, kind = (bool(orc.all(orc.adj(op, x))) if n > 1 else True), "all"
            else:
                op, v = str(rng.choice(list(CMP))), int(rng.choice([-5, 0, 1, 500, 999, 1000, 2000]))
                m = sg.sg_enqueue(c.ctx, CMP[op], [hx, imm(v)])
                mask = orc.cmp_scalar(op, x, float(v) if is_f else v)
                if rng.random() < 0.5:
                    h, truth, kind = sg.sg_forall(c.ctx, m), bool(orc.all(mask)), "all"
                else:
                    h, truth, kind = sg.sg_exists(c.ctx, m), bool(orc.any(mask)), "any"
                sg.sg_release(c.ctx, m)
            reg = rng.random() < 0.5
            if reg:
                sg.sg_contract(c.ctx, h, sg.SG_CONTRACT_PRE if rng.random() < 0.5 else sg.SG_CONTRACT_POST, "q%d" % len(quants))
            quants.append((h, truth, kind, reg))
        body = sg.sg_reduce(c.ctx, hx, sg.SG_SUM) if rng.random() < 0.5 else None        # a reduction body in the same flush
        violated = [k for k, (_, truth, _, reg) in enumerate(quants) if reg and not truth]
        try:
            sg.sg_flush(c.ctx)
            raised = False
        except sg.SgError as e:
            assert e.status == sg.SG_ERR_CONTRACT, (seed, str(e))
            raised = True
        assert raised == bool(violated), (seed, "flush status", raised, violated)
        violated_all = [k for k in violated if quants[k][2] == "all"]       # only a violated for_all contract ends a pass early
        decided_violations = 0
        for k, (h, truth, kind, reg) in enumerate(quants):
            try:
                got = c.get(h)
            except sg.SgError as e:
                assert e.status == sg.SG_ERR_CONTRACT and "not evaluated" in str(e), (seed, k, str(e))
                assert violated_all and not flags, (seed, k, "not evaluated without an early exit")
                # an undecided quantifier reads for_all = true / exists = false so far: one that is false / true on the whole vector —
                # a SECOND violated contract whose violation lies further on, too — may still be undecided on the prefix
                continue
            assert got is truth, (seed, k, kind, got, truth)
            decided_violations += k in violated_all
        if violated_all and not flags:
            assert decided_violations >= 1, (seed, "the contract that ended the pass must be readable (and false)")
        if body is not None:
            check_sum(c.get(body), x, 1e-12 if dtype is np.float64 else 1e-5, (seed, "body sum"))


# ----------------------------------------------------------------------------------------------------------------------------------
# the filter's protocols (look-back over tile states, runs of tiles, the compaction ring, epoch-tagged states) under BURSTY masks:
# kept elements come in random runs (a two-state Markov chain with random switch probabilities: from almost nothing kept to long
# stretches where everything is kept, which fill the ring and shrink the runs), several launches of different lengths per context,
# misaligned views, all four element types, output into a caller buffer of exactly the needed capacity.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(120 * FUZZ))
def test_random_bursty_filters_match_the_oracle(seed):
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(90000 + seed)
    dtype = DTYPES[seed % 4]
    is_f = np.dtype(dtype).kind == "f"
    with Ctx() as c:
        for launch in range(int(rng.integers(2, 6))):
            n = int(rng.choice([1, 100, 8191, 8192, 8193, 70001, int(rng.integers(1, 3_000_000))]))
            p_on, p_off = 10.0 ** -rng.uniform(0.3, 4.5), 10.0 ** -rng.uniform(0.3, 4.5)
            # run lengths of the two states are geometric: build the pattern from run lengths (fast), trim to n
            runs, state, total = [], bool(rng.random() < 0.5), 0
            while total < n:
                ln = int(rng.geometric(p_off if state else p_on))
                runs.append((state, ln)); total += ln; state = not state
            pattern = np.concatenate([np.full(ln, st) for st, ln in runs])[:n]
            mag = rng.integers(1, 1000, n)
            x = np.where(pattern, mag, -mag).astype(dtype)
            off = int(rng.integers(0, 5))
            buf = np.zeros(n + 8, dtype=dtype)
            buf[off:off + n] = x
            t = dev(buf)
            c.keep.append(t)
            hx = sg.sg_vec_subset(c.ctx, sg.sg_vec_create(c.ctx, NP2SG[np.dtype(dtype)], n + 8, t.data_ptr()), off, off + n)
            m = sg.sg_enqueue(c.ctx, sg.SG_GT, [hx, sg.F(0.0) if is_f else sg.I(0)])
            want = orc.filter(x, orc.cmp_scalar("gt", x, 0.0 if is_f else 0))
            assert want.size == int(pattern.sum())
            if rng.random() < 0.5:                                   # into a caller buffer with exactly the capacity needed
                to = dev(np.full(want.size + 4, 77, dtype=dtype))
                c.keep.append(to)
                fv, fc = sg.sg_filter(c.ctx, hx, m, to.data_ptr(), want.size)
            else:
                to = None
                fv, fc = sg.sg_filter(c.ctx, hx, m)
            sg.sg_release(c.ctx, m)
            s, mx = sg.sg_reduce(c.ctx, fv, sg.SG_SUM), (sg.sg_reduce(c.ctx, fv, sg.SG_RMAX) if want.size else None)
            cnt = c.get(fc)
            ctx = (seed, launch, n, np.dtype(dtype).name, float(p_on), float(p_off))
            assert cnt == want.size, (ctx, cnt, want.size)
            assert bits_equal(c.read_vec(fv, dtype, cnt), want), ctx
            check_sum(c.get(s), want, 1e-12 if dtype is np.float64 else 1e-5, ctx)
            if mx is not None:
                assert dtype(c.get(mx)) == orc.max(want), ctx
            if to is not None:
                c.torch.cuda.synchronize()
                assert (to.cpu().numpy()[want.size:] == 77).all(), (ctx, "wrote past the capacity")
            for h in (fv, fc, s) + ((mx,) if mx is not None else ()):
                sg.sg_release(c.ctx, h)


@pytest.mark.parametrize("seed", range(60 * FUZZ))
def test_random_bursty_filters_through_the_template_instance(seed):
    """The same bursty masks through config 2's own chain (x mod 7 == 3, count, kept-sum: the TEMPLATE filter kernel with its TMA
    stages, look-back warp and compaction ring), several launches of different lengths in one context."""
    from paper_1410_6685_b200 import workloads as W
    from gpu_util import dev
    rng = np.random.default_rng(95000 + seed)
    with Ctx() as c:
        for launch in range(int(rng.integers(2, 6))):
            n = int(rng.choice([8192, 70001, 1 << 20, int(rng.integers(1, 6_000_000))]))
            p_on, p_off = 10.0 ** -rng.uniform(0.3, 5.0), 10.0 ** -rng.uniform(0.3, 5.0)
            runs, state, total = [], bool(rng.random() < 0.5), 0
            while total < n:
                ln = int(rng.geometric(p_off if state else p_on))
                runs.append((state, ln)); total += ln; state = not state
            pattern = np.concatenate([np.full(ln, st) for st, ln in runs])[:n]
            k = rng.integers(0, 1 << 27, n)
            x = (7 * k + np.where(pattern, 3, rng.choice([0, 1, 2, 4, 5, 6], n))).astype(np.int32)
            t = dev(x)
            c.keep.append(t)
            want = orc.filter(x, orc.cmp_scalar("eq", orc.scalar("mod", x, 7), 3))
            assert want.size == int(pattern.sum())
            to = None
            if rng.random() < 0.5:
                to = dev(np.full(want.size + 4, 77, dtype=np.int32))
                c.keep.append(to)
            r = W.cfg2(c.ctx, n, t.data_ptr(), to.data_ptr() if to is not None else None, want.size if to is not None else 0)
            cnt = c.get(r["count"])
            ctx = (seed, launch, n, float(p_on), float(p_off))
            assert sg.sg_plan_stats(c.ctx).n_template == 1, ctx
            assert cnt == want.size, (ctx, cnt, want.size)
            assert bits_equal(c.read_vec(r["kept"], np.int32, cnt), want), ctx
            assert c.get(r["sum"]) == orc.sum(want), ctx
            if to is not None:
                c.torch.cuda.synchronize()
                assert (to.cpu().numpy()[want.size:] == 77).all(), (ctx, "wrote past the capacity")
            for h in r.values():
                sg.sg_release(c.ctx, h)


# ----------------------------------------------------------------------------------------------------------------------------------
# the TEMPLATE matrix kernels and the movers on random shapes: config 4's step (staged pass with row maxima and column sums), the
# matrix-vector products, transpose (incl. the pair kernel of 4-byte elements) — any rows / columns / leading dimensions / pivot.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(60 * FUZZ))
def test_random_shapes_through_the_matrix_templates(seed):
    from oracle import configs as ocfg
    from paper_1410_6685_b200 import inputs, workloads as W
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(97000 + seed)
    # config 4's step
    n = int(rng.choice([int(rng.integers(2, 70)), int(rng.integers(70, 600)), int(rng.integers(600, 2300))]))
    k = int(rng.integers(0, n))
    ld = n + int(rng.choice([0, 0, 1, 2, 5]))
    M = inputs.boosted_matrix_f64(int(rng.integers(1, 1000)), 0, n)
    want = ocfg.cfg4(M, k)
    with Ctx() as c:
        buf = np.full((n, ld), 7.25)
        buf[:, :n] = M
        t = dev(buf)
        c.keep.append(t)
        r = W.cfg4(c.ctx, n, t.data_ptr(), k, ld=ld)
        sg.sg_flush(c.ctx)
        c.torch.cuda.synchronize()
        full = t.cpu().numpy()
        assert bits_equal(np.ascontiguousarray(full[:, :n]), want["M"]) and (full[:, n:] == 7.25).all(), (seed, "cfg4", n, k, ld)
        if k + 1 < n:
            assert bits_equal(c.read_vec(r["rowmax"], np.float64), want["rowmax"]), (seed, "rowmax", n, k, ld)
            cs, scale = c.read_vec(r["colsum"], np.float64), np.abs(want["M"][k + 1:]).sum(axis=0)
            assert np.all(np.abs(cs - want["colsum"]) <= 1e-12 * np.maximum(np.abs(want["colsum"]), 1e-300) + 2.0 ** -64 * scale), (seed, "colsum", n, k, ld)
    # matrix-vector products, exact in the integer regime
    rows, cols = int(rng.integers(1, 1500)), int(rng.integers(1, 1500))
    ld = cols + int(rng.choice([0, 0, 1, 3]))
    A = rng.integers(-8, 9, (rows, cols)).astype(np.float64)
    v, w = rng.integers(-8, 9, cols).astype(np.float64), rng.integers(-8, 9, rows).astype(np.float64)
    with Ctx() as c:
        Ap = np.zeros((rows, ld))
        Ap[:, :cols] = A
        tA, tv, tw = dev(Ap), dev(v), dev(w)
        c.keep += [tA, tv, tw]
        r = W.right_multiply(c.ctx, rows, cols, tA.data_ptr(), tv.data_ptr(), ld)
        sg.sg_flush(c.ctx)
        l = W.left_multiply(c.ctx, rows, cols, tw.data_ptr(), tA.data_ptr(), ld)
        got_r, got_l = c.read_vec(r["out"], np.float64, rows), c.read_vec(l["out"], np.float64, cols)
        assert bits_equal(got_r, ocfg.right_multiply(A, v)) and bits_equal(got_l, ocfg.left_multiply(w, A)), (seed, "matvec", rows, cols, ld)
    # transpose, every element type
    dtype = DTYPES[seed % 4]
    rows, cols = int(rng.integers(1, 700)), int(rng.integers(1, 700))
    ld, ldo = cols + int(rng.choice([0, 0, 1, 2, 6])), rows + int(rng.choice([0, 0, 1, 2, 6]))
    B = rng.integers(-10**6, 10**6, (rows, cols)).astype(dtype)
    with Ctx() as c:
        Bp = np.full((rows, ld), -7, dtype=dtype)
        Bp[:, :cols] = B
        tB, tout = dev(Bp), dev(np.full((cols, ldo), -9, dtype=dtype))
        c.keep += [tB, tout]
        W.transpose(c.ctx, NP2SG[np.dtype(dtype)], rows, cols, tB.data_ptr(), tout.data_ptr(), ld, ldo)
        c.torch.cuda.synchronize()
        got = tout.cpu().numpy()
        assert bits_equal(np.ascontiguousarray(got[:, :rows]), ocfg.transpose(B)) and np.all(got[:, rows:] == -9), (seed, "transpose", rows, cols, ld, ldo)


# ----------------------------------------------------------------------------------------------------------------------------------
# Listing 5's determinant loop (one persistent kernel) and Listing 3's quicksort (one launch per recursion level) on random inputs:
# random orders and leading dimensions, planted rank deficiencies, exact zeros below pivots, eps = 0 and eps > 0, the loop split
# over two calls; keys with few distinct values, runs, signed zeros, every element type.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(40 * FUZZ))
def test_random_determinants_and_sorts_match_the_oracle(seed):
    from oracle import configs as ocfg
    from paper_1410_6685_b200 import inputs, workloads as W
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(98000 + seed)
    n = int(rng.choice([int(rng.integers(1, 40)), int(rng.integers(40, 330)), int(rng.integers(330, 700))]))
    ld = n + int(rng.choice([0, 0, 1, 3]))
    M = inputs.boosted_matrix_f64(int(rng.integers(1, 1000)), 0, n) / float(n)
    eps = float(rng.choice([0.0, 0.0, 1e-12, 1e-6]))
    q = rng.random()
    if q < 0.3 and n > 3:                                           # rank deficient: one row a combination of two others
        i, j, k = (int(x) for x in rng.choice(n, 3, replace=False))
        M[i] = 0.5 * M[j] + 0.25 * M[k]
    elif q < 0.6 and n > 2:                                         # exact zeros strewn about (guarded rows), a clean diagonal
        M[rng.integers(0, n, 2 * n), rng.integers(0, n, 2 * n)] = 0.0
        M[np.arange(n), np.arange(n)] = 1.0 + np.arange(n) / n
    want_det, want_E, zs = orc.ge_determinant(M, eps=eps)
    with Ctx() as c:
        buf = np.zeros((n, ld))
        buf[:, :n] = M
        t = dev(buf)
        det, minpiv = c.torch.ones(1, dtype=c.torch.float64, device="cuda"), c.torch.full((1,), float("inf"), dtype=c.torch.float64, device="cuda")
        c.keep += [t, det, minpiv]
        got, ok = W.ge_determinant(c.ctx, n, t.data_ptr(), det.data_ptr(), minpiv.data_ptr(), ld=ld, eps=eps)
        E = t.cpu().numpy()
        ctx = (seed, "determinant", n, ld, eps, zs)
        assert ok == (zs < 0), ctx
        assert bits_equal(np.array([got]), np.array([want_det])), (ctx, got, want_det)
        assert bits_equal(np.ascontiguousarray(E[:, :n]), want_E) and not E[:, n:].any(), ctx
    # quicksort
    dtype = DTYPES[seed % 4]
    m = int(rng.choice([int(rng.integers(1, 3000)), int(rng.integers(3000, 60000))]))
    style = int(rng.integers(0, 5))
    if style == 0:
        keys = rng.integers(-5, 6, m)                               # few distinct keys
    elif style == 1:
        keys = np.repeat(rng.integers(-1000, 1000, m // 50 + 1), 50)[:m]      # runs of equal keys
    elif style == 2:
        keys = np.sort(rng.integers(-10**6, 10**6, m))[::int(rng.choice([1, -1]))]      # sorted / reversed
    else:
        keys = rng.integers(-10**6, 10**6, m)
    keys = keys.astype(dtype)
    if np.dtype(dtype).kind == "f" and m > 4:
        keys[rng.integers(0, m, max(1, m // 10))] = rng.choice(np.array([0.0, -0.0], dtype=dtype))     # signed zeros: equal keys, stable order
    want = ocfg.quicksort(keys)
    with Ctx() as c:
        hk = c.vec(keys)
        out = sg.sg_vec_quicksort(c.ctx, hk)
        got = c.read_vec(out, dtype)
    assert bits_equal(got, want), (seed, "quicksort", np.dtype(dtype).name, m, style)


# ----------------------------------------------------------------------------------------------------------------------------------
# the plan cache: the same random program enqueued again over the same buffers takes its pass assignment from the
# cache (a hit) — every round's results must still be the oracle's, with the cache and with SG_FLAG_NO_PLAN_CACHE.
# ----------------------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(120 * FUZZ))
def test_random_chains_replayed_through_the_plan_cache(seed):
    from gpu_util import NP2SG, dev
    rng = np.random.default_rng(1000 + seed)                 # the DAGs of test_random_chains_match_the_oracle
    dtype = DTYPES[seed % 4]
    n = int(SIZES[(seed // 4) % len(SIZES)])
    inputs = [make_input(rng, dtype, n) for _ in range(int(rng.integers(1, 4)))]
    steps, keep, reds, want, storage, filt = build_dag(rng, dtype, inputs, rich=True)
    tol = {np.float32: 1e-5, np.float64: 1e-12}.get(dtype, 0)
    rounds = 3
    for flags in (0, sg.SG_FLAG_NO_PLAN_CACHE):
        with Ctx(flags) as c:
            tens = [dev(a) for a in inputs]
            c.keep += tens

            class Round:                                     # what run_gpu needs of a context: the SAME device buffers every round
                ctx = c.ctx

                def __init__(self):
                    self.k = 0

                def vec(self, a):
                    t = tens[self.k]
                    self.k += 1
                    return sg.sg_vec_create(c.ctx, NP2SG[np.dtype(dtype)], a.size, t.data_ptr())

                def get(self, h):
                    return c.get(h)
            for rnd in range(rounds):
                for t, a in zip(tens, inputs):               # in-place steps overwrote the inputs: restore them
                    t.copy_(c.torch.from_numpy(a))
                c.torch.cuda.synchronize()
                h, scal, st, fres = run_gpu(Round(), steps, keep, reds, inputs, dtype, filt)
                for i in sorted(keep | storage):
                    assert bits_equal(c.read_vec(h[i], want[i].dtype), want[i]), (flags, seed, rnd, "stored value", i, steps)
                for (kind, src, _), got in zip(reds, scal):
                    w = want[src]
                    if kind == "sum":
                        check_sum(got, w, tol, (flags, seed, rnd, kind))
                    elif kind == "count":
                        assert got == orc.count(w), (flags, seed, rnd, kind)
                    elif kind in ("all", "any"):
                        assert got == (orc.all(w) if kind == "all" else orc.any(w)), (flags, seed, rnd, kind)
                    elif kind.startswith("adj_"):
                        assert got == (orc.all(orc.adj(kind[4:], w)) if w.size > 1 else True), (flags, seed, rnd, kind)
                    elif not (w.dtype.kind == "f" and np.isnan(w).any()):
                        assert bits_equal(np.array([got], dtype=dtype), np.array([(orc.max if kind == "max" else orc.min)(w)], dtype=dtype)), (flags, seed, rnd, kind)
                if fres is not None:
                    kept = orc.filter(want[filt[0]], want[filt[1]])
                    cnt = c.get(fres[1])
                    assert cnt == kept.size and bits_equal(c.read_vec(fres[0], kept.dtype, cnt), kept), (flags, seed, rnd, "filter")
                    for x in fres:
                        sg.sg_release(c.ctx, x)
                for x in {h[i] for i in range(len(inputs))} | {h[i] for i in keep}:      # what the caller still holds (run_gpu released the rest)
                    sg.sg_release(c.ctx, x)
            hits, misses = sg.sg_plan_cache_stats(c.ctx)
            if flags:
                assert hits == 0 and misses == 0
            else:
                assert hits >= rounds - 1 and misses >= 1, (seed, hits, misses)
