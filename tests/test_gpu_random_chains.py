"""Randomised differential test (SURVEY.md §8(c) pin table: "bytecode vs template ... and on random chains"): seeded random
operation DAGs over the C ABI against the CPU oracle, primitive by primitive.  A DAG mixes value operations, immediates, comparisons,
logic, stored and released intermediates, IN-PLACE results (dst_or_0), device scalars used as operands (an exact reduction of one
value broadcast into a later operation: a scalar edge, so the flush has several passes), reductions, quantifiers, the neighbour
predicate and a stable filter with its count and kept-sum — all pending in ONE flush.  No template instance matches such chains, so
what is exercised is the plan builder (pass assignment, spills, hazards, register allocation) and the bytecode evaluators; the same
DAG also runs unfused (one launch per operation) and must give the same bits.

Bars as everywhere: stored values, extrema, counts, filter outputs and quantifiers bit-exact; sums 1e-12 (fp64) / 1e-5 (fp32)."""
import numpy as np
import pytest

import oracle as orc
from paper_1410_6685_b200 import sg
from gpu_util import Ctx, rel_err

pytestmark = pytest.mark.gpu

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
            assert rel_err(got, ws, float(np.abs(w.astype(np.float64)).sum())) <= tol, (ctx, got, ws)
    else:
        assert got == ws, (ctx, got, ws)


@pytest.mark.parametrize("seed", range(400))
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
                if mode == "unfused" and e.status == sg.SG_ERR_CAPACITY:    # one launch per operation: more than 16 passes in one flush (a plan limit)
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
