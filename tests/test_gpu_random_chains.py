"""Randomised differential test (SURVEY.md §8(c) pin table: "bytecode vs template ... and on random chains"): seeded random
operation DAGs over the C ABI — value ops, immediates, comparisons, logic, stored and released intermediates, reductions and
quantifiers in one flush — against the CPU oracle, primitive by primitive.  No template instance matches such chains, so the plan
builder's pass splitting / spilling and the bytecode evaluator are what is exercised; the same DAG also runs unfused (one launch per
operation) and must give the same bits.

Bars as everywhere: stored values, extrema, counts and quantifiers bit-exact; sums 1e-12 (fp64) / 1e-5 (fp32) relative."""
import numpy as np
import pytest

import oracle as orc
from paper_1410_6685_b200 import sg
from gpu_util import Ctx, rel_err

pytestmark = pytest.mark.gpu

BIN = {"add": sg.SG_ADD, "sub": sg.SG_SUB, "mul": sg.SG_MUL, "div": sg.SG_DIV, "min": sg.SG_MIN, "max": sg.SG_MAX, "mod": sg.SG_MOD}
CMP = {"eq": sg.SG_EQ, "ne": sg.SG_NE, "lt": sg.SG_LT, "le": sg.SG_LE, "gt": sg.SG_GT, "ge": sg.SG_GE}
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


def build_dag(rng, dtype, n_inputs):
    """A list of steps (kind, op, operand indices / immediate); value ids index one list that starts with the inputs."""
    is_f = np.dtype(dtype).kind == "f"
    vals, bools, steps = list(range(n_inputs)), [], []
    nid = n_inputs
    for _ in range(int(rng.integers(4, 15))):
        r = rng.random()
        if r < 0.45 or (r < 0.75 and not bools and rng.random() < 0.5):
            op = str(rng.choice(list(BIN) if not is_f else [k for k in BIN if k != "mod"]))
            a = int(rng.choice(vals))
            if rng.random() < 0.35:
                imm = float(rng.choice([0.5, 2.0, -3.25, 7.0])) if is_f else int(rng.choice([2, 3, 7, -5, 1]))
                steps.append(("bin_imm", op, a, imm, bool(rng.random() < 0.3), nid))
            else:
                steps.append(("bin", op, a, int(rng.choice(vals)), nid))
            vals.append(nid)
        elif r < 0.58:
            op = str(rng.choice(["neg", "abs"] + (["sqrt"] if is_f else [])))
            steps.append(("un", op, int(rng.choice(vals)), nid))
            vals.append(nid)
        elif r < 0.80:
            op = str(rng.choice(list(CMP)))
            a = int(rng.choice(vals))
            if rng.random() < 0.4:
                imm = float(rng.choice([0.0, 1.0, -2.5])) if is_f else int(rng.choice([0, 3, -7]))
                steps.append(("cmp_imm", op, a, imm, nid))
            else:
                steps.append(("cmp", op, a, int(rng.choice(vals)), nid))
            bools.append(nid)
        elif bools:
            op = str(rng.choice(["and", "or", "not"]))
            a = int(rng.choice(bools))
            steps.append(("logic", op, a, int(rng.choice(bools)) if op != "not" else -1, nid))
            bools.append(nid)
        else:
            continue
        nid += 1
    if not steps:                                          # every draw was a logic op without a BOOL to apply it to
        steps.append(("un", "neg", 0, nid))
        vals.append(nid)
    produced_v = [v for v in vals if v >= n_inputs]
    produced_b = list(bools)
    keep = set(int(x) for x in rng.choice(produced_v, min(len(produced_v), int(rng.integers(0, 3))), replace=False)) if produced_v else set()
    if produced_b and rng.random() < 0.4:
        keep.add(int(rng.choice(produced_b)))
    reds = []
    for _ in range(int(rng.integers(1, 4))):
        if produced_v:
            reds.append((str(rng.choice(["sum", "max", "min"])), int(rng.choice(produced_v))))
    for _ in range(int(rng.integers(0, 3))):
        if produced_b:
            reds.append((str(rng.choice(["all", "any", "count"])), int(rng.choice(produced_b))))
    if not keep and not reds:
        keep.add(produced_v[-1] if produced_v else produced_b[-1])
    return steps, keep, reds


def run_oracle(steps, inputs):
    v = dict(enumerate(inputs))
    for st in steps:
        kind = st[0]
        if kind == "bin":
            v[st[4]] = orc.zip(st[1], v[st[2]], v[st[3]])
        elif kind == "bin_imm":
            v[st[5]] = orc.scalar(st[1], v[st[2]], st[3], reversed=st[4])
        elif kind == "un":
            v[st[3]] = orc.unary(st[1], v[st[2]])
        elif kind == "cmp":
            v[st[4]] = orc.cmp(st[1], v[st[2]], v[st[3]])
        elif kind == "cmp_imm":
            v[st[4]] = orc.cmp_scalar(st[1], v[st[2]], st[3])
        else:
            v[st[4]] = orc.logic(st[1], v[st[2]], v[st[3]] if st[3] >= 0 else None)
    return v


RED = {"sum": sg.SG_SUM, "max": sg.SG_RMAX, "min": sg.SG_RMIN}


def run_gpu(c, steps, keep, reds, inputs, dtype):
    is_f = np.dtype(dtype).kind == "f"
    imm = (lambda x: sg.F(x)) if is_f else (lambda x: sg.I(x))
    h = {i: c.vec(a) for i, a in enumerate(inputs)}
    for st in steps:
        kind = st[0]
        if kind == "bin":
            h[st[4]] = sg.sg_enqueue(c.ctx, BIN[st[1]], [h[st[2]], h[st[3]]])
        elif kind == "bin_imm":
            ops = [imm(st[3]), h[st[2]]] if st[4] else [h[st[2]], imm(st[3])]
            h[st[5]] = sg.sg_enqueue(c.ctx, BIN[st[1]], ops)
        elif kind == "un":
            h[st[3]] = sg.sg_enqueue(c.ctx, {"neg": sg.SG_NEG, "abs": sg.SG_ABS, "sqrt": sg.SG_SQRT}[st[1]], [h[st[2]]])
        elif kind == "cmp":
            h[st[4]] = sg.sg_enqueue(c.ctx, CMP[st[1]], [h[st[2]], h[st[3]]])
        elif kind == "cmp_imm":
            h[st[4]] = sg.sg_enqueue(c.ctx, CMP[st[1]], [h[st[2]], imm(st[3])])
        else:
            op = {"and": sg.SG_AND, "or": sg.SG_OR, "not": sg.SG_NOT}[st[1]]
            h[st[4]] = sg.sg_enqueue(c.ctx, op, [h[st[2]]] + ([h[st[3]]] if st[3] >= 0 else []))
    rh = []
    for kind, src in reds:
        if kind in RED:
            rh.append(sg.sg_reduce(c.ctx, h[src], RED[kind]))
        elif kind == "count":
            rh.append(sg.sg_reduce(c.ctx, h[src], sg.SG_COUNT))
        else:
            rh.append((sg.sg_forall if kind == "all" else sg.sg_exists)(c.ctx, h[src]))
    for i, hv in h.items():                                 # anonymous intermediates: everything produced that is not kept
        if i >= len(inputs) and i not in keep:
            sg.sg_release(c.ctx, hv)
    sg.sg_flush(c.ctx)
    st = sg.sg_plan_stats(c.ctx)
    return h, [c.get(r) for r in rh], st


@pytest.mark.parametrize("seed", range(160))
def test_random_chains_match_the_oracle(seed):
    rng = np.random.default_rng(1000 + seed)
    dtype = DTYPES[seed % 4]
    n = int(SIZES[(seed // 4) % len(SIZES)])
    n_inputs = int(rng.integers(1, 4))
    inputs = [make_input(rng, dtype, n) for _ in range(n_inputs)]
    steps, keep, reds = build_dag(rng, dtype, n_inputs)
    want = run_oracle(steps, inputs)
    tol = {np.float32: 1e-5, np.float64: 1e-12}.get(dtype, 0)
    results = {}
    for mode, flags in (("fused", 0), ("unfused", sg.SG_FLAG_UNFUSED)):
        with Ctx(flags) as c:
            h, scal, st = run_gpu(c, steps, keep, reds, inputs, dtype)
            assert st.n_passes >= 1
            for i in sorted(keep):
                got = c.read_vec(h[i], want[i].dtype)
                assert bits_equal(got, want[i]), (mode, seed, "stored value", i, steps)
            for (kind, src), got in zip(reds, scal):
                w = want[src]
                if kind == "sum":
                    ws = orc.sum(w)
                    if np.dtype(dtype).kind == "f":
                        if not np.isfinite(ws):
                            assert (np.isnan(ws) and np.isnan(got)) or ws == got, (mode, seed, kind, got, ws)
                        else:
                            assert rel_err(got, ws, float(np.abs(w.astype(np.float64)).sum())) <= tol, (mode, seed, kind, got, ws, steps)
                    else:
                        assert got == ws, (mode, seed, kind, got, ws)
                elif kind in ("max", "min"):
                    ext = orc.max if kind == "max" else orc.min
                    # extrema follow the total order on bit patterns (R15: -NaN below -inf, +NaN above +inf); the SIGN of a
                    # generated NaN (sqrt of a negative) is the hardware's: x86 makes -NaN, the GPU +NaN — both readings are accepted
                    cands = [ext(w)]
                    if w.dtype.kind == "f" and np.isnan(w).any():
                        cands = [ext(np.where(np.isnan(w), np.copysign(np.nan, sgn), w).astype(w.dtype)) for sgn in (1.0, -1.0)]
                    assert any(bits_equal(np.array([got], dtype=dtype), np.array([wv], dtype=dtype)) for wv in cands), (mode, seed, kind, got, cands, steps)
                elif kind == "count":
                    assert got == orc.count(w), (mode, seed, kind)
                else:
                    assert got == (orc.all(w) if kind == "all" else orc.any(w)), (mode, seed, kind, steps)
            results[mode] = scal
    # fused and unfused plans of the same DAG: exact results are the same bits (sums only within the tolerance: another order)
    for (kind, _), a, b in zip(reds, results["fused"], results["unfused"]):
        if kind != "sum" or np.dtype(dtype).kind != "f":
            assert a == b or (a != a and b != b), (seed, kind, a, b)
