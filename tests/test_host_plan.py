"""Host-side tests (no GPU): the C-ABI library loads and exports every symbol include/sg.h declares, the
scalar contracts are checked at enqueue, and the plan builder produces the plans the paper describes
(PAPER.md:284 deferred execution, :301-309 merged kernels, :315-322 fused row operation).  Plan-only contexts
(device -1) build plans without touching CUDA."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

from paper_1410_6685_b200 import sg
from paper_1410_6685_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def built():
    from paper_1410_6685_b200 import build
    build.build()


def plan(builder, flags=0):
    ctx = sg.sg_ctx_create(-1)
    sg.sg_ctx_set_flags(ctx, flags)
    try:
        builder(ctx)
        sg.sg_flush(ctx)
        st = sg.sg_plan_stats(ctx)
        dumps = [sg.sg_plan_dump(ctx, p) for p in range(st.n_passes)]
        return st, dumps
    finally:
        sg.sg_ctx_destroy(ctx)


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "sg.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)          # prototypes only, not names mentioned in comments
    declared = set(re.findall(r"\b(sg_[a-z0-9_]+)\s*\(", header))
    assert len(declared) >= 30
    lib = ctypes.CDLL(sg.lib_path())
    for name in sorted(declared):
        assert hasattr(lib, name), name
    assert declared == set(sg.EXPORTS)                               # the binding has the same names
    for name in sg.EXPORTS:
        assert callable(getattr(sg, name)), name
    assert "sm_100a" in sg.sg_version()


def test_kernels_are_compiled_for_sm_100a_only():
    out = subprocess.run(["cuobjdump", "--list-elf", sg.lib_path()], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\d+a?", out))
    assert archs == {"sm_100a"}, archs


def test_no_device_means_failure_not_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(sg.SgError) as ei:
        sg.sg_ctx_create(0)
    assert ei.value.status == sg.SG_ERR_CUDA


def test_noalloc_sum_checks_its_arguments_before_it_touches_a_device():
    """sg_vec_sum_noalloc (include/sg.h): size limit, dtype, pointers and the device ordinal are rejected on the host, with a message;
    without a GPU the call fails with SG_ERR_CUDA — there is no CPU fallback."""
    import torch
    for args, status, word in (((0, 0, sg.SG_F32, 16, sg.SG_NOALLOC_MAX_N + 1, 16), sg.SG_ERR_CAPACITY, "SG_NOALLOC_MAX_N"),
                               ((0, 0, sg.SG_I64, 16, 8, 16), sg.SG_ERR_DTYPE, "SG_F32"),
                               ((0, 0, sg.SG_F64, 0, 8, 16), sg.SG_ERR_ARG, "null"),
                               ((0, 0, sg.SG_F64, 16, 8, 0), sg.SG_ERR_ARG, "null"),
                               ((0, 0, sg.SG_F64, 16, -1, 16), sg.SG_ERR_ARG, "negative"),
                               ((0, 0, sg.SG_F64, 12, 8, 16), sg.SG_ERR_ARG, "aligned"),
                               ((99, 0, sg.SG_F64, 16, 8, 16), sg.SG_ERR_ARG, "device")):
        with pytest.raises(sg.SgError) as ei:
            sg.sg_vec_sum_noalloc(*args)
        assert ei.value.status == status and word in str(ei.value), (args, str(ei.value))
    assert sg.SG_NOALLOC_SCRATCH_BYTES == 256 + 16 * (sg.SG_NOALLOC_MAX_N // 8192)
    if not torch.cuda.is_available():
        with pytest.raises(sg.SgError) as ei:
            sg.sg_vec_sum_noalloc(0, 0, sg.SG_F32, 16, 8, 16)
        assert ei.value.status == sg.SG_ERR_CUDA


def test_template_registry_is_current():
    assert sg.sg_template_count() >= 25
    rc = subprocess.run([sys.executable, "-m", "paper_1410_6685_b200.gen_templates", "--check"], cwd=ROOT).returncode
    assert rc == 0


def test_nothing_runs_before_a_trigger():
    # a call is added to the pending list; update / a scalar read / to_array trigger execution
    ctx = sg.sg_ctx_create(-1)
    r = W.dot_product(ctx, sg.SG_F64, 1000, None, None)
    assert sg.sg_plan_stats(ctx).n_passes == 0 and sg.sg_plan_stats(ctx).launches_total == 0
    sg.sg_scalar_get(ctx, r["sum"])                                  # trigger (1)
    st = sg.sg_plan_stats(ctx)
    assert st.n_passes == 1 and st.n_nodes == 2
    sg.sg_flush(ctx)                                                 # nothing pending: no new plan
    assert sg.sg_plan_stats(ctx).n_passes == 1
    sg.sg_ctx_destroy(ctx)


def test_dot_product_two_kernels_become_one():
    # Figure 2: cmult and sum are merged; the product is never materialised
    st, dumps = plan(lambda c: W.dot_product(c, sg.SG_F64, 1 << 20, None, None))
    assert st.n_passes == 1 and st.pass_n_in[0] == 2 and st.pass_n_instr[0] == 1 and st.pass_n_out[0] == 1
    assert "OUT_STORE" not in dumps[0] and "OP_MUL" in dumps[0] and "OUT_SUM" in dumps[0]
    assert st.bytes_min == 2 * 8 * (1 << 20)
    stu, _ = plan(lambda c: W.dot_product(c, sg.SG_F64, 1 << 20, None, None), sg.SG_FLAG_UNFUSED)
    assert stu.n_passes == 2 and stu.bytes_min == 4 * 8 * (1 << 20)   # a*b stored, then read again


def test_axpy_is_one_kernel_with_one_more_argument():
    # Figure 3: X[i]+Y[i] becomes a*X[i]+Y[i]; the scalar is one extra kernel argument
    st_add, _ = plan(lambda c: sg.sg_enqueue(c, sg.SG_ADD, [sg.sg_vec_create(c, sg.SG_F64, 100, None), sg.sg_vec_create(c, sg.SG_F64, 100, None)]))
    st_axpy, dumps = plan(lambda c: W.axpy(c, sg.SG_F64, 100, 2.0, None, None))
    assert st_add.n_passes == st_axpy.n_passes == 1
    assert st_axpy.pass_n_args[0] == st_add.pass_n_args[0] + 1
    assert st_axpy.pass_n_instr[0] == 2 and "IN_IMM" in dumps[0]


def test_row_divide_then_subtract_is_one_expression():
    # row(i).divided_by(pivot); row(i).in_place_minus(row(step)) -> (A[i]/pivot) - A[step]
    st, dumps = plan(lambda c: W.ge_row_op(c, 4096, None, None, 3.0))
    assert st.n_passes == 1 and st.pass_n_instr[0] == 2 and st.pass_n_out[0] == 1
    assert dumps[0].count("OUT_STORE") == 1 and "OP_DIV" in dumps[0] and "OP_SUB" in dumps[0]
    assert st.bytes_min == 3 * 8 * 4096                              # read row i, read row step, write row i


def test_cfg0_plans():
    n = 1 << 20
    st, dumps = plan(lambda c: W.cfg0(c, n, None, None, None))          # P2: z stored, postcondition re-reads it
    assert st.n_passes == 2 and st.n_template == 2
    assert st.pass_n_in[0] == 3 and st.pass_n_out[0] == 5 and dumps[0].count("OUT_STORE") == 1
    assert st.pass_n_in[1] == 4 and st.pass_n_out[1] == 1 and "OUT_ALL" in dumps[1]
    assert st.bytes_min == (4 + 4) * 8 * n                           # pass A 3R+1W, pass B 4R
    st, dumps = plan(lambda c: W.cfg0(c, n, None, None, None, keep_z=False))   # P1: everything in one pass
    assert st.n_passes == 1 and st.bytes_min == 3 * 8 * n and "OUT_STORE" not in dumps[0]


def test_cfg1_to_cfg4_plans():
    st, dumps = plan(lambda c: W.cfg1(c, 1 << 26, None, None))
    assert st.n_passes == 1 and st.pass_n_instr[0] == 10 and st.pass_n_out[0] == 2 and st.bytes_min == 8 << 26 and st.n_template == 1
    stu, _ = plan(lambda c: W.cfg1(c, 1 << 26, None, None), sg.SG_FLAG_UNFUSED)
    assert stu.n_passes == 12 and stu.bytes_min == 27 * (4 << 26)     # 27 vector units
    st, dumps = plan(lambda c: W.cfg2(c, 1 << 27, None))
    assert st.n_passes == 1 and "OUT_FILTER" in dumps[0] and st.n_template == 1
    st, dumps = plan(lambda c: W.cfg3(c, 1 << 28, None))
    assert st.n_passes == 1 and st.pass_n_in[0] == 1 and "IN_SHIFT" in dumps[0] and st.bytes_min == 4 << 28 and st.n_template == 1
    st, dumps = plan(lambda c: W.cfg4(c, 16384, None, 0))
    assert st.n_passes == 2 and "IN_STRIDED" in dumps[0] and "IN_COLB" in dumps[1] and "IN_ROWB" in dumps[1] and st.n_template == 2
    rows = 16383
    assert st.bytes_min == 8 * rows + 8 * rows + (2 * 8 * rows * 16384 + 8 * 16384 + 8 * rows) + 8 * rows + 8 * 16384


def test_ge_loop_entry_point_checks_its_arguments():
    """sg_mat_ge_steps: the whole loop of Listing 5 as one composite call (a persistent kernel on a device; nothing on a plan-only context)."""
    ctx = sg.sg_ctx_create(-1)
    try:
        n = 64
        M = sg.sg_mat_create(ctx, sg.SG_F64, n, n, n, None)
        det = sg.sg_vec_create(ctx, sg.SG_F64, 1, None)
        mp = sg.sg_vec_create(ctx, sg.SG_F64, 1, None)
        before = sg.sg_plan_stats(ctx).launches_total
        sg.sg_mat_ge_steps(ctx, M, det, mp, 0.0, 0, n)
        assert sg.sg_plan_stats(ctx).launches_total == before + 1          # ONE launch for n steps
        for bad in (dict(eps=-1.0), dict(eps=float("nan")), dict(k0=-1), dict(k1=n + 1), dict(k0=5, k1=4)):
            kw = dict(eps=0.0, k0=0, k1=n)
            kw.update(bad)
            with pytest.raises(sg.SgError) as e:
                sg.sg_mat_ge_steps(ctx, M, det, mp, kw["eps"], kw["k0"], kw["k1"])
            assert e.value.status == sg.SG_ERR_ARG
        with pytest.raises(sg.SgError) as e:
            sg.sg_mat_ge_steps(ctx, sg.sg_mat_create(ctx, sg.SG_F64, 4, 6, 6, None), det, mp, 0.0, 0, 4)
        assert e.value.status == sg.SG_ERR_SHAPE
        with pytest.raises(sg.SgError) as e:
            sg.sg_mat_ge_steps(ctx, sg.sg_mat_create(ctx, sg.SG_F32, 4, 4, 4, None), det, mp, 0.0, 0, 4)
        assert e.value.status == sg.SG_ERR_DTYPE
        with pytest.raises(sg.SgError) as e:
            sg.sg_mat_ge_steps(ctx, M, sg.sg_vec_create(ctx, sg.SG_F64, 2, None), mp, 0.0, 0, n)
        assert e.value.status == sg.SG_ERR_SHAPE
    finally:
        sg.sg_ctx_destroy(ctx)


def test_ge_step_is_two_passes_with_no_read_back():
    """Listing 5's loop body: the paper launches one kernel per row and reads two scalars back per
    row (its slow case); here a step is a scalar + factor pass and ONE matrix pass over all rows."""
    def step(k):
        def build(c):
            M = sg.sg_mat_create(c, sg.SG_F64, 1000, 1000, 1000, None)
            det, mp = sg.sg_vec_create(c, sg.SG_F64, 1, None), sg.sg_vec_create(c, sg.SG_F64, 1, None)
            for h in W.ge_step(c, M, 1000, k, det, mp):
                sg.sg_release(c, h)
        return build
    rows = 989
    for _ in (0,):
        st, dumps = plan(step(10))
        # det, min |pivot| and the factors share one pass (values of different lengths; it has no precompiled instance and runs
        # on the bytecode kernel); the rows change in place in the second (template instance)
        assert st.n_passes == 2 and st.n_template == 1
        assert "OP_MUL" in dumps[0] and "OP_MIN" in dumps[0] and "IN_STRIDED" in dumps[0] and "IN_SCALAR" in dumps[0] and dumps[0].count("OUT_STORE") == 3
        assert "IN_COLB" in dumps[1] and "IN_ROWB" in dumps[1] and dumps[1].count("OUT_STORE") == 1
        assert abs(st.bytes_min - ((3 * 8 + 2 * 8) + (8 * rows + 8 + 8 * rows) + (2 * 8 * rows * 1000 + 8 * 1000 + 8 * rows))) <= 8
    st, dumps = plan(step(999))                                       # last step: only the scalar pass
    assert st.n_passes == 1 and "IN_COLB" not in dumps[0]
    def far(c):                                                       # factor column much longer than one element: three passes, all instances
        M = sg.sg_mat_create(c, sg.SG_F64, 4096, 4096, 4096, None)
        det, mp = sg.sg_vec_create(c, sg.SG_F64, 1, None), sg.sg_vec_create(c, sg.SG_F64, 1, None)
        for h in W.ge_step(c, M, 4096, 6, det, mp):
            sg.sg_release(c, h)
    st, dumps = plan(far)
    assert st.n_passes == 3 and st.n_template == 3


def test_force_bytecode_and_unknown_chains_use_the_bytecode_kernel():
    st, _ = plan(lambda c: W.cfg1(c, 1 << 20, None, None), sg.SG_FLAG_FORCE_BYTECODE)
    assert st.n_bytecode == 1 and st.n_template == 0

    def odd_chain(c):
        a = sg.sg_vec_create(c, sg.SG_F32, 1000, None)
        t = sg.sg_enqueue(c, sg.SG_MAX, [a, sg.F(0.25)])
        u = sg.sg_enqueue(c, sg.SG_NEG, [t])
        sg.sg_release(c, t)
        return sg.sg_reduce(c, u, sg.SG_RMIN)
    st, _ = plan(odd_chain)
    assert st.n_passes == 1 and st.n_bytecode == 1


def test_scalar_contracts_at_enqueue():
    ctx = sg.sg_ctx_create(-1)
    a = sg.sg_vec_create(ctx, sg.SG_F32, 10, None)
    b = sg.sg_vec_create(ctx, sg.SG_F32, 11, None)
    d = sg.sg_vec_create(ctx, sg.SG_F64, 10, None)
    m = sg.sg_mat_create(ctx, sg.SG_F64, 4, 6, 6, None)
    for ops, code in [([a, b], sg.SG_ERR_SHAPE), ([a, d], sg.SG_ERR_DTYPE), ([sg.F(1.0), sg.F(2.0)], sg.SG_ERR_ARG)]:
        with pytest.raises(sg.SgError) as ei:
            sg.sg_enqueue(ctx, sg.SG_ADD, ops)
        assert ei.value.status == code
    with pytest.raises(sg.SgError) as ei:
        sg.sg_enqueue(ctx, sg.SG_AND, [a, a])                        # logic needs BOOL
    assert ei.value.status == sg.SG_ERR_DTYPE
    with pytest.raises(sg.SgError) as ei:
        sg.sg_enqueue(ctx, sg.SG_MUL, [m, sg.H(d, sg.SG_BCAST_ROW)])  # ROW-broadcast length must equal columns (6)
    assert ei.value.status == sg.SG_ERR_SHAPE
    with pytest.raises(sg.SgError) as ei:
        sg.sg_vec_subset(ctx, a, 3, 11)
    assert ei.value.status == sg.SG_ERR_ARG
    with pytest.raises(sg.SgError) as ei:
        sg.sg_reduce(ctx, sg.sg_vec_create(ctx, sg.SG_F32, 0, None), sg.SG_RMAX)
    assert ei.value.status == sg.SG_ERR_EMPTY
    assert sg.sg_plan_stats(ctx).n_passes == 0                        # failed calls left the pending list unchanged
    assert sg.sg_vec_count(ctx, a) == 10 and sg.sg_vec_count(ctx, m) == 24
    sg.sg_ctx_destroy(ctx)


def test_memory_hazards_order_the_passes():
    # a read of column k must precede the in-place update of the rows it crosses (WAR through memory)
    st, dumps = plan(lambda c: W.cfg4(c, 512, None, 3))
    assert st.n_passes == 2 and "OUT_STORE" in dumps[0] and dumps[1].count("OUT_STORE") == 1

    # a view read after an in-place write through another handle sees the new data: it lands in a later pass
    def raw(c):
        x = sg.sg_vec_create(c, sg.SG_F64, 1000, None)
        y = sg.sg_vec_create(c, sg.SG_F64, 1000, None)
        head = sg.sg_vec_subset(c, x, 0, 500)
        sg.sg_enqueue(c, sg.SG_ADD, [x, y], dst_or_0=x)
        return sg.sg_reduce(c, head, sg.SG_SUM)
    st, _ = plan(raw)
    assert st.n_passes == 2

    # an in-place result may not alias a shifted view of its own destination
    ctx = sg.sg_ctx_create(-1)
    x = sg.sg_vec_create(ctx, sg.SG_F64, 1000, None)
    lo, hi = sg.sg_vec_subset(ctx, x, 0, 999), sg.sg_vec_subset(ctx, x, 1, 1000)
    sg.sg_enqueue(ctx, sg.SG_ADD, [lo, hi], dst_or_0=lo)
    with pytest.raises(sg.SgError) as ei:
        sg.sg_flush(ctx)
    assert ei.value.status == sg.SG_ERR_ALIAS
    sg.sg_ctx_destroy(ctx)


def test_released_intermediates_are_never_materialised():
    def chain(c, release):
        a = sg.sg_vec_create(c, sg.SG_F32, 4096, None)
        t = sg.sg_enqueue(c, sg.SG_MUL, [a, a])
        u = sg.sg_enqueue(c, sg.SG_ADD, [t, sg.F(1.0)])
        if release:
            sg.sg_release(c, t)
        return u
    st_kept, d_kept = plan(lambda c: chain(c, False))
    st_rel, d_rel = plan(lambda c: chain(c, True))
    assert d_kept[0].count("OUT_STORE") == 2 and d_rel[0].count("OUT_STORE") == 1
    assert st_kept.bytes_min - st_rel.bytes_min == 4 * 4096


# ----------------------------------------------------------------------------------------------------------
# plans of the rest of the vector API
# ----------------------------------------------------------------------------------------------------------
def test_vector_api_plans():
    n = 1 << 16
    st, dumps = plan(lambda c: W.project_sqrt(c, sg.SG_F32, n, None))
    assert st.n_passes == 1 and "OP_SQRT" in dumps[0]
    # avg: the vector pass produces the sum, a one-element pass divides it on the device (scalar consumed elementwise)
    st, dumps = plan(lambda c: W.avg(c, sg.SG_F64, n, None))
    assert st.n_passes == 2 and "OUT_SUM" in dumps[0] and "OP_DIV" in dumps[1] and "IN_SCALAR" in dumps[1]
    st, dumps = plan(lambda c: W.norm2(c, sg.SG_F32, n, None))
    assert st.n_passes == 2 and "OP_MUL" in dumps[0] and "OP_SQRT" in dumps[1]
    # Listing 2: the precondition is fused into the dividing pass (fresh output); the registered postcondition re-reads the
    # stored quotient in a second pass (R17); unregistered (exact EQ) it shares the pass
    st, dumps = plan(lambda c: W.compwise_divide(c, sg.SG_F64, n, None, None, eps=1e-12))
    assert st.n_passes == 2 and st.pass_n_in[0] == 2 and st.pass_n_in[1] == 3 and st.bytes_min == 6 * 8 * n
    assert all(k in dumps[0] for k in ("OP_DIV", "OUT_ANY", "OUT_ALL", "OUT_STORE")) and "OP_ABS" not in dumps[0]
    assert all(k in dumps[1] for k in ("OP_MUL", "OP_ABS", "OP_LE", "OUT_ALL")) and "OP_DIV" not in dumps[1]
    st, dumps = plan(lambda c: W.compwise_divide(c, sg.SG_F64, n, None, None))
    assert st.n_passes == 1 and st.bytes_min == 3 * 8 * n and dumps[0].count("OUT_ALL") == 2
    st, dumps = plan(lambda c: W.approx_equal(c, sg.SG_F32, n, None, None, 1e-5))
    assert st.n_passes == 1 and st.pass_n_in[0] == 2 and "OUT_MAX" in dumps[0] and "OUT_ALL" in dumps[0]


def test_sqrt_and_scalar_only_operands_are_checked_at_enqueue():
    ctx = sg.sg_ctx_create(-1)
    try:
        vi = sg.sg_vec_create(ctx, sg.SG_I32, 8, None)
        vb = sg.sg_enqueue(ctx, sg.SG_GT, [vi, sg.I(0)])
        with pytest.raises(sg.SgError) as e:
            sg.sg_enqueue(ctx, sg.SG_SQRT, [vb])               # BOOL: undefined
        assert e.value.status == sg.SG_ERR_DTYPE
        mi = sg.sg_mat_create(ctx, sg.SG_I32, 4, 4, 4, None)
        with pytest.raises(sg.SgError) as e:
            sg.sg_enqueue(ctx, sg.SG_SQRT, [mi])               # integer MATRIX: the promoting form is a vector operation
        assert e.value.status == sg.SG_ERR_DTYPE
        with pytest.raises(sg.SgError) as e:
            sg.sg_enqueue(ctx, 18, [vi])                       # reserved op code
        assert e.value.status == sg.SG_ERR_ARG
        with pytest.raises(sg.SgError) as e:
            sg.sg_enqueue(ctx, sg.SG_ADD, [sg.F(1.0), sg.F(2.0)])   # no handle at all
        assert e.value.status == sg.SG_ERR_ARG
        vf = sg.sg_vec_create(ctx, sg.SG_F64, 8, None)
        s = sg.sg_reduce(ctx, vf, sg.SG_SUM)
        r = sg.sg_enqueue(ctx, sg.SG_DIV, [s, sg.F(8.0)])
        assert sg.sg_vec_count(ctx, r) == 1                    # device scalars only -> a one-element vector
    finally:
        sg.sg_ctx_destroy(ctx)


# ----------------------------------------------------------------------------------------------------------
# dtype-changing project: the conversion happens at load, inside the consumer's pass
# ----------------------------------------------------------------------------------------------------------
def test_integer_sqrt_is_one_pass_with_a_converting_load():
    n = 1 << 16
    st, dumps = plan(lambda c: sg.sg_enqueue(c, sg.SG_SQRT, [sg.sg_vec_create(c, sg.SG_I32, n, None)]))
    assert st.n_passes == 1 and "IN_VEC_CVT,2" in dumps[0] and "OP_SQRT" in dumps[0] and "DT_F64" in dumps[0]
    assert st.bytes_min == 4 * n + 8 * n                     # int32 read once, double written once: 12 B per element

    def chain(c):                                           # a PENDING integer operand is stored first: a pass has one value type
        x = sg.sg_vec_create(c, sg.SG_I32, n, None)
        y = sg.sg_enqueue(c, sg.SG_ADD, [x, sg.I(1)])
        f = sg.sg_cast(c, y, sg.SG_F32)
        sg.sg_release(c, y)
        return sg.sg_reduce(c, f, sg.SG_SUM)
    st, dumps = plan(chain)
    assert st.n_passes == 2 and "DT_I32" in dumps[0] and "OUT_STORE" in dumps[0] and "DT_F32" in dumps[1] and "IN_VEC_CVT,2" in dumps[1]
    ctx = sg.sg_ctx_create(-1)
    try:
        x = sg.sg_vec_create(ctx, sg.SG_F64, 8, None)
        assert sg.sg_vec_count(ctx, sg.sg_cast(ctx, x, sg.SG_I64)) == 8
        with pytest.raises(sg.SgError) as e:
            sg.sg_cast(ctx, x, sg.SG_BOOL)
        assert e.value.status == sg.SG_ERR_DTYPE
        with pytest.raises(sg.SgError) as e:
            sg.sg_cast(ctx, sg.sg_mat_create(ctx, sg.SG_F64, 2, 2, 2, None), sg.SG_F32)
        assert e.value.status == sg.SG_ERR_UNSUPPORTED
        with pytest.raises(sg.SgError) as e:
            sg.sg_reduce(ctx, x, sg.SG_SUM, acc=sg.SG_F32)   # a narrower accumulator is rejected, not emulated
        assert e.value.status == sg.SG_ERR_DTYPE
        sg.sg_reduce(ctx, x, sg.SG_SUM, acc=sg.SG_F64)
        sg.sg_reduce(ctx, x, sg.SG_RMAX, acc=sg.SG_F64)
    finally:
        sg.sg_ctx_destroy(ctx)


# ----------------------------------------------------------------------------------------------------------
# plan hazards and context robustness (round-1 review)
# ----------------------------------------------------------------------------------------------------------
def test_inplace_update_never_shares_a_pass_with_a_neighbour_read_of_the_same_storage():
    """is_sorted(x) reads x[i+1], which belongs to another thread / warp / block: x *= 2 in place must wait for that pass."""
    n = 1 << 16

    def prog(c):
        x = sg.sg_vec_create(c, sg.SG_F32, n, None)
        srt = sg.sg_forall_adjacent(c, x, sg.SG_LE)
        sg.sg_enqueue(c, sg.SG_MUL, [x, sg.F(2.0)], dst_or_0=x)
        return srt
    st, dumps = plan(prog)
    assert st.n_passes == 2
    assert "IN_SHIFT" in dumps[0] and "OUT_STORE" not in dumps[0] and "OUT_STORE" in dumps[1]

    def prog2(c):                                           # an index-for-index reader of the same view still fuses
        x = sg.sg_vec_create(c, sg.SG_F32, n, None)
        pos = sg.sg_enqueue(c, sg.SG_GE, [x, sg.F(0.0)])
        ok = sg.sg_forall(c, pos)
        sg.sg_release(c, pos)
        sg.sg_enqueue(c, sg.SG_MUL, [x, sg.F(2.0)], dst_or_0=x)
        return ok
    st, dumps = plan(prog2)
    assert st.n_passes == 1 and "OUT_ALL" in dumps[0] and "OUT_STORE" in dumps[0]


def test_release_before_flush_keeps_storage_for_pending_readers():
    ctx = sg.sg_ctx_create(-1)
    try:
        x = sg.sg_vec_create(ctx, sg.SG_F32, 1024, None)     # context-owned storage
        y = sg.sg_enqueue(ctx, sg.SG_ADD, [x, sg.F(1.0)])
        sg.sg_release(ctx, x)                               # released while y = x + 1 is pending
        sg.sg_flush(ctx)
        assert sg.sg_plan_stats(ctx).n_passes == 1
        s = sg.sg_reduce(ctx, y, sg.SG_SUM)
        sg.sg_flush(ctx)
        a = sg.sg_enqueue(ctx, sg.SG_DIV, [s, sg.F(4.0)])    # a materialised scalar consumed by a new chain ...
        sg.sg_release(ctx, s)                               # ... and released before the flush
        sg.sg_flush(ctx)
        assert sg.sg_plan_stats(ctx).n_passes == 1 and sg.sg_vec_count(ctx, a) == 1
    finally:
        sg.sg_ctx_destroy(ctx)


def test_handle_slots_are_recycled_and_stale_handles_are_unknown():
    """A long-running loop must not grow the handle table: the slot of a dead value is reused once no pending operation can name
    it, under a new generation — the released handle is then an unknown handle, never an alias of the slot's new value."""
    ctx = sg.sg_ctx_create(-1)
    try:
        x = sg.sg_vec_create(ctx, sg.SG_F32, 4096, None)
        slots, first = set(), None
        for it in range(200):                                 # x -> (x + 1) * 2 -> sum, everything released every step
            t = sg.sg_enqueue(ctx, sg.SG_ADD, [x, sg.F(1.0)])
            u = sg.sg_enqueue(ctx, sg.SG_MUL, [t, sg.F(2.0)])
            s = sg.sg_reduce(ctx, u, sg.SG_SUM)
            sg.sg_release(ctx, t)
            sg.sg_flush(ctx)
            assert sg.sg_plan_stats(ctx).n_passes == 1
            assert sg.sg_vec_count(ctx, u) == 4096 and sg.sg_vec_count(ctx, s) == 1
            for h in (t, u, s):
                slots.add(h & 0xffffffff)
            first = first or (t, u, s)
            sg.sg_release(ctx, u)
            sg.sg_release(ctx, s)
        assert len(slots) <= 9, slots                          # 600 handles lived in a handful of slots (at most three steps' worth)
        assert sg.sg_vec_count(ctx, x) == 4096                 # a handle that was never released still answers
        for h in first:                                        # the first step's handles: their slots hold other values now
            with pytest.raises(sg.SgError) as e:
                sg.sg_vec_count(ctx, h)
            assert e.value.status == sg.SG_ERR_ARG
            with pytest.raises(sg.SgError):
                sg.sg_enqueue(ctx, sg.SG_ADD, [h, sg.F(1.0)])
        # a slot is not reused while a pending operation still reads its value
        y = sg.sg_enqueue(ctx, sg.SG_ADD, [x, sg.F(3.0)])
        z = sg.sg_enqueue(ctx, sg.SG_MUL, [y, y])
        sg.sg_release(ctx, y)
        fresh = [sg.sg_enqueue(ctx, sg.SG_SUB, [x, sg.F(float(k))]) for k in range(8)]
        assert all((f & 0xffffffff) != (y & 0xffffffff) for f in fresh)
        sg.sg_flush(ctx)
        assert sg.sg_vec_count(ctx, z) == 4096
    finally:
        sg.sg_ctx_destroy(ctx)


_VALUE_OPS = {"OP_ADD", "OP_SUB", "OP_MUL", "OP_DIV", "OP_MIN", "OP_MAX", "OP_MOD", "OP_NEG", "OP_ABS", "OP_MOV", "OP_SQRT"}


def _input_registers_are_never_written(dump: str) -> bool:
    """Every input of a tile is loaded before the first instruction runs, so no instruction may write a register an input lives in."""
    groups = re.findall(r"\{(IN_[A-Z_]+),(\d+),(\d+),(\d+)\}", dump)
    v_in = {int(reg) for kind, _, reg, _ in groups if kind != "IN_BOOLVEC"}
    p_in = {int(reg) for kind, _, reg, _ in groups if kind == "IN_BOOLVEC"}
    for op, dst, _, _ in re.findall(r"\{(OP_[A-Z]+),(\d+),(\d+),(\d+)\}", dump):
        if int(dst) in (v_in if op in _VALUE_OPS else p_in):
            return False
    return True


def test_an_input_never_shares_a_register_with_an_earlier_temporary():
    """`(a+b)*(c+d) + e`: the multiplication gives two registers back, and e — first named afterwards — must not move into the one
    c+d was computed in (it is loaded at the start of the tile and would be overwritten).  Checked on that chain, on 200 random
    operation DAGs (the generator of tests/test_gpu_random_chains.py, planned on a plan-only context) and on every registered
    template program."""
    def chain(ctx):
        v = [sg.sg_vec_create(ctx, sg.SG_F64, 4096, None) for _ in range(5)]
        t1 = sg.sg_enqueue(ctx, sg.SG_ADD, [v[0], v[1]])
        t2 = sg.sg_enqueue(ctx, sg.SG_ADD, [v[2], v[3]])
        t3 = sg.sg_enqueue(ctx, sg.SG_MUL, [t1, t2])
        t4 = sg.sg_enqueue(ctx, sg.SG_ADD, [t3, v[4]])
        t5 = sg.sg_enqueue(ctx, sg.SG_MUL, [t4, sg.F(3.0)])
        for t in (t1, t2, t3, t4):
            sg.sg_release(ctx, t)
        return t5
    st, dumps = plan(chain)
    assert st.n_passes == 1 and _input_registers_are_never_written(dumps[0]), dumps[0]

    import numpy as np
    import test_gpu_random_chains as R

    class PlanOnly:                       # the slice of tests/gpu_util.Ctx that run_gpu uses, on a context without a device
        def __init__(self):
            self.ctx = sg.sg_ctx_create(-1)

        def vec(self, a):
            return sg.sg_vec_create(self.ctx, {"float32": sg.SG_F32, "float64": sg.SG_F64, "int32": sg.SG_I32, "int64": sg.SG_I64}[a.dtype.name], a.size, None)

        def get(self, h):
            return 0
    for seed in range(200):
        rng = np.random.default_rng(5000 + seed)
        dtype = R.DTYPES[seed % 4]
        inputs = [R.make_input(rng, dtype, 64) for _ in range(int(rng.integers(1, 4)))]
        steps, keep, reds, _, _, filt = R.build_dag(rng, dtype, inputs)
        c = PlanOnly()
        try:
            # every DAG plans: a pass that a later spill would overfill (more than SG_MAX_OUT outputs) is re-planned with outputs held
            # in reserve — seeds 16, 42, 53, 77, ... failed with SG_ERR_CAPACITY "too many outputs in one pass" before
            _, _, stats, _ = R.run_gpu(c, steps, keep, reds, inputs, dtype, filt)
            assert 1 <= stats.n_passes <= 32
            for p in range(stats.n_passes):
                d = sg.sg_plan_dump(c.ctx, p)
                assert _input_registers_are_never_written(d), (seed, d)
        finally:
            sg.sg_ctx_destroy(c.ctx)
    inc = open(os.path.join(ROOT, "paper_1410_6685_b200", "csrc", "sg_templates_gen.inc")).read()
    progs = inc.split("SG_TEMPLATE(")[1:]
    assert len(progs) >= 50 and all(_input_registers_are_never_written(pr) for pr in progs)


def test_chains_beyond_the_limits_of_one_pass_are_split_not_rejected():
    """A pass holds at most 10 distinct inputs, 8 outputs, 32 operations and the evaluator's registers.  A chain that needs more is
    planned as several passes (the assignment repeats with fewer operations per pass; round 2 failed such a flush with SG_ERR_CAPACITY)."""
    def many_inputs(ctx):                       # v0 + v1 + ... + v13: fourteen distinct vectors in one expression
        v = [sg.sg_vec_create(ctx, sg.SG_F64, 4096, None) for _ in range(14)]
        acc = v[0]
        for x in v[1:]:
            nxt = sg.sg_enqueue(ctx, sg.SG_ADD, [acc, x])
            if acc != v[0]:
                sg.sg_release(ctx, acc)
            acc = nxt
        return acc
    st, dumps = plan(many_inputs)
    assert 2 <= st.n_passes <= 4 and st.n_nodes == 13
    assert all(len(re.findall(r"\{IN_", d)) <= 10 for d in dumps)

    def many_registers(ctx):                    # thirteen temporaries a + i alive at once, each with its own immediate
        a = sg.sg_vec_create(ctx, sg.SG_F32, 4096, None)
        t = [sg.sg_enqueue(ctx, sg.SG_ADD, [a, sg.F(float(i))]) for i in range(13)]
        acc = t[0]
        for x in t[1:]:
            nxt = sg.sg_enqueue(ctx, sg.SG_MUL, [acc, x])
            if acc != t[0]:
                sg.sg_release(ctx, acc)
            acc = nxt
        for x in t:
            sg.sg_release(ctx, x)
        return acc
    st, dumps = plan(many_registers)
    assert st.n_passes >= 2 and st.n_nodes == 25


def test_plan_cache_hits_on_the_same_list_and_misses_on_a_different_one():
    """the pass assignment is remembered under the signature of the pending list — operations, identity pattern,
    storage and liveness of the values, contracts, flags; immediates excluded."""
    ctx = sg.sg_ctx_create(-1)
    try:
        bufs = [0x7000000000, 0x7100000000, 0x7200000000]     # (away from a plan-only context's made-up addresses)

        def step(k=2.5, keep_t=False, ptr0=None):
            a, b, c3 = (sg.sg_vec_create(ctx, sg.SG_F64, 1 << 20, p) for p in ([ptr0 or bufs[0]] + bufs[1:]))
            t = sg.sg_enqueue(ctx, sg.SG_ADD, [a, b])
            u = sg.sg_enqueue(ctx, sg.SG_MUL, [t, sg.F(k)])
            z = sg.sg_enqueue(ctx, sg.SG_SUB, [u, c3])
            s = sg.sg_reduce(ctx, z, sg.SG_SUM)
            if not keep_t:
                sg.sg_release(ctx, t)
            sg.sg_release(ctx, u)
            sg.sg_flush(ctx)
            st = sg.sg_plan_stats(ctx)
            dumps = [sg.sg_plan_dump(ctx, p) for p in range(st.n_passes)]
            for h in (a, b, c3, z, s) + ((t,) if keep_t else ()):
                sg.sg_release(ctx, h)
            return dumps
        first = step()
        assert sg.sg_plan_cache_stats(ctx) == (0, 1)
        assert step() == first and sg.sg_plan_cache_stats(ctx) == (1, 1)             # the same list again: a hit, the same programs
        assert step(k=7.0) == first and sg.sg_plan_cache_stats(ctx) == (2, 1)        # another immediate: still a hit
        kept = step(keep_t=True)                                                     # t stays alive: one more stored output, another list
        assert kept != first and sg.sg_plan_cache_stats(ctx) == (2, 2)
        step(ptr0=0x7300000000)                                                        # another buffer: another signature
        assert sg.sg_plan_cache_stats(ctx) == (2, 3)
        assert step() == first and step(keep_t=True) == kept and sg.sg_plan_cache_stats(ctx) == (4, 3)    # both lists are remembered
        sg.sg_ctx_set_flags(ctx, sg.SG_FLAG_NO_PLAN_CACHE)
        assert step() == first and sg.sg_plan_cache_stats(ctx) == (4, 3)             # switched off: planned from scratch, not counted
    finally:
        sg.sg_ctx_destroy(ctx)


def test_a_failed_flush_discards_the_pending_list_and_leaves_the_context_usable():
    ctx = sg.sg_ctx_create(-1)
    try:
        x = sg.sg_vec_create(ctx, sg.SG_F64, 1024, None)
        bad = x
        for _ in range(40):                                  # a chain longer than one pass holds (SG_MAX_INSTR) ...
            nxt = sg.sg_enqueue(ctx, sg.SG_ADD, [bad, x])
            if bad != x:
                sg.sg_release(ctx, bad)
            bad = nxt
        pend = [sg.sg_reduce(ctx, bad, k) for k in (sg.SG_SUM, sg.SG_RMAX, sg.SG_RMIN)] * 1
        many = [sg.sg_reduce(ctx, sg.sg_enqueue(ctx, sg.SG_MUL, [x, sg.F(float(i))]), sg.SG_SUM) for i in range(2200)]   # ... and > 256 passes
        with pytest.raises(sg.SgError) as e:
            sg.sg_flush(ctx)
        assert e.value.status == sg.SG_ERR_CAPACITY and "discarded" in str(e.value)
        sg.sg_flush(ctx)                                    # nothing is pending any more: the error does not come back
        y = sg.sg_enqueue(ctx, sg.SG_MUL, [x, sg.F(3.0)])    # unrelated later work runs
        sg.sg_flush(ctx)
        st = sg.sg_plan_stats(ctx)
        assert st.n_passes == 1 and st.n_nodes == 1 and sg.sg_vec_count(ctx, y) == 1024
        for h in pend + many:
            sg.sg_release(ctx, h)
    finally:
        sg.sg_ctx_destroy(ctx)


def test_composite_entry_points_on_a_plan_only_context():
    """sg_vec_quicksort / sg_mat_transpose / sg_replay_last_graph check their arguments and flush pending work without a device."""
    ctx = sg.sg_ctx_create(-1)
    try:
        v = sg.sg_vec_create(ctx, sg.SG_F32, 1000, None)
        w = sg.sg_enqueue(ctx, sg.SG_MUL, [v, sg.F(2.0)])           # pending: the composite flushes it first (trigger (2))
        before = sg.sg_plan_stats(ctx).launches_total
        out = sg.sg_vec_quicksort(ctx, w)
        assert sg.sg_vec_count(ctx, out) == 1000 and sg.sg_plan_stats(ctx).n_passes == 1
        assert sg.sg_plan_stats(ctx).launches_total > before
        with pytest.raises(sg.SgError) as e:
            sg.sg_vec_quicksort(ctx, sg.sg_vec_create(ctx, sg.SG_F32, 0, None))     # require a.count > 0
        assert e.value.status == sg.SG_ERR_EMPTY
        b = sg.sg_enqueue(ctx, sg.SG_GT, [v, sg.F(0.0)])
        with pytest.raises(sg.SgError) as e:
            sg.sg_vec_quicksort(ctx, b)
        assert e.value.status == sg.SG_ERR_DTYPE
        with pytest.raises(sg.SgError) as e:
            sg.sg_vec_quicksort(ctx, sg.sg_mat_create(ctx, sg.SG_F32, 4, 4, 4, None))
        assert e.value.status == sg.SG_ERR_ARG
        sg.sg_enqueue(ctx, sg.SG_ADD, [v, sg.F(1.0)])
        sg.sg_flush(ctx)
        assert sg.sg_replay_last_graph(ctx, 5) == (0.0, 0.0)       # nothing is launched on a plan-only context
    finally:
        sg.sg_ctx_destroy(ctx)
