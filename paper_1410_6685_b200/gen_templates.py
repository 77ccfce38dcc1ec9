"""Writes csrc/sg_templates_gen.inc: the registry of precompiled template instances.

Each registered chain is built through the C ABI on a PLAN-ONLY context (device -1, nothing is launched), and the
canonical program the plan builder produced for every pass is dumped as a C++ initialiser.  Because the registry
comes from the plan builder's own output, a registered chain always matches its signature at run time.

    python -m paper_1410_6685_b200.gen_templates          # rewrite the file (then rebuild the library)
    python -m paper_1410_6685_b200.gen_templates --check  # exit 1 if the committed file is stale

Bootstrap: the library must exist to run this (its plan builder is what is being dumped); with a stale or empty
registry the library still builds and every chain runs on the bytecode kernel.
"""
from __future__ import annotations

import os
import sys

from . import sg
from . import workloads as W

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "sg_templates_gen.inc")

# tuning per instance: (unroll = 128-bit accesses per operand per thread per tile, min blocks per SM, rows per stage, shared-memory stages of a matrix pass)
DEFAULT_TUNE = (2, 3, 4, 3)
TUNE = {
    "cfg1": (2, 4, 4),
    "cfg3": (4, 4, 4),
    "cfg3sum": (4, 4, 4),
    "red": (4, 4, 4),
    "extrema": (4, 4, 4),
    "sorted_f32": (4, 4, 4),
    "cfg4": (2, 2, 4),      # measured at 16384^2 (k = 0 / k = 8191): (2,2,4,3) 0.765 / 0.393 ms; (1,4,4,3) 0.780 / 0.400; (2,3,4,2) 0.772 / 0.406 (80 registers, spills); (1,4,8,2) 0.813 / 0.418
    "matvec": (2, 2, 4, 3),   # measured: (2, 4, 2, 3) is slower (0.430 / 0.379 ms vs 0.376 / 0.343 ms right / left at 16384^2)
    "matvec_right": (2, 3, 4, 2),   # per-row double-double sums are latency-bound: TWO stages and three blocks per SM: 0.374 -> 0.343 ms (left: 0.341 -> 0.359, kept at three stages)
    "cfg2": (2, 2, 2),      # filter: tile = 4*unroll steps, min blocks per SM, input stages
}

N = 1 << 20


def _chains():
    """(name, flags, builder) — builder(ctx) enqueues the chain; the flush is done by the caller."""
    f32, f64, i32 = sg.SG_F32, sg.SG_F64, sg.SG_I32
    yield "dot_f64", 0, lambda c: W.dot_product(c, f64, N, None, None)                      # Listing 4
    yield "dot_f32", 0, lambda c: W.dot_product(c, f32, N, None, None)
    yield "axpy_f64", 0, lambda c: W.axpy(c, f64, N, 2.0, None, None)
    yield "axpy_f32", 0, lambda c: W.axpy(c, f32, N, 2.0, None, None)
    yield "axpy_inplace_f64", 0, lambda c: _axpy_inplace(c, f64)
    yield "scale_inplace_f64", 0, lambda c: _scale_inplace(c, f64)                          # x := x * a in place (for_each): the 1R+1W same-buffer ceiling
    yield "scale_f64", 0, lambda c: sg.sg_enqueue(c, sg.SG_MUL, [sg.sg_vec_create(c, f64, N, None), sg.F(2.0)], dst_or_0=sg.sg_vec_create(c, f64, N, 0x7000000))
    yield "ge_row_f64", 0, lambda c: W.ge_row_op(c, N, None, None, 3.0)
    yield "cfg0", 0, lambda c: W.cfg0(c, N, None, None, None)                               # plan P2: pass A + pass B
    yield "cfg0_zbuf", 0, lambda c: W.cfg0(c, N, None, None, None, pz=0x7000000)
    yield "cfg0_nocontract", 0, lambda c: W.cfg0(c, N, None, None, None, contracts=False)
    yield "cfg0_onepass", 0, lambda c: W.cfg0(c, N, None, None, None, keep_z=False)              # plan P1: one pass
    yield "cfg1", 0, lambda c: W.cfg1(c, N, None, None)
    yield "cfg1_keep", 0, lambda c: W.cfg1(c, N, None, None, keep_w=True)
    yield "cfg1_unfused", sg.SG_FLAG_UNFUSED, lambda c: W.cfg1(c, N, None, None)            # one kernel per op
    yield "cfg2", 0, lambda c: W.cfg2(c, N, None)
    yield "cfg3", 0, lambda c: W.cfg3(c, N, None)
    yield "cfg3sum", 0, lambda c: _cfg3_sum(c)                                              # a body (sum) with config 3's two PRE contracts fused into its pass
    yield "sorted_f32", 0, lambda c: _sorted_only(c, f32)
    yield "sorted_f64", 0, lambda c: _sorted_only(c, f64)
    yield "cfg4", 0, lambda c: W.cfg4(c, 4096, None, 0)
    yield "cfg4_gestep", 0, lambda c: _ge_step(c, 0)                                        # Listing 5 loop body
    # matrix-vector products, PAPER.md:217 (without an instance they would run on the 2-D bytecode evaluator)
    yield "matvec_right", 0, lambda c: W.right_multiply(c, 4096, 4096, None, None)
    yield "matvec_left", 0, lambda c: W.left_multiply(c, 4096, 4096, None, None)
    # the rest of the vector API
    yield "isqrt_i32", 0, lambda c: W.project_sqrt(c, i32, N, None, pout=0x7000000)                      # INT -> DOUBLE sqrt
    yield "isqrt_i64", 0, lambda c: W.project_sqrt(c, sg.SG_I64, N, None, pout=0x7000000)
    yield "cast_i32_f32", 0, lambda c: sg.sg_cast(c, sg.sg_vec_create(c, i32, N, None), f32, sg.sg_vec_create(c, f32, N, 0x7000000))
    yield "cast_f64_i32", 0, lambda c: sg.sg_cast(c, sg.sg_vec_create(c, f64, N, None), i32, sg.sg_vec_create(c, i32, N, 0x7000000))
    # the terminal reductions of a stored vector in one pass: integer sum + extrema, float extrema — exact in any
    # order, so these passes take the last part of their tiles through tickets (sg_kernels.cu)
    yield "red_i32", 0, lambda c: _reduce_all(c, i32, (sg.SG_SUM, sg.SG_RMAX, sg.SG_RMIN))
    yield "red_i64", 0, lambda c: _reduce_all(c, sg.SG_I64, (sg.SG_SUM, sg.SG_RMAX, sg.SG_RMIN))
    yield "extrema_f32", 0, lambda c: _reduce_all(c, f32, (sg.SG_RMAX, sg.SG_RMIN))
    yield "extrema_f64", 0, lambda c: _reduce_all(c, f64, (sg.SG_RMAX, sg.SG_RMIN))
    for tag, dt in (("f32", f32), ("f64", f64)):
        yield f"sqrt_{tag}", 0, lambda c, dt=dt: W.project_sqrt(c, dt, N, None, pout=0x7000000)
        yield f"avg_{tag}", 0, lambda c, dt=dt: W.avg(c, dt, N, None)
        yield f"norm_{tag}", 0, lambda c, dt=dt: W.norm2(c, dt, N, None)
        yield f"cdiv_{tag}", 0, lambda c, dt=dt: W.compwise_divide(c, dt, N, None, None, pout=0x7000000, eps=1e-9)  # Listing 2
        yield f"approx_{tag}", 0, lambda c, dt=dt: W.approx_equal(c, dt, N, None, None, 1e-9)


def _axpy_inplace(c, dt):
    x = sg.sg_vec_create(c, dt, N, None)
    y = sg.sg_vec_create(c, dt, N, None)
    ax = sg.sg_enqueue(c, sg.SG_MUL, [x, sg.F(2.0)])
    sg.sg_enqueue(c, sg.SG_ADD, [ax, y], dst_or_0=y)
    sg.sg_release(c, ax)


def _reduce_all(c, dt, kinds):
    x = sg.sg_vec_create(c, dt, N, None)
    return [sg.sg_reduce(c, x, k) for k in kinds]


def _scale_inplace(c, dt):
    x = sg.sg_vec_create(c, dt, N, None)
    sg.sg_enqueue(c, sg.SG_MUL, [x, sg.F(2.0)], dst_or_0=x)


def _ge_step(c, k):
    M = sg.sg_mat_create(c, sg.SG_F64, 4096, 4096, 4096, None)
    det = sg.sg_vec_create(c, sg.SG_F64, 1, None)
    minpiv = sg.sg_vec_create(c, sg.SG_F64, 1, None)
    for h in W.ge_step(c, M, 4096, k, det, minpiv):
        sg.sg_release(c, h)


def _cfg3_sum(c):
    r = W.cfg3(c, N, None, contracts=True)
    return sg.sg_reduce(c, r["x"], sg.SG_SUM)


def _sorted_only(c, dt):
    x = sg.sg_vec_create(c, dt, N, None)
    return sg.sg_forall_adjacent(c, x, sg.SG_LE)


def generate() -> str:
    seen = {}
    lines = [
        "// GENERATED by paper_1410_6685_b200/gen_templates.py from the plan builder's canonical output — do not edit.",
        "// SG_TEMPLATE(index, name, unroll, min_blocks_per_sm, row_unroll, stages, {program})",
    ]
    for name, flags, builder in _chains():
        ctx = sg.sg_ctx_create(-1)
        sg.sg_ctx_set_flags(ctx, flags | sg.SG_FLAG_FORCE_BYTECODE)
        builder(ctx)
        sg.sg_flush(ctx)
        st = sg.sg_plan_stats(ctx)
        for p in range(st.n_passes):
            text = sg.sg_plan_dump(ctx, p)
            if text in seen:
                continue
            tune = TUNE.get(name, TUNE.get(name.split("_")[0]))
            if tune is None:
                # measured and rejected (2^26 fp32 / 2^25 fp64, of the measured peak): unroll 8 for passes with ONE vector input — sqrt 0.94 ->
                # 0.88 / 0.97 -> 0.90, scale 0.92 -> 0.935, sums unchanged: the default stays
                tune = DEFAULT_TUNE
            inst = f"{name}_p{p}"
            seen[text] = inst
            tune = tuple(tune) + (3,) * (4 - len(tune))
            lines.append(f"SG_TEMPLATE({len(seen) - 1}, {inst}, {tune[0]}, {tune[1]}, {tune[2]}, {tune[3]}, {text})")
        sg.sg_ctx_destroy(ctx)
    return "\n".join(lines) + "\n"


def main(argv) -> int:
    text = generate()
    if "--check" in argv:
        cur = open(OUT).read() if os.path.exists(OUT) else ""
        if cur != text:
            print("sg_templates_gen.inc is stale: run python -m paper_1410_6685_b200.gen_templates and rebuild")
            return 1
        return 0
    with open(OUT, "w") as f:
        f.write(text)
    print(f"wrote {OUT}: {text.count('SG_TEMPLATE(') - 1} instances")
    return 0


if __name__ == "__main__":
    sys.exit(main(sys.argv[1:]))
