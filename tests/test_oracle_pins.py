"""Pins for the CPU oracle (no GPU).  Each test checks an oracle primitive against something other than
itself: exact rational arithmetic + correct rounding, closed forms, hand-listed special cases, library
routines (numpy / math.fsum), invariants and brute force on tiny inputs (SURVEY.md §8(c) pin table)."""
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle as orc
from oracle import configs as ocfg

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
RNG = np.random.default_rng(12345)


# ----------------------------------------------------------------------------------------------------------
# helpers: correctly rounded results from exact rationals (independent of the oracle's C arithmetic)
# ----------------------------------------------------------------------------------------------------------
def round_f64(q: Fraction) -> float:
    return q.numerator / q.denominator          # python int/int true division is correctly rounded


def round_f32(q: Fraction) -> np.float32:
    # for one +,-,*,/ of two binary32 operands, rounding to binary64 first is innocuous (53 >= 2*24+2)
    return np.float32(round_f64(q))


def exact(op, a, b):
    fa, fb = Fraction(float(a)), Fraction(float(b))
    return {"add": fa + fb, "sub": fa - fb, "mul": fa * fb, "div": fa / fb if fb else None}[op]


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("op", ["add", "sub", "mul", "div"])
def test_float_arith_is_correctly_rounded(dtype, op):
    a = RNG.standard_normal(64).astype(dtype) * dtype(1e3)
    b = RNG.standard_normal(64).astype(dtype)
    a[:4] = [1.0, -0.0, 3.0, 1e-30]
    b[:4] = [3.0, 7.0, -1e30, 1e30 if dtype is np.float64 else 3e8]
    got = orc.zip(op, a, b)
    rnd = round_f32 if dtype is np.float32 else round_f64
    for i in range(a.size):
        q = exact(op, a[i], b[i])
        want = dtype(rnd(q))
        if q != 0:
            assert got[i] == want and np.signbit(got[i]) == np.signbit(want), (op, a[i], b[i], got[i], want)
        else:
            # an exactly-zero result: the rational has no sign, IEEE 754 fixes it — products and quotients take the XOR of the
            # operand signs; a sum x + y that cancels is +0 under round-to-nearest unless both addends are -0
            sa, sb = bool(np.signbit(a[i])), bool(np.signbit(b[i]))
            if op in ("mul", "div"):
                neg = sa != sb
            else:
                sb_eff = sb if op == "add" else not sb
                neg = sa and sb_eff and a[i] == 0 and b[i] == 0
            assert got[i] == 0 and bool(np.signbit(got[i])) == neg, (op, a[i], b[i], got[i])
    # scalar forms, both operand orders
    s = dtype(2.5)
    got = orc.scalar(op, a, s)
    got_r = orc.scalar(op, a, s, reversed=True)
    for i in range(a.size):
        assert got[i] == dtype(rnd(exact(op, a[i], s)))
        if not (op == "div" and a[i] == 0):
            assert got_r[i] == dtype(rnd(exact(op, s, a[i])))


def test_scalar_is_converted_to_vector_dtype():
    # 0.1 is not representable: a float32 chain must use float32(0.1), never the double (DESIGN.md R-imm)
    a = np.array([1.0, 3.0, 9.0], dtype=np.float32)
    got = orc.scalar("mul", a, 0.1)
    s = np.float32(0.1)
    for i in range(3):
        assert got[i] == round_f32(Fraction(float(a[i])) * Fraction(float(s)))
    # 9 * float32(0.1) = 0.90000004f, whereas a double-promoted 9 * 0.1 rounds to 0.9f: the two readings differ here
    assert got[2] == np.float32(0.90000004) and got[2] != np.float32(9.0 * 0.1)


def test_dyadic_inputs_are_exact():
    a = np.array([0.5, 1.25, -3.0, 1024.0, 2.0 ** -20], dtype=np.float64)
    b = np.array([0.25, -8.0, 0.75, 2.0 ** -10, 4.0], dtype=np.float64)
    assert np.array_equal(orc.zip("add", a, b), [0.75, -6.75, -2.25, 1024.0 + 2.0 ** -10, 4.0 + 2.0 ** -20])
    assert np.array_equal(orc.zip("mul", a, b), [0.125, -10.0, -2.25, 1.0, 2.0 ** -18])
    assert np.array_equal(orc.zip("div", a, b), [2.0, -0.15625, -4.0, 2.0 ** 20, 2.0 ** -22])


def test_fma_canaries_no_contraction():
    # fp32: x = 1+2^-12, c = -(1+2^-11): fl(x*x) + c == 0; a contracted fma gives 2^-24
    x = np.array([1.0 + 2.0 ** -12], dtype=np.float32)
    c = np.array([-(1.0 + 2.0 ** -11)], dtype=np.float32)
    assert orc.zip("add", orc.zip("mul", x, x), c)[0] == 0.0
    xd = np.array([1.0 + 2.0 ** -27], dtype=np.float64)
    cd = np.array([-(1.0 + 2.0 ** -26)], dtype=np.float64)
    assert orc.zip("add", orc.zip("mul", xd, xd), cd)[0] == 0.0
    # the same canary inside the one loop that does multiply-then-subtract in a single C statement pair
    xv = 1.0 + 2.0 ** -27
    M = np.array([[1.0, xv], [xv, 1.0 + 2.0 ** -26]])
    Mo, rowmax, colsum = orc.mat_step(M, 0)
    assert Mo[1, 1] == 0.0            # contracted: -(2^-54)
    assert Mo[1, 0] == 0.0 and rowmax[0] == 0.0 and colsum[1] == 0.0


def test_axpy_matches_blas_definition():
    # aX+Y: y_i + fl(a*x_i), each rounded once
    x = RNG.standard_normal(50)
    y = RNG.standard_normal(50)
    a = 1.7
    got = ocfg.axpy(a, x, y)
    for i in range(50):
        ax = round_f64(Fraction(a) * Fraction(float(x[i])))
        assert got[i] == round_f64(Fraction(ax) + Fraction(float(y[i])))


# ----------------------------------------------------------------------------------------------------------
# integers: wrap-around, truncating division (brute force against python big ints)
# ----------------------------------------------------------------------------------------------------------
def wrap(v, bits):
    v &= (1 << bits) - 1
    return v - (1 << bits) if v >> (bits - 1) else v


def py_int_op(op, a, b, bits):
    lo = -(1 << (bits - 1))
    if op == "add":
        return wrap(a + b, bits)
    if op == "sub":
        return wrap(a - b, bits)
    if op == "mul":
        return wrap(a * b, bits)
    if op == "div":
        if b == 0:
            return 0
        if a == lo and b == -1:
            return lo
        q = abs(a) // abs(b)
        return q if (a < 0) == (b < 0) else -q
    if op == "mod":
        if b == 0 or b == -1:
            return 0
        r = abs(a) % abs(b)
        return -r if a < 0 else r
    raise KeyError(op)


@pytest.mark.parametrize("dtype,bits", [(np.int32, 32), (np.int64, 64)])
def test_int_arith_brute_force(dtype, bits):
    lo, hi = -(1 << (bits - 1)), (1 << (bits - 1)) - 1
    special = [0, 1, -1, 2, -2, 7, -7, 3, lo, hi, lo + 1, hi - 1, 123456789, -987654321]
    a = np.array([x for x in special for _ in special], dtype=dtype)
    b = np.array([y for _ in special for y in special], dtype=dtype)
    for op in ["add", "sub", "mul", "div", "mod"]:
        got = orc.zip(op, a, b)
        for i in range(a.size):
            assert int(got[i]) == py_int_op(op, int(a[i]), int(b[i]), bits), (op, a[i], b[i])
    got = orc.scalar("mod", a, 7)
    for i in range(a.size):
        assert int(got[i]) == py_int_op("mod", int(a[i]), 7, bits)
    got = orc.scalar("sub", a, 5, reversed=True)
    for i in range(a.size):
        assert int(got[i]) == wrap(5 - int(a[i]), bits)


def test_int_abs_neg():
    a = np.array([0, 5, -5, -(2 ** 31), 2 ** 31 - 1], dtype=np.int32)
    assert orc.unary("abs", a).tolist() == [0, 5, 5, -(2 ** 31), 2 ** 31 - 1]
    assert orc.unary("neg", a).tolist() == [0, -5, 5, -(2 ** 31), -(2 ** 31 - 1)]


# ----------------------------------------------------------------------------------------------------------
# unary, elementwise min/max, comparisons: hand-listed special cases
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_float_abs_neg_sign_bit(dtype):
    a = np.array([0.0, -0.0, 1.5, -1.5, np.inf, -np.inf], dtype=dtype)
    r = orc.unary("abs", a)
    assert np.array_equal(r, [0.0, 0.0, 1.5, 1.5, np.inf, np.inf]) and not np.signbit(r).any()
    r = orc.unary("neg", a)
    assert np.array_equal(r, [-0.0, 0.0, -1.5, 1.5, -np.inf, np.inf])
    assert np.signbit(r).tolist() == [True, False, True, False, True, False]
    assert np.isnan(orc.unary("abs", np.array([np.nan], dtype=dtype))[0])


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_elementwise_min_max_ternary(dtype):
    # MIN(a,b) = (b<a)?b:a ; MAX(a,b) = (a<b)?b:a   (DESIGN.md R-minmax)
    nan = np.nan
    a = np.array([1.0, 2.0, 0.0, -0.0, nan, 1.0, 3.0], dtype=dtype)
    b = np.array([2.0, 1.0, -0.0, 0.0, 1.0, nan, 3.0], dtype=dtype)
    mn = orc.zip("min", a, b)
    mx = orc.zip("max", a, b)
    assert mn[0] == 1 and mn[1] == 1 and mx[0] == 2 and mx[1] == 2
    assert not np.signbit(mn[2]) and np.signbit(mn[3])          # equal zeros: first operand is returned
    assert not np.signbit(mx[2]) and np.signbit(mx[3])
    assert np.isnan(mn[4]) and mn[5] == 1.0                      # a NaN first operand is returned, a NaN second is not
    assert np.isnan(mx[4]) and mx[5] == 1.0
    assert mn[6] == 3 and mx[6] == 3
    # on NaN-free data without signed-zero ties it is the library minimum/maximum
    x = RNG.standard_normal(200).astype(dtype)
    y = RNG.standard_normal(200).astype(dtype)
    assert np.array_equal(orc.zip("min", x, y), np.minimum(x, y))
    assert np.array_equal(orc.zip("max", x, y), np.maximum(x, y))


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
def test_comparisons_vs_library(dtype):
    a = (RNG.integers(-5, 5, 300)).astype(dtype)
    b = (RNG.integers(-5, 5, 300)).astype(dtype)
    lib = {"eq": np.equal, "ne": np.not_equal, "lt": np.less, "le": np.less_equal, "gt": np.greater, "ge": np.greater_equal}
    for op, f in lib.items():
        assert np.array_equal(orc.cmp(op, a, b).astype(bool), f(a, b)), op
        assert np.array_equal(orc.cmp_scalar(op, a, 1).astype(bool), f(a, dtype(1))), op


def test_comparisons_nan_and_signed_zero():
    a = np.array([np.nan, np.nan, 0.0, -0.0], dtype=np.float64)
    b = np.array([np.nan, 1.0, -0.0, 0.0], dtype=np.float64)
    assert orc.cmp("eq", a, b).tolist() == [0, 0, 1, 1]
    assert orc.cmp("ne", a, b).tolist() == [1, 1, 0, 0]
    for op in ["lt", "gt"]:
        assert orc.cmp(op, a, b).tolist() == [0, 0, 0, 0]
    for op in ["le", "ge"]:
        assert orc.cmp(op, a, b).tolist() == [0, 0, 1, 1]


def test_logic_truth_tables():
    a = np.array([0, 0, 1, 1], dtype=np.uint8)
    b = np.array([0, 1, 0, 1], dtype=np.uint8)
    assert orc.logic("and", a, b).tolist() == [0, 0, 0, 1]
    assert orc.logic("or", a, b).tolist() == [0, 1, 1, 1]
    assert orc.logic("not", a).tolist() == [1, 1, 0, 0]


# ----------------------------------------------------------------------------------------------------------
# sum
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
@pytest.mark.parametrize("n", [0, 1, 2, 1000, 4097, 1 << 20])
def test_sum_arithmetic_sequence_closed_form(dtype, n):
    if dtype is np.float32 and n > (1 << 24):
        pytest.skip("iota not exact in float32")
    a = np.arange(n).astype(dtype)
    assert orc.sum(a) == n * (n - 1) // 2


def test_sum_constant_dyadic():
    assert orc.sum(np.full(12345, 0.375)) == 12345 * 0.375
    assert orc.sum(np.full(777, np.float32(-2.0 ** -9))) == -777 * 2.0 ** -9


def test_sum_ill_conditioned_matches_exact_fsum():
    # math.fsum returns the correctly rounded exact sum: an independent library routine
    x = np.array([1e100, 1.0, -1e100, 1e-30, 3.0, -4.0, 2.0 ** -60] * 37, dtype=np.float64)
    RNG.shuffle(x)
    got = orc.sum(x)
    want = math.fsum(x.tolist())
    assert want != 0.0
    assert abs(got - want) <= 2.0 ** -63 * float(np.abs(x).sum())   # long double resolution of the compensated loop
    y = RNG.standard_normal(100000) * np.exp(RNG.uniform(-20, 20, 100000))
    assert orc.sum(y) == pytest.approx(math.fsum(y.tolist()), rel=1e-15)
    z = (RNG.standard_normal(100000)).astype(np.float32)
    assert orc.sum(z) == math.fsum(z.astype(np.float64).tolist())    # n * 2^-64 relative: rounds to the same double


def test_sum_int_wraps_in_int64():
    a = np.full(5, np.iinfo(np.int64).max, dtype=np.int64)
    assert orc.sum(a) == wrap(5 * (2 ** 63 - 1), 64)
    b = np.array([-(2 ** 31), 2 ** 31 - 1, -1], dtype=np.int32)
    assert orc.sum(b) == -2                     # widened to int64 before adding: no int32 wrap


def test_dot_product_listing4_matches_exact():
    # Listing 4: compwise_multiply then sum; products rounded once, then summed
    a = RNG.standard_normal(5000)
    b = RNG.standard_normal(5000)
    prods = [round_f64(Fraction(float(x)) * Fraction(float(y))) for x, y in zip(a, b)]
    assert ocfg.dot_product(a, b) == math.fsum(prods)
    # and it is the library inner product up to summation order
    assert ocfg.dot_product(a, b) == pytest.approx(float(np.dot(a, b)), rel=1e-12)


# ----------------------------------------------------------------------------------------------------------
# max / min
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
def test_extremum_of_permutation(dtype):
    n = 10007
    p = RNG.permutation(n).astype(dtype)
    assert orc.max(p) == n - 1 and orc.min(p) == 0
    for pos in [0, 1, 31, 32, 1023, 1024, n - 1]:
        q = p.copy()
        q[pos] = n + 5
        assert orc.max(q) == n + 5
        q[pos] = -7
        assert orc.min(q) == -7
    x = (RNG.standard_normal(5000) * 100).astype(dtype)
    assert orc.max(x) == np.max(x) and orc.min(x) == np.min(x)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_extremum_total_order(dtype):
    z = np.array([0.0, -0.0], dtype=dtype)
    assert np.signbit(orc.min(z)) and not np.signbit(orc.max(z))
    z = z[::-1].copy()
    assert np.signbit(orc.min(z)) and not np.signbit(orc.max(z))
    w = np.array([1.0, np.inf, -np.inf, np.nan, -2.0], dtype=dtype)      # +NaN sorts above +inf
    assert np.isnan(orc.max(w)) and orc.min(w) == -np.inf
    w[3] = -np.nan                                                       # -NaN sorts below -inf
    w[3] = np.copysign(np.nan, -1.0)
    assert np.isnan(orc.min(w)) and orc.max(w) == np.inf


def test_extremum_empty_is_an_error():
    with pytest.raises(ValueError):
        orc.max(np.empty(0, dtype=np.float64))
    with pytest.raises(ValueError):
        orc.min(np.empty(0, dtype=np.int32))


# ----------------------------------------------------------------------------------------------------------
# for_all / exists / count / neighbour predicates
# ----------------------------------------------------------------------------------------------------------
def test_quantifiers_vs_library_and_duality():
    for n in [0, 1, 2, 33, 1025]:
        for trial in range(6):
            m = (RNG.random(n) < [0.0, 1.0, 0.5, 0.02, 0.98, 0.5][trial]).astype(np.uint8)
            assert orc.all(m) == bool(np.all(m))
            assert orc.any(m) == bool(np.any(m))
            assert orc.count(m) == int(np.count_nonzero(m))
            assert orc.all(m) == (not orc.any(orc.logic("not", m)))      # for_all(p) == !exists(!p)
    assert orc.all(np.empty(0, dtype=np.uint8)) is True and orc.any(np.empty(0, dtype=np.uint8)) is False


def test_single_witness_every_position_class():
    n = 4099
    for pos in [0, 1, 31, 32, 33, 1023, 1024, 1025, 4096, n - 1]:
        m = np.ones(n, dtype=np.uint8)
        m[pos] = 0
        assert orc.all(m) is False and orc.any(orc.logic("not", m)) is True and orc.count(m) == n - 1


@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32])
def test_is_sorted(dtype):
    n = 3001
    iota = np.arange(n).astype(dtype)
    assert orc.all(orc.adj("le", iota)) is True
    assert orc.all(orc.adj("le", iota[::-1].copy())) is False
    assert orc.all(orc.adj("le", np.full(n, 7).astype(dtype))) is True
    assert orc.all(orc.adj("lt", np.full(n, 7).astype(dtype))) is False
    assert orc.adj("le", iota[:1]).size == 0 and orc.all(orc.adj("le", iota[:1])) is True   # n <= 1 => sorted
    assert orc.all(orc.adj("le", iota[:0])) is True
    for j in [1, 2, 32, 33, 1024, n - 1]:
        x = iota.copy()
        x[j] = x[j - 1] - 1                       # exactly one descent, at the pair (j-1, j)
        b = orc.adj("le", x)
        assert b.size == n - 1
        viol = np.flatnonzero(b == 0)
        assert orc.all(b) is False and viol.tolist()[0] == j - 1
    x = np.sort(RNG.standard_normal(n)).astype(dtype)
    assert orc.all(orc.adj("le", x)) == bool(np.all(np.diff(x) >= 0))
    y = RNG.standard_normal(n).astype(dtype)
    assert np.array_equal(orc.adj("le", y).astype(bool), y[:-1] <= y[1:])
    assert np.array_equal(orc.adj("gt", y).astype(bool), y[:-1] > y[1:])


# ----------------------------------------------------------------------------------------------------------
# filter
# ----------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [np.float32, np.float64, np.int32, np.int64])
def test_filter_vs_copy_if(dtype):
    for n in [0, 1, 2, 31, 32, 33, 1000, 4097]:
        a = RNG.integers(-1000, 1000, n).astype(dtype)
        m = (RNG.random(n) < 0.3).astype(np.uint8)
        got = orc.filter(a, m)
        assert np.array_equal(got, a[m.astype(bool)])
        assert got.size == orc.count(m)
        assert np.array_equal(orc.filter(a, np.ones(n, dtype=np.uint8)), a)
        assert orc.filter(a, np.zeros(n, dtype=np.uint8)).size == 0


@pytest.mark.parametrize("n", [0, 3, 4, 10, 11, 7000, 100003])
def test_filter_closed_form_mod7(n):
    # x = 0..n-1 keeping x mod 7 == 3: m = floor((n+3)/7) items 3, 10, 17, ...; sum = 3m + 7m(m-1)/2
    r = ocfg.cfg2(np.arange(n, dtype=np.int32))
    m = (n + 3) // 7
    assert r["count"] == m and r["count_mask"] == m
    assert r["sum"] == 3 * m + 7 * m * (m - 1) // 2
    assert r["kept"].tolist() == list(range(3, n, 7))        # stable: ascending order preserved


def test_filter_is_stable_subsequence():
    a = RNG.integers(0, 2 ** 31, 5000).astype(np.int32)
    r = ocfg.cfg2(a)
    it = iter(a.tolist())
    assert all(any(v == w for w in it) for v in r["kept"].tolist())       # subsequence test
    assert all(v % 7 == 3 for v in r["kept"].tolist())
    assert r["count"] == sum(1 for v in a.tolist() if v % 7 == 3)
    assert r["sum"] == sum(v for v in a.tolist() if v % 7 == 3)


# ----------------------------------------------------------------------------------------------------------
# matrix step
# ----------------------------------------------------------------------------------------------------------
def load_matstep_golden():
    cases, cur = [], {}
    for line in open(os.path.join(GOLDEN, "matstep_4x4.txt")):
        if line.startswith("#") or not line.strip():
            continue
        key, *vals = line.split()
        if key == "k" and cur:
            cases.append(cur)
            cur = {}
        cur[key] = int(vals[0]) if key == "k" else np.array([float(v) for v in vals])
    cases.append(cur)
    return cases


def test_matstep_hand_derived_golden():
    for case in load_matstep_golden():
        k = case["k"]
        for impl in (ocfg.cfg4, ocfg.cfg4_unfused):
            r = impl(case["M"].reshape(4, 4), k)
            assert np.array_equal(r["M"], case["Mout"].reshape(4, 4))
            assert np.array_equal(r["rowmax"], case["rowmax"])
            assert np.array_equal(r["colsum"], case["colsum"])


def test_matstep_exact_rational_and_invariants():
    n, k = 9, 3
    M = RNG.standard_normal((n, n))
    M[np.arange(n), np.arange(n)] += n
    r = ocfg.cfg4(M, k)
    r2 = ocfg.cfg4_unfused(M, k)
    for key in ("M", "rowmax", "colsum"):
        assert np.array_equal(r[key], r2[key]), key                       # plain loop == primitive-by-primitive
    assert np.array_equal(r["M"][: k + 1], M[: k + 1])                     # rows <= k untouched bit for bit
    piv = Fraction(float(M[k, k]))
    for j in range(k + 1, n):
        f = round_f64(Fraction(float(M[j, k])) / piv)
        for c in range(n):
            t = round_f64(Fraction(f) * Fraction(float(M[k, c])))
            assert r["M"][j, c] == round_f64(Fraction(float(M[j, c])) - Fraction(t))
        assert r["rowmax"][j - k - 1] == np.max(np.abs(r["M"][j]))
        assert abs(r["M"][j, k]) <= 4 * np.finfo(float).eps * abs(M[j, k])     # eliminated entry is rounding-small
    for c in range(n):
        assert r["colsum"][c] == math.fsum(r["M"][k + 1:, c].tolist())
    last = ocfg.cfg4(M, n - 1)                                             # k = n-1: nothing changes
    assert np.array_equal(last["M"], M) and last["rowmax"].size == 0 and not last["colsum"].any()


def test_matstep_column_sampled_form_equals_full():
    # the sampled-column check used at 16384^2: run the definition on columns [k] + S with pivot column 0
    n, k = 40, 7
    M = RNG.standard_normal((n, n))
    M[np.arange(n), np.arange(n)] += n
    full = ocfg.cfg4(M, k)
    S = [0, 5, 7, 8, 39]
    Ms, rowmax_s, colsum_s = orc.mat_step(M[:, [k] + S], k, 0)
    assert np.array_equal(Ms[:, 1:], full["M"][:, S])
    assert np.array_equal(colsum_s[1:], full["colsum"][S])


# ----------------------------------------------------------------------------------------------------------
# configs 0, 1, 3 (composition order / parenthesisation)
# ----------------------------------------------------------------------------------------------------------
def test_cfg0_chain_exact_rational():
    a, b, c = (RNG.uniform(-1, 1, 40) for _ in range(3))
    r = ocfg.cfg0(a, b, c)
    for i in range(40):
        t1 = round_f64(Fraction(float(a[i])) + Fraction(float(b[i])))
        t2 = round_f64(Fraction(t1) * Fraction(2.5))
        assert r["z"][i] == round_f64(Fraction(t2) - Fraction(float(c[i])))
    assert r["post"] is True
    assert r["pre"] == bool((a > 0.99).any())
    assert r["max"] == r["z"].max() and r["min"] == r["z"].min()
    assert r["sum"] == math.fsum(r["z"].tolist())


def test_cfg1_chain_exact_rational():
    x = RNG.standard_normal(40).astype(np.float32)
    y = RNG.standard_normal(40).astype(np.float32)
    w = ocfg.cfg1_chain(x, y)
    F = lambda v: Fraction(float(v))
    for i in range(40):
        t1 = round_f32(F(x[i]) * F(y[i]))
        t2 = round_f32(F(t1) + F(np.float32(0.5)))
        t3 = abs(t2)
        t4 = y[i] if y[i] < x[i] else x[i]
        t5 = round_f32(F(t4) * 3)
        t6 = round_f32(F(t3) - F(t5))
        t7 = round_f32(F(y[i]) * F(y[i]))
        t8 = round_f32(1 + F(t7))
        t9 = round_f32(F(x[i]) / F(t8))
        assert w[i] == round_f32(F(t6) + F(t9)), i
    r = ocfg.cfg1(x, y)
    assert r["sum"] == math.fsum(w.astype(np.float64).tolist()) and r["max"] == w.max()


def test_cfg3_clean_and_injected():
    from paper_1410_6685_b200 import inputs
    n = 1 << 16
    x = inputs.sorted_cumsum_f32(4, 0, n)
    assert ocfg.cfg3(x) == {"pre": True, "post": True}
    j = inputs.violation_index(4, n)
    assert 1 <= j <= n - 2
    inputs.inject_unsorted(x, j)
    assert ocfg.cfg3(x) == {"pre": True, "post": False}
    assert np.flatnonzero(orc.adj("le", x) == 0).tolist() == [j - 1]      # only the pair (j-1, j) is broken
    x[5] = -1.0
    assert ocfg.cfg3(x)["pre"] is False


# ---------------------------------------------------------------------------------------------------------
# Determinant by Gaussian elimination (Listing 5) — SURVEY.md §8(f)(1)
# ---------------------------------------------------------------------------------------------------------
def _leibniz_det(A):
    """Brute force: sum over all permutations, exact rational arithmetic."""
    import itertools
    n = len(A)
    total = Fraction(0)
    for perm in itertools.permutations(range(n)):
        sign = 1
        for i in range(n):
            for j in range(i + 1, n):
                if perm[i] > perm[j]:
                    sign = -sign
        term = Fraction(sign)
        for i in range(n):
            term *= Fraction(float(A[i][perm[i]]))
        total += term
    return total


def _exact_lu_matrix(n, rng):
    """M = L @ U with unit-lower L and upper U of small dyadic entries and power-of-two pivots: every quotient, product
    and difference of the elimination is exact in fp64, so it must return U bit for bit and det = prod(diag U)."""
    L = np.tril(rng.integers(-4, 5, (n, n)) / 4.0, -1) + np.eye(n)
    U = np.triu(rng.integers(-8, 9, (n, n)) / 2.0, 1) + np.diag(2.0 ** rng.integers(-2, 3, n) * rng.choice([-1.0, 1.0], n))
    return L, U, L @ U


def test_ge_determinant_exact_lu_and_brute_force():
    rng = np.random.default_rng(11)
    for n in (1, 2, 3, 4, 5, 6):
        L, U, M = _exact_lu_matrix(n, rng)
        det, E, zs = orc.ge_determinant(M)
        assert zs == -1
        assert np.array_equal(np.triu(E), U)                               # elimination recovers U exactly
        assert not np.tril(E, -1).any()                                    # and exact zeros below the diagonal
        assert Fraction(det) == math.prod(Fraction(float(u)) for u in np.diag(U))
        assert Fraction(det) == _leibniz_det(M.tolist())                   # == the definition of the determinant


def test_ge_determinant_hand_values_triangular_and_singular():
    det, E, zs = orc.ge_determinant([[2.0, 3.0], [4.0, 5.0]])              # f = 2, row 1 -> [0, -1]; 2 * -1
    assert det == -2.0 and np.array_equal(E, [[2.0, 3.0], [0.0, -1.0]]) and zs == -1
    T = np.triu(RNG.standard_normal((7, 7))) + 3 * np.eye(7)
    det, E, zs = orc.ge_determinant(T)                                     # upper triangular: nothing to eliminate
    ref = 1.0
    for d in np.diag(T):
        ref = ref * d                                                      # PAPER.md:338, in step order
    assert det == ref and np.array_equal(E, T)
    # Zero pivots, derived from the listing's statement order: `Result := Result * pivot` comes BEFORE
    # `if not double_approx_equals (pivot, 0.0)`, whose else-branch ends the loop.
    det, E, zs = orc.ge_determinant([[1.0, 2.0], [2.0, 4.0]])              # step 0: Result = 1, row 1 -> [0, 0]; step 1: pivot 0 -> Result = 1 * 0
    assert det == 0.0 and not np.signbit(det) and zs == 1 and np.array_equal(E, [[1.0, 2.0], [0.0, 0.0]])
    det, E, zs = orc.ge_determinant([[-1.0, 2.0], [3.0, -6.0]])            # step 0: Result = -1, f = -3, row 1 -> [0, 0]; step 1: Result = -1 * 0 = -0
    assert det == 0.0 and np.signbit(det) and zs == 1 and np.array_equal(E, [[-1.0, 2.0], [0.0, 0.0]])
    M = [[1e-9, 1.0], [1.0, 1.0]]
    det, E, zs = orc.ge_determinant(M, eps=1e-6)                           # approximately zero with an explicit eps: Result = 1 * 1e-9, loop ends,
    assert det == 1e-9 and zs == 0 and np.array_equal(E, M)                # no row has been touched — NOT a hard-wired 0.0
    det, E, zs = orc.ge_determinant([[2.0, 1.0], [4.0, 2.0 + 2.0 ** -40]], eps=1e-6)   # step 0: Result = 2, f = 2, row 1 -> [0, 2^-40]; step 1: Result = 2 * 2^-40
    assert det == 2.0 ** -39 and zs == 1 and np.array_equal(E, [[2.0, 1.0], [0.0, 2.0 ** -40]])
    # the per-row guard: a row whose entry below the pivot is approximately zero is left as it is
    M = [[2.0, 1.0], [1e-9, 3.0]]
    det, E, zs = orc.ge_determinant(M, eps=1e-6)
    assert det == 6.0 and zs == -1 and np.array_equal(E, M)                # without the guard row 1 would become [~0, 3 - 5e-10] and det 5.999999999
    det, E, zs = orc.ge_determinant(M, eps=0.0)                            # eps = 0: 1e-9 is not zero, the row IS eliminated
    f = 1e-9 / 2.0
    assert np.array_equal(E, [[2.0, 1.0], [1e-9 - f * 2.0, 3.0 - f * 1.0]]) and det == 2.0 * (3.0 - f * 1.0) and zs == -1
    det, _, zs = orc.ge_determinant(np.zeros((0, 0)))                      # empty product
    assert det == 1.0 and zs == -1


def test_ge_determinant_steps_are_matstep_and_library_det():
    n = 48
    M = RNG.uniform(-1, 1, (n, n)) / n + np.eye(n)
    det, E, zs = orc.ge_determinant(M)
    A = M.copy()                                                           # the loop is n applications of the cfg4 step
    ref = 1.0
    for k in range(n):
        ref = ref * A[k, k]
        A = orc.mat_step(A, k)[0]
    assert det == ref and np.array_equal(E, A) and zs == -1
    assert abs(det - np.linalg.det(M)) <= 1e-12 * abs(det)                 # LAPACK (partial pivoting): same value to rounding
    sign, logabs = np.linalg.slogdet(M)
    assert sign == np.sign(det) and abs(math.log(abs(det)) - logabs) <= 1e-12
    s = 0.5                                                                # det(s*M) = s^n det(M): exact for a power of two
    assert orc.ge_determinant(s * M)[0] == det * s ** n


# ----------------------------------------------------------------------------------------------------------
# rest of the vector API — sqrt projection, avg,
# compwise_divide with its built-in non-zero contract (Listing 2), approximate equality
#
# ----------------------------------------------------------------------------------------------------------
def _is_correctly_rounded_sqrt(x: float, r: float, dtype) -> bool:
    """r == RN(sqrt(x)) decided in exact integer/rational arithmetic: the two neighbours' midpoints bracket sqrt(x),
    i.e. ((r_prev + r)/2)^2 <= x <= ((r + r_next)/2)^2 (a tie cannot occur for sqrt of a binary float)."""
    lo = np.nextafter(dtype(r), dtype(-np.inf))
    hi = np.nextafter(dtype(r), dtype(np.inf))
    X, R, LO, HI = Fraction(float(x)), Fraction(float(r)), Fraction(float(lo)), Fraction(float(hi))
    return ((LO + R) / 2) ** 2 < X < ((R + HI) / 2) ** 2 or R * R == X


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_sqrt_is_correctly_rounded(dtype):
    a = np.concatenate([RNG.uniform(0, 4, 300), RNG.uniform(0, 1e-30, 50), RNG.uniform(1e30, 1e38, 50),
                        [2.0, 3.0, 0.5, 1e-40 if dtype is np.float32 else 5e-324]]).astype(dtype)
    r = orc.unary("sqrt", a)
    assert r.dtype == a.dtype
    for x, y in zip(a, r):
        assert _is_correctly_rounded_sqrt(x, y, dtype), (x, y)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_sqrt_perfect_squares_and_special_values(dtype):
    k = np.arange(0, 4096, dtype=np.int64)
    assert np.array_equal(orc.unary("sqrt", (k * k).astype(dtype)), k.astype(dtype))          # exact (k^2 < 2^24)
    p = np.array([4.0 ** e for e in range(-20, 21)], dtype=dtype)
    assert np.array_equal(orc.unary("sqrt", p), np.array([2.0 ** e for e in range(-20, 21)], dtype=dtype))
    s = orc.unary("sqrt", np.array([0.0, -0.0, np.inf, -1.0, np.nan], dtype=dtype))
    assert s[0] == 0 and not np.signbit(s[0]) and s[1] == 0 and np.signbit(s[1]) and s[2] == np.inf
    assert np.isnan(s[3]) and np.isnan(s[4])
    with pytest.raises(TypeError):
        orc.unary("sqrt", np.arange(4, dtype=np.int32))


def test_sqrt_matches_library_routine():
    for dtype in (np.float32, np.float64):
        a = np.abs(RNG.standard_normal(5000)).astype(dtype)
        assert np.array_equal(orc.unary("sqrt", a), np.sqrt(a))
    assert orc.unary("sqrt", np.array([2.0]))[0] == math.sqrt(2.0)


def test_avg_closed_forms():
    for n in (1, 2, 1000, 4097):
        assert orc.avg(np.arange(n, dtype=np.float64)) == (n - 1) / 2                        # n(n-1)/2 / n, exact
        assert orc.avg(np.arange(n, dtype=np.int32)) == (n - 1) / 2
    assert orc.avg(np.full(777, 0.375, dtype=np.float32)) == 0.375
    a = RNG.uniform(-1, 1, 3001)
    exact_avg = sum(Fraction(float(v)) for v in a) / len(a)
    assert abs(Fraction(orc.avg(a)) - exact_avg) <= abs(exact_avg) * Fraction(1, 2 ** 50)
    with pytest.raises(ValueError):
        orc.avg(np.zeros(0))


def test_compwise_divide_contract_listing2():
    """Listing 2: require not other.exists(is_zero); ensure Result * other = Current (read as the
    approximate equality of PAPER.md:339, since a/b*b rounds twice)."""
    a = RNG.uniform(-4, 4, 2000)
    b = RNG.uniform(0.5, 2, 2000)
    pre_violated = orc.any(orc.cmp_scalar("eq", b, 0.0))
    assert pre_violated is False
    q = orc.zip("div", a, b)
    for x, y, z in zip(a[:200], b[:200], q[:200]):
        assert z == round_f64(Fraction(float(x)) / Fraction(float(y)))
    back = orc.zip("mul", q, b)
    approx = orc.cmp_scalar("le", orc.unary("abs", orc.zip("sub", back, a)), 1e-12)
    assert orc.all(approx) is True
    assert orc.all(orc.cmp("eq", back, a)) == bool(np.all(q * b == a))                       # exact EQ is a different predicate
    b2 = b.copy(); b2[1234] = 0.0
    assert orc.any(orc.cmp_scalar("eq", b2, 0.0)) is True
    b3 = b.copy(); b3[7] = -0.0
    assert orc.any(orc.cmp_scalar("eq", b3, 0.0)) is True                                    # -0 == +0


def test_vector_norm_pythagorean():
    """sqrt(sum(x*x)) on integer vectors whose norm is an integer: (3,4)->5, (1,2,2)->3, (2,3,6)->7, k copies of (3,4)*..."""
    for v, nrm in (([3, 4], 5), ([1, 2, 2], 3), ([2, 3, 6], 7), ([1, 4, 8], 9), ([3, 4] * 4, 10)):
        x = np.array(v, dtype=np.float64)
        s = np.array([orc.sum(orc.zip("mul", x, x))])
        assert orc.unary("sqrt", s)[0] == nrm


# ----------------------------------------------------------------------------------------------------------
# quicksort (Listing 3) and concatenate
# ----------------------------------------------------------------------------------------------------------
def test_concatenate_vs_list_semantics():
    a, b = np.arange(5, dtype=np.float32), np.arange(7, 10, dtype=np.float32)
    assert ocfg.concatenate(a, b).tolist() == a.tolist() + b.tolist()
    assert ocfg.concatenate(a[:0], b).tolist() == b.tolist() and ocfg.concatenate(a, b[:0]).tolist() == a.tolist()


@pytest.mark.parametrize("n", [1, 2, 3, 10, 257, 3000])
def test_quicksort_matches_library_sort_and_listing3_postconditions(n):
    for a in (RNG.standard_normal(n).astype(np.float32),
              RNG.integers(-5, 6, n).astype(np.float32),                    # many duplicates
              np.arange(n, dtype=np.float32), np.arange(n, dtype=np.float32)[::-1].copy(), np.zeros(n, dtype=np.float32)):
        r = ocfg.quicksort(a)
        assert r.dtype == a.dtype and r.size == a.size                       # ensure Result.count = a.count
        assert orc.all(orc.adj("le", r))                                     # ensure Result.is_sorted
        assert np.array_equal(r, np.sort(a, kind="stable"))
        assert sorted(r.tolist()) == r.tolist() and sorted(a.tolist()) == r.tolist()


def test_quicksort_equal_keys_keep_their_order_and_empty_is_rejected():
    a = np.array([0.0, 3.0, -0.0, 1.0, 0.0, -0.0, 3.0], dtype=np.float32)     # -0 == +0: one `mid`, stable filter keeps the order
    r = ocfg.quicksort(a)
    assert r.tolist() == [0.0, 0.0, 0.0, 0.0, 1.0, 3.0, 3.0]
    assert np.signbit(r[:4]).tolist() == [False, True, False, True]
    with pytest.raises(ValueError):
        ocfg.quicksort(np.zeros(0, dtype=np.float32))


# ----------------------------------------------------------------------------------------------------------
# matrix-vector products
# ----------------------------------------------------------------------------------------------------------
def test_matvec_exact_integer_regime_identity_and_hand_values():
    M = RNG.integers(-8, 9, (37, 53)).astype(np.float64)
    v, w = RNG.integers(-8, 9, 53).astype(np.float64), RNG.integers(-8, 9, 37).astype(np.float64)
    assert np.array_equal(ocfg.right_multiply(M, v), (M.astype(np.int64) @ v.astype(np.int64)).astype(np.float64))   # exact: any order agrees
    assert np.array_equal(ocfg.left_multiply(w, M), (w.astype(np.int64) @ M.astype(np.int64)).astype(np.float64))
    x = RNG.standard_normal(9)
    assert np.array_equal(ocfg.right_multiply(np.eye(9), x), x) and np.array_equal(ocfg.left_multiply(x, np.eye(9)), x)
    A = np.array([[1.0, 2.0, 3.0], [4.0, 5.0, 6.0]])
    assert ocfg.right_multiply(A, np.array([1.0, 0.5, -1.0])).tolist() == [-1.0, 0.5]      # not symmetric: a transposed operand fails
    assert ocfg.left_multiply(np.array([2.0, -1.0]), A).tolist() == [-2.0, -1.0, 0.0]


def test_matvec_general_values_against_exact_rationals():
    M, v, w = RNG.standard_normal((5, 7)), RNG.standard_normal(7), RNG.standard_normal(5)
    r, l = ocfg.right_multiply(M, v), ocfg.left_multiply(w, M)
    for i in range(5):      # each product rounds once, the sum of the ROUNDED products is then (nearly) exact
        ex = sum(Fraction(float(M[i, c] * v[c])) for c in range(7))
        assert abs(Fraction(float(r[i])) - ex) <= abs(ex) * Fraction(1, 2 ** 51)
    for c in range(7):
        ex = sum(Fraction(float(w[i] * M[i, c])) for i in range(5))
        assert abs(Fraction(float(l[c])) - ex) <= abs(ex) * Fraction(1, 2 ** 51)


def test_transpose_hand_values_involution_and_library():
    A = np.array([[1.0, 2.0, 3.0], [4.0, 5.0, 6.0]])
    assert ocfg.transpose(A).tolist() == [[1.0, 4.0], [2.0, 5.0], [3.0, 6.0]]
    for shape in ((1, 1), (1, 7), (7, 1), (33, 65), (130, 64)):
        for dt in (np.float32, np.float64, np.int32):
            M = RNG.integers(-1000, 1000, shape).astype(dt)
            T = ocfg.transpose(M)
            assert T.shape == shape[::-1] and T.dtype == M.dtype and T.flags["C_CONTIGUOUS"]
            assert np.array_equal(ocfg.transpose(T), M)                     # involution
            assert np.array_equal(T, M.T)                                   # library view
            assert all(T[j, i] == M[i, j] for i in range(0, shape[0], 5) for j in range(0, shape[1], 3))


# ----------------------------------------------------------------------------------------------------------
# the dtype-changing projection (R23)
# ----------------------------------------------------------------------------------------------------------
def _nearest_even(q: Fraction, mant_bits: int) -> Fraction:
    """q rounded to `mant_bits` significant bits, ties to even, from the definition (no floating point involved)."""
    if q == 0:
        return Fraction(0)
    sign, q = (-1 if q < 0 else 1), abs(q)
    e = q.numerator.bit_length() - q.denominator.bit_length()
    if Fraction(2) ** e > q:
        e -= 1
    ulp = Fraction(2) ** (e - mant_bits + 1)
    k, r = divmod(q, ulp)
    if r > ulp / 2 or (r == ulp / 2 and k % 2 == 1):
        k += 1
    return sign * k * ulp


def test_cast_int_to_float_rounds_to_nearest_even():
    i32 = np.array([0, 1, -1, 2 ** 24, 2 ** 24 + 1, 2 ** 24 + 2, 2 ** 24 + 3, -(2 ** 24 + 1), -(2 ** 24 + 3), 2 ** 31 - 1, -2 ** 31, 123456789], dtype=np.int32)
    got = orc.cast(i32, np.float32)
    for x, g in zip(i32.tolist(), got.tolist()):
        assert Fraction(g) == _nearest_even(Fraction(x), 24), (x, g)
    assert got[4] == 2.0 ** 24 and got[6] == 2.0 ** 24 + 4                # the two ties: 2^24+1 -> even 2^24, 2^24+3 -> even 2^24+4
    assert orc.cast(i32, np.float64).tolist() == [float(x) for x in i32.tolist()]      # every int32 is exact in a double
    i64 = np.array([2 ** 53, 2 ** 53 + 1, 2 ** 53 + 2, 2 ** 53 + 3, -(2 ** 53 + 1), 2 ** 63 - 1, -2 ** 63, 2 ** 62 + 2 ** 8, 987654321987654321], dtype=np.int64)
    got = orc.cast(i64, np.float64)
    for x, g in zip(i64.tolist(), got.tolist()):
        assert Fraction(g) == _nearest_even(Fraction(x), 53), (x, g)
    assert got[1] == 2.0 ** 53 and got[3] == 2.0 ** 53 + 4 and got[5] == 2.0 ** 63
    got = orc.cast(i64, np.float32)
    for x, g in zip(i64.tolist(), got.tolist()):
        assert Fraction(g) == _nearest_even(Fraction(x), 24), (x, g)      # ONE rounding from the integer (not via double)
    # a value where rounding through double first would give another float: 2^24 + 1 + 2^-30 cannot be an integer, so take an
    # int64 just above a float32 tie: 2^40 + 2^16 + 1 -> above the midpoint between 2^40 and 2^40 + 2^17 -> rounds UP
    x = 2 ** 40 + 2 ** 16 + 1
    assert orc.cast(np.array([x], dtype=np.int64), np.float32)[0] == np.float32(2 ** 40 + 2 ** 17)


def test_cast_float_to_int_truncates_saturates_and_nan_is_zero():
    f64 = np.array([0.0, -0.0, 0.9, -0.9, 1.5, -1.5, 2.5, -2.5, 2147483647.0, 2147483647.9, 2147483648.0, -2147483648.0, -2147483648.9,
                    -2147483649.0, 3e9, -3e9, 1e300, -1e300, np.inf, -np.inf, np.nan])
    want32 = [0, 0, 0, 0, 1, -1, 2, -2, 2147483647, 2147483647, 2147483647, -2147483648, -2147483648,
              -2147483648, 2147483647, -2147483648, 2147483647, -2147483648, 2147483647, -2147483648, 0]
    assert orc.cast(f64, np.int32).tolist() == want32
    want64 = [0, 0, 0, 0, 1, -1, 2, -2, 2147483647, 2147483647, 2147483648, -2147483648, -2147483648,
              -2147483649, 3000000000, -3000000000, 2 ** 63 - 1, -2 ** 63, 2 ** 63 - 1, -2 ** 63, 0]
    assert orc.cast(f64, np.int64).tolist() == want64
    edge = np.array([2.0 ** 63, -(2.0 ** 63), 2.0 ** 63 - 1024.0, -(2.0 ** 63) - 2048.0, 2.0 ** 62])
    assert orc.cast(edge, np.int64).tolist() == [2 ** 63 - 1, -2 ** 63, 2 ** 63 - 1024, -2 ** 63, 2 ** 62]
    f32 = np.array([16777216.0, 16777218.0, -7.75, 2147483520.0, 2147483648.0, -2147483648.0, 3.4e38, np.nan], dtype=np.float32)
    assert orc.cast(f32, np.int32).tolist() == [16777216, 16777218, -7, 2147483520, 2147483647, -2147483648, 2147483647, 0]
    # in range, truncation == math.trunc of the exact value (brute force over random values)
    x = (RNG.standard_normal(500) * 1e6)
    assert orc.cast(x, np.int32).tolist() == [math.trunc(v) for v in x.tolist()]
    assert orc.cast(x.astype(np.float32), np.int64).tolist() == [math.trunc(float(v)) for v in x.astype(np.float32).tolist()]


def test_cast_between_floats_and_between_ints():
    d = np.array([1.0, 1.0 + 2.0 ** -24, 1.0 + 2.0 ** -23 + 2.0 ** -24, 1.0 + 2.0 ** -24 + 2.0 ** -50, 1e40, -1e40, 1e-50, np.inf, 0.1])
    got = orc.cast(d, np.float32)
    # ties to even: 1 + 2^-24 -> 1 (even), 1 + 2^-23 + 2^-24 -> 1 + 2^-22 (even); just above a tie rounds up; overflow -> inf; underflow -> 0
    assert got.tolist()[:8] == [1.0, 1.0, 1.0 + 2.0 ** -22, 1.0 + 2.0 ** -23, np.inf, -np.inf, 0.0, np.inf]
    assert Fraction(float(got[8])) == _nearest_even(Fraction(0.1), 24)
    f = RNG.standard_normal(64).astype(np.float32)
    up = orc.cast(f, np.float64)
    assert up.dtype == np.float64 and [Fraction(float(v)) for v in up] == [Fraction(float(v)) for v in f]     # widening is exact
    i32 = np.array([0, -1, 2 ** 31 - 1, -2 ** 31, 12345], dtype=np.int32)
    assert orc.cast(i32, np.int64).tolist() == i32.tolist()                                                   # sign extension
    i64 = np.array([5, -1, 2 ** 31, 2 ** 32 + 5, -(2 ** 31) - 1, 2 ** 63 - 1, -2 ** 63], dtype=np.int64)
    want = [((v + 2 ** 31) % 2 ** 32) - 2 ** 31 for v in i64.tolist()]                                        # the low 32 bits, two's complement
    assert orc.cast(i64, np.int32).tolist() == want
    for dt in (np.float32, np.float64, np.int32, np.int64):
        a = (RNG.standard_normal(16) * 100).astype(dt)
        assert orc.cast(a, dt).tobytes() == a.tobytes()                                                       # same type: identity
    assert orc.cast(np.zeros(0, dtype=np.int32), np.float64).size == 0


def test_project_sqrt_of_integers_gives_doubles():
    """`c.project (agent (a: INT): DOUBLE do Result := sqrt (a) end)`."""
    c = np.array([0, 1, 4, 9, 16, 2, 3, 10 ** 6, 2 ** 31 - 1, 46340 ** 2], dtype=np.int32)
    got = orc.project_sqrt(c)
    assert got.dtype == np.float64
    assert got.tolist()[:5] == [0.0, 1.0, 2.0, 3.0, 4.0] and got[7] == 1000.0 and got[9] == 46340.0      # perfect squares are exact
    for x, r in zip(c.tolist(), got.tolist()):                                                           # correct rounding by the exact bracket
        lo, hi = np.nextafter(r, -np.inf), np.nextafter(r, np.inf)
        if x > 0:
            assert ((Fraction(float(lo)) + Fraction(r)) / 2) ** 2 <= x <= ((Fraction(r) + Fraction(float(hi))) / 2) ** 2
    big = np.array([2 ** 53 + 1, 2 ** 62], dtype=np.int64)                 # int64: the conversion rounds first (2^53+1 -> 2^53), then the root
    assert orc.project_sqrt(big).tolist() == [math.sqrt(2.0 ** 53), 2.0 ** 31]
    assert np.isnan(orc.project_sqrt(np.array([-4], dtype=np.int32))[0])   # sqrt of a negative number: NaN (R20)
