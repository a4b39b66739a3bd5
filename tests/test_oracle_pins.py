"""Pins of the CPU oracle against what the mathematics fixes (no GPU, no CUDA library).

The paper (arxiv 1405.2915) prints no worked example for any skeleton (it names them only,
PAPER.md L75/L83), so the pins are the ones BASELINE.json L5 names (dot(x_i=i, ones) = n(n-1)/2,
scan(ones) = indices, stencil(const) = const * sum w) plus: impulse / one-hot shifts (orientation,
indexing, edge policy), invariants (split, permutation, separable identity, transpose symmetry),
library special cases (numpy cumsum / correlate, math.fsum) and pure-Python brute force on tiny
inputs. The golden closed-form values live in tests/golden/closed_forms.txt.
"""
import math
import os

import numpy as np
import pytest

import oracle as O
import skel_inputs as I

GOLD = os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")
BOUNDARY_N = [1, 2, 3, 4, 5, 7, 8, 31, 32, 33, 127, 128, 129, 1023, 1024, 1025]


def wrap32(v: int) -> int:
    v &= 0xFFFFFFFF
    return v - (1 << 32) if v >= (1 << 31) else v


def golden():
    out = {}
    with open(GOLD) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                out[k] = int(v)
    return out


# ------------------------------------------------------------------ generators (host logic)
def test_generator_is_stateless_and_in_range():
    a = I.uniform_pm1_f32(7, 1000)
    b = I.uniform_pm1_f32(7, 2000)[:1000]
    assert np.array_equal(a, b)
    assert a.min() >= -1.0 and a.max() < 1.0 and abs(a.mean()) < 0.1
    assert not np.array_equal(a, I.uniform_pm1_f32(8, 1000))
    # streams of neighbouring seeds are not shifted copies of each other
    c = I.uniform_pm1_f32(8, 1001)
    assert not np.array_equal(a[1:], c[:999]) and not np.array_equal(a[:999], c[1:1000])
    v = I.uniform_int_i32(9, 100000, 15)
    assert v.min() == 0 and v.max() == 15 and abs(v.mean() - 7.5) < 0.1
    w = I.positive_weights_f32(3, 33)
    assert (w > 0).all() and abs(w.astype(np.float64).sum() - 1.0) < 33 * 2.0 ** -24
    p = I.permutation(4, 1000)
    assert np.array_equal(np.sort(p), np.arange(1000))


def test_generator_crosses_chunk_boundary_consistently():
    n = (1 << 24) + 5
    a = I.raw_u64(11, n)
    assert np.array_equal(a[-10:], I.raw_u64(11, 10, start=n - 10))


# ------------------------------------------------------------------ Map
def test_map_saxpy_closed_form_exact():
    # x_i = i, y = 1, c = 2.5 -> 2.5 i + 1, exactly representable for i < 2^22 (SURVEY (c).1 pins)
    n = 1 << 16
    x = np.arange(n, dtype=np.float32)
    y = np.ones(n, np.float32)
    out = O.map_f32(O.FN_SAXPY, 2.5, x, y)
    assert np.array_equal(out, 2.5 * np.arange(n, dtype=np.float64) + 1.0)


def test_map_identities_and_constant_rounding():
    x = I.uniform_pm1_f32(21, 1025)
    assert np.array_equal(O.map_f32(O.FN_MULT, 1.0, x), x.astype(np.float64))
    assert np.array_equal(O.map_f32(O.FN_ADD, 0.0, x), x.astype(np.float64))
    # the constant is rounded to fp32 first (reading (c).1 iii): x * (double)(float)1.0001
    c32 = float(np.float32(1.0001))
    assert c32 != 1.0001
    assert np.array_equal(O.map_f32(O.FN_MULT, 1.0001, x), x.astype(np.float64) * c32)


@pytest.mark.parametrize("fn", [O.FN_ADD, O.FN_MULT, O.FN_MAX, O.FN_SAXPY])
def test_map_brute_force(fn):
    for n in [0] + BOUNDARY_N[:9]:
        a = I.uniform_pm1_f32(30 + n, n)
        b = I.uniform_pm1_f32(31 + n, n)
        c = float(np.float32(0.3))
        exp = []
        for i in range(n):
            ai, bi = float(a[i]), float(b[i])
            exp.append({O.FN_ADD: ai + bi, O.FN_MULT: ai * bi, O.FN_MAX: max(ai, bi), O.FN_SAXPY: c * ai + bi}[fn])
        assert np.array_equal(O.map_f32(fn, 0.3, a, b), np.array(exp, np.float64))


def test_map_i32_wraps():
    a = np.array([2 ** 31 - 1, -2 ** 31, 70000, -5], np.int32)
    b = np.array([1, -1, 70000, 3], np.int32)
    assert O.map_i32(O.FN_ADD, 0, a, b).tolist() == [wrap32(int(x) + int(y)) for x, y in zip(a, b)]
    assert O.map_i32(O.FN_MULT, 0, a, b).tolist() == [wrap32(int(x) * int(y)) for x, y in zip(a, b)]
    assert O.map_i32(O.FN_MAX, 0, a, b).tolist() == [max(int(x), int(y)) for x, y in zip(a, b)]
    assert O.map_i32(O.FN_SAXPY, 3, a, b).tolist() == [wrap32(3 * int(x) + int(y)) for x, y in zip(a, b)]
    assert O.map_i32(O.FN_ADD, 7, a).tolist() == [wrap32(int(x) + 7) for x in a]


def test_map3_muladd_exact_against_rationals_and_python_ints():
    """Three-vector Map (MULADD): the fp64 result must be the correctly rounded exact value a*b + c (the product of
    two fp32 numbers is exact in fp64, so one rounding happens), checked with Python's exact rationals; closed
    forms; exact cancellation; int32 wraps like Python integers modulo 2^32. Swapping operands is caught (b != c)."""
    from fractions import Fraction
    n = 300
    a, b, c = I.uniform_pm1_f32(81, n), I.uniform_pm1_f32(82, n), I.uniform_pm1_f32(83, n)
    got = O.map3_muladd_f32(a, b, c)
    for i in range(n):
        exact = Fraction(float(a[i])) * Fraction(float(b[i])) + Fraction(float(c[i]))
        assert got[i] == float(exact), i          # float(Fraction) rounds to nearest even
    i32s = np.arange(1000, dtype=np.float32)
    assert np.array_equal(O.map3_muladd_f32(i32s, np.full(1000, 2, np.float32), np.ones(1000, np.float32)), 2.0 * np.arange(1000) + 1)
    p = (a.astype(np.float64) * b.astype(np.float64))
    exact_prod = p.astype(np.float32).astype(np.float64) == p   # products that happen to be fp32 numbers
    cc = (-p).astype(np.float32)
    assert np.all(O.map3_muladd_f32(a, b, cc)[exact_prod] == 0.0)
    x = (I.raw_u64(84, 64) % np.uint64(1 << 32)).astype(np.uint32).view(np.int32)
    y = (I.raw_u64(85, 64) % np.uint64(1 << 32)).astype(np.uint32).view(np.int32)
    z = (I.raw_u64(86, 64) % np.uint64(1 << 32)).astype(np.uint32).view(np.int32)
    assert O.map3_muladd_i32(x, y, z).tolist() == [wrap32(int(p) * int(q) + int(r)) for p, q, r in zip(x, y, z)]
    assert O.map3_muladd_f32(a[:0], b[:0], c[:0]).size == 0


# ------------------------------------------------------------------ Reduce
def test_reduce_closed_forms():
    g = golden()
    for n in BOUNDARY_N + [1 << 20]:
        ones = np.ones(n, np.float32)
        assert O.reduce_f32(O.FN_ADD, ones)[0] == n
        idx = np.arange(n, dtype=np.int32)
        r, exact = O.reduce_i32(O.FN_ADD, idx)
        assert exact == n * (n - 1) // 2 and r == wrap32(n * (n - 1) // 2)
    n = 1 << 20
    assert O.reduce_i32(O.FN_ADD, np.arange(n, dtype=np.int32))[1] == g["sum_i_lt_2p20"]
    # wraps: sum of 2^17 copies of 2^20 = 2^37 = 0 mod 2^32
    assert O.reduce_i32(O.FN_ADD, np.full(1 << 17, 1 << 20, np.int32)) == (0, 1 << 37)
    assert g["sum_i_lt_2p17_mod32"] == wrap32((1 << 17) * ((1 << 17) - 1) // 2)
    assert O.reduce_i32(O.FN_ADD, np.arange(1 << 17, dtype=np.int32))[0] == g["sum_i_lt_2p17_mod32"]


def test_reduce_max_of_permutation_wherever_it_sits():
    n = 4099
    base = I.permutation(5, n).astype(np.int32)
    for pos in [0, 1, n // 2, 1023, 1024, n - 2, n - 1]:
        p = base.copy()
        j = int(np.argmax(p))
        p[j], p[pos] = p[pos], p[j]
        assert O.reduce_i32(O.FN_MAX, p)[0] == n - 1
        assert O.reduce_f32(O.FN_MAX, p.astype(np.float32))[0] == n - 1


def test_reduce_split_and_permutation_invariants():
    n = 5003
    v = I.full_range_i32(6, n)
    total = O.reduce_i32(O.FN_ADD, v)[0]
    for k in [1, 17, 2500, n - 1]:
        a = O.reduce_i32(O.FN_ADD, v[:k])[0]
        b = O.reduce_i32(O.FN_ADD, v[k:])[0]
        assert wrap32(a + b) == total
    assert O.reduce_i32(O.FN_ADD, v[I.permutation(7, n)])[0] == total
    small = (v % 7).astype(np.int32)
    prod = O.reduce_i32(O.FN_MULT, small)[0]
    assert O.reduce_i32(O.FN_MULT, small[I.permutation(8, n)])[0] == prod
    x = I.uniform_pm1_f32(9, n)
    s, a = O.reduce_f32(O.FN_ADD, x)
    s1 = O.reduce_f32(O.FN_ADD, x[:1234])[0] + O.reduce_f32(O.FN_ADD, x[1234:])[0]
    assert abs(s - s1) <= 1e-14 * a
    assert abs(O.reduce_f32(O.FN_ADD, x[I.permutation(10, n)])[0] - s) <= 1e-14 * a


def test_reduce_matches_fsum_and_python_loops():
    for n in BOUNDARY_N:
        x = I.uniform_pm1_f32(40 + n, n)
        s, a = O.reduce_f32(O.FN_ADD, x)
        exact = math.fsum(float(t) for t in x)
        assert abs(s - exact) <= 4e-16 * max(a, 1e-300)
        assert a == pytest.approx(math.fsum(abs(float(t)) for t in x), rel=1e-15)
        assert O.reduce_f32(O.FN_MAX, x)[0] == max(float(t) for t in x)
        v = I.full_range_i32(41 + n, n)
        acc = int(v[0])
        for t in v[1:]:
            acc = wrap32(acc + int(t))
        assert O.reduce_i32(O.FN_ADD, v)[0] == acc
    with pytest.raises(ValueError):
        O.reduce_f32(O.FN_ADD, np.zeros(0, np.float32))
    with pytest.raises(ValueError):
        O.reduce_i32(O.FN_ADD, np.zeros(0, np.int32))


def test_reduce_config2_semantics_overflow_is_wrap():
    # BJ:L8 inputs uniform{0..1000}: at n = 2^26 the sum exceeds 2^32; check the wrap on a
    # scaled-down instance whose exact sum is known from the int64 path
    v = I.uniform_int_i32(I.config_seed(2, 2), 1 << 18, 1000) * 20000
    r, exact = O.reduce_i32(O.FN_ADD, v)
    assert exact == int(v.astype(np.int64).sum()) and exact > 2 ** 32 and r == wrap32(exact)


# ------------------------------------------------------------------ MapReduce
def test_dot_closed_form_and_unit_vectors():
    g = golden()
    for n in BOUNDARY_N + [1 << 20]:
        x = np.arange(n, dtype=np.float32)  # exact for n <= 2^24
        ones = np.ones(n, np.float32)
        r, a = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, ones)
        assert r == n * (n - 1) // 2 and a == r
    assert O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, np.arange(1 << 20, dtype=np.float32), np.ones(1 << 20, np.float32))[0] == g["sum_i_lt_2p20"]
    x = I.uniform_pm1_f32(50, 777)
    for j in [0, 5, 776]:
        e = np.zeros(777, np.float32)
        e[j] = 1.0
        assert O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, e)[0] == float(x[j])
    r, a = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, x)
    assert r >= 0 and r == pytest.approx(a, rel=1e-15)


def test_reduce_rows_closed_forms_library_and_brute_force():
    """Row-wise Reduce: closed forms, numpy's axis reductions and math.fsum (independent
    library routines), Python-int brute force for the int32 wrap, and the transposition / vector-Reduce
    invariants. A dropped row, a row/column mix-up or a wrong stride fails one of them."""
    rows, cols = 37, 129
    # closed forms: X[i][j] = i -> cols * i; X[i][j] = j -> cols (cols - 1) / 2 in every row
    Xi = np.repeat(np.arange(rows, dtype=np.float32)[:, None], cols, axis=1)
    r, a = O.reduce_rows_f32(O.FN_ADD, Xi)
    assert r.tolist() == [float(cols * i) for i in range(rows)] and a.tolist() == r.tolist()
    Xj = np.repeat(np.arange(cols, dtype=np.int32)[None, :], rows, axis=0)
    assert O.reduce_rows_i32(O.FN_ADD, Xj).tolist() == [cols * (cols - 1) // 2] * rows
    assert O.reduce_rows_i32(O.FN_MAX, Xj).tolist() == [cols - 1] * rows
    # library routines on random data (not symmetric under transposition: a swapped axis is caught)
    X = I.uniform_pm1_f32(71, rows * cols).reshape(rows, cols)
    r, a = O.reduce_rows_f32(O.FN_ADD, X)
    for i in range(rows):
        assert r[i] == pytest.approx(math.fsum(float(v) for v in X[i]), rel=0, abs=1e-12)
        assert a[i] == pytest.approx(math.fsum(abs(float(v)) for v in X[i]), rel=1e-15)
    assert np.array_equal(O.reduce_rows_f32(O.FN_MAX, X)[0], X.max(axis=1).astype(np.float64))
    P = 1.0 + 0.001 * X[:5, :40]
    assert np.allclose(O.reduce_rows_f32(O.FN_MULT, P)[0], np.prod(P.astype(np.float64), axis=1), rtol=1e-13)
    # every row is the vector Reduce of that row; the row-wise Reduce of X^T reduces the columns of X
    for i in (0, 7, rows - 1):
        assert O.reduce_f32(O.FN_ADD, X[i])[0] == r[i]
    rt, _ = O.reduce_rows_f32(O.FN_ADD, np.ascontiguousarray(X.T))
    assert np.allclose(rt, X.astype(np.float64).sum(axis=0), rtol=0, atol=1e-12)
    # int32: wraps modulo 2^32 (Python integers are exact)
    V = (I.raw_u64(72, 6 * 50) % np.uint64(1 << 31)).astype(np.int64).reshape(6, 50)
    V32 = V.astype(np.int32)
    assert O.reduce_rows_i32(O.FN_ADD, V32).tolist() == [wrap32(sum(int(v) for v in row)) for row in V32]
    assert O.reduce_rows_i32(O.FN_MULT, V32[:, :5]).tolist() == [wrap32(math.prod(int(v) for v in row[:5])) for row in V32]
    # shapes: a single column is the identity, a single row is the vector Reduce; empty rows are an error
    assert np.array_equal(O.reduce_rows_f32(O.FN_ADD, X[:, :1])[0], X[:, 0].astype(np.float64))
    assert O.reduce_rows_f32(O.FN_ADD, X[:1])[0][0] == O.reduce_f32(O.FN_ADD, X[0])[0]
    with pytest.raises(ValueError):
        O.reduce_rows_f32(O.FN_ADD, np.zeros((3, 0), np.float32))
    # the OpenMP build computes the same rows
    O.use_openmp(True)
    try:
        assert np.array_equal(O.reduce_rows_f32(O.FN_ADD, X)[0], r)
    finally:
        O.use_openmp(False)


def test_mapreduce_fusion_invariant_and_brute_force():
    for n in BOUNDARY_N:
        x = I.uniform_pm1_f32(60 + n, n)
        y = I.uniform_pm1_f32(61 + n, n)
        r, a = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, y)
        exact = math.fsum(float(p) * float(q) for p, q in zip(x, y))  # products exact in fp64
        assert abs(r - exact) <= 4e-16 * max(a, 1e-300)
        # max of sums
        r2, _ = O.mapreduce_f32(O.FN_ADD, O.FN_MAX, 0.0, x, y)
        assert r2 == max(float(p) + float(q) for p, q in zip(x, y))
        # saxpy then add: c*sum x + sum y
        r3, _ = O.mapreduce_f32(O.FN_SAXPY, O.FN_ADD, 2.5, x, y)
        assert r3 == pytest.approx(math.fsum(2.5 * float(p) + float(q) for p, q in zip(x, y)), abs=1e-12)
        a_i = I.full_range_i32(62 + n, n)
        b_i = I.full_range_i32(63 + n, n)
        fused = O.mapreduce_i32(O.FN_MULT, O.FN_ADD, 0, a_i, b_i)
        assert fused == O.reduce_i32(O.FN_ADD, O.map_i32(O.FN_MULT, 0, a_i, b_i))[0]
        assert fused == wrap32(sum(int(p) * int(q) for p, q in zip(a_i, b_i)))


def test_mapreduce_constant_second_operand():
    """in1 = None: the second operand of the user function is the constant c, rounded to fp32 first
    (reading (c).1 iii). Pinned against math.fsum / exact Python integers, never against the oracle."""
    c = 1.0001
    c32 = float(np.float32(c))
    assert c32 != c  # the rounding is visible, so using the unrounded constant fails below
    for n in BOUNDARY_N:
        x = I.uniform_pm1_f32(64 + n, n)
        xs = [float(t) for t in x]
        r, a = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, c, x)          # sum_i c32 * x_i (products exact in fp64)
        assert abs(r - math.fsum(c32 * t for t in xs)) <= 4e-16 * max(a, 1e-300)
        assert a == pytest.approx(math.fsum(abs(c32 * t) for t in xs), rel=1e-15)
        r, _ = O.mapreduce_f32(O.FN_ADD, O.FN_ADD, c, x)           # sum_i (x_i + c32)
        assert r == pytest.approx(math.fsum(t + c32 for t in xs), abs=1e-12)
        r, _ = O.mapreduce_f32(O.FN_MAX, O.FN_ADD, 0.25, x)        # sum_i max(x_i, 0.25)
        assert r == pytest.approx(math.fsum(max(t, 0.25) for t in xs), abs=1e-12)
        r, _ = O.mapreduce_f32(O.FN_MULT, O.FN_MAX, -2.0, x)       # max_i (-2 x_i) = -2 min x
        assert r == -2.0 * min(xs)
        r, _ = O.mapreduce_f32(O.FN_ADD, O.FN_MULT, 1.0, 0.001 * x)  # prod_i (1 + x_i/1000): left to right in fp64
        acc = None
        for t in (0.001 * x).astype(np.float32):
            acc = float(t) + 1.0 if acc is None else acc * (float(t) + 1.0)
        assert r == acc
        v = I.full_range_i32(65 + n, n)
        vi = [int(t) for t in v]
        assert O.mapreduce_i32(O.FN_MULT, O.FN_ADD, 3, v) == wrap32(sum(3 * t for t in vi))
        assert O.mapreduce_i32(O.FN_ADD, O.FN_ADD, -7, v) == wrap32(sum(t - 7 for t in vi))
        assert O.mapreduce_i32(O.FN_MAX, O.FN_MAX, 12345, v) == max(max(vi), 12345)
        assert O.mapreduce_i32(O.FN_ADD, O.FN_MAX, 1, v) == max(wrap32(t + 1) for t in vi)
    # closed form: sum_i c * i with c = 2 over i < n -> n (n - 1); the constant really is the SECOND operand
    n = 1000
    assert O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 2.0, np.arange(n, dtype=np.float32))[0] == n * (n - 1)
    assert O.mapreduce_i32(O.FN_MULT, O.FN_ADD, 2, np.arange(n, dtype=np.int32)) == n * (n - 1)


def test_reduce_f32_mult_on_a_vector():
    """Reduce(mult) over a vector: plain left-to-right fp64 product (reading (c).2), against math.prod,
    numpy.prod and the closed form n!."""
    for n in BOUNDARY_N:
        x = (1.0 + 0.001 * I.uniform_pm1_f32(66 + n, n)).astype(np.float32)
        r, a = O.reduce_f32(O.FN_MULT, x)
        acc = float(x[0])
        for t in x[1:]:
            acc *= float(t)
        assert r == acc
        assert r == pytest.approx(float(np.prod(x.astype(np.float64))), rel=1e-12)
        assert a == pytest.approx(math.fsum(abs(float(t)) for t in x), rel=1e-15)
    f = np.arange(1, 19, dtype=np.float32)
    assert O.reduce_f32(O.FN_MULT, f)[0] == float(math.factorial(18))  # 18! < 2^53: exact
    assert O.reduce_f32(O.FN_MULT, np.array([3.0, -2.0, 0.5], np.float32))[0] == -3.0


# ------------------------------------------------------------------ Scan
def test_scan_closed_forms():
    for n in [0] + BOUNDARY_N + [4096, 4097, 1 << 18]:
        ones = np.ones(n, np.int32)
        assert np.array_equal(O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, ones), np.arange(1, n + 1, dtype=np.int32))
        assert np.array_equal(O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, 0, ones), np.arange(0, n, dtype=np.int32))
    n = 1 << 17  # i(i+1)/2 exceeds 2^32 -> wraps
    i = np.arange(n, dtype=np.int64)
    exp = ((i * (i + 1) // 2) & 0xFFFFFFFF).astype(np.uint32).view(np.int32)
    assert np.array_equal(O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, np.arange(n, dtype=np.int32)), exp)


def test_scan_matches_cumsum_and_invariants():
    for n in BOUNDARY_N + [5000]:
        x = I.full_range_i32(70 + n, n)
        inc = O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, x)
        exc = O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, 5, x)
        lib = np.cumsum(x.astype(np.int64)).astype(np.uint64).astype(np.uint32).view(np.int32)
        assert np.array_equal(inc, lib)
        assert exc[0] == 5
        assert np.array_equal(exc[1:], (inc[:-1].astype(np.int64) + 5).astype(np.uint64).astype(np.uint32).view(np.int32))
        assert inc[-1] == O.reduce_i32(O.FN_ADD, x)[0]
        mx = O.scan_i32(O.FN_MAX, O.SCAN_INCLUSIVE, 0, x)
        assert np.array_equal(mx, np.maximum.accumulate(x))
        mxe = O.scan_i32(O.FN_MAX, O.SCAN_EXCLUSIVE, -7, x)
        assert mxe[0] == -7 and np.array_equal(mxe[1:], np.maximum(np.maximum.accumulate(x)[:-1], -7))


def test_scan_brute_force_every_small_n():
    for n in range(0, 70):
        x = I.uniform_int_i32(80 + n, n, 15)
        acc, inc, exc = 0, [], []
        e = 3
        for t in x:
            exc.append(e)
            e = wrap32(e + int(t))
            acc = wrap32(acc + int(t))
            inc.append(acc)
        assert O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, x).tolist() == inc
        assert O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, 3, x).tolist() == exc


def test_scan_i32_mult_wraps_like_python_ints():
    """Scan(mult) on int32: running product modulo 2^32 (reading (c).2 ii), against exact Python
    integers and the closed form i! mod 2^32."""
    for n in list(range(0, 40)) + [127, 128, 129, 1025]:
        x = (I.full_range_i32(84 + n, n) | 1)  # odd factors: the product never collapses to 0
        acc, inc, exc = None, [], []
        e = 3
        for t in x:
            exc.append(wrap32(e))
            e = wrap32(e * int(t))
            acc = int(t) if acc is None else wrap32(acc * int(t))
            inc.append(acc)
        assert O.scan_i32(O.FN_MULT, O.SCAN_INCLUSIVE, 0, x).tolist() == inc
        assert O.scan_i32(O.FN_MULT, O.SCAN_EXCLUSIVE, 3, x).tolist() == exc
    k = np.arange(1, 21, dtype=np.int32)
    assert O.scan_i32(O.FN_MULT, O.SCAN_INCLUSIVE, 0, k).tolist() == [wrap32(math.factorial(int(j))) for j in k]
    assert O.scan_i32(O.FN_MULT, O.SCAN_EXCLUSIVE, 1, k).tolist() == [wrap32(math.factorial(int(j) - 1)) for j in k]


def test_scan_f32_max_and_mult():
    """fp32 Scan with max / mult in fp64: numpy's accumulate routines (independent library) and closed forms;
    the exclusive forms fold the fp32-rounded init into every prefix (reading (c).4 ii)."""
    x = I.uniform_pm1_f32(91, 2500)
    x64 = x.astype(np.float64)
    out, ab = O.scan_f32(O.FN_MAX, O.SCAN_INCLUSIVE, 0.0, x)
    assert np.array_equal(out, np.maximum.accumulate(x64))
    assert np.allclose(ab, np.cumsum(np.abs(x64)), rtol=1e-14)
    init = 0.3
    i32 = float(np.float32(init))
    oute, abe = O.scan_f32(O.FN_MAX, O.SCAN_EXCLUSIVE, init, x)
    assert oute[0] == i32 and np.array_equal(oute[1:], np.maximum(np.maximum.accumulate(x64)[:-1], i32))
    assert abe[0] == abs(i32) and np.allclose(abe[1:], abs(i32) + np.cumsum(np.abs(x64))[:-1], rtol=1e-14)
    # a strictly decreasing input: the running max is the first element; increasing: the identity
    dec = np.arange(100, 0, -1).astype(np.float32)
    assert np.array_equal(O.scan_f32(O.FN_MAX, O.SCAN_INCLUSIVE, 0.0, dec)[0], np.full(100, 100.0))
    assert np.array_equal(O.scan_f32(O.FN_MAX, O.SCAN_INCLUSIVE, 0.0, dec[::-1].copy())[0], dec[::-1].astype(np.float64))
    p = (1.0 + 0.01 * x[:600]).astype(np.float32)
    out, _ = O.scan_f32(O.FN_MULT, O.SCAN_INCLUSIVE, 0.0, p)
    assert np.allclose(out, np.cumprod(p.astype(np.float64)), rtol=1e-13, atol=0)
    acc = None
    for k, t in enumerate(p[:50]):
        acc = float(t) if acc is None else acc * float(t)
        assert out[k] == acc  # left to right, one rounding per step
    oute, _ = O.scan_f32(O.FN_MULT, O.SCAN_EXCLUSIVE, 2.0, p)
    assert oute[0] == 2.0 and np.allclose(oute[1:], 2.0 * np.cumprod(p.astype(np.float64))[:-1], rtol=1e-13)
    two = np.full(40, 2.0, np.float32)  # closed form 2^(i+1), exact
    assert O.scan_f32(O.FN_MULT, O.SCAN_INCLUSIVE, 0.0, two)[0].tolist() == [2.0 ** (k + 1) for k in range(40)]


def test_scan_f32_against_cumsum():
    x = I.uniform_pm1_f32(90, 3000)
    out, ab = O.scan_f32(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, x)
    assert np.allclose(out, np.cumsum(x.astype(np.float64)), rtol=0, atol=1e-12)
    assert np.allclose(ab, np.cumsum(np.abs(x.astype(np.float64))), rtol=1e-14)
    oute, _ = O.scan_f32(O.FN_ADD, O.SCAN_EXCLUSIVE, 1.5, x)
    assert oute[0] == 1.5 and np.allclose(oute[1:], 1.5 + out[:-1], atol=1e-12)


# ------------------------------------------------------------------ MapOverlap 1D
EDGES = [O.EDGE_CONSTANT, O.EDGE_DUPLICATE]


@pytest.mark.parametrize("r", [0, 1, 4, 16])
def test_overlap1d_constant_input_closed_form(r):
    n, K = 100, 3.0
    w = I.positive_weights_f32(100 + r, 2 * r + 1)
    wd = w.astype(np.float64)
    x = np.full(n, K, np.float32)
    out, ab = O.mapoverlap_1d(w, r, O.EDGE_DUPLICATE, 0.0, x)
    seq = 0.0
    for k in range(2 * r + 1):
        seq += wd[k] * K
    assert np.all(out == seq) and abs(seq - K) < 1e-5 and np.array_equal(out, ab)
    out0, _ = O.mapoverlap_1d(w, r, O.EDGE_CONSTANT, 0.0, x)
    for i in range(n):
        exp = K * math.fsum(wd[k + r] for k in range(-r, r + 1) if 0 <= i + k < n)
        assert out0[i] == pytest.approx(exp, rel=1e-14)
    # non-zero pad: border cells see the pad value
    outp, _ = O.mapoverlap_1d(w, r, O.EDGE_CONSTANT, 7.0, x)
    for i in [0, n - 1]:
        exp = math.fsum(wd[k + r] * (K if 0 <= i + k < n else 7.0) for k in range(-r, r + 1))
        assert outp[i] == pytest.approx(exp, rel=1e-14)


@pytest.mark.parametrize("edge", EDGES)
def test_overlap1d_impulse_pins_orientation(edge):
    # x = e_j -> out[i] = w[(j - i) + r] for |i-j| <= r else 0: correlation, not convolution
    r, n = 4, 41
    w = I.signed_weights_f32(110, 2 * r + 1)
    for j in [0, 1, 3, 20, n - 2, n - 1]:
        x = np.zeros(n, np.float32)
        x[j] = 1.0
        out, _ = O.mapoverlap_1d(w, r, edge, 0.0, x)
        for i in range(n):
            exp = float(w[(j - i) + r]) if abs(i - j) <= r else 0.0
            if edge == O.EDGE_DUPLICATE and j in (0, n - 1):
                # the impulse sits on the border and is replicated outwards
                exp = math.fsum(float(w[k + r]) for k in range(-r, r + 1) if min(max(i + k, 0), n - 1) == j)
            assert out[i] == pytest.approx(exp, abs=1e-15)


@pytest.mark.parametrize("edge", EDGES)
@pytest.mark.parametrize("r", [1, 3, 16])
def test_overlap1d_one_hot_weights_are_a_shift_bit_exact(edge, r):
    for n in [1, 2, r, r + 1, 2 * r + 1, 50]:
        x = I.uniform_pm1_f32(120 + n, n)
        for m in range(2 * r + 1):
            w = np.zeros(2 * r + 1, np.float32)
            w[m] = 1.0
            out, _ = O.mapoverlap_1d(w, r, edge, 0.25, x)
            for i in range(n):
                j = i + m - r
                if 0 <= j < n:
                    exp = float(x[j])
                elif edge == O.EDGE_CONSTANT:
                    exp = 0.25
                else:
                    exp = float(x[min(max(j, 0), n - 1)])
                assert out[i] == exp


def test_overlap1d_identity_linearity_convexity_and_numpy_correlate():
    x = I.uniform01_f32(130, 500)
    y = I.uniform01_f32(131, 500)
    out, _ = O.mapoverlap_1d(np.ones(1, np.float32), 0, O.EDGE_DUPLICATE, 0.0, x)
    assert np.array_equal(out, x.astype(np.float64))
    r = 4
    w = I.positive_weights_f32(132, 2 * r + 1)
    a, b = 2.0, -0.5  # exactly representable scalings keep the fp32 combination exact
    ox, _ = O.mapoverlap_1d(w, r, O.EDGE_DUPLICATE, 0.0, x)
    oy, _ = O.mapoverlap_1d(w, r, O.EDGE_DUPLICATE, 0.0, y)
    z = (a * x.astype(np.float64) + b * y.astype(np.float64))
    z32 = z.astype(np.float32)
    oz, _ = O.mapoverlap_1d(w, r, O.EDGE_DUPLICATE, 0.0, z32)
    assert np.allclose(oz, a * ox + b * oy, atol=1e-6)
    assert ox.min() >= x.min() - 1e-6 and ox.max() <= x.max() + 1e-6
    # library special case: constant-0 edges == numpy.correlate(..., 'same') on zero-padded input
    lib = np.correlate(x.astype(np.float64), w.astype(np.float64), mode="same")
    o0, _ = O.mapoverlap_1d(w, r, O.EDGE_CONSTANT, 0.0, x)
    assert np.allclose(o0, lib, rtol=0, atol=1e-14)
    # duplicate edges == correlate 'valid' on an edge-padded copy
    xp = np.pad(x.astype(np.float64), r, mode="edge")
    assert np.allclose(ox, np.correlate(xp, w.astype(np.float64), mode="valid"), rtol=0, atol=1e-14)


@pytest.mark.parametrize("edge", EDGES)
def test_overlap1d_brute_force_small(edge):
    for r in [0, 1, 2, 5, 16]:
        w = I.signed_weights_f32(140 + r, 2 * r + 1)
        for n in [1, 2, 3, r, r + 1, 2 * r, 2 * r + 1, 2 * r + 2, 70]:
            if n == 0:
                continue
            x = I.uniform_pm1_f32(141 + n, n)
            out, ab = O.mapoverlap_1d(w, r, edge, -0.5, x)
            for i in range(n):
                acc = 0.0
                aacc = 0.0
                for k in range(-r, r + 1):
                    j = i + k
                    if 0 <= j < n:
                        v = float(x[j])
                    elif edge == O.EDGE_CONSTANT:
                        v = -0.5
                    else:
                        v = float(x[min(max(j, 0), n - 1)])
                    acc += float(w[k + r]) * v
                    aacc += abs(float(w[k + r]) * v)
                assert out[i] == acc and ab[i] == aacc
            # range form agrees with the full call
            if n > 3:
                part, _ = O.mapoverlap_1d(w, r, edge, -0.5, x, 1, n - 1)
                assert np.array_equal(part, out[1:n - 1])


@pytest.mark.parametrize("edge", EDGES)
def test_overlap1d_matrix_axes(edge):
    rows, cols, r = 13, 17, 3
    w = I.signed_weights_f32(150, 2 * r + 1)
    X = I.uniform_pm1_f32(151, rows * cols).reshape(rows, cols)
    rw, _ = O.mapoverlap_1d_matrix(w, r, edge, 0.5, O.AXIS_ROW, X)
    for i in range(rows):
        assert np.array_equal(rw[i], O.mapoverlap_1d(w, r, edge, 0.5, X[i])[0])
    cw, _ = O.mapoverlap_1d_matrix(w, r, edge, 0.5, O.AXIS_COL, X)
    # col-wise on X == transpose(row-wise on X^T)
    assert np.array_equal(cw, O.mapoverlap_1d_matrix(w, r, edge, 0.5, O.AXIS_ROW, np.ascontiguousarray(X.T))[0].T)
    # 1 x n matrix row-wise == vector call; fp64-input entry == fp32 entry on widened data
    v = X.reshape(1, -1)
    assert np.array_equal(O.mapoverlap_1d_matrix(w, r, edge, 0.5, O.AXIS_ROW, v)[0][0], O.mapoverlap_1d(w, r, edge, 0.5, v[0])[0])
    assert np.array_equal(O.mapoverlap_1d_matrix(w, r, edge, 0.5, O.AXIS_COL, X.astype(np.float64))[0], cw)


# ------------------------------------------------------------------ MapOverlap 2D
@pytest.mark.parametrize("edge", EDGES)
def test_overlap2d_brute_force_small(edge):
    for (ry, rx) in [(0, 0), (1, 0), (0, 2), (1, 1), (2, 2), (4, 4), (3, 1)]:
        W = I.signed_weights_f32(160 + ry * 5 + rx, (2 * ry + 1) * (2 * rx + 1)).reshape(2 * ry + 1, 2 * rx + 1)
        for (rows, cols) in [(1, 1), (2, 3), (5, 4), (9, 11), (20, 23)]:
            X = I.uniform_pm1_f32(161 + rows, rows * cols).reshape(rows, cols)
            out, ab = O.mapoverlap_2d(W, ry, rx, edge, 0.75, X)
            for i in range(rows):
                for j in range(cols):
                    acc = 0.0
                    for a in range(-ry, ry + 1):
                        for b in range(-rx, rx + 1):
                            p, q = i + a, j + b
                            if 0 <= p < rows and 0 <= q < cols:
                                v = float(X[p, q])
                            elif edge == O.EDGE_CONSTANT:
                                v = 0.75
                            else:
                                v = float(X[min(max(p, 0), rows - 1), min(max(q, 0), cols - 1)])
                            acc += float(W[a + ry, b + rx]) * v
                    assert out[i, j] == acc
            if rows > 2:
                part, _ = O.mapoverlap_2d(W, ry, rx, edge, 0.75, X, 1, rows - 1)
                assert np.array_equal(part, out[1:rows - 1])


def test_overlap2d_constant_impulse_onehot():
    ry, rx = 2, 2
    W = I.positive_weights_f32(170, 25).reshape(5, 5)
    X = np.full((12, 9), 2.0, np.float32)
    out, _ = O.mapoverlap_2d(W, ry, rx, O.EDGE_DUPLICATE, 0.0, X)
    assert np.allclose(out, 2.0 * W.astype(np.float64).sum(), rtol=1e-15)
    Wsg = I.signed_weights_f32(171, 25).reshape(5, 5)
    X = np.zeros((12, 9), np.float32)
    X[6, 4] = 1.0
    out, _ = O.mapoverlap_2d(Wsg, ry, rx, O.EDGE_CONSTANT, 0.0, X)
    for i in range(12):
        for j in range(9):
            exp = float(Wsg[6 - i + ry, 4 - j + rx]) if abs(i - 6) <= ry and abs(j - 4) <= rx else 0.0
            assert out[i, j] == pytest.approx(exp, abs=1e-15)
    X = I.uniform_pm1_f32(172, 7 * 6).reshape(7, 6)
    for edge in EDGES:
        for a in range(5):
            for b in range(5):
                W1 = np.zeros((5, 5), np.float32)
                W1[a, b] = 1.0
                out, _ = O.mapoverlap_2d(W1, ry, rx, edge, 0.125, X)
                for i in range(7):
                    for j in range(6):
                        p, q = i + a - ry, j + b - rx
                        if 0 <= p < 7 and 0 <= q < 6:
                            exp = float(X[p, q])
                        elif edge == O.EDGE_CONSTANT:
                            exp = 0.125
                        else:
                            exp = float(X[min(max(p, 0), 6), min(max(q, 0), 5)])
                        assert out[i, j] == exp


@pytest.mark.parametrize("edge", EDGES)
def test_overlap2d_degenerate_axes_separable_identity_transpose(edge):
    rows, cols = 19, 21
    X = I.uniform01_f32(180, rows * cols).reshape(rows, cols)
    wr = I.positive_weights_f32(181, 7)
    wc = I.positive_weights_f32(182, 5)
    # ry = 0 == row-wise 1D; rx = 0 == col-wise 1D
    assert np.array_equal(O.mapoverlap_2d(wr.reshape(1, 7), 0, 3, edge, 0.0, X)[0], O.mapoverlap_1d_matrix(wr, 3, edge, 0.0, O.AXIS_ROW, X)[0])
    assert np.array_equal(O.mapoverlap_2d(wc.reshape(5, 1), 2, 0, edge, 0.0, X)[0], O.mapoverlap_1d_matrix(wc, 2, edge, 0.0, O.AXIS_COL, X)[0])
    # separable identity: row pass then column pass (fp64 intermediate) == dense outer-product
    # filter; holds for duplicate edges and for constant-0 edges (SURVEY (c).6 pins). The outer
    # product is rounded to fp32 for the dense call, hence the 1e-6 slack.
    T, _ = O.mapoverlap_1d_matrix(wr, 3, edge, 0.0, O.AXIS_ROW, X)
    S, _ = O.mapoverlap_1d_matrix(wc, 2, edge, 0.0, O.AXIS_COL, T)
    Wd = np.outer(wc.astype(np.float64), wr.astype(np.float64))
    D, _ = O.mapoverlap_2d(Wd.astype(np.float32), 2, 3, edge, 0.0, X)
    assert np.allclose(S, D, rtol=0, atol=1e-6)
    # transpose symmetry
    W = I.signed_weights_f32(183, 15).reshape(3, 5)
    A, _ = O.mapoverlap_2d(W, 1, 2, edge, 0.5, X)
    B, _ = O.mapoverlap_2d(np.ascontiguousarray(W.T), 2, 1, edge, 0.5, np.ascontiguousarray(X.T))
    assert np.allclose(A, B.T, rtol=0, atol=1e-14)


def test_openmp_build_matches_single_thread():
    x = I.uniform01_f32(190, 10007)
    w = I.positive_weights_f32(191, 9)
    X = x[:10000].reshape(100, 100)
    W = I.positive_weights_f32(192, 25)
    O.use_openmp(False)
    a = O.mapoverlap_1d(w, 4, O.EDGE_DUPLICATE, 0.0, x)[0]
    b = O.mapoverlap_2d(W, 2, 2, O.EDGE_DUPLICATE, 0.0, X)[0]
    c = O.map_f32(O.FN_SAXPY, 2.5, x, x)
    try:
        O.use_openmp(True)
        assert np.array_equal(a, O.mapoverlap_1d(w, 4, O.EDGE_DUPLICATE, 0.0, x)[0])
        assert np.array_equal(b, O.mapoverlap_2d(W, 2, 2, O.EDGE_DUPLICATE, 0.0, X)[0])
        assert np.array_equal(c, O.map_f32(O.FN_SAXPY, 2.5, x, x))
    finally:
        O.use_openmp(False)


# ---- CYCLIC edge policy (reading 19) --------------------------------------
@pytest.mark.parametrize("r", [0, 1, 4, 16])
def test_overlap1d_cyclic_is_circular_correlation(r):
    # pin: out = sum_k w[k+r] * roll(x, -k) (numpy roll is the textbook circular shift); the one-hot
    # weight case is a pure rotation and must be bit-exact
    n = 257
    x = I.uniform01_f32(4200 + r, n)
    w = I.signed_weights_f32(4300 + r, 2 * r + 1)
    got, ab = O.mapoverlap_1d(w, r, O.EDGE_CYCLIC, 0.0, x)
    ref = np.zeros(n)
    for k in range(-r, r + 1):
        ref += float(w[k + r]) * np.roll(x.astype(np.float64), -k)
    assert np.allclose(got, ref, rtol=0, atol=1e-13)
    for m in range(2 * r + 1):
        e = np.zeros(2 * r + 1, np.float32)
        e[m] = 1.0
        got, _ = O.mapoverlap_1d(e, r, O.EDGE_CYCLIC, 0.0, x)
        assert np.array_equal(got.astype(np.float32), np.roll(x, -(m - r)))


def test_overlap1d_cyclic_short_vector_wraps_more_than_once():
    # n < r: indices wrap several times (mathematical modulo, never negative)
    x = np.array([1.0, 10.0, 100.0], np.float32)
    r = 5
    w = np.arange(1, 2 * r + 2, dtype=np.float32)
    got, _ = O.mapoverlap_1d(w, r, O.EDGE_CYCLIC, 0.0, x)
    for i in range(3):
        brute = sum(float(w[k + r]) * float(x[(i + k) % 3]) for k in range(-r, r + 1))  # Python % is non-negative
        assert got[i] == brute


def test_overlap2d_cyclic_matches_rolls_and_constant_input():
    rows, cols, ry, rx = 13, 17, 2, 3
    X = I.uniform01_f32(4400, rows * cols).reshape(rows, cols)
    W = I.signed_weights_f32(4401, (2 * ry + 1) * (2 * rx + 1)).reshape(2 * ry + 1, 2 * rx + 1)
    got, _ = O.mapoverlap_2d(W.ravel(), ry, rx, O.EDGE_CYCLIC, 0.0, X)
    ref = np.zeros((rows, cols))
    for a in range(-ry, ry + 1):
        for b in range(-rx, rx + 1):
            ref += float(W[a + ry, b + rx]) * np.roll(X.astype(np.float64), (-a, -b), axis=(0, 1))
    assert np.allclose(got, ref, rtol=0, atol=1e-13)
    # a constant stays constant * sum(W) everywhere (no border at all)
    got, _ = O.mapoverlap_2d(W.ravel(), ry, rx, O.EDGE_CYCLIC, 0.0, np.full((rows, cols), 2.0, np.float32))
    assert np.allclose(got, 2.0 * W.astype(np.float64).sum(), rtol=0, atol=1e-13)
    # column-wise 1D on a matrix == 2D with rx = 0
    wc = I.signed_weights_f32(4402, 5)
    a1, _ = O.mapoverlap_1d_matrix(wc, 2, O.EDGE_CYCLIC, 0.0, O.AXIS_COL, X)
    a2, _ = O.mapoverlap_2d(wc, 2, 0, O.EDGE_CYCLIC, 0.0, X)
    assert np.array_equal(a1, a2)


# ------------------------------------------------------------------ int32 MapOverlap (wraps mod 2^32)
def _py_ext(x, j, edge, pad):
    n = len(x)
    if 0 <= j < n:
        return int(x[j])
    if edge == O.EDGE_CONSTANT:
        return int(pad)
    if edge == O.EDGE_CYCLIC:
        return int(x[j % n])
    return int(x[min(max(j, 0), n - 1)])


ALL_EDGES = [O.EDGE_CONSTANT, O.EDGE_DUPLICATE, O.EDGE_CYCLIC]


@pytest.mark.parametrize("edge", ALL_EDGES)
def test_overlap1d_i32_brute_force_python_ints(edge):
    """Exact Python integers, full-range data and weights (every product and the sum overflow): a dropped tap, a
    flipped filter, a wrong clamp or a missing wrap fails."""
    for r in (0, 1, 2, 5, 16):
        w = I.full_range_i32(300 + r, 2 * r + 1)
        for n in (1, 2, 3, 7, 33, 70):   # n < r included: the index clamps / wraps more than once
            x = I.full_range_i32(301 + n + r, n)
            pad = -123456789
            got = O.mapoverlap_1d_i32(w, r, edge, pad, x)
            exp = [wrap32(sum(int(w[k + r]) * _py_ext(x, i + k, edge, pad) for k in range(-r, r + 1))) for i in range(n)]
            assert got.tolist() == exp, (r, n)
            # a sub-range of the outputs is the same numbers
            if n > 4:
                assert O.mapoverlap_1d_i32(w, r, edge, pad, x, 2, n - 1).tolist() == exp[2:n - 1]


def test_overlap1d_i32_one_hot_shift_impulse_constant_and_library():
    n, r = 257, 4
    x = I.full_range_i32(310, n)
    for m in range(2 * r + 1):                       # one-hot weights: a pure shift, bit-exact, no flip
        w = np.zeros(2 * r + 1, np.int32)
        w[m] = 1
        j = np.arange(n) + m - r
        assert np.array_equal(O.mapoverlap_1d_i32(w, r, O.EDGE_DUPLICATE, 0, x), x[np.clip(j, 0, n - 1)])
        assert np.array_equal(O.mapoverlap_1d_i32(w, r, O.EDGE_CYCLIC, 0, x), x[j % n])
        exp = np.where((j >= 0) & (j < n), x[np.clip(j, 0, n - 1)], np.int32(77))
        assert np.array_equal(O.mapoverlap_1d_i32(w, r, O.EDGE_CONSTANT, 77, x), exp)
    w = I.uniform_int_i32(311, 2 * r + 1, 1000) - 500
    e = np.zeros(n, np.int32)                        # impulse at j: out[i] = w[(j - i) + r] (orientation)
    e[100] = 1
    out = O.mapoverlap_1d_i32(w, r, O.EDGE_CONSTANT, 0, e)
    assert out[100 - r:100 + r + 1].tolist() == w[::-1].tolist() and out.sum() == w.sum()
    K = 123457                                        # constant input: K * sum(w) mod 2^32 everywhere (DUPLICATE)
    assert O.mapoverlap_1d_i32(w, r, O.EDGE_DUPLICATE, 0, np.full(n, K, np.int32)).tolist() == [wrap32(K * int(w.sum()))] * n
    # library special case: numpy.correlate on int64 (no overflow for small values) == interior outputs
    xs = I.uniform_int_i32(312, n, 1000)
    lib = np.correlate(xs.astype(np.int64), w.astype(np.int64), mode="valid")
    assert np.array_equal(O.mapoverlap_1d_i32(w, r, O.EDGE_CONSTANT, 0, xs)[r:n - r].astype(np.int64), lib)
    # small values: the fp64 oracle of the same numbers is exact and must agree, every edge policy
    for edge in ALL_EDGES:
        f, _ = O.mapoverlap_1d(w.astype(np.float32), r, edge, 3.0, xs.astype(np.float32))
        assert np.array_equal(O.mapoverlap_1d_i32(w, r, edge, 3, xs).astype(np.float64), f)


@pytest.mark.parametrize("edge", ALL_EDGES)
def test_overlap_matrix_and_2d_i32(edge):
    rows, cols = 9, 13
    X = I.full_range_i32(320, rows * cols).reshape(rows, cols)
    pad = 40000
    for r in (1, 3, 10):                              # 10 > rows: clamps / wraps through the whole matrix
        w = I.full_range_i32(321 + r, 2 * r + 1)
        got_r = O.mapoverlap_1d_matrix_i32(w, r, edge, pad, O.AXIS_ROW, X)
        got_c = O.mapoverlap_1d_matrix_i32(w, r, edge, pad, O.AXIS_COL, X)
        for i in range(rows):                          # every row / column is the vector call on that row / column
            assert np.array_equal(got_r[i], O.mapoverlap_1d_i32(w, r, edge, pad, X[i]))
        for j in range(cols):
            assert np.array_equal(got_c[:, j], O.mapoverlap_1d_i32(w, r, edge, pad, np.ascontiguousarray(X[:, j])))
        assert np.array_equal(got_c, O.mapoverlap_1d_matrix_i32(w, r, edge, pad, O.AXIS_ROW, np.ascontiguousarray(X.T)).T)
    for ry, rx in ((0, 0), (1, 2), (2, 2), (4, 1)):
        W = I.full_range_i32(330 + 9 * ry + rx, (2 * ry + 1) * (2 * rx + 1)).reshape(2 * ry + 1, 2 * rx + 1)
        got = O.mapoverlap_2d_i32(W, ry, rx, edge, pad, X)

        def ext(p, q):
            if 0 <= p < rows and 0 <= q < cols:
                return int(X[p, q])
            if edge == O.EDGE_CONSTANT:
                return pad
            if edge == O.EDGE_CYCLIC:
                return int(X[p % rows, q % cols])
            return int(X[min(max(p, 0), rows - 1), min(max(q, 0), cols - 1)])

        exp = [[wrap32(sum(int(W[a + ry, b + rx]) * ext(i + a, j + b) for a in range(-ry, ry + 1) for b in range(-rx, rx + 1)))
                for j in range(cols)] for i in range(rows)]
        assert got.tolist() == exp, (ry, rx)
    # degenerate axes: ry = 0 is the row-wise 1D call, rx = 0 the column-wise one; one-hot 2D weights shift both ways
    w = I.full_range_i32(340, 5)
    assert np.array_equal(O.mapoverlap_2d_i32(w.reshape(1, 5), 0, 2, edge, pad, X), O.mapoverlap_1d_matrix_i32(w, 2, edge, pad, O.AXIS_ROW, X))
    assert np.array_equal(O.mapoverlap_2d_i32(w.reshape(5, 1), 2, 0, edge, pad, X), O.mapoverlap_1d_matrix_i32(w, 2, edge, pad, O.AXIS_COL, X))
    W = np.zeros((3, 3), np.int32)
    W[0, 2] = 1                                       # out[i][j] = X~[i-1][j+1]
    p, q = np.arange(rows)[:, None] - 1, np.arange(cols)[None, :] + 1
    if edge == O.EDGE_DUPLICATE:
        exp = X[np.clip(p, 0, rows - 1), np.clip(q, 0, cols - 1)]
    elif edge == O.EDGE_CYCLIC:
        exp = X[p % rows, q % cols]
    else:
        exp = np.where((p >= 0) & (q < cols), X[np.clip(p, 0, rows - 1), np.clip(q, 0, cols - 1)], np.int32(pad))
    assert np.array_equal(O.mapoverlap_2d_i32(W, 1, 1, edge, pad, X), exp)
    # small values agree with the (exact) fp64 oracle; the OpenMP build computes the same numbers
    Xs = I.uniform_int_i32(341, rows * cols, 100).reshape(rows, cols)
    Ws = (I.uniform_int_i32(342, 25, 20) - 10).reshape(5, 5)
    f, _ = O.mapoverlap_2d(Ws.astype(np.float32), 2, 2, edge, 7.0, Xs.astype(np.float32))
    assert np.array_equal(O.mapoverlap_2d_i32(Ws, 2, 2, edge, 7, Xs).astype(np.float64), f)
    O.use_openmp(True)
    try:
        assert np.array_equal(O.mapoverlap_2d_i32(Ws, 2, 2, edge, 7, Xs).astype(np.float64), f)
    finally:
        O.use_openmp(False)


# ------------------------------------------------------------------ fp64 elements (binary128 oracle)
from fractions import Fraction  # noqa: E402


def _rn(fr: Fraction) -> float:
    """Exact rational -> nearest fp64 (Python's int / int true division is correctly rounded)."""
    return fr.numerator / fr.denominator


def test_f64_map_is_the_exact_result_rounded_once():
    n = 300
    x, y = I.uniform_pm1_f64(400, n), I.uniform_pm1_f64(401, n)
    c = 2.5000000000000004   # not a short binary fraction
    for fn, f in ((O.FN_ADD, lambda a, b: a + b), (O.FN_MULT, lambda a, b: a * b), (O.FN_SAXPY, lambda a, b: Fraction(c) * a + b)):
        got = O.map_f64(fn, c, x, y)
        assert got.tolist() == [_rn(f(Fraction(float(a)), Fraction(float(b)))) for a, b in zip(x, y)], fn
    assert np.array_equal(O.map_f64(O.FN_MAX, 0.0, x, y), np.maximum(x, y))
    assert O.map_f64(O.FN_MULT, c, x).tolist() == [_rn(Fraction(float(a)) * Fraction(c)) for a in x]   # constant operand
    # cancellation: c*x + y with y = -RN(c*x): the exact residual, which a separate multiply and add returns as 0
    yc = -(c * x)
    res = O.map_f64(O.FN_SAXPY, c, x, yc)
    assert res.tolist() == [_rn(Fraction(c) * Fraction(float(a)) + Fraction(float(b))) for a, b in zip(x, yc)]
    assert np.count_nonzero(res) > n // 2
    z = I.uniform_pm1_f64(402, n)
    assert O.map3_muladd_f64(x, y, z).tolist() == [_rn(Fraction(float(a)) * Fraction(float(b)) + Fraction(float(d))) for a, b, d in zip(x, y, z)]


def test_f64_reduce_mapreduce_against_exact_rationals_and_cancellation():
    assert O.reduce_f64(O.FN_ADD, np.array([1e16, 1.0, -1e16]))[0] == 1.0          # a plain fp64 loop returns 0
    r, a = O.mapreduce_f64(O.FN_MULT, O.FN_ADD, 0.0, np.array([2.0 ** 27 + 1, -2.0 ** 54]), np.array([2.0 ** 27 + 1, 1.0]))
    assert r == 2.0 ** 28 + 1                                                       # the product needs 55 bits
    for n in BOUNDARY_N:
        x, y = I.uniform_pm1_f64(410 + n, n), I.uniform_pm1_f64(411 + n, n)
        fx, fy = [Fraction(float(t)) for t in x], [Fraction(float(t)) for t in y]
        r, a = O.reduce_f64(O.FN_ADD, x)
        assert r == _rn(sum(fx)) and a == _rn(sum(abs(t) for t in fx))
        assert O.reduce_f64(O.FN_MAX, x)[0] == float(x.max())
        r, a = O.mapreduce_f64(O.FN_MULT, O.FN_ADD, 0.0, x, y)
        assert r == _rn(sum(p * q for p, q in zip(fx, fy))) and a == _rn(sum(abs(p * q) for p, q in zip(fx, fy)))
        r, _ = O.mapreduce_f64(O.FN_SAXPY, O.FN_ADD, 0.75, x, y)
        assert r == _rn(sum(Fraction(0.75) * p + q for p, q in zip(fx, fy)))
        r, _ = O.mapreduce_f64(O.FN_MULT, O.FN_ADD, 3.0, x)                        # constant second operand
        assert r == _rn(3 * sum(fx))
    n = 1 << 16                                                                    # closed form: sum i = n (n - 1) / 2
    assert O.reduce_f64(O.FN_ADD, np.arange(n, dtype=np.float64))[0] == n * (n - 1) // 2
    assert O.mapreduce_f64(O.FN_MULT, O.FN_ADD, 0.0, np.arange(n, dtype=np.float64), np.ones(n))[0] == n * (n - 1) // 2
    p = 1.0 + 1e-3 * I.uniform_pm1_f64(412, 40)
    prod = Fraction(1)
    for t in p:
        prod *= Fraction(float(t))
    assert O.reduce_f64(O.FN_MULT, p)[0] == pytest.approx(_rn(prod), rel=1e-30, abs=0)  # ~1e-34 per step
    with pytest.raises(ValueError):
        O.reduce_f64(O.FN_ADD, np.zeros(0))


def test_f64_scan_against_exact_rationals():
    for n in (0, 1, 2, 3, 33, 257):
        x = I.uniform_pm1_f64(420 + n, n)
        fx = [Fraction(float(t)) for t in x]
        inc, ab = O.scan_f64(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, x)
        acc, exp, expa, aa = Fraction(0), [], [], Fraction(0)
        for t in fx:
            acc += t
            aa += abs(t)
            exp.append(_rn(acc))
            expa.append(_rn(aa))
        assert inc.tolist() == exp and ab.tolist() == expa
        exc, abe = O.scan_f64(O.FN_ADD, O.SCAN_EXCLUSIVE, 0.3, x)
        init = Fraction(0.3)
        assert exc.tolist() == [_rn(init + sum(fx[:i])) for i in range(n)]
        assert abe.tolist() == [_rn(abs(init) + sum(abs(t) for t in fx[:i])) for i in range(n)]
        if n:
            assert np.array_equal(O.scan_f64(O.FN_MAX, O.SCAN_INCLUSIVE, 0.0, x)[0], np.maximum.accumulate(x))
            mxe = O.scan_f64(O.FN_MAX, O.SCAN_EXCLUSIVE, -0.25, x)[0]
            assert mxe[0] == -0.25 and np.array_equal(mxe[1:], np.maximum(np.maximum.accumulate(x)[:-1], -0.25))
    big = np.array([1e16, 1.0, 1.0, -1e16, 1.0])
    assert O.scan_f64(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, big)[0].tolist() == [1e16, 1e16, 1e16 + 2, 2.0, 3.0]
    two = np.full(60, 2.0)
    assert O.scan_f64(O.FN_MULT, O.SCAN_INCLUSIVE, 0.0, two)[0].tolist() == [2.0 ** (k + 1) for k in range(60)]
    assert O.scan_f64(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, np.ones(5000))[0].tolist() == list(range(1, 5001))


@pytest.mark.parametrize("edge", ALL_EDGES)
def test_f64_overlap_against_exact_rationals_shifts_and_the_f32_oracle(edge):
    pad = 0.37
    fpad = Fraction(pad)

    def ext(x, j):
        n = len(x)
        if 0 <= j < n:
            return Fraction(float(x[j]))
        if edge == O.EDGE_CONSTANT:
            return fpad
        if edge == O.EDGE_CYCLIC:
            return Fraction(float(x[j % n]))
        return Fraction(float(x[min(max(j, 0), n - 1)]))

    for r in (0, 1, 3, 16):
        w = I.uniform_pm1_f64(430 + r, 2 * r + 1)
        fw = [Fraction(float(t)) for t in w]
        for n in (1, 2, 5, 40):
            x = I.uniform_pm1_f64(431 + n + r, n)
            got, ab = O.mapoverlap_1d_f64(w, r, edge, pad, x)
            assert got.tolist() == [_rn(sum(fw[k + r] * ext(x, i + k) for k in range(-r, r + 1))) for i in range(n)], (r, n)
            assert ab.tolist() == [_rn(sum(abs(fw[k + r] * ext(x, i + k)) for k in range(-r, r + 1))) for i in range(n)]
    rows, cols = 7, 9
    X = I.uniform_pm1_f64(440, rows * cols).reshape(rows, cols)
    w = I.uniform_pm1_f64(441, 5)
    got_r, _ = O.mapoverlap_1d_matrix_f64(w, 2, edge, pad, O.AXIS_ROW, X)
    got_c, _ = O.mapoverlap_1d_matrix_f64(w, 2, edge, pad, O.AXIS_COL, X)
    for i in range(rows):
        assert np.array_equal(got_r[i], O.mapoverlap_1d_f64(w, 2, edge, pad, X[i])[0])
    for j in range(cols):
        assert np.array_equal(got_c[:, j], O.mapoverlap_1d_f64(w, 2, edge, pad, np.ascontiguousarray(X[:, j]))[0])
    W = I.uniform_pm1_f64(442, 15).reshape(3, 5)

    def ext2(p, q):
        if 0 <= p < rows and 0 <= q < cols:
            return Fraction(float(X[p, q]))
        if edge == O.EDGE_CONSTANT:
            return fpad
        if edge == O.EDGE_CYCLIC:
            return Fraction(float(X[p % rows, q % cols]))
        return Fraction(float(X[min(max(p, 0), rows - 1), min(max(q, 0), cols - 1)]))

    got, _ = O.mapoverlap_2d_f64(W, 1, 2, edge, pad, X)
    exp = [[_rn(sum(Fraction(float(W[a + 1, b + 2])) * ext2(i + a, j + b) for a in (-1, 0, 1) for b in range(-2, 3)))
            for j in range(cols)] for i in range(rows)]
    assert got.tolist() == exp
    # one-hot weights: a pure shift (orientation, edge policy), bit-exact; degenerate axes
    W1 = np.zeros((3, 3))
    W1[2, 0] = 1.0                                  # out[i][j] = X~[i+1][j-1]
    sh, _ = O.mapoverlap_2d_f64(W1, 1, 1, edge, pad, X)
    assert sh.tolist() == [[float(ext2(i + 1, j - 1)) for j in range(cols)] for i in range(rows)]
    assert np.array_equal(O.mapoverlap_2d_f64(w.reshape(1, 5), 0, 2, edge, pad, X)[0], got_r)
    assert np.array_equal(O.mapoverlap_2d_f64(w.reshape(5, 1), 2, 0, edge, pad, X)[0], got_c)
    # fp32-representable data: the fp32-element oracle (fp64 accumulation) and this one agree to ~1e-16 relative
    Xs, Ws = X.astype(np.float32), W.astype(np.float32)
    a32, ab32 = O.mapoverlap_2d(Ws, 1, 2, edge, float(np.float32(pad)), Xs)
    a64, _ = O.mapoverlap_2d_f64(Ws.astype(np.float64), 1, 2, edge, float(np.float32(pad)), Xs.astype(np.float64))
    assert np.all(np.abs(a32 - a64) <= 4e-16 * ab32)
