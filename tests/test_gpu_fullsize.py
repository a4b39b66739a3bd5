"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same plan file,
same containers): results the oracle can produce in seconds are compared whole (integer Reduce / Scan,
dot), the others on sampled windows the oracle computes one by one (windows at both ends and around
tile boundaries in the middle)."""
import os

import numpy as np
import pytest

import oracle as O
from helpers import assert_map_f32, assert_overlap, assert_reduce_f32
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PLAN = os.path.join(ROOT, "paper_1405_2915_b200", "plans", "b200.plan")
N26, N28, SIDE = 1 << 26, 1 << 28, 8192


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    if os.path.exists(PLAN):
        c.plan_load(PLAN)
    O.use_openmp(True)   # same loops, independent outputs in parallel (tests/test_oracle_pins.py checks equality)
    yield c
    O.use_openmp(False)
    c.close()


def windows(n, width=3000):
    """Index windows: both ends and a few places around power-of-two tile boundaries."""
    mids = [n // 2, n // 3, (n // 4096 // 2) * 4096, (n // 65536 // 3) * 65536 + 16384, n - (1 << 20)]
    w = [(0, min(width, n)), (max(0, n - width), n)]
    for m in mids:
        w.append((max(0, m - width // 2), min(n, m + width // 2)))
    return w


def test_map_saxpy_2p26(ctx):
    x, y = I.uniform_pm1_f32(I.config_seed(2, 0), N26), I.uniform_pm1_f32(I.config_seed(2, 1), N26)
    vx, vy, vr = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(N26)
    ctx.map(S.FN_SAXPY, 2.5, vx, vy, vr)
    got = vr.numpy()
    for lo, hi in windows(N26, 100000):
        assert_map_f32(got[lo:hi], O.map_f32(O.FN_SAXPY, 2.5, x[lo:hi], y[lo:hi]))
    idx = I.raw_u64(99, 1 << 16) % np.uint64(N26)
    assert_map_f32(got[idx], O.map_f32(O.FN_SAXPY, 2.5, x[idx], y[idx]))
    # MapReduce dot on the same operands: whole result against the compensated fp64 oracle
    dot = ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vx, vy)
    r, ab = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, y)
    assert_reduce_f32(dot, r, ab)
    for c in (vx, vy, vr):
        c.destroy()


def test_reduce_i32_2p26_bit_exact(ctx):
    v = I.uniform_int_i32(I.config_seed(2, 2), N26, 1000)
    vi = ctx.vector_from(v)
    assert ctx.reduce(S.FN_ADD, vi) == O.reduce_i32(O.FN_ADD, v)[0]   # wraps: the int64 sum is ~7.8 * 2^32
    assert ctx.reduce(S.FN_MAX, vi) == O.reduce_i32(O.FN_MAX, v)[0] == int(v.max())
    vi.destroy()


def test_scan_i32_2p28_bit_exact(ctx):
    x = I.uniform_int_i32(I.config_seed(5, 0), N28, 15)
    assert int(x.astype(np.int64).sum()) < 2**31 - 1    # DESIGN.md reading 7: no wrap occurs on this input
    vx, vo = ctx.vector_from(x), ctx.vector(N28, S.I32)
    ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, vx, vo)
    sk, v = ctx.last_variant()
    ref = O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, x)
    got = vo.numpy()
    assert np.array_equal(got, ref), f"inclusive scan differs (variant {S.variant_names(sk)[v]})"
    ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 0, vx, vo)
    got = vo.numpy()
    assert got[0] == 0 and np.array_equal(got[1:], ref[:-1]), "exclusive scan differs"
    vx.destroy()
    vo.destroy()


@pytest.mark.parametrize("r", [1, 4, 16])
@pytest.mark.parametrize("edge", [S.EDGE_CONSTANT, S.EDGE_DUPLICATE])
def test_overlap1d_2p26_windows(ctx, r, edge):
    x = I.uniform01_f32(I.config_seed(3, 0), N26)
    w = I.positive_weights_f32(I.config_seed(3, 10 + r), 2 * r + 1)
    vx, vo = ctx.vector_from(x), ctx.vector(N26)
    ctx.mapoverlap_1d(w, r, edge, 0.0, vx, vo)
    got = vo.numpy()
    for lo, hi in windows(N26, 20000):
        ref, ab = O.mapoverlap_1d(w, r, edge, 0.0, x, lo, hi)
        assert_overlap(got[lo:hi], ref, ab)
    vx.destroy()
    vo.destroy()


def test_overlap2d_and_separable_8192(ctx):
    X = I.uniform01_f32(I.config_seed(4, 0), SIDE * SIDE).reshape(SIDE, SIDE)
    mx, mt, mo = ctx.matrix_from(X), ctx.matrix(SIDE, SIDE), ctx.matrix(SIDE, SIDE)
    bands = [(0, 24), (4084, 4108), (SIDE - 24, SIDE)]
    for ry, seed in ((2, 1), (4, 2)):
        W = I.positive_weights_f32(I.config_seed(4, seed), (2 * ry + 1) ** 2)
        ctx.mapoverlap_2d(W, ry, ry, S.EDGE_DUPLICATE, 0.0, mx, mo)
        got = mo.numpy()
        for lo, hi in bands:
            ref, ab = O.mapoverlap_2d(W, ry, ry, O.EDGE_DUPLICATE, 0.0, X, lo, hi)
            assert_overlap(got[lo:hi], ref, ab)
    # separable pair (two calls, fp32 intermediate): each pass against its own input, on sampled rows / columns
    wr, wc = I.positive_weights_f32(I.config_seed(4, 3), 17), I.positive_weights_f32(I.config_seed(4, 4), 17)
    ctx.mapoverlap_1d_matrix(wr, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
    ctx.mapoverlap_1d_matrix(wc, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
    T, out = mt.numpy(), mo.numpy()
    for i in (0, 1, 4095, 4096, SIDE - 1):
        ref, ab = O.mapoverlap_1d(wr, 8, O.EDGE_DUPLICATE, 0.0, X[i])
        assert_overlap(T[i], ref, ab)
    for j in (0, 3, 127, 128, 4097, SIDE - 1):
        col = np.ascontiguousarray(T[:, j])
        ref, ab = O.mapoverlap_1d(wc, 8, O.EDGE_DUPLICATE, 0.0, col)
        assert_overlap(np.ascontiguousarray(out[:, j]), ref, ab)
    for c in (mx, mt, mo):
        c.destroy()


def test_fused_separable_8192(ctx):
    """skel_mapoverlap_separable at the bench size, with the variant the plan picks: whole result bit-identical to
    the two public 1D calls (same taps, same order, same fp32 intermediate), sampled columns against the oracle's
    row pass (fp32) fed to its column pass."""
    X = I.uniform01_f32(I.config_seed(4, 0), SIDE * SIDE).reshape(SIDE, SIDE)
    wr, wc = I.positive_weights_f32(I.config_seed(4, 3), 17), I.positive_weights_f32(I.config_seed(4, 4), 17)
    mx, mt, mo, mf = ctx.matrix_from(X), ctx.matrix(SIDE, SIDE), ctx.matrix(SIDE, SIDE), ctx.matrix(SIDE, SIDE)
    ctx.mapoverlap_separable(wr, 8, wc, 8, S.EDGE_DUPLICATE, 0.0, mx, mf)
    sk, v = ctx.last_variant()
    assert sk == S.SK_SEPARABLE and S.variant_names(sk)[v].startswith("fused")
    ctx.mapoverlap_1d_matrix(wr, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
    ctx.mapoverlap_1d_matrix(wc, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
    fused = mf.numpy()
    assert np.array_equal(fused, mo.numpy())
    for j in (0, 5, 127, 128, 4097, SIDE - 1):
        # the row pass of column j reads columns j-8 .. j+8 (clamped): cut a block that contains them and whose own
        # clamping coincides with the matrix's (it starts at column 0 / ends at the last column) or is never reached
        lo = 0 if j < 16 else j - 8
        hi = SIDE if j >= SIDE - 16 else j + 9
        sub = np.ascontiguousarray(X[:, lo:hi])
        jj = j - lo
        t64, tabs = O.mapoverlap_1d_matrix(wr, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_ROW, sub)
        tcol = np.ascontiguousarray(t64[:, jj]).astype(np.float32)
        ref, ab = O.mapoverlap_1d(wc, 8, O.EDGE_DUPLICATE, 0.0, tcol)
        carried, _ = O.mapoverlap_1d(wc, 8, O.EDGE_DUPLICATE, 0.0, np.ascontiguousarray(tabs[:, jj]).astype(np.float32))
        err = np.abs(np.ascontiguousarray(fused[:, j]).astype(np.float64) - ref)
        assert np.all(err <= 2e-6 * (ab + 1.000001 * carried)), (j, float((err / (ab + carried)).max()))
    for c in (mx, mt, mo, mf):
        c.destroy()


def test_fused_chain_2p26(ctx):
    """The chained pipeline iteration of BASELINE.json configs[4] as ONE kernel (skel_ctx_set_fusion) at the bench
    size: A' bit-identical to the oracle's Map, B on sampled windows, the sum against the oracle chain."""
    x = I.uniform01_f32(I.config_seed(5, 1), N26)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    a, b = ctx.vector_from(x), ctx.vector(N26)
    ctx.set_fusion(True)
    try:
        ctx.reset_stats()
        ctx.map(S.FN_MULT, 1.0001, a, None, a)
        ctx.mapoverlap_1d(w, 4, S.EDGE_DUPLICATE, 0.0, a, b)
        s = ctx.reduce(S.FN_ADD, b)
        st = ctx.stats()
    finally:
        ctx.set_fusion(False)
    assert st["fused_launches"] == 1 and st["launches"] == 1
    a1 = O.map_f32(O.FN_MULT, 1.0001, x).astype(np.float32)
    assert np.array_equal(a.numpy(), a1)
    ref, ab = O.mapoverlap_1d(w, 4, O.EDGE_DUPLICATE, 0.0, a1)
    got = b.numpy()
    for lo, hi in windows(N26, 50000):
        assert_overlap(got[lo:hi], ref[lo:hi], ab[lo:hi])
    r, asum = O.reduce_f32(O.FN_ADD, ref.astype(np.float32))
    assert abs(s - r) <= 1e-5 * asum + 2e-6 * float(ab.sum()), (s, r)
    a.destroy()
    b.destroy()
