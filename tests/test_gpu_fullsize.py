"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same plan file,
same containers). Every result is compared WHOLE, element by element, against the oracle: the sequential
build for Reduce / Scan / dot, the OpenMP build of the same loops (independent outputs in parallel;
tests/test_oracle_pins.py checks the two builds agree) for Map and the stencils, which it finishes in seconds."""
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


def test_map_saxpy_2p26(ctx):
    x, y = I.uniform_pm1_f32(I.config_seed(2, 0), N26), I.uniform_pm1_f32(I.config_seed(2, 1), N26)
    vx, vy, vr = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(N26)
    ctx.map(S.FN_SAXPY, 2.5, vx, vy, vr)
    assert_map_f32(vr.numpy(), O.map_f32(O.FN_SAXPY, 2.5, x, y))   # whole output
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
def test_overlap1d_2p26_whole(ctx, r, edge):
    x = I.uniform01_f32(I.config_seed(3, 0), N26)
    w = I.positive_weights_f32(I.config_seed(3, 10 + r), 2 * r + 1)
    vx, vo = ctx.vector_from(x), ctx.vector(N26)
    ctx.mapoverlap_1d(w, r, edge, 0.0, vx, vo)
    ref, ab = O.mapoverlap_1d(w, r, edge, 0.0, x)
    assert_overlap(vo.numpy(), ref, ab)   # whole output
    vx.destroy()
    vo.destroy()


def test_overlap2d_and_separable_8192(ctx):
    X = I.uniform01_f32(I.config_seed(4, 0), SIDE * SIDE).reshape(SIDE, SIDE)
    mx, mt, mo = ctx.matrix_from(X), ctx.matrix(SIDE, SIDE), ctx.matrix(SIDE, SIDE)
    for ry, seed in ((2, 1), (4, 2)):
        W = I.positive_weights_f32(I.config_seed(4, seed), (2 * ry + 1) ** 2)
        ctx.mapoverlap_2d(W, ry, ry, S.EDGE_DUPLICATE, 0.0, mx, mo)
        ref, ab = O.mapoverlap_2d(W, ry, ry, O.EDGE_DUPLICATE, 0.0, X)
        assert_overlap(mo.numpy(), ref, ab)   # whole output
        del ref, ab
    # separable pair (two calls, fp32 intermediate): each pass against its own input (lock-step), whole outputs
    wr, wc = I.positive_weights_f32(I.config_seed(4, 3), 17), I.positive_weights_f32(I.config_seed(4, 4), 17)
    ctx.mapoverlap_1d_matrix(wr, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
    ctx.mapoverlap_1d_matrix(wc, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
    T = mt.numpy().copy()
    ref, ab = O.mapoverlap_1d_matrix(wr, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_ROW, X)
    assert_overlap(T, ref, ab)
    ref2, ab2 = O.mapoverlap_1d_matrix(wc, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, T)
    assert_overlap(mo.numpy(), ref2, ab2)
    del ref2, ab2
    # ... and the pair against the oracle's fp64 chain (intermediate kept in fp64, SURVEY 8(c).6 iii)
    ref3, ab3 = O.mapoverlap_1d_matrix(wc, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, ref)
    assert_overlap(mo.numpy(), ref3, ab3)
    for c in (mx, mt, mo):
        c.destroy()


def test_fused_separable_8192(ctx):
    """skel_mapoverlap_separable at the bench size, with the variant the plan picks: the WHOLE result against the
    oracle's row pass (rounded to fp32, reading 20) fed to its column pass; then, as a second and weaker
    check, bit-identical to the two public 1D calls (same taps, same order, same fp32 intermediate)."""
    X = I.uniform01_f32(I.config_seed(4, 0), SIDE * SIDE).reshape(SIDE, SIDE)
    wr, wc = I.positive_weights_f32(I.config_seed(4, 3), 17), I.positive_weights_f32(I.config_seed(4, 4), 17)
    mx, mt, mo, mf = ctx.matrix_from(X), ctx.matrix(SIDE, SIDE), ctx.matrix(SIDE, SIDE), ctx.matrix(SIDE, SIDE)
    ctx.mapoverlap_separable(wr, 8, wc, 8, S.EDGE_DUPLICATE, 0.0, mx, mf)
    sk, v = ctx.last_variant()
    assert sk == S.SK_SEPARABLE and S.variant_names(sk)[v].startswith(("fused", "march"))  # one launch, not two_pass
    fused = mf.numpy().copy()
    t64, tabs = O.mapoverlap_1d_matrix(wr, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_ROW, X)
    ref, ab = O.mapoverlap_1d_matrix(wc, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, t64.astype(np.float32))
    del t64
    carried, _ = O.mapoverlap_1d_matrix(wc, 8, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, tabs.astype(np.float32))
    del tabs
    assert_overlap(fused, ref, ab + 1.000001 * carried)   # whole output; tolerance: tests/test_gpu_separable.py
    del ref, ab, carried
    ctx.mapoverlap_1d_matrix(wr, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
    ctx.mapoverlap_1d_matrix(wc, 8, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
    assert np.array_equal(fused, mo.numpy())
    for c in (mx, mt, mo, mf):
        c.destroy()


def test_fused_chain_2p26(ctx):
    """The chained pipeline iteration of BASELINE.json configs[4] as ONE kernel (skel_ctx_set_fusion) at the bench
    size: A' bit-identical to the oracle's Map, B whole, the sum against the oracle chain."""
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
    assert_overlap(b.numpy(), ref, ab)   # whole output
    r, asum = O.reduce_f32(O.FN_ADD, ref.astype(np.float32))
    assert abs(s - r) <= 1e-5 * asum + 2e-6 * float(ab.sum()), (s, r)
    a.destroy()
    b.destroy()
