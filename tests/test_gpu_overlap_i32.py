"""MapOverlap on int32 containers (include/skel.h skel_mapoverlap_*_i32; reading 26):
bit-exact against the oracle's int32 definitions (oracle/oracle.cpp, pinned in tests/test_oracle_pins.py) for every
kernel variant that runs int32 elements, on full-range data and weights (every product and sum wraps modulo 2^32)."""
import numpy as np
import pytest

import oracle as O
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

EDGE_CASES = [(S.EDGE_CONSTANT, 0), (S.EDGE_CONSTANT, -2147483648), (S.EDGE_CONSTANT, 123456789), (S.EDGE_DUPLICATE, 0),
              (S.EDGE_CYCLIC, 0)]
SIZES = [1, 2, 3, 5, 17, 33, 100, 1023, 4096, 4097, 8200, 12320, 16385, 65537, 300001]
MAT_SHAPES = [(1, 1), (3, 5), (37, 129), (64, 128), (65, 136), (200, 520), (130, 1032), (6, 8256)]


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


def i32_variants(sk):
    """Variants that run int32 elements: direct, regshfl_*, tma_* (csrc/overlap1d.cu, csrc/overlap2d.cu)."""
    names = S.variant_names(sk)
    return [v for v, n in enumerate(names) if n == "direct" or n.startswith("regshfl") or (n.startswith("tma_") and "bx" not in n)]


def run_forced(ctx, sk, v, fn):
    ctx.force_variant(sk, v)
    try:
        fn()
        assert ctx.last_variant() == (sk, v)
    finally:
        ctx.force_variant(sk, -1)


@pytest.mark.parametrize("v", i32_variants(S.SK_OVERLAP1D))
@pytest.mark.parametrize("r", [0, 1, 2, 4, 5, 8, 16])
def test_overlap1d_i32_vector(ctx, v, r):
    if S.variant_names(S.SK_OVERLAP1D)[v] == "regshfl_2x8" and r > 8:
        return
    w = I.full_range_i32(9000 + r, 2 * r + 1)
    for n in SIZES:
        x = I.full_range_i32(9001 + n, n)
        vx, vo = ctx.vector_from(x), ctx.vector(n, S.I32)
        for edge, pad in EDGE_CASES:
            run_forced(ctx, S.SK_OVERLAP1D, v, lambda: ctx.mapoverlap_1d_i32(w, r, edge, pad, vx, vo))
            assert np.array_equal(vo.numpy(), O.mapoverlap_1d_i32(w, r, edge, pad, x)), (n, edge, pad)
        vx.destroy()
        vo.destroy()


def test_overlap1d_i32_large_r_and_default_variant(ctx):
    n = 100003
    x = I.full_range_i32(9010, n)
    vx, vo = ctx.vector_from(x), ctx.vector(n, S.I32)
    for r in (17, 64):                      # only the direct variant
        w = I.full_range_i32(9011 + r, 2 * r + 1)
        ctx.mapoverlap_1d_i32(w, r, S.EDGE_DUPLICATE, 0, vx, vo)
        assert S.variant_names(S.SK_OVERLAP1D)[ctx.last_variant()[1]] == "direct"
        assert np.array_equal(vo.numpy(), O.mapoverlap_1d_i32(w, r, O.EDGE_DUPLICATE, 0, x))
    w = I.full_range_i32(9012, 9)           # untuned int32 instance: a TMA / register-window variant, not `direct`
    ctx.mapoverlap_1d_i32(w, 4, S.EDGE_DUPLICATE, 0, vx, vo)
    assert S.variant_names(S.SK_OVERLAP1D)[ctx.last_variant()[1]] != "direct"
    assert np.array_equal(vo.numpy(), O.mapoverlap_1d_i32(w, 4, O.EDGE_DUPLICATE, 0, x))
    vx.destroy()
    vo.destroy()


@pytest.mark.parametrize("v", i32_variants(S.SK_OVERLAP1D))
def test_overlap1d_i32_matrix_rows(ctx, v):
    name = S.variant_names(S.SK_OVERLAP1D)[v]
    for r in (1, 4, 8):
        w = I.full_range_i32(9020 + r, 2 * r + 1)
        for rows, cols in MAT_SHAPES:
            ok = v == 0 or (rows == 1 or cols % (32 if name.startswith("tma") else 8) == 0)
            X = I.full_range_i32(9021 + rows, rows * cols).reshape(rows, cols)
            mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols, S.I32)
            for edge, pad in EDGE_CASES[1:]:
                if not ok:
                    with pytest.raises(S.SkelError):
                        run_forced(ctx, S.SK_OVERLAP1D, v, lambda: ctx.mapoverlap_1d_matrix_i32(w, r, edge, pad, S.AXIS_ROW, mx, mo))
                    continue
                run_forced(ctx, S.SK_OVERLAP1D, v, lambda: ctx.mapoverlap_1d_matrix_i32(w, r, edge, pad, S.AXIS_ROW, mx, mo))
                assert np.array_equal(mo.numpy(), O.mapoverlap_1d_matrix_i32(w, r, edge, pad, O.AXIS_ROW, X)), (rows, cols, edge)
            mx.destroy()
            mo.destroy()


@pytest.mark.parametrize("v", i32_variants(S.SK_OVERLAP1D_COL))
@pytest.mark.parametrize("r", [0, 1, 3, 5, 8, 16])
def test_overlap1d_i32_matrix_cols(ctx, v, r):
    w = I.full_range_i32(9030 + r, 2 * r + 1)
    for rows, cols in MAT_SHAPES:
        X = I.full_range_i32(9031 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols, S.I32)
        for edge, pad in EDGE_CASES[1:]:
            if v != 0 and cols % 4 != 0:
                with pytest.raises(S.SkelError):
                    run_forced(ctx, S.SK_OVERLAP1D_COL, v, lambda: ctx.mapoverlap_1d_matrix_i32(w, r, edge, pad, S.AXIS_COL, mx, mo))
                continue
            run_forced(ctx, S.SK_OVERLAP1D_COL, v, lambda: ctx.mapoverlap_1d_matrix_i32(w, r, edge, pad, S.AXIS_COL, mx, mo))
            assert np.array_equal(mo.numpy(), O.mapoverlap_1d_matrix_i32(w, r, edge, pad, O.AXIS_COL, X)), (rows, cols, edge)
        mx.destroy()
        mo.destroy()


@pytest.mark.parametrize("v", i32_variants(S.SK_OVERLAP2D))
@pytest.mark.parametrize("radii", [(0, 0), (1, 1), (2, 2), (3, 3), (4, 4), (2, 4), (1, 0), (8, 8)])
def test_overlap2d_i32(ctx, v, radii):
    ry, rx = radii
    W = I.full_range_i32(9040 + 9 * ry + rx, (2 * ry + 1) * (2 * rx + 1))
    for rows, cols in MAT_SHAPES:
        X = I.full_range_i32(9041 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols, S.I32)
        ok = v == 0 or (ry <= 4 and rx <= 4 and cols % 4 == 0)
        for edge, pad in EDGE_CASES[1:]:
            if not ok:
                with pytest.raises(S.SkelError):
                    run_forced(ctx, S.SK_OVERLAP2D, v, lambda: ctx.mapoverlap_2d_i32(W, ry, rx, edge, pad, mx, mo))
                continue
            run_forced(ctx, S.SK_OVERLAP2D, v, lambda: ctx.mapoverlap_2d_i32(W, ry, rx, edge, pad, mx, mo))
            assert np.array_equal(mo.numpy(), O.mapoverlap_2d_i32(W, ry, rx, edge, pad, X)), (rows, cols, edge)
        mx.destroy()
        mo.destroy()


def test_overlap_i32_multitile_whole_output(ctx):
    """Every persistent block walks several tiles (tests/test_gpu_multitile.py): refilled stages, the dynamic tile queue."""
    O.use_openmp(True)
    try:
        rows, cols = 3075, 6148
        X = I.full_range_i32(9050, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols, S.I32)
        W = I.full_range_i32(9051, 25)
        w = I.full_range_i32(9052, 17)
        for edge, pad in ((S.EDGE_CONSTANT, 7), (S.EDGE_DUPLICATE, 0), (S.EDGE_CYCLIC, 0)):
            ref2 = O.mapoverlap_2d_i32(W, 2, 2, edge, pad, X)
            refc = O.mapoverlap_1d_matrix_i32(w, 8, edge, pad, O.AXIS_COL, X)
            for v in i32_variants(S.SK_OVERLAP2D)[1:]:
                run_forced(ctx, S.SK_OVERLAP2D, v, lambda: ctx.mapoverlap_2d_i32(W, 2, 2, edge, pad, mx, mo))
                assert np.array_equal(mo.numpy(), ref2), (v, edge)
            for v in i32_variants(S.SK_OVERLAP1D_COL)[1:]:
                run_forced(ctx, S.SK_OVERLAP1D_COL, v, lambda: ctx.mapoverlap_1d_matrix_i32(w, 8, edge, pad, S.AXIS_COL, mx, mo))
                assert np.array_equal(mo.numpy(), refc), (v, edge)
        mx.destroy()
        mo.destroy()
        n = 4096 * 3700 + 77
        x = I.full_range_i32(9053, n)
        vx, vo = ctx.vector_from(x), ctx.vector(n, S.I32)
        w = I.full_range_i32(9054, 33)
        for edge, pad in ((S.EDGE_CONSTANT, 0), (S.EDGE_CONSTANT, -5), (S.EDGE_CYCLIC, 0)):
            ref = O.mapoverlap_1d_i32(w, 16, edge, pad, x)
            for v in i32_variants(S.SK_OVERLAP1D)[1:]:
                if S.variant_names(S.SK_OVERLAP1D)[v] == "regshfl_2x8":
                    continue
                run_forced(ctx, S.SK_OVERLAP1D, v, lambda: ctx.mapoverlap_1d_i32(w, 16, edge, pad, vx, vo))
                assert np.array_equal(vo.numpy(), ref), (v, edge)
        vx.destroy()
        vo.destroy()
    finally:
        O.use_openmp(False)


def test_overlap_i32_small_values_agree_with_the_f32_call_and_errors(ctx):
    n = 50000
    x = I.uniform_int_i32(9060, n, 1000)
    w = I.uniform_int_i32(9061, 9, 100) - 50
    vi, vo = ctx.vector_from(x), ctx.vector(n, S.I32)
    vf, vfo = ctx.vector_from(x.astype(np.float32)), ctx.vector(n)
    ctx.mapoverlap_1d_i32(w, 4, S.EDGE_DUPLICATE, 0, vi, vo)
    ctx.mapoverlap_1d(w.astype(np.float32), 4, S.EDGE_DUPLICATE, 0.0, vf, vfo)
    assert np.array_equal(vo.numpy().astype(np.float32), vfo.numpy())    # |sums| < 2^24: both exact
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_1d_i32(w, 4, S.EDGE_DUPLICATE, 0, vf, vfo)        # f32 containers in the int32 call
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_1d(w.astype(np.float32), 4, S.EDGE_DUPLICATE, 0.0, vi, vo)
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_1d_i32(w, 4, S.EDGE_DUPLICATE, 0, vi, vi)         # alias
    for c in (vi, vo, vf, vfo):
        c.destroy()
