"""Whole-output parity of the PERSISTENT 2D kernels on matrices that give every resident block several tiles.

VERDICT r1 weak point 3 / ADVICE r1: the shapes of test_gpu_parity.py / test_gpu_separable.py top out at 99 tiles,
fewer than the 148 x occupancy blocks a persistent kernel launches, so every block walks exactly one tile there and
the refill path (the `empty` mbarrier wait of the producer, the TMA refill of a stage that generic-proxy writes have
patched, both mbarrier parities, the cp.async double buffer's second half) is never reached by a whole-output
comparison. Here: 3072 x 6144 (96 x 48 tiles of 32 x 128 = 4608 tiles >= 4 x 148 x 5 blocks; 48 x 48 tiles of
64 x 128 = 2304 >= 4 x 148 x 3) and the ragged 3075 x 6148 (partial tiles on both axes, cols % 128 = 4), every tiled
variant of MapOverlap 2D, of the column pass and of the fused separable pair, all edge cases, element by element
against the OpenMP build of the oracle (the same loops; tests/test_oracle_pins.py checks the two builds agree).
"""
import numpy as np
import pytest

import oracle as O
import skel_inputs as I
from helpers import assert_overlap
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

SHAPES = [(3072, 6144), (3075, 6148)]
EDGE_CASES = [(S.EDGE_CONSTANT, 0.0), (S.EDGE_CONSTANT, 0.75), (S.EDGE_DUPLICATE, 0.0), (S.EDGE_CYCLIC, 0.0)]


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    O.use_openmp(True)
    yield c
    O.use_openmp(False)
    c.close()


def tiled_variants(sk):
    return [v for v in range(1, S.lib.skel_variant_count(sk))]


def tiles_per_block(rows, cols, tile_h, blocks_per_sm=5, sms=148):
    return (-(-rows // tile_h)) * (-(-cols // 128)) / (sms * blocks_per_sm)


def test_shapes_give_every_block_at_least_four_tiles():
    for rows, cols in SHAPES:
        assert tiles_per_block(rows, cols, 32, 5) >= 4      # 32-row tiles, at most 5 resident blocks per SM
        assert tiles_per_block(rows, cols, 64, 3) >= 4      # 64-row tiles, at most 3


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("r", [2, 4, 1])
def test_overlap2d_persistent_whole_output(ctx, shape, r):
    rows, cols = shape
    X = I.uniform01_f32(8100 + rows, rows * cols).reshape(rows, cols)
    W = I.signed_weights_f32(8101 + r, (2 * r + 1) ** 2)
    mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
    names = S.variant_names(S.SK_OVERLAP2D)
    ran = 0
    for edge, pad in EDGE_CASES:
        ref, ab = O.mapoverlap_2d(W, r, r, edge, pad, X)
        for v in tiled_variants(S.SK_OVERLAP2D):
            ctx.force_variant(S.SK_OVERLAP2D, v)
            try:
                ctx.mapoverlap_2d(W, r, r, edge, pad, mx, mo)
                assert ctx.last_variant() == (S.SK_OVERLAP2D, v)
            except S.SkelError:
                continue   # variant not instantiated for this radius (checked by test_gpu_parity.py)
            finally:
                ctx.force_variant(S.SK_OVERLAP2D, -1)
            ran += 1
            try:
                assert_overlap(mo.numpy(), ref, ab)
            except AssertionError as e:
                raise AssertionError(f"{names[v]} r={r} edge={edge} pad={pad} {rows}x{cols}: {e}") from None
    assert ran >= 4 * 5
    mx.destroy()
    mo.destroy()


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("r", [8, 16, 2])
def test_overlap1d_cols_persistent_whole_output(ctx, shape, r):
    rows, cols = shape
    X = I.uniform01_f32(8200 + rows, rows * cols).reshape(rows, cols)
    w = I.signed_weights_f32(8201 + r, 2 * r + 1)
    mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
    names = S.variant_names(S.SK_OVERLAP1D_COL)
    ran = 0
    for edge, pad in EDGE_CASES:
        ref, ab = O.mapoverlap_1d_matrix(w, r, edge, pad, O.AXIS_COL, X)
        for v in tiled_variants(S.SK_OVERLAP1D_COL):
            ctx.force_variant(S.SK_OVERLAP1D_COL, v)
            try:
                ctx.mapoverlap_1d_matrix(w, r, edge, pad, S.AXIS_COL, mx, mo)
                assert ctx.last_variant() == (S.SK_OVERLAP1D_COL, v)
            except S.SkelError:
                continue
            finally:
                ctx.force_variant(S.SK_OVERLAP1D_COL, -1)
            ran += 1
            try:
                assert_overlap(mo.numpy(), ref, ab)
            except AssertionError as e:
                raise AssertionError(f"{names[v]} r={r} edge={edge} pad={pad} {rows}x{cols}: {e}") from None
    assert ran >= 4 * 5
    mx.destroy()
    mo.destroy()


@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("r", [8, 4])
def test_separable_fused_whole_output(ctx, shape, r):
    """Every fused variant: bit-identical to the two public 1D calls (whole output), and the two calls themselves within
    tolerance of the oracle's fp64 chain (whole output)."""
    rows, cols = shape
    X = I.uniform01_f32(8300 + rows, rows * cols).reshape(rows, cols)
    wr, wc = I.positive_weights_f32(8301 + r, 2 * r + 1), I.signed_weights_f32(8302 + r, 2 * r + 1)
    mx, mt, mo, mf = ctx.matrix_from(X), ctx.matrix(rows, cols), ctx.matrix(rows, cols), ctx.matrix(rows, cols)
    names = S.variant_names(S.SK_SEPARABLE)
    for (edge, pad), oe in zip(EDGE_CASES, (O.EDGE_CONSTANT, O.EDGE_CONSTANT, O.EDGE_DUPLICATE, O.EDGE_CYCLIC)):
        t64, tabs = O.mapoverlap_1d_matrix(wr, r, oe, pad, O.AXIS_ROW, X)
        ref, ab = O.mapoverlap_1d_matrix(wc, r, oe, pad, O.AXIS_COL, t64.astype(np.float32))
        carried, _ = O.mapoverlap_1d_matrix(np.abs(wc), r, oe, 0.0, O.AXIS_COL, tabs.astype(np.float32))
        tol = ab + 1.000001 * np.abs(carried)
        ctx.mapoverlap_1d_matrix(wr, r, edge, pad, S.AXIS_ROW, mx, mt)
        ctx.mapoverlap_1d_matrix(wc, r, edge, pad, S.AXIS_COL, mt, mo)
        two = mo.numpy().copy()
        assert_overlap(mt.numpy(), t64, tabs)
        assert_overlap(two, ref, tol)
        ran = 0
        for v in tiled_variants(S.SK_SEPARABLE):
            ctx.force_variant(S.SK_SEPARABLE, v)
            try:
                ctx.mapoverlap_separable(wr, r, wc, r, edge, pad, mx, mf)
            except S.SkelError:
                continue
            finally:
                ctx.force_variant(S.SK_SEPARABLE, -1)
            ran += 1
            got = mf.numpy()
            assert_overlap(got, ref, tol)
            assert np.array_equal(got, two), f"{names[v]} r={r} edge={edge} pad={pad}: differs from the two 1D calls"
        assert ran >= 2 or cols % 4 != 0
    for m in (mx, mt, mo, mf):
        m.destroy()
