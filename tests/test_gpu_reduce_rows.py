"""skel_reduce_rows against the CPU oracle: int32 bit-exact (wraps), fp32 max exact, fp32 add / mult
within the Reduce tolerance (1e-5 * sum|terms| per row; BASELINE.json L5), every variant forced, ragged shapes."""
import numpy as np
import pytest

import oracle as O
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

SHAPES = [(1, 1), (1, 5), (3, 4), (7, 33), (37, 129), (64, 128), (65, 136), (9, 4100), (300, 1027), (1030, 264),
          (2, 70000), (5000, 12)]


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


@pytest.mark.parametrize("v", [0, 1, 2, 3])
def test_reduce_rows_matches_oracle(ctx, v):
    names = S.variant_names(S.SK_REDUCE_ROWS)
    assert names == ["warp_scalar", "warp_v4", "block_v4", "block_v4_row"]
    for rows, cols in SHAPES:
        X = I.uniform_pm1_f32(800 + rows, rows * cols).reshape(rows, cols)
        Xi = (I.raw_u64(801 + rows, rows * cols) % np.uint64(1 << 31)).astype(np.int32).reshape(rows, cols)
        mx, mi = ctx.matrix_from(X), ctx.matrix_from(Xi)
        of, oi = ctx.vector(rows), ctx.vector(rows, S.I32)
        vec_ok = v == 0 or cols % 4 == 0
        ctx.force_variant(S.SK_REDUCE_ROWS, v)
        try:
            if not vec_ok:
                with pytest.raises(S.SkelError):
                    ctx.reduce_rows(S.FN_ADD, mx, of)
                continue
            ctx.reduce_rows(S.FN_ADD, mx, of)
            assert ctx.last_variant() == (S.SK_REDUCE_ROWS, v)
            r, a = O.reduce_rows_f32(O.FN_ADD, X)
            got = of.numpy()
            assert np.all(np.abs(got.astype(np.float64) - r) <= 1e-5 * a), (rows, cols)
            ctx.reduce_rows(S.FN_MAX, mx, of)
            assert np.array_equal(of.numpy().astype(np.float64), O.reduce_rows_f32(O.FN_MAX, X)[0])
            P = (1.0 + 1e-3 * X).astype(np.float32)
            mx.write(P)
            ctx.reduce_rows(S.FN_MULT, mx, of)
            r, _ = O.reduce_rows_f32(O.FN_MULT, P)
            assert np.allclose(of.numpy(), r, rtol=1e-5 * max(1, cols // 64), atol=0)
            for op, oop in ((S.FN_ADD, O.FN_ADD), (S.FN_MAX, O.FN_MAX), (S.FN_MULT, O.FN_MULT)):
                ctx.reduce_rows(op, mi, oi)
                assert np.array_equal(oi.numpy(), O.reduce_rows_i32(oop, Xi)), (rows, cols, op)
        finally:
            ctx.force_variant(S.SK_REDUCE_ROWS, -1)
            for c in (mx, mi, of, oi):
                c.destroy()


def test_reduce_rows_closed_forms_determinism_and_errors(ctx):
    rows, cols = 513, 2052
    Xj = np.repeat(np.arange(cols, dtype=np.int32)[None, :], rows, axis=0)
    mi, oi = ctx.matrix_from(Xj), ctx.vector(rows, S.I32)
    ctx.reduce_rows(S.FN_ADD, mi, oi)
    assert oi.numpy().tolist() == [cols * (cols - 1) // 2] * rows
    X = I.uniform_pm1_f32(810, rows * cols).reshape(rows, cols)
    mx, of = ctx.matrix_from(X), ctx.vector(rows)
    ctx.reduce_rows(S.FN_ADD, mx, of)
    first = of.numpy().copy()
    for _ in range(3):
        ctx.reduce_rows(S.FN_ADD, mx, of)
        assert np.array_equal(of.numpy(), first), "row-wise reduce is not deterministic run to run"
    # each row equals the vector Reduce of that row within the tolerance (the matrix as_vector view, first row)
    r, a = O.reduce_rows_f32(O.FN_ADD, X)
    assert np.all(np.abs(first.astype(np.float64) - r) <= 1e-5 * a)
    bad = ctx.vector(rows + 1)
    with pytest.raises(S.SkelError):
        ctx.reduce_rows(S.FN_ADD, mx, bad)            # one element per row
    with pytest.raises(S.SkelError):
        ctx.reduce_rows(S.FN_ADD, mx, oi)             # element types differ
    with pytest.raises(S.SkelError):
        ctx.reduce_rows(S.FN_SAXPY, mx, of)           # not a reduction operator
    for c in (mi, oi, mx, of, bad):
        c.destroy()
