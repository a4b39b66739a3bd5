"""skel_mapoverlap_separable (include/skel.h): out = colpass(RN_f32(rowpass(X))).
The expected value is the oracle's row pass, rounded to fp32, fed to the oracle's column pass.
Tolerance per element: the column pass's own 2e-6 * sum_a |wc_a T~[i+a][j]|, plus what the row pass's
tolerance lets the GPU's intermediate differ from the oracle's, carried through the column filter:
sum_a |wc_a| * 2e-6 * (sum_b |wr_b X~|)[i+a][j] (the oracle's column pass applied to the row pass's
absolute-term sums with |wc|; for CONSTANT edges the padded rows of T are exact)."""
import numpy as np
import pytest

import oracle as O
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

SHAPES = [(1, 4), (3, 8), (9, 128), (33, 132), (64, 256), (70, 136), (150, 520), (257, 1028), (40, 30)]
EDGES = [(S.EDGE_CONSTANT, O.EDGE_CONSTANT, 0.0), (S.EDGE_CONSTANT, O.EDGE_CONSTANT, 0.5),
         (S.EDGE_DUPLICATE, O.EDGE_DUPLICATE, 0.0), (S.EDGE_CYCLIC, O.EDGE_CYCLIC, 0.0)]


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


def oracle_separable(wr, rr, wc, rc, oe, pad, X):
    t64, tabs = O.mapoverlap_1d_matrix(wr, rr, oe, pad, O.AXIS_ROW, X)
    t32 = t64.astype(np.float32)
    ref, ab = O.mapoverlap_1d_matrix(wc, rc, oe, pad, O.AXIS_COL, t32)
    # the row pass's absolute-term sums seen through |wc| (pad cells of a CONSTANT edge carry no error)
    carried, _ = O.mapoverlap_1d_matrix(np.abs(wc), rc, oe, 0.0, O.AXIS_COL, tabs.astype(np.float32))
    return ref, ab + np.abs(carried) * 1.000001


@pytest.mark.parametrize("v", list(range(S.lib.skel_variant_count(S.SK_SEPARABLE))))
@pytest.mark.parametrize("radii", [(1, 1), (2, 2), (3, 3), (4, 4), (8, 8), (0, 0), (8, 2), (5, 5), (3, 6), (16, 16), (9, 1)])
def test_separable_matches_oracle(ctx, v, radii):
    rr, rc = radii
    wr = I.positive_weights_f32(700 + rr, 2 * rr + 1)
    wc = I.signed_weights_f32(701 + rc, 2 * rc + 1)
    assert S.variant_names(S.SK_SEPARABLE)[:3] == ["two_pass", "fused_oy4", "fused_oy8"]
    for rows, cols in SHAPES:
        X = I.uniform01_f32(702 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
        fused_ok = rr <= 8 and rc <= 8 and cols % 4 == 0   # unequal / other radii run zero-padded (csrc/kernels.hpp)
        ctx.force_variant(S.SK_SEPARABLE, v)
        try:
            for ge, oe, pad in EDGES:
                if v != 0 and not fused_ok:
                    with pytest.raises(S.SkelError):
                        ctx.mapoverlap_separable(wr, rr, wc, rc, ge, pad, mx, mo)
                    continue
                ctx.mapoverlap_separable(wr, rr, wc, rc, ge, pad, mx, mo)
                assert ctx.last_variant()[1] == v or v == 0  # two_pass reports the column kernel's variant
                ref, tol_abs = oracle_separable(wr, rr, wc, rc, oe, pad, X)
                err = np.abs(mo.numpy().astype(np.float64) - ref)
                bad = err > 2e-6 * tol_abs
                assert not bad.any(), (rows, cols, ge, pad, int(bad.sum()), float((err / np.maximum(tol_abs, 1e-300)).max()))
        finally:
            ctx.force_variant(S.SK_SEPARABLE, -1)
        mx.destroy()
        mo.destroy()


def test_separable_fused_is_bit_identical_to_the_two_passes_and_plan_default(ctx):
    rows, cols, r = 300, 1024, 8
    X = I.uniform01_f32(710, rows * cols).reshape(rows, cols)
    wr, wc = I.positive_weights_f32(711, 17), I.positive_weights_f32(712, 17)
    mx, mt, mo = ctx.matrix_from(X), ctx.matrix(rows, cols), ctx.matrix(rows, cols)
    outs = []
    for v in list(range(S.lib.skel_variant_count(S.SK_SEPARABLE))) + [-1]:
        ctx.force_variant(S.SK_SEPARABLE, v)
        ctx.reset_stats()
        ctx.mapoverlap_separable(wr, r, wc, r, S.EDGE_DUPLICATE, 0.0, mx, mo)
        # two_pass: the two 1D kernels; every fused form is one launch (march_r8 applies DUPLICATE in registers when
        # cols % 128 == 0, as here; CYCLIC and ragged column counts would add the border-tile launch)
        if v >= 0:
            assert ctx.stats()["launches"] == (2 if v == 0 else 1)
        outs.append(mo.numpy().copy())
    ctx.force_variant(S.SK_SEPARABLE, -1)
    # the same taps in the same order with the same fp32 intermediate: every variant gives the same bits
    for o in outs[1:]:
        assert np.array_equal(outs[0], o)
    # ... and so do the two public 1D calls the definition names
    ctx.mapoverlap_1d_matrix(wr, r, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
    ctx.mapoverlap_1d_matrix(wc, r, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
    assert np.array_equal(outs[0], mo.numpy())
    for m in (mx, mt, mo):
        m.destroy()


def test_separable_march_policies_and_launch_counts(ctx):
    """march_r8: CONSTANT / DUPLICATE on cols % 128 == 0 are applied in registers (one launch), CYCLIC and ragged column
    counts take the border-tile launch as well (two), and both give the bits of the two 1D calls; matrices tall enough
    for several segments per strip and exactly one strip wide (both border fix-ups in the same warp)."""
    names = S.variant_names(S.SK_SEPARABLE)
    v = names.index("march_r8")
    for rows, cols in ((700, 128), (1000, 384), (517, 1024), (300, 1028), (97, 640)):
        X = I.uniform_pm1_f32(720 + rows, rows * cols).reshape(rows, cols)
        mx, mt, mo = ctx.matrix_from(X), ctx.matrix(rows, cols), ctx.matrix(rows, cols)
        for r in (8, 3):
            wr, wc = I.signed_weights_f32(721 + r, 2 * r + 1), I.signed_weights_f32(722 + r, 2 * r + 1)
            for ge, oe, pad in EDGES:
                ctx.mapoverlap_1d_matrix(wr, r, ge, pad, S.AXIS_ROW, mx, mt)
                ctx.mapoverlap_1d_matrix(wc, r, ge, pad, S.AXIS_COL, mt, mo)
                want = mo.numpy().copy()
                ctx.force_variant(S.SK_SEPARABLE, v)
                try:
                    ctx.reset_stats()
                    ctx.mapoverlap_separable(wr, r, wc, r, ge, pad, mx, mo)
                    launches = ctx.stats()["launches"]
                finally:
                    ctx.force_variant(S.SK_SEPARABLE, -1)
                assert np.array_equal(mo.numpy(), want), (rows, cols, r, ge, pad)
                in_registers = (ge == S.EDGE_CONSTANT or ge == S.EDGE_DUPLICATE) and cols % 128 == 0
                zeros = ge == S.EDGE_CONSTANT and pad == 0.0
                tiled_alone = not zeros and not in_registers and (rows % 32 not in (0,) and rows % 32 < 8 or cols % 128 not in (0,) and cols % 128 < 8
                                                                  or -(-cols // 128) <= 2 or -(-rows // 32) <= 2)
                assert launches == (1 if zeros or in_registers or tiled_alone else 2), (rows, cols, r, ge, pad, launches)
        for m in (mx, mt, mo):
            m.destroy()


def test_separable_errors(ctx):
    X = np.ones((8, 8), np.float32)
    mx, mo = ctx.matrix_from(X), ctx.matrix(8, 8)
    w = np.ones(3, np.float32)
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_separable(w, 1, w, 1, S.EDGE_DUPLICATE, 0.0, mx, mx)  # alias
    m2 = ctx.matrix(8, 12)
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_separable(w, 1, w, 1, S.EDGE_DUPLICATE, 0.0, mx, m2)  # shape
    for m in (mx, mo, m2):
        m.destroy()
