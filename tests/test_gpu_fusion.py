"""Cross-call fusion (include/skel.h skel_ctx_set_fusion): the chain
Map(f, c) -> MapOverlap1D -> Reduce runs as ONE kernel and must give what the three separate
skeletons give. The expected values come from the CPU oracle alone, chained on the oracle side:
  A'_o = RN_f32(oracle Map(A))            (add / mult / max with a constant are correctly rounded: the
                                           GPU must match bit for bit, so both sides feed the same A')
  B_o  = oracle MapOverlap1D(A'_o)        GPU B within 2e-6 * sum|w x| per element (BASELINE.json)
  s_o  = oracle Reduce(RN_f32(B_o))       GPU s within 1e-5 * sum|B_o| (the Reduce tolerance)
                                           + sum_i 2e-6 * sum|w x|_i (what the MapOverlap tolerance lets
                                           the GPU's B differ from B_o, summed; for max: the largest)."""
import numpy as np
import pytest

import oracle as O
from helpers import assert_map_f32, assert_overlap
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

EDGES = [(S.EDGE_CONSTANT, O.EDGE_CONSTANT, 0.25), (S.EDGE_DUPLICATE, O.EDGE_DUPLICATE, 0.0),
         (S.EDGE_CYCLIC, O.EDGE_CYCLIC, 0.0)]
MAPS = [(S.FN_MULT, O.FN_MULT, 1.0001), (S.FN_ADD, O.FN_ADD, -0.375), (S.FN_MAX, O.FN_MAX, 0.5)]
REDS = [(S.FN_ADD, O.FN_ADD), (S.FN_MAX, O.FN_MAX)]


@pytest.fixture()
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    c.set_fusion(True)
    made = []
    for name in ("vector", "vector_from", "vector_adopt"):  # remember the containers: destroyed at teardown
        orig = getattr(c, name)
        setattr(c, name, lambda *a, _o=orig, **k: (made.append(_o(*a, **k)) or made[-1]))
    yield c
    for v in made:
        if v.h:
            v.destroy()
    c.close()


def oracle_chain(x, mapf, c, w, r, edge, pad, redop):
    a1 = O.map_f32(mapf, c, x).astype(np.float32) if mapf is not None else x
    b64, absref = O.mapoverlap_1d(w, r, edge, pad, a1)
    s, abs_sum = O.reduce_f32(redop, b64.astype(np.float32)) if redop is not None else (None, None)
    return a1, b64, absref, s, abs_sum


def check_chain(got_a, got_b, got_s, ref, redop):
    a1, b64, absref, s, abs_sum = ref
    if got_a is not None:
        assert np.array_equal(got_a.view(np.uint32), a1.view(np.uint32)), "fused Map is not bit-identical to the oracle"
    assert_overlap(got_b, b64, absref)
    if got_s is not None:
        slack = 2e-6 * (float(absref.sum()) if redop == O.FN_ADD else float(absref.max()))
        assert abs(float(got_s) - s) <= 1e-5 * abs_sum + slack, (got_s, s, abs_sum, slack)


@pytest.mark.parametrize("n", [1, 5, 33, 4097, 100003, (1 << 20) + 1])
@pytest.mark.parametrize("r", [1, 4, 5, 8, 16])
def test_fused_inplace_chain_matches_oracle(ctx, n, r):
    x = I.uniform01_f32(I.config_seed(5, 1) + n + r, n)
    w = I.positive_weights_f32(I.config_seed(3, 20 + r), 2 * r + 1)
    for (ge, oe, pad), (gm, om, c), (gr, orr) in zip(EDGES, MAPS, REDS + REDS[:1]):
        a, b = ctx.vector_from(x), ctx.vector(n)
        ctx.reset_stats()
        ctx.map(gm, c, a, None, a)
        ctx.mapoverlap_1d(w, r, ge, pad, a, b)
        s = ctx.reduce(gr, b)
        st = ctx.stats()
        if r <= 8:   # r = 5 runs the r = 8 kernel zero-padded
            assert st["fused_launches"] == 1 and st["fused_calls"] == 3 and st["launches"] == 1, st
            assert ctx.last_variant() == (S.SK_OVERLAP1D, -2)
        else:        # beyond r = 8 the chain runs call by call (the separate TMA-fed MapOverlap kernel is faster)
            assert st["fused_launches"] == 0 and st["launches"] == 3, st
        check_chain(a.numpy(), b.numpy(), s, oracle_chain(x, om, c, w, r, oe, pad, orr), orr)
        a.destroy()
        b.destroy()


def test_fused_out_of_place_map_and_reduce_to(ctx):
    n, r = 70001, 4
    x = I.uniform_pm1_f32(I.config_seed(5, 2), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    a, a2, b, res1, res4 = ctx.vector_from(x), ctx.vector(n), ctx.vector(n), ctx.vector(1), ctx.vector(4)
    ref = oracle_chain(x, O.FN_MULT, 1.0001, w, r, O.EDGE_DUPLICATE, 0.0, O.FN_ADD)
    # a one-element result vector is write-only: nothing is uploaded, the whole chain fuses
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a, None, a2)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a2, b)
    ctx.reduce_to(S.FN_ADD, b, res1, 0)
    st = ctx.stats()
    assert st["fused_launches"] == 1 and st["fused_calls"] == 3 and st["launches"] == 1
    check_chain(a2.numpy(), b.numpy(), res1.numpy()[0], ref, O.FN_ADD)
    assert np.array_equal(a.numpy(), x), "the Map input was modified"
    # a host-written result vector must be uploaded first: the upload flushes Map + MapOverlap (fused as a
    # pair, stream order kept), the Reduce then runs alone and leaves the other elements untouched
    res4.write(np.arange(4, dtype=np.float32))
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a, None, a2)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a2, b)
    ctx.reduce_to(S.FN_ADD, b, res4, 2)
    st = ctx.stats()
    assert st["fused_launches"] == 1 and st["fused_calls"] == 2 and st["launches"] == 2
    out = res4.numpy()
    assert out[0] == 0 and out[1] == 1 and out[3] == 3
    check_chain(a2.numpy(), b.numpy(), out[2], ref, O.FN_ADD)


def test_fused_pairs(ctx):
    n, r = 50021, 8
    x = I.uniform01_f32(I.config_seed(5, 3), n)
    w = I.positive_weights_f32(I.config_seed(3, 15), 2 * r + 1)
    # MapOverlap1D -> Reduce (no Map)
    a, b = ctx.vector_from(x), ctx.vector(n)
    ctx.reset_stats()
    ctx.mapoverlap_1d(w, r, S.EDGE_CONSTANT, 0.0, a, b)
    s = ctx.reduce(S.FN_MAX, b)
    st = ctx.stats()
    assert st["fused_launches"] == 1 and st["fused_calls"] == 2 and st["launches"] == 1
    check_chain(None, b.numpy(), s, oracle_chain(x, None, 0.0, w, r, O.EDGE_CONSTANT, 0.0, O.FN_MAX), O.FN_MAX)
    # Map -> MapOverlap1D, flushed by an unrelated call (a Scan on other containers)
    v = I.uniform_int_i32(I.config_seed(5, 4), 1000, 15)
    vi, vo = ctx.vector_from(v), ctx.vector(1000, S.I32)
    ctx.reset_stats()
    ctx.map(S.FN_ADD, 2.0, a, None, a)
    ctx.mapoverlap_1d(w, r, S.EDGE_CYCLIC, 0.0, a, b)
    ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, vi, vo)
    st = ctx.stats()
    assert st["fused_launches"] == 1 and st["fused_calls"] == 2
    assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, v))
    check_chain(a.numpy(), b.numpy(), None, oracle_chain(x, O.FN_ADD, 2.0, w, r, O.EDGE_CYCLIC, 0.0, None), None)


def test_chain_broken_by_host_access_runs_call_by_call(ctx):
    n, r = 30011, 2
    x = I.uniform01_f32(I.config_seed(5, 5), n)
    w = I.positive_weights_f32(I.config_seed(3, 16), 5)
    a, b = ctx.vector_from(x), ctx.vector(n)
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a, None, a)
    mid = a.numpy().copy()  # host read: the held-back Map must run first
    assert_map_f32(mid, O.map_f32(O.FN_MULT, 1.0001, x))
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a, b)
    ctx.flush()
    s = ctx.reduce(S.FN_ADD, b)  # its MapOverlap is already launched: a lone Reduce
    st = ctx.stats()
    assert st["fused_launches"] == 0 and st["fused_calls"] == 0 and st["launches"] >= 3
    check_chain(a.numpy(), b.numpy(), s, oracle_chain(x, O.FN_MULT, 1.0001, w, r, O.EDGE_DUPLICATE, 0.0, O.FN_ADD), O.FN_ADD)


def test_not_fusible_chains_fall_back(ctx):
    import torch
    n, r = 40009, 4
    x = I.uniform01_f32(I.config_seed(5, 6), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    ref = oracle_chain(x, O.FN_MULT, 1.0001, w, r, O.EDGE_DUPLICATE, 0.0, O.FN_ADD)
    # (1) an adopted (caller-owned) buffer cannot be swapped: an in-place Map on it runs call by call
    t = torch.from_numpy(x).cuda()
    a, b = ctx.vector_adopt(t), ctx.vector(n)
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a, None, a)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a, b)
    s = ctx.reduce(S.FN_ADD, b)
    st = ctx.stats()
    assert st["fused_launches"] == 0 and st["launches"] >= 3
    ctx.sync()
    check_chain(t.cpu().numpy(), b.numpy(), s, ref, O.FN_ADD)
    # (2) Reduce(MULT) is not part of the fusible chain: Map+MapOverlap fuse, the Reduce runs alone
    a2, b2 = ctx.vector_from(x), ctx.vector(n)
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a2, None, a2)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a2, b2)
    p = ctx.reduce(S.FN_MULT, b2)
    st = ctx.stats()
    assert st["fused_launches"] == 1 and st["fused_calls"] == 2
    check_chain(a2.numpy(), b2.numpy(), None, ref, None)
    pr, _ = O.reduce_f32(O.FN_MULT, ref[1].astype(np.float32))
    assert p == pytest.approx(pr, rel=1e-3, abs=1e-30)
    # (3) a forced variant is honoured: nothing is held back
    ctx.force_variant(S.SK_OVERLAP1D, 0)
    a3, b3 = ctx.vector_from(x), ctx.vector(n)
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a3, None, a3)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a3, b3)
    assert ctx.last_variant() == (S.SK_OVERLAP1D, 0)
    s3 = ctx.reduce(S.FN_ADD, b3)
    assert ctx.stats()["fused_launches"] == 0
    ctx.force_variant(S.SK_OVERLAP1D, -1)
    check_chain(a3.numpy(), b3.numpy(), s3, ref, O.FN_ADD)


def test_fusion_off_by_default_and_same_results_as_unfused():
    n, r = 123457, 4
    x = I.uniform01_f32(I.config_seed(5, 7), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    out = {}
    for fused in (False, True):
        c = S.Context()
        if fused:
            c.set_fusion(True)
        a, b = c.vector_from(x), c.vector(n)
        c.map(S.FN_MULT, 1.0001, a, None, a)
        c.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a, b)
        s = c.reduce(S.FN_ADD, b)
        assert c.stats()["fused_launches"] == (1 if fused else 0)
        out[fused] = (a.numpy().copy(), b.numpy().copy(), s)
        a.destroy(); b.destroy(); c.close()
    assert np.array_equal(out[False][0], out[True][0])
    # the fused kernel accumulates the taps in the same order as the register-window variant the plan picks here
    assert np.array_equal(out[False][1], out[True][1])
    assert abs(out[False][2] - out[True][2]) <= 1e-5 * float(np.abs(out[True][1]).sum())


def test_fused_pipeline_iterations_ping_pong(ctx):
    """BASELINE.json configs[4] pipeline with fusion on: A and B swap roles, the in-place Map swaps
    buffers every iteration; one upload, no download, one launch per iteration."""
    n, iters, r = (1 << 18) + 37, 6, 4
    x0 = I.uniform01_f32(I.config_seed(5, 1), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    a, b = ctx.vector_from(x0), ctx.vector(n)
    ctx.reset_stats()
    scal = []
    for _ in range(iters):
        ctx.map(S.FN_MULT, 1.0001, a, None, a)
        ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a, b)
        scal.append(ctx.reduce(S.FN_ADD, b))
        a, b = b, a
    st = ctx.stats()
    assert st["h2d_count"] == 1 and st["d2h_count"] == 0 and st["scalar_d2h_count"] == iters
    assert st["fused_launches"] == iters and st["launches"] == iters
    # oracle chain, free running in fp32 containers like the GPU's
    xa = x0
    for k in range(iters):
        a1, b64, absref, s, abs_sum = oracle_chain(xa, O.FN_MULT, 1.0001, w, r, O.EDGE_DUPLICATE, 0.0, O.FN_ADD)
        # the GPU's B of iteration k feeds iteration k+1: its rounding differences (<= 2e-6 relative per
        # element, positive weights summing to 1) propagate, so the bound grows by one such term per iteration
        tol = (k + 1) * 2e-6 * float(absref.sum()) + 1e-5 * abs_sum
        assert abs(scal[k] - s) <= tol, (k, scal[k], s, tol)
        xa = b64.astype(np.float32)
    final = a.numpy()
    assert np.allclose(final, xa, rtol=iters * 4e-6, atol=0)


def test_fusion_with_eager_coherence_and_result_inside_the_chain(ctx):
    n, r = 20011, 4
    x = I.uniform01_f32(I.config_seed(5, 8), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    ref = oracle_chain(x, O.FN_MULT, 1.0001, w, r, O.EDGE_DUPLICATE, 0.0, O.FN_ADD)
    # EAGER coherence uploads and downloads around every call: every transfer flushes, nothing fuses
    ctx.set_coherence(S.EAGER)
    a, b = ctx.vector_from(x), ctx.vector(n)
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a, None, a)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a, b)
    s = ctx.reduce(S.FN_ADD, b)
    ctx.set_coherence(S.LAZY)
    assert ctx.stats()["fused_launches"] == 0
    check_chain(a.numpy(), b.numpy(), s, ref, O.FN_ADD)
    # the Reduce writes its result INTO the Map's container: call-by-call order is kept (Map + MapOverlap fuse)
    a2, b2 = ctx.vector_from(x), ctx.vector(n)
    ctx.reset_stats()
    ctx.map(S.FN_MULT, 1.0001, a2, None, a2)
    ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, a2, b2)
    ctx.reduce_to(S.FN_ADD, b2, a2, 7)
    st = ctx.stats()
    assert st["fused_launches"] == 0 and st["launches"] == 3
    got_a = a2.numpy()
    exp_a = ref[0].copy()
    s2 = got_a[7]
    exp_a[7] = s2
    assert np.array_equal(got_a, exp_a)
    check_chain(None, b2.numpy(), s2, ref, O.FN_ADD)
