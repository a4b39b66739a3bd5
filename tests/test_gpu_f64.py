"""fp64 elements (SKEL_F64, reading 27) against the binary128 oracle
(oracle/oracle.cpp, pinned with exact rationals in tests/test_oracle_pins.py). Tolerances = the fp32 contract of
BASELINE.json scaled to the fp64 unit round-off u = 2^-53: Map <= 1 ulp; Reduce / MapReduce / Scan
1e-5 / 2^-24 * u = 168 u -> 2e-14 * sum|terms|; MapOverlap 2e-6 / 2^-24 * u = 33.5 u -> 3.72e-15 * sum|w x|; max exact."""
import numpy as np
import pytest

import oracle as O
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

SIZES = [1, 2, 3, 4, 5, 7, 8, 33, 1023, 1024, 1025, 2047, 2049, 8191, 8193, 100003, (1 << 20) + 1]
RED_TOL, OVL_TOL = 2e-14, 3.72e-15


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


def ulp64(got, ref):
    def ordered(a):
        i = np.ascontiguousarray(a).view(np.int64)
        return np.where(i < 0, -(i & np.int64(0x7FFFFFFFFFFFFFFF)), i)
    return np.abs(ordered(got) - ordered(ref))


def test_map_f64_all_functions_one_ulp_and_fma(ctx):
    for n in SIZES:
        x, y = I.uniform_pm1_f64(9500 + n, n), I.uniform_pm1_f64(9501 + n, n)
        vx, vy, vo = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(n, S.F64)
        for fn, of in ((S.FN_ADD, O.FN_ADD), (S.FN_MULT, O.FN_MULT), (S.FN_MAX, O.FN_MAX), (S.FN_SAXPY, O.FN_SAXPY)):
            ctx.map(fn, 2.5000000000000004, vx, vy, vo)
            d = ulp64(vo.numpy(), O.map_f64(of, 2.5000000000000004, x, y))
            assert d.max() == 0, (fn, n, int(d.max()))       # correctly rounded operations: 0 ulp
        for fn, of in ((S.FN_ADD, O.FN_ADD), (S.FN_MULT, O.FN_MULT), (S.FN_MAX, O.FN_MAX)):
            ctx.map(fn, 0.3, vx, None, vo)
            assert ulp64(vo.numpy(), O.map_f64(of, 0.3, x)).max() == 0
        ctx.map(S.FN_MULT, 1.0001, vx, None, vx)               # in place
        assert np.array_equal(vx.numpy(), O.map_f64(O.FN_MULT, 1.0001, x))
        z = I.uniform_pm1_f64(9502 + n, n)
        vz = ctx.vector_from(z)
        ctx.map3(S.FN_MULADD, vy, vz, vy, vo)
        assert np.array_equal(vo.numpy(), O.map3_muladd_f64(y, z, y))
        for c in (vx, vy, vz, vo):
            c.destroy()
    # cancellation: c*x + y with y = -RN(c*x) is the rounding residual; a separate multiply and add would return 0
    n = 50000
    x = I.uniform_pm1_f64(9503, n)
    c = 1.0000000000000002
    y = -(c * x)
    vx, vy, vo = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(n, S.F64)
    ctx.map(S.FN_SAXPY, c, vx, vy, vo)
    assert np.array_equal(vo.numpy(), O.map_f64(O.FN_SAXPY, c, x, y)) and np.count_nonzero(vo.numpy()) > n // 4
    for h in (vx, vy, vo):
        h.destroy()


def test_reduce_mapreduce_f64(ctx):
    for n in SIZES + [1 << 22]:
        x, y = I.uniform_pm1_f64(9510 + n, n), I.uniform_pm1_f64(9511 + n, n)
        vx, vy, res = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(4, S.F64)
        r, a = O.reduce_f64(O.FN_ADD, x)
        s = ctx.reduce(S.FN_ADD, vx)
        assert abs(s - r) <= RED_TOL * a, (n, s, r)
        assert ctx.reduce(S.FN_ADD, vx) == s                                  # bitwise deterministic
        assert ctx.reduce(S.FN_MAX, vx) == O.reduce_f64(O.FN_MAX, x)[0]       # max does not round
        r, a = O.mapreduce_f64(O.FN_MULT, O.FN_ADD, 0.0, x, y)
        assert abs(ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vx, vy) - r) <= RED_TOL * a
        r, a = O.mapreduce_f64(O.FN_SAXPY, O.FN_ADD, 0.75, x, y)
        assert abs(ctx.mapreduce(S.FN_SAXPY, S.FN_ADD, 0.75, vx, vy) - r) <= RED_TOL * a
        r, a = O.mapreduce_f64(O.FN_MULT, O.FN_ADD, 3.0, x)                   # constant second operand
        ctx.mapreduce_to(S.FN_MULT, S.FN_ADD, 3.0, vx, None, res, 2)
        f = ctx.mapreduce_async(S.FN_MULT, S.FN_ADD, 3.0, vx, None)
        got = res.numpy()[2]
        assert abs(got - r) <= RED_TOL * a and f.result() == got
        for c in (vx, vy, res):
            c.destroy()
    p = 1.0 + 1e-4 * I.uniform_pm1_f64(9512, 5000)
    vp = ctx.vector_from(p)
    r, _ = O.reduce_f64(O.FN_MULT, p)
    assert abs(ctx.reduce(S.FN_MULT, vp) - r) <= 5000 * 2.3e-16 * abs(r)
    # cancellation a plain fp64 loop cannot survive either: only the tolerance relative to sum|x| is promised
    big = np.concatenate([np.full(1000, 1e16), np.ones(1000), np.full(1000, -1e16)])
    vb = ctx.vector_from(big)
    r, a = O.reduce_f64(O.FN_ADD, big)
    assert r == 1000.0 and abs(ctx.reduce(S.FN_ADD, vb) - r) <= RED_TOL * a
    e = ctx.vector_from(np.zeros(0))
    with pytest.raises(S.SkelError):
        ctx.reduce(S.FN_ADD, e)
    e.destroy()
    vp.destroy()
    vb.destroy()


def test_scan_f64(ctx):
    for n in [0] + SIZES + [(1 << 22) + 5]:
        x = I.uniform_pm1_f64(9520 + n, n)
        vx, vo = ctx.vector_from(x), ctx.vector(n, S.F64)
        ref, ab = O.scan_f64(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, x)
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        got = vo.numpy().copy()
        assert np.all(np.abs(got - ref) <= RED_TOL * ab), n
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert np.array_equal(vo.numpy(), got)                                # deterministic
        ref, ab = O.scan_f64(O.FN_ADD, O.SCAN_EXCLUSIVE, 0.3, x)
        ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 0.3, vx, vo)
        assert np.all(np.abs(vo.numpy() - ref) <= RED_TOL * ab)
        ctx.scan(S.FN_MAX, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert np.array_equal(vo.numpy(), O.scan_f64(O.FN_MAX, O.SCAN_INCLUSIVE, 0.0, x)[0])
        ctx.scan(S.FN_MAX, S.SCAN_EXCLUSIVE, -0.25, vx, vo)
        assert np.array_equal(vo.numpy(), O.scan_f64(O.FN_MAX, O.SCAN_EXCLUSIVE, -0.25, x)[0])
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vx)                     # in place
        assert np.array_equal(vx.numpy(), got)
        vx.destroy()
        vo.destroy()
    ones = np.ones(300001)
    vx, vo = ctx.vector_from(ones), ctx.vector(ones.size, S.F64)
    ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
    assert np.array_equal(vo.numpy(), np.arange(1, ones.size + 1, dtype=np.float64))   # exact integers
    p = 1.0 + 1e-5 * I.uniform_pm1_f64(9521, 20000)
    vp, vq = ctx.vector_from(p), ctx.vector(p.size, S.F64)
    ctx.scan(S.FN_MULT, S.SCAN_INCLUSIVE, 0.0, vp, vq)
    ref = O.scan_f64(O.FN_MULT, O.SCAN_INCLUSIVE, 0.0, p)[0]
    assert np.all(np.abs(vq.numpy() - ref) <= np.arange(1, p.size + 1) * 2.3e-16 * np.abs(ref))
    for c in (vx, vo, vp, vq):
        c.destroy()


def test_scan_f64_single_pass_path(ctx):
    """n >= 2^20 takes the single-pass kernel (f64.cu scan_l2_f64_kernel): several tiles per CTA (296 CTAs x 4096
    elements), ragged tails, all operators, in place, and the tile states of earlier launches (tagged with their launch
    number, never cleared) must not leak into later launches of other sizes and other data."""
    sizes = [1 << 20, (1 << 20) + 4096 * 300 + 17, (1 << 23) + 1, (1 << 21) - 3, 1 << 20]
    for rep, n in enumerate(sizes):
        x = I.uniform_pm1_f64(9600 + rep, n)
        vx, vo = ctx.vector_from(x), ctx.vector(n, S.F64)
        ref, ab = O.scan_f64(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, x)
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        got = vo.numpy().copy()
        assert np.all(np.abs(got - ref) <= RED_TOL * ab), n
        for _ in range(3):
            ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
            assert np.array_equal(vo.numpy(), got)                            # bitwise deterministic
        ref, ab = O.scan_f64(O.FN_ADD, O.SCAN_EXCLUSIVE, -1.75, x)
        ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, -1.75, vx, vo)
        assert np.all(np.abs(vo.numpy() - ref) <= RED_TOL * ab), n
        ctx.scan(S.FN_MAX, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert np.array_equal(vo.numpy(), np.maximum.accumulate(x))
        ctx.scan(S.FN_MAX, S.SCAN_EXCLUSIVE, 0.5, vx, vo)
        assert np.array_equal(vo.numpy(), O.scan_f64(O.FN_MAX, O.SCAN_EXCLUSIVE, 0.5, x)[0])
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vx)                     # in place
        assert np.array_equal(vx.numpy(), got)
        vx.destroy()
        vo.destroy()
    # operands that are 16- but not 32-byte aligned (adopted pointers) take the 128-bit form of the kernel; 8-byte
    # aligned ones the three-kernel form
    import torch
    n = (1 << 21) + 77
    x = I.uniform_pm1_f64(9620, n)
    ref, ab = O.scan_f64(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, x)
    for off in (2, 1):
        t, to = torch.zeros(n + 8, dtype=torch.float64, device="cuda"), torch.zeros(n + 8, dtype=torch.float64, device="cuda")
        t[off:n + off] = torch.from_numpy(x).cuda()
        vx, vo = ctx.vector_adopt(t[off:n + off]), ctx.vector_adopt(to[off:n + off])
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        ctx.sync()
        assert np.all(np.abs(to[off:n + off].cpu().numpy() - ref) <= RED_TOL * ab), off
        assert float(to[off - 1]) == 0.0 and float(to[n + off]) == 0.0       # nothing written outside
        vx.destroy()
        vo.destroy()
    n = (1 << 22) + 4099
    ones = np.ones(n)
    vx, vo = ctx.vector_from(ones), ctx.vector(n, S.F64)
    ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
    assert np.array_equal(vo.numpy(), np.arange(1, n + 1, dtype=np.float64))  # exact integers: any dropped tile shows
    ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 7.0, vx, vo)
    assert np.array_equal(vo.numpy(), np.arange(7, n + 7, dtype=np.float64))
    p = 1.0 + 1e-7 * I.uniform_pm1_f64(9610, 1 << 21)
    vp, vq = ctx.vector_from(p), ctx.vector(p.size, S.F64)
    ctx.scan(S.FN_MULT, S.SCAN_INCLUSIVE, 0.0, vp, vq)
    ref = O.scan_f64(O.FN_MULT, O.SCAN_INCLUSIVE, 0.0, p)[0]
    assert np.all(np.abs(vq.numpy() - ref) <= np.arange(1, p.size + 1) * 2.3e-16 * np.abs(ref))   # i roundings at element i
    for c in (vx, vo, vp, vq):
        c.destroy()


EDGES = [(S.EDGE_CONSTANT, 0.0), (S.EDGE_CONSTANT, -0.75), (S.EDGE_DUPLICATE, 0.0), (S.EDGE_CYCLIC, 0.0)]


@pytest.mark.parametrize("r", [0, 1, 3, 4, 5, 8, 11, 16, 17, 64])
def test_overlap1d_f64(ctx, r):
    w = I.uniform_pm1_f64(9530 + r, 2 * r + 1)
    # n % 4 == 0 and n >= 64 with r <= 16: the 256-bit row form (zero-padded to radius 4, 8 or 16); everything else: scalar form
    for n in (1, 2, 3, 17, 64, 100, 4096, 4097, 100003, 100004):
        x = I.uniform_pm1_f64(9531 + n, n)
        vx, vo = ctx.vector_from(x), ctx.vector(n, S.F64)
        for edge, pad in EDGES:
            ctx.mapoverlap_1d_f64(w, r, edge, pad, vx, vo)
            ref, ab = O.mapoverlap_1d_f64(w, r, edge, pad, x)
            err = np.abs(vo.numpy() - ref)
            assert np.all(err <= OVL_TOL * ab), (n, edge, float((err / np.maximum(ab, 1e-300)).max()))
        vx.destroy()
        vo.destroy()
    # one-hot weights: a pure shift, bit-exact
    n = 5003
    x = I.uniform_pm1_f64(9532, n)
    vx, vo = ctx.vector_from(x), ctx.vector(n, S.F64)
    for m in (0, r, 2 * r):
        w1 = np.zeros(2 * r + 1)
        w1[m] = 1.0
        ctx.mapoverlap_1d_f64(w1, r, S.EDGE_DUPLICATE, 0.0, vx, vo)
        assert np.array_equal(vo.numpy(), x[np.clip(np.arange(n) + m - r, 0, n - 1)])
    vx.destroy()
    vo.destroy()


def test_overlap_matrix_and_2d_f64(ctx):
    for rows, cols in ((1, 1), (3, 5), (37, 129), (200, 520), (6, 8256)):
        X = I.uniform_pm1_f64(9540 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols, S.F64)
        for edge, pad in EDGES:
            for r in (1, 8, 13):
                w = I.uniform_pm1_f64(9541 + r, 2 * r + 1)
                for axis, oax in ((S.AXIS_ROW, O.AXIS_ROW), (S.AXIS_COL, O.AXIS_COL)):
                    ctx.mapoverlap_1d_matrix_f64(w, r, edge, pad, axis, mx, mo)
                    ref, ab = O.mapoverlap_1d_matrix_f64(w, r, edge, pad, oax, X)
                    assert np.all(np.abs(mo.numpy() - ref) <= OVL_TOL * ab), (rows, cols, edge, r, axis)
            for ry, rx in ((0, 0), (2, 2), (4, 4), (1, 3), (8, 8)):
                W = I.uniform_pm1_f64(9542 + 9 * ry + rx, (2 * ry + 1) * (2 * rx + 1))
                ctx.mapoverlap_2d_f64(W, ry, rx, edge, pad, mx, mo)
                ref, ab = O.mapoverlap_2d_f64(W, ry, rx, edge, pad, X)
                assert np.all(np.abs(mo.numpy() - ref) <= OVL_TOL * ab), (rows, cols, edge, ry, rx)
        mx.destroy()
        mo.destroy()


def test_f64_containers_coherence_ranges_and_errors(ctx):
    n = 100000
    x = I.uniform_pm1_f64(9550, n)
    vx, vo = ctx.vector_from(x), ctx.vector(n, S.F64)
    ctx.reset_stats()
    ctx.map(S.FN_ADD, 1.0, vx, None, vo)
    ctx.map(S.FN_ADD, 1.0, vo, None, vo)
    st = ctx.stats()
    assert st["h2d_count"] == 1 and st["h2d_bytes"] == 8 * n and st["h2d_elided"] == 1
    assert np.array_equal(vo.numpy(), (x + 1.0) + 1.0)
    assert ctx.stats()["d2h_bytes"] == 8 * n
    # range access moves 8-byte elements
    v = vx.host_view_range(S.READWRITE, 1000, 16)
    v[:] = 7.0
    vx.release()
    ctx.reset_stats()
    s = ctx.reduce(S.FN_ADD, vx)
    assert ctx.stats()["h2d_bytes"] == 16 * 8
    x2 = x.copy()
    x2[1000:1016] = 7.0
    r, a = O.reduce_f64(O.FN_ADD, x2)
    assert abs(s - r) <= RED_TOL * a
    # element types must match; f32-only entry points refuse fp64 containers
    vf = ctx.vector(n)
    with pytest.raises(S.SkelError):
        ctx.map(S.FN_ADD, 1.0, vx, None, vf)
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_1d(np.ones(3, np.float32), 1, S.EDGE_DUPLICATE, 0.0, vx, vo)
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_1d_f64(np.ones(3), 1, S.EDGE_DUPLICATE, 0.0, vf, vf)
    with pytest.raises(S.SkelError):
        ctx.force_variant(S.SK_MAP, 2), ctx.map(S.FN_ADD, 1.0, vx, None, vo)
    ctx.force_variant(S.SK_MAP, -1)
    for c in (vx, vo, vf):
        c.destroy()
