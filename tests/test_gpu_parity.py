"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs. Sizes span several tiles and ragged tails; every kernel variant is forced
through the same checks. Tolerances: BASELINE.json L5 (integers bit-exact; Map <= 1 ulp; fp32
Reduce/MapReduce <= 1e-5 * sum|terms|; MapOverlap <= 2e-6 * sum|w x|)."""
import numpy as np
import pytest

import oracle as O
from helpers import SIZES, SIZES_SHORT, assert_map_f32, assert_overlap, assert_reduce_f32
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


def variants(sk):
    return list(range(S.lib.skel_variant_count(sk)))


def o1_radius_ok(v, r):
    """Radii a MapOverlap 1D variant runs (direct: any; tiled: r <= 16, radii between the instantiated ones
    {1,2,3,4,8,16} zero-padded to the next one, csrc/kernels.hpp; regshfl_2x8: r <= 8)."""
    if v == 0:
        return True
    if S.variant_names(S.SK_OVERLAP1D)[v] == "regshfl_2x8":
        return 0 <= r <= 8
    return 0 <= r <= 16


class forced:
    def __init__(self, ctx, sk, v):
        self.ctx, self.sk, self.v = ctx, sk, v

    def __enter__(self):
        self.ctx.force_variant(self.sk, self.v)

    def __exit__(self, *a):
        self.ctx.force_variant(self.sk, -1)


# ------------------------------------------------------------------ Map
@pytest.mark.parametrize("v", variants(S.SK_MAP))
def test_map_f32_all_functions(ctx, v):
    with forced(ctx, S.SK_MAP, v):
        for n in SIZES:
            x, y = I.uniform_pm1_f32(100 + n, n), I.uniform_pm1_f32(101 + n, n)
            vx, vy, vo = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(n)
            for fn in (S.FN_ADD, S.FN_MULT, S.FN_MAX, S.FN_SAXPY):
                ctx.map(fn, 2.5, vx, vy, vo)
                assert ctx.last_variant() == (S.SK_MAP, v)
                assert_map_f32(vo.numpy(), O.map_f32(fn, 2.5, x, y))
            for fn in (S.FN_ADD, S.FN_MULT, S.FN_MAX):
                ctx.map(fn, 1.0001, vx, None, vo)
                assert_map_f32(vo.numpy(), O.map_f32(fn, 1.0001, x))
            for c in (vx, vy, vo):
                c.destroy()


def test_map_saxpy_cancellation_needs_fma(ctx):
    # c*x ~ -y: a separate multiply and add would be hundreds of ulps off (reading (c).1 ii)
    n = 50000
    x = I.uniform_pm1_f32(110, n)
    c32 = np.float32(2.5000001)
    y = (-(c32 * x)).astype(np.float32)
    vx, vy, vo = ctx.vector_from(x), ctx.vector_from(y), ctx.vector(n)
    ctx.map(S.FN_SAXPY, float(c32), vx, vy, vo)
    assert_map_f32(vo.numpy(), O.map_f32(O.FN_SAXPY, float(c32), x, y))
    for c in (vx, vy, vo):
        c.destroy()


@pytest.mark.parametrize("v", variants(S.SK_MAP))
def test_map_i32_and_in_place(ctx, v):
    with forced(ctx, S.SK_MAP, v):
        for n in SIZES_SHORT:
            a, b = I.full_range_i32(120 + n, n), I.full_range_i32(121 + n, n)
            va, vb, vo = ctx.vector_from(a), ctx.vector_from(b), ctx.vector(n, S.I32)
            for fn in (S.FN_ADD, S.FN_MULT, S.FN_MAX, S.FN_SAXPY):
                ctx.map(fn, -7, va, vb, vo)
                assert np.array_equal(vo.numpy(), O.map_i32(fn, -7, a, b))
            ctx.map(S.FN_ADD, 12345, va, None, vo)
            assert np.array_equal(vo.numpy(), O.map_i32(O.FN_ADD, 12345, a))
            # in place: out aliases in0, then in1, then both
            ctx.map(S.FN_MULT, 0, va, vb, va)
            a1 = O.map_i32(O.FN_MULT, 0, a, b)
            assert np.array_equal(va.numpy(), a1)
            ctx.map(S.FN_ADD, 0, va, vb, vb)
            b1 = O.map_i32(O.FN_ADD, 0, a1, b)
            assert np.array_equal(vb.numpy(), b1)
            ctx.map(S.FN_ADD, 0, vb, vb, vb)
            assert np.array_equal(vb.numpy(), O.map_i32(O.FN_ADD, 0, b1, b1))
            for c in (va, vb, vo):
                c.destroy()


def test_map_closed_form_and_empty(ctx):
    n = 1 << 20
    x = np.arange(n, dtype=np.float32)
    vx, vy, vo = ctx.vector_from(x), ctx.vector_from(np.ones(n, np.float32)), ctx.vector(n)
    ctx.map(S.FN_SAXPY, 2.5, vx, vy, vo)
    assert np.array_equal(vo.numpy(), (2.5 * np.arange(n, dtype=np.float64) + 1).astype(np.float32))
    ctx.map(S.FN_MULT, 1.0, vx, None, vo)
    assert np.array_equal(vo.numpy(), x)
    e0, e1 = ctx.vector_from(np.zeros(0, np.float32)), ctx.vector(0)
    ctx.map(S.FN_ADD, 1.0, e0, None, e1)
    assert e1.numpy().size == 0
    for c in (vx, vy, vo, e0, e1):
        c.destroy()


def test_map_misaligned_adopted_pointer_falls_back(ctx):
    import torch
    n = 10001
    x = I.uniform_pm1_f32(130, n + 3)
    t = torch.from_numpy(x).cuda()
    to = torch.empty(n + 3, dtype=torch.float32, device="cuda")
    vx, vo = ctx.vector_adopt(t[1:n + 1]), ctx.vector_adopt(to[3:n + 3])
    ctx.map(S.FN_MULT, 3.0, vx, None, vo)
    assert ctx.last_variant() == (S.SK_MAP, 0)  # the any-alignment variant
    ctx.sync()
    assert_map_f32(to[3:n + 3].cpu().numpy(), O.map_f32(O.FN_MULT, 3.0, x[1:n + 1]))
    with forced(ctx, S.SK_MAP, 2):
        with pytest.raises(S.SkelError) as ei:
            ctx.map(S.FN_MULT, 3.0, vx, None, vo)
        assert ei.value.status == S.ERR_UNSUPPORTED
    vx.destroy()
    vo.destroy()


# ------------------------------------------------------------------ Reduce / MapReduce
@pytest.mark.parametrize("v", variants(S.SK_REDUCE))
def test_reduce_i32_bit_exact(ctx, v):
    with forced(ctx, S.SK_REDUCE, v):
        for n in SIZES:
            a = I.full_range_i32(200 + n, n)
            va = ctx.vector_from(a)
            assert ctx.reduce(S.FN_ADD, va) == O.reduce_i32(O.FN_ADD, a)[0]
            assert ctx.reduce(S.FN_MAX, va) == O.reduce_i32(O.FN_MAX, a)[0]
            small = (a % 5 + 1).astype(np.int32)
            va.write(small)
            assert ctx.reduce(S.FN_MULT, va) == O.reduce_i32(O.FN_MULT, small)[0]
            va.destroy()


@pytest.mark.parametrize("v", variants(S.SK_REDUCE))
def test_reduce_f32_tolerance_and_determinism(ctx, v):
    with forced(ctx, S.SK_REDUCE, v):
        for n in SIZES_SHORT + [(1 << 22) + 7]:
            x = I.uniform_pm1_f32(210 + n, n)
            vx = ctx.vector_from(x)
            got = ctx.reduce(S.FN_ADD, vx)
            ref, ab = O.reduce_f32(O.FN_ADD, x)
            assert_reduce_f32(got, ref, ab)
            assert all(ctx.reduce(S.FN_ADD, vx) == got for _ in range(3))  # bitwise run-to-run
            assert ctx.reduce(S.FN_MAX, vx) == O.reduce_f32(O.FN_MAX, x)[0]
            y = (1.0 + x * 2.0 ** -12).astype(np.float32)[: min(n, 5000)]
            vy = ctx.vector_from(y)
            refm, _ = O.reduce_f32(O.FN_MULT, y)
            assert abs(ctx.reduce(S.FN_MULT, vy) - refm) <= 1e-4 * abs(refm)
            vx.destroy()
            vy.destroy()


def test_reduce_i32_atomic_end_chain_resets_its_scratch_word(ctx):
    """The *_iatom variants keep (sum, count of arrived blocks) in one scratch word that the last block zeroes: launches
    of different sizes, operators and element types in any order must each start from a clean word."""
    names = S.variant_names(S.SK_REDUCE)
    sizes = [(1 << 20) + 5, 8192 * 3, (1 << 22) + 4097, 8193, 1 << 21, 100003, (1 << 23) + 1]
    data = {n: I.full_range_i32(240 + n, n) for n in sizes}
    vecs = {n: ctx.vector_from(a) for n, a in data.items()}
    xf = I.uniform_pm1_f32(241, 1 << 20)
    vf = ctx.vector_from(xf)
    reff, abf = O.reduce_f32(O.FN_ADD, xf)
    for v in [i for i, nm in enumerate(names) if nm.endswith("_iatom")]:
        with forced(ctx, S.SK_REDUCE, v):
            for rep in range(3):
                for n in sizes if rep % 2 == 0 else reversed(sizes):
                    assert ctx.reduce(S.FN_ADD, vecs[n]) == O.reduce_i32(O.FN_ADD, data[n])[0], (names[v], n)
                    if n % 3 == 0:
                        assert ctx.reduce(S.FN_MAX, vecs[n]) == O.reduce_i32(O.FN_MAX, data[n])[0]
                    if n % 2 == 1:
                        assert_reduce_f32(ctx.reduce(S.FN_ADD, vf), reff, abf)
    for c in list(vecs.values()) + [vf]:
        c.destroy()


def test_reduce_tagged_end_across_launches(ctx):
    """The *_tag variants end a max / mult / fp32 Reduce with one (partial, launch number) word per block and a fold by
    the block that STARTED last; the slots are never cleared. Launches of different sizes (odd and even block counts,
    more and fewer blocks than the launch before, so stale slots of earlier launches sit beside fresh ones), operators
    and element types, back to back: exact for int32, fp32 inside the tolerance and bitwise equal run to run."""
    names = S.variant_names(S.SK_REDUCE)
    tagged = [i for i, nm in enumerate(names) if nm.endswith("_tag")]
    assert tagged
    sizes = [(1 << 23) + 1, 8192 * 3, (1 << 22) + 4097, 8193, 1 << 21, 100003, (1 << 20) + 5, 3 * 8192 + 1, 1 << 24]
    data = {n: I.full_range_i32(250 + n, n) for n in sizes}
    vecs = {n: ctx.vector_from(a) for n, a in data.items()}
    xf = I.uniform_pm1_f32(251, (1 << 22) + 12345)
    vf, vg = ctx.vector_from(xf), ctx.vector_from(xf[::-1].copy())
    reff, abf = O.reduce_f32(O.FN_ADD, xf)
    dref, dabs = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, xf, xf[::-1].copy())
    for v in tagged:
        with forced(ctx, S.SK_REDUCE, v), forced(ctx, S.SK_MAPREDUCE, v):
            first = None
            for rep in range(4):
                for n in sizes if rep % 2 == 0 else reversed(sizes):
                    assert ctx.reduce(S.FN_MAX, vecs[n]) == O.reduce_i32(O.FN_MAX, data[n])[0], (names[v], n)
                    if n % 2 == 1:
                        assert ctx.reduce(S.FN_ADD, vecs[n]) == O.reduce_i32(O.FN_ADD, data[n])[0]
                        got = ctx.reduce(S.FN_ADD, vf)
                        assert_reduce_f32(got, reff, abf)
                        first = got if first is None else first
                        assert got == first
                    if n % 3 == 0:
                        assert ctx.reduce(S.FN_MAX, vf) == O.reduce_f32(O.FN_MAX, xf)[0]
                        d = ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vf, vg)
                        assert abs(d - dref) <= 1e-5 * dabs
            # many launches in a row without a host read in between: futures resolved at the end
            outs = [ctx.vector(1, S.I32) for _ in range(64)]
            for k, o in enumerate(outs):
                ctx.reduce_to(S.FN_MAX, vecs[sizes[k % len(sizes)]], o)
            for k, o in enumerate(outs):
                assert int(o.numpy()[0]) == O.reduce_i32(O.FN_MAX, data[sizes[k % len(sizes)]])[0]
                o.destroy()
    for c in list(vecs.values()) + [vf, vg]:
        c.destroy()


def test_reduce_l2_aware_direction_keeps_the_bits(ctx):
    """skel_ctx_set_l2_reuse: a Reduce / MapReduce that follows a launch on the same operand walks it from the end to
    the front. Every chunk variant, sizes with a ragged last chunk and odd chunk counts: int32 exact, and the fp32 sum
    and dot product have the SAME BITS with the setting on (directions alternate call by call) and off (all forward)."""
    names = S.variant_names(S.SK_REDUCE)
    chunked = [i for i, nm in enumerate(names) if "chunk" in nm]
    sizes = [(1 << 22) + 4097, 8192 * 3 + 1, (1 << 24) + 5, 100003]
    for n in sizes:
        a = I.full_range_i32(260 + n, n)
        x, y = I.uniform_pm1_f32(261 + n, n), I.uniform_pm1_f32(262 + n, n)
        va, vx, vy = ctx.vector_from(a), ctx.vector_from(x), ctx.vector_from(y)
        ref_add, ref_max = O.reduce_i32(O.FN_ADD, a)[0], O.reduce_i32(O.FN_MAX, a)[0]
        rf, af = O.reduce_f32(O.FN_ADD, x)
        rd, ad = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, y)
        for v in chunked:
            with forced(ctx, S.SK_REDUCE, v), forced(ctx, S.SK_MAPREDUCE, v):
                got = {}
                for on in (False, True):
                    ctx.set_l2_reuse(on)
                    for _ in range(3):  # forward, backward, forward when on
                        assert ctx.reduce(S.FN_ADD, va) == ref_add, (names[v], n, on)
                        assert ctx.reduce(S.FN_MAX, va) == ref_max, (names[v], n, on)
                    fs = [ctx.reduce(S.FN_ADD, vx) for _ in range(3)]
                    ds = [ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vx, vy) for _ in range(3)]
                    assert_reduce_f32(fs[0], rf, af)
                    assert abs(ds[0] - rd) <= 1e-5 * ad
                    assert fs[0] == fs[1] == fs[2] and ds[0] == ds[1] == ds[2]
                    got[on] = (fs[0], ds[0])
                assert got[False] == got[True], (names[v], n)
        ctx.set_l2_reuse(True)
        for c in (va, vx, vy):
            c.destroy()


def test_reduce_closed_forms_and_max_position(ctx):
    for n in [1, 1000, 4096, (1 << 20) + 3]:
        v = ctx.vector_from(np.ones(n, np.float32))
        assert ctx.reduce(S.FN_ADD, v) == n
        v.destroy()
        idx = np.arange(n, dtype=np.int32)
        vi = ctx.vector_from(idx)
        exp = (n * (n - 1) // 2) & 0xFFFFFFFF
        assert ctx.reduce(S.FN_ADD, vi) & 0xFFFFFFFF == exp
        vi.destroy()
    n = 70001
    base = I.permutation(220, n).astype(np.int32)
    for pos in [0, 1, 255, 256, 4095, 4096, n // 2, n - 1]:
        p = base.copy()
        j = int(np.argmax(p))
        p[j], p[pos] = p[pos], p[j]
        vp = ctx.vector_from(p)
        assert ctx.reduce(S.FN_MAX, vp) == n - 1
        vp.destroy()


def test_reduce_to_device_slot_and_errors(ctx):
    x = I.uniform_int_i32(230, 5000, 1000)
    vx = ctx.vector_from(x)
    res = ctx.vector(4, S.I32)
    ctx.reduce_to(S.FN_ADD, vx, res, 2)
    ctx.reduce_to(S.FN_MAX, vx, res, 0)
    got = res.numpy()
    assert got[2] == O.reduce_i32(O.FN_ADD, x)[0] and got[0] == O.reduce_i32(O.FN_MAX, x)[0]
    with pytest.raises(S.SkelError) as ei:
        ctx.reduce_to(S.FN_ADD, vx, res, 4)
    assert ei.value.status == S.ERR_INVALID_ARG
    un = ctx.vector(10, S.I32)
    with pytest.raises(S.SkelError) as ei:
        ctx.reduce(S.FN_ADD, un)
    assert ei.value.status == S.ERR_UNINIT
    for c in (vx, res, un):
        c.destroy()


@pytest.mark.parametrize("v", variants(S.SK_MAPREDUCE))
def test_mapreduce_dot_and_friends(ctx, v):
    with forced(ctx, S.SK_MAPREDUCE, v):
        for n in SIZES_SHORT + [1 << 20]:
            x, y = I.uniform_pm1_f32(300 + n, n), I.uniform_pm1_f32(301 + n, n)
            vx, vy = ctx.vector_from(x), ctx.vector_from(y)
            got = ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vx, vy)
            ref, ab = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, y)
            assert_reduce_f32(got, ref, ab)
            assert ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vx, vy) == got
            got = ctx.mapreduce(S.FN_ADD, S.FN_MAX, 0.0, vx, vy)
            assert got == np.float32(O.mapreduce_f32(O.FN_ADD, O.FN_MAX, 0.0, x, y)[0])
            got = ctx.mapreduce(S.FN_SAXPY, S.FN_ADD, 2.5, vx, vy)
            ref, ab = O.mapreduce_f32(O.FN_SAXPY, O.FN_ADD, 2.5, x, y)
            assert_reduce_f32(got, ref, ab)
            got = ctx.mapreduce(S.FN_MULT, S.FN_ADD, 3.0, vx, None)  # sum of 3*x
            ref, ab = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 3.0, x, None)
            assert_reduce_f32(got, ref, ab)
            a, b = I.full_range_i32(302 + n, n), I.full_range_i32(303 + n, n)
            va, vb = ctx.vector_from(a), ctx.vector_from(b)
            assert ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0, va, vb) == O.mapreduce_i32(O.FN_MULT, O.FN_ADD, 0, a, b)
            assert ctx.mapreduce(S.FN_ADD, S.FN_MAX, 0, va, vb) == O.mapreduce_i32(O.FN_ADD, O.FN_MAX, 0, a, b)
            for c in (vx, vy, va, vb):
                c.destroy()


def test_dot_closed_form_and_fusion_invariant(ctx):
    n = 1 << 20
    vx, vy = ctx.vector_from(np.arange(n, dtype=np.float32)), ctx.vector_from(np.ones(n, np.float32))
    exact = n * (n - 1) // 2
    assert abs(ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, vx, vy) - exact) <= 1e-5 * exact
    a, b = I.full_range_i32(310, 99999), I.full_range_i32(311, 99999)
    va, vb, vt = ctx.vector_from(a), ctx.vector_from(b), ctx.vector(99999, S.I32)
    ctx.map(S.FN_MULT, 0, va, vb, vt)
    assert ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0, va, vb) == ctx.reduce(S.FN_ADD, vt)
    for c in (vx, vy, va, vb, vt):
        c.destroy()


# ------------------------------------------------------------------ Scan
SCAN_SIZES = SIZES + [(1 << 21) + 13]


@pytest.mark.parametrize("v", variants(S.SK_SCAN))
def test_scan_i32_bit_exact(ctx, v):
    with forced(ctx, S.SK_SCAN, v):
        for n in SCAN_SIZES:
            x = I.full_range_i32(400 + n, n)
            vx, vo = ctx.vector_from(x), ctx.vector(n, S.I32)
            ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, vx, vo)
            assert ctx.last_variant() == (S.SK_SCAN, v)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, x))
            ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, -12345, vx, vo)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, -12345, x))
            ctx.scan(S.FN_MAX, S.SCAN_INCLUSIVE, 0, vx, vo)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_MAX, O.SCAN_INCLUSIVE, 0, x))
            ctx.scan(S.FN_MAX, S.SCAN_EXCLUSIVE, 77, vx, vo)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_MAX, O.SCAN_EXCLUSIVE, 77, x))
            ctx.scan(S.FN_MULT, S.SCAN_INCLUSIVE, 0, vx, vo)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_MULT, O.SCAN_INCLUSIVE, 0, x))
            # in place
            ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 5, vx, vx)
            assert np.array_equal(vx.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, 5, x))
            vx.destroy()
            vo.destroy()


@pytest.mark.parametrize("v", variants(S.SK_SCAN))
def test_scan_every_small_n_and_tile_boundaries(ctx, v):
    with forced(ctx, S.SK_SCAN, v):
        sizes = list(range(0, 70)) + [4096 * k + d for k in (1, 2, 3) for d in (-1, 0, 1)] + [8192 * 3 + 1, 16384 + 1]
        for n in sizes:
            x = I.uniform_int_i32(410 + n, n, 15)
            vx, vo = ctx.vector_from(x), ctx.vector(n, S.I32)
            ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, vx, vo)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, x))
            ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 3, vx, vo)
            assert np.array_equal(vo.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_EXCLUSIVE, 3, x))
            vx.destroy()
            vo.destroy()


def test_scan_closed_forms_many_repeats(ctx):
    # ones -> indices; repeated launches exercise the epoch-tagged tile states and the ticket reset
    n = (1 << 22) + 5
    vx, vo = ctx.vector_from(np.ones(n, np.int32)), ctx.vector(n, S.I32)
    for v in variants(S.SK_SCAN):
        with forced(ctx, S.SK_SCAN, v):
            for rep in range(6):
                ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, vx, vo)
            assert np.array_equal(vo.numpy(), np.arange(1, n + 1, dtype=np.int32))
            ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 0, vx, vo)
            assert np.array_equal(vo.numpy(), np.arange(0, n, dtype=np.int32))
    vx.destroy()
    vo.destroy()


def test_scan_f32_three_kernel(ctx):
    for n in SIZES_SHORT:
        x = I.uniform_pm1_f32(420 + n, n)
        vx, vo = ctx.vector_from(x), ctx.vector(n)
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert S.variant_names(S.SK_SCAN)[ctx.last_variant()[1]].startswith("three_kernel")
        ref, ab = O.scan_f32(O.FN_ADD, O.SCAN_INCLUSIVE, 0.0, x)
        got = vo.numpy()
        assert np.all(np.abs(got - ref) <= 1e-5 * ab)
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert np.array_equal(vo.numpy(), got)  # deterministic
        ctx.scan(S.FN_ADD, S.SCAN_EXCLUSIVE, 1.5, vx, vo)
        ref, ab = O.scan_f32(O.FN_ADD, O.SCAN_EXCLUSIVE, 1.5, x)
        assert np.all(np.abs(vo.numpy() - ref) <= 1e-5 * ab)
        ctx.scan(S.FN_MAX, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert np.array_equal(vo.numpy(), O.scan_f32(O.FN_MAX, O.SCAN_INCLUSIVE, 0.0, x)[0].astype(np.float32))
        vx.destroy()
        vo.destroy()
    with forced(ctx, S.SK_SCAN, 0):  # look-back variants are int32 only
        vx, vo = ctx.vector_from(np.ones(10, np.float32)), ctx.vector(10)
        with pytest.raises(S.SkelError) as ei:
            ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0.0, vx, vo)
        assert ei.value.status == S.ERR_UNSUPPORTED
        vx.destroy()
        vo.destroy()


# ------------------------------------------------------------------ MapOverlap 1D
EDGE_CASES = [(S.EDGE_CONSTANT, 0.0), (S.EDGE_CONSTANT, -0.75), (S.EDGE_DUPLICATE, 0.0), (S.EDGE_CYCLIC, 0.0)]
O1_SIZES = [1, 2, 3, 5, 16, 17, 33, 100, 1023, 4096, 4097, 8200, 12320, 16385, 65537, 300001]


@pytest.mark.parametrize("v,r", [(v, r) for r in [0, 1, 2, 3, 4, 5, 6, 8, 12, 16, 17, 64]
                                  for v in variants(S.SK_OVERLAP1D) if o1_radius_ok(v, r)])
def test_overlap1d_vector(ctx, v, r):
    w = I.positive_weights_f32(500 + r, 2 * r + 1)
    ws = I.signed_weights_f32(501 + r, 2 * r + 1)
    with forced(ctx, S.SK_OVERLAP1D, v):
        for n in O1_SIZES:
            x = I.uniform01_f32(502 + n, n)
            vx, vo = ctx.vector_from(x), ctx.vector(n)
            for edge, pad in EDGE_CASES:
                ctx.mapoverlap_1d(w, r, edge, pad, vx, vo)
                assert ctx.last_variant() == (S.SK_OVERLAP1D, v)
                ref, ab = O.mapoverlap_1d(w, r, edge, pad, x)
                assert_overlap(vo.numpy(), ref, ab)
            ctx.mapoverlap_1d(ws, r, S.EDGE_DUPLICATE, 0.0, vx, vo)
            ref, ab = O.mapoverlap_1d(ws, r, S.EDGE_DUPLICATE, 0.0, x)
            assert_overlap(vo.numpy(), ref, ab)
            vx.destroy()
            vo.destroy()


@pytest.mark.parametrize("v", variants(S.SK_OVERLAP1D))
def test_overlap1d_one_hot_weights_shift_bit_exact(ctx, v):
    with forced(ctx, S.SK_OVERLAP1D, v):
        for r in (1, 4, 5, 12, 16):   # 5 and 12 run zero-padded to 8 and 16: the shift must not move
            if not o1_radius_ok(v, r):
                continue
            for n in (3, 50, 4099, 8193):
                x = I.uniform_pm1_f32(510 + n, n)
                vx, vo = ctx.vector_from(x), ctx.vector(n)
                for m in range(2 * r + 1):
                    w = np.zeros(2 * r + 1, np.float32)
                    w[m] = 1.0
                    for edge, pad in ((S.EDGE_CONSTANT, 0.25), (S.EDGE_DUPLICATE, 0.0)):
                        ctx.mapoverlap_1d(w, r, edge, pad, vx, vo)
                        j = np.arange(n) + m - r
                        if edge == S.EDGE_CONSTANT:
                            exp = np.where((j >= 0) & (j < n), x[np.clip(j, 0, n - 1)], np.float32(pad))
                        else:
                            exp = x[np.clip(j, 0, n - 1)]
                        assert np.array_equal(vo.numpy(), exp.astype(np.float32))
                vx.destroy()
                vo.destroy()


def test_overlap1d_constant_input_and_impulse(ctx):
    for v in variants(S.SK_OVERLAP1D):
        with forced(ctx, S.SK_OVERLAP1D, v):
            for r in (1, 4, 16):
                if not o1_radius_ok(v, r):
                    continue
                n = 20000
                w = I.positive_weights_f32(520 + r, 2 * r + 1)
                vx, vo = ctx.vector_from(np.full(n, 3.0, np.float32)), ctx.vector(n)
                ctx.mapoverlap_1d(w, r, S.EDGE_DUPLICATE, 0.0, vx, vo)
                got = vo.numpy()
                assert np.all(np.abs(got - 3.0 * w.astype(np.float64).sum()) <= 2e-6 * 3.0)
                assert np.all(got == got[0])
                x = np.zeros(n, np.float32)
                j = 8192
                x[j] = 1.0
                vx.write(x)
                ctx.mapoverlap_1d(w, r, S.EDGE_CONSTANT, 0.0, vx, vo)
                got = vo.numpy()
                exp = np.zeros(n, np.float32)
                for i in range(j - r, j + r + 1):
                    exp[i] = w[(j - i) + r]
                assert np.array_equal(got, exp)
                vx.destroy()
                vo.destroy()


@pytest.mark.parametrize("name", ["tma_swz_o16_s2", "tma_swz_o16_s3"])
def test_overlap1d_tma_pipeline_wraps(ctx, name):
    """Every persistent block of the TMA kernel walks >= 4 tiles (at most 148 x 6 blocks): the stages are refilled, both
    mbarrier parities are used, and a ragged tail (n % 32 != 0) ends the walk. Element by element against the oracle."""
    v = S.variant_names(S.SK_OVERLAP1D).index(name)
    n = 4096 * 3700 + 77
    x = I.uniform01_f32(7300, n)
    vx, vo = ctx.vector_from(x), ctx.vector(n)
    with forced(ctx, S.SK_OVERLAP1D, v):
        for r, edge, pad in ((16, S.EDGE_CYCLIC, 0.0), (16, S.EDGE_CONSTANT, 0.0), (8, S.EDGE_DUPLICATE, 0.0), (4, S.EDGE_CONSTANT, 1.5)):
            w = I.signed_weights_f32(7301 + r, 2 * r + 1)
            ctx.mapoverlap_1d(w, r, edge, pad, vx, vo)
            assert ctx.last_variant() == (S.SK_OVERLAP1D, v)
            ref, ab = O.mapoverlap_1d(w, r, edge, pad, x)
            assert_overlap(vo.numpy(), ref, ab)
    vx.destroy()
    vo.destroy()
    # rows of a matrix: two tiles per row (the second one 32 columns wide), > 4 tiles per block
    rows, cols = 3800, 4128
    X = I.uniform01_f32(7310, rows * cols).reshape(rows, cols)
    mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
    with forced(ctx, S.SK_OVERLAP1D, v):
        for r, edge, pad in ((8, S.EDGE_DUPLICATE, 0.0), (16, S.EDGE_CONSTANT, 0.0), (16, S.EDGE_CYCLIC, 0.0)):
            w = I.positive_weights_f32(7311 + r, 2 * r + 1)
            ctx.mapoverlap_1d_matrix(w, r, edge, pad, S.AXIS_ROW, mx, mo)
            assert ctx.last_variant() == (S.SK_OVERLAP1D, v)
            ref, ab = O.mapoverlap_1d_matrix(w, r, edge, pad, O.AXIS_ROW, X)
            assert_overlap(mo.numpy(), ref, ab)
    mx.destroy()
    mo.destroy()


MAT_SHAPES = [(1, 1), (3, 5), (37, 129), (64, 128), (65, 136), (200, 520), (130, 1032), (1030, 264), (6, 8256)]


@pytest.mark.parametrize("v", variants(S.SK_OVERLAP1D))
@pytest.mark.parametrize("r", [1, 4, 8, 16, 5])
def test_overlap1d_matrix_rows(ctx, v, r):
    w = I.positive_weights_f32(530 + r, 2 * r + 1)
    for rows, cols in MAT_SHAPES:
        X = I.uniform01_f32(531 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
        tiled_ok = o1_radius_ok(v, r) and (rows == 1 or cols % 8 == 0)
        if S.variant_names(S.SK_OVERLAP1D)[v].startswith("tma_swz"):
            tiled_ok = o1_radius_ok(v, r) and (rows == 1 or cols % 32 == 0)  # a matrix row must be whole 128-byte rows
        with forced(ctx, S.SK_OVERLAP1D, v):
            for edge, pad in EDGE_CASES:
                if v != 0 and not tiled_ok:
                    with pytest.raises(S.SkelError):
                        ctx.mapoverlap_1d_matrix(w, r, edge, pad, S.AXIS_ROW, mx, mo)
                    continue
                ctx.mapoverlap_1d_matrix(w, r, edge, pad, S.AXIS_ROW, mx, mo)
                ref, ab = O.mapoverlap_1d_matrix(w, r, edge, pad, O.AXIS_ROW, X)
                assert_overlap(mo.numpy(), ref, ab)
        mx.destroy()
        mo.destroy()


@pytest.mark.parametrize("v", variants(S.SK_OVERLAP1D_COL))
@pytest.mark.parametrize("r", [0, 1, 2, 3, 4, 8, 16, 5, 40])
def test_overlap1d_matrix_cols(ctx, v, r):
    w = I.positive_weights_f32(540 + r, 2 * r + 1)
    for rows, cols in MAT_SHAPES:
        X = I.uniform01_f32(541 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
        tiled_ok = 0 <= r <= 16 and cols % 4 == 0   # radii between the instantiated ones run zero-padded
        with forced(ctx, S.SK_OVERLAP1D_COL, v):
            for edge, pad in EDGE_CASES:
                if v != 0 and not tiled_ok:
                    with pytest.raises(S.SkelError):
                        ctx.mapoverlap_1d_matrix(w, r, edge, pad, S.AXIS_COL, mx, mo)
                    continue
                ctx.mapoverlap_1d_matrix(w, r, edge, pad, S.AXIS_COL, mx, mo)
                assert ctx.last_variant() == (S.SK_OVERLAP1D_COL, v)
                ref, ab = O.mapoverlap_1d_matrix(w, r, edge, pad, O.AXIS_COL, X)
                assert_overlap(mo.numpy(), ref, ab)
        mx.destroy()
        mo.destroy()


# ------------------------------------------------------------------ MapOverlap 2D
@pytest.mark.parametrize("v", variants(S.SK_OVERLAP2D))
@pytest.mark.parametrize("radii", [(0, 0), (1, 1), (2, 2), (3, 3), (4, 4), (2, 4), (1, 0), (0, 3), (4, 1), (8, 8), (5, 2)])
def test_overlap2d(ctx, v, radii):
    ry, rx = radii
    W = I.positive_weights_f32(600 + ry * 9 + rx, (2 * ry + 1) * (2 * rx + 1))
    Ws = I.signed_weights_f32(601 + ry * 9 + rx, (2 * ry + 1) * (2 * rx + 1))
    for rows, cols in MAT_SHAPES:
        X = I.uniform01_f32(602 + rows, rows * cols).reshape(rows, cols)
        mx, mo = ctx.matrix_from(X), ctx.matrix(rows, cols)
        tiled_ok = ry <= 4 and rx <= 4 and cols % 4 == 0   # rectangular filters run the zero-padded square one
        with forced(ctx, S.SK_OVERLAP2D, v):
            for edge, pad in EDGE_CASES:
                if v != 0 and not tiled_ok:
                    with pytest.raises(S.SkelError):
                        ctx.mapoverlap_2d(W, ry, rx, edge, pad, mx, mo)
                    continue
                ctx.mapoverlap_2d(W, ry, rx, edge, pad, mx, mo)
                assert ctx.last_variant() == (S.SK_OVERLAP2D, v)
                ref, ab = O.mapoverlap_2d(W, ry, rx, edge, pad, X)
                assert_overlap(mo.numpy(), ref, ab)
            if v == 0 or tiled_ok:
                ctx.mapoverlap_2d(Ws, ry, rx, S.EDGE_DUPLICATE, 0.0, mx, mo)
                ref, ab = O.mapoverlap_2d(Ws, ry, rx, O.EDGE_DUPLICATE, 0.0, X)
                assert_overlap(mo.numpy(), ref, ab)
        mx.destroy()
        mo.destroy()


@pytest.mark.parametrize("v", variants(S.SK_OVERLAP2D))
def test_overlap2d_one_hot_shift_bit_exact_and_separable_identity(ctx, v):
    rows, cols = 70, 136
    X = I.uniform_pm1_f32(610, rows * cols).reshape(rows, cols)
    mx, mo, mt = ctx.matrix_from(X), ctx.matrix(rows, cols), ctx.matrix(rows, cols)
    with forced(ctx, S.SK_OVERLAP2D, v):
        for a in range(5):
            for b in range(5):
                W = np.zeros((5, 5), np.float32)
                W[a, b] = 1.0
                for edge, pad in ((S.EDGE_CONSTANT, 0.125), (S.EDGE_DUPLICATE, 0.0)):
                    ctx.mapoverlap_2d(W, 2, 2, edge, pad, mx, mo)
                    p = np.arange(rows)[:, None] + a - 2
                    q = np.arange(cols)[None, :] + b - 2
                    inside = (p >= 0) & (p < rows) & (q >= 0) & (q < cols)
                    val = X[np.clip(p, 0, rows - 1), np.clip(q, 0, cols - 1)]
                    exp = val if edge == S.EDGE_DUPLICATE else np.where(inside, val, np.float32(pad))
                    assert np.array_equal(mo.numpy(), exp.astype(np.float32))
        # row pass then column pass == dense outer-product filter (within tolerance)
        X01 = np.abs(X)
        mx.write(X01)
        wr, wc = I.positive_weights_f32(611, 9), I.positive_weights_f32(612, 9)
        ctx.mapoverlap_1d_matrix(wr, 4, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
        ctx.mapoverlap_1d_matrix(wc, 4, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
        sep = mo.numpy()
        Wd = np.outer(wc.astype(np.float64), wr.astype(np.float64)).astype(np.float32)
        ctx.mapoverlap_2d(Wd, 4, 4, S.EDGE_DUPLICATE, 0.0, mx, mo)
        assert np.allclose(sep, mo.numpy(), rtol=0, atol=4e-6)
    for c in (mx, mo, mt):
        c.destroy()


def test_separable_pair_lock_step(ctx):
    # BJ:L10 "separable row-then-column 1D passes of radius 8": two calls, fp32 intermediate;
    # each pass is checked against the oracle fed with that pass's actual input (reading (c).6 iii)
    rows, cols, r = 300, 520, 8
    X = I.uniform01_f32(620, rows * cols).reshape(rows, cols)
    wr, wc = I.positive_weights_f32(621, 17), I.positive_weights_f32(622, 17)
    mx, mt, mo = ctx.matrix_from(X), ctx.matrix(rows, cols), ctx.matrix(rows, cols)
    ctx.mapoverlap_1d_matrix(wr, r, S.EDGE_DUPLICATE, 0.0, S.AXIS_ROW, mx, mt)
    ctx.mapoverlap_1d_matrix(wc, r, S.EDGE_DUPLICATE, 0.0, S.AXIS_COL, mt, mo)
    T = mt.numpy()
    ref, ab = O.mapoverlap_1d_matrix(wr, r, O.EDGE_DUPLICATE, 0.0, O.AXIS_ROW, X)
    assert_overlap(T, ref, ab)
    ref2, ab2 = O.mapoverlap_1d_matrix(wc, r, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, T)
    assert_overlap(mo.numpy(), ref2, ab2)
    # against the oracle's fp64 chain: the fp32 rounding of the intermediate stays inside 2e-6
    ref3, ab3 = O.mapoverlap_1d_matrix(wc, r, O.EDGE_DUPLICATE, 0.0, O.AXIS_COL, ref)
    assert_overlap(mo.numpy(), ref3, ab3)
    for c in (mx, mt, mo):
        c.destroy()


# ------------------------------------------------------------------ CYCLIC edge policy
@pytest.mark.parametrize("v", variants(S.SK_OVERLAP1D))
def test_overlap1d_cyclic_one_hot_is_a_rotation_bit_exact(ctx, v):
    r = 4
    with forced(ctx, S.SK_OVERLAP1D, v):
        for n in (3, 9, 4097, 100003):  # n < r: the index wraps more than once
            x = I.uniform01_f32(7000 + n, n)
            vx, vo = ctx.vector_from(x), ctx.vector(n)
            for m in (0, 3, 4, 8):
                w = np.zeros(2 * r + 1, np.float32)
                w[m] = 1.0
                ctx.mapoverlap_1d(w, r, S.EDGE_CYCLIC, 0.0, vx, vo)
                assert np.array_equal(vo.numpy(), np.roll(x, -(m - r))), (n, m)
            vx.destroy()
            vo.destroy()


@pytest.mark.parametrize("v", variants(S.SK_OVERLAP2D))
def test_overlap2d_cyclic_constant_input_has_no_border(ctx, v):
    rows, cols = 70, 260
    W = I.positive_weights_f32(7100, 25)
    with forced(ctx, S.SK_OVERLAP2D, v):
        mx, mo = ctx.matrix_from(np.full((rows, cols), 0.5, np.float32)), ctx.matrix(rows, cols)
        ctx.mapoverlap_2d(W, 2, 2, S.EDGE_CYCLIC, 0.0, mx, mo)
        got = mo.numpy()
        assert np.all(np.abs(got - 0.5 * W.astype(np.float64).sum()) <= 2e-6 * 0.5)
        assert np.all(got == got[0, 0])  # every output saw the same 25 values in the same order
        mx.destroy()
        mo.destroy()


# ------------------------------------------------------------------ three-vector Map
@pytest.mark.parametrize("v", variants(S.SK_MAP))
def test_map3_muladd(ctx, v):
    with forced(ctx, S.SK_MAP, v):
        for n in SIZES_SHORT + [4096, 65536 + 3]:
            a, b, c = I.uniform_pm1_f32(900 + n, n), I.uniform_pm1_f32(901 + n, n), I.uniform_pm1_f32(902 + n, n)
            va, vb, vc, vo = ctx.vector_from(a), ctx.vector_from(b), ctx.vector_from(c), ctx.vector(n)
            ctx.map3(S.FN_MULADD, va, vb, vc, vo)
            assert ctx.last_variant() == (S.SK_MAP, v)
            assert_map_f32(vo.numpy(), O.map3_muladd_f32(a, b, c))
            ctx.map3(S.FN_MULADD, va, vb, vc, vc)      # in place on the addend
            assert_map_f32(vc.numpy(), O.map3_muladd_f32(a, b, c))
            x = (I.raw_u64(903 + n, n) % np.uint64(1 << 32)).astype(np.uint32).view(np.int32)
            y = (I.raw_u64(904 + n, n) % np.uint64(1 << 32)).astype(np.uint32).view(np.int32)
            z = (I.raw_u64(905 + n, n) % np.uint64(1 << 32)).astype(np.uint32).view(np.int32)
            vx, vy, vz, vi = ctx.vector_from(x), ctx.vector_from(y), ctx.vector_from(z), ctx.vector(n, S.I32)
            ctx.map3(S.FN_MULADD, vx, vy, vz, vi)
            assert np.array_equal(vi.numpy(), O.map3_muladd_i32(x, y, z))
            for h in (va, vb, vc, vo, vx, vy, vz, vi):
                h.destroy()


def test_map3_cancellation_needs_fma_and_errors(ctx):
    n = 50000
    a, b = I.uniform_pm1_f32(910, n), I.uniform_pm1_f32(911, n)
    c = (-(a.astype(np.float64) * b.astype(np.float64))).astype(np.float32)   # a*b + c ~ the product's rounding error
    va, vb, vc, vo = ctx.vector_from(a), ctx.vector_from(b), ctx.vector_from(c), ctx.vector(n)
    ctx.map3(S.FN_MULADD, va, vb, vc, vo)
    assert_map_f32(vo.numpy(), O.map3_muladd_f32(a, b, c))   # a separate multiply and add would return 0 everywhere
    assert np.count_nonzero(vo.numpy()) > n // 2
    with pytest.raises(S.SkelError):
        ctx.map3(S.FN_ADD, va, vb, vc, vo)
    short = ctx.vector(n - 1)
    with pytest.raises(S.SkelError):
        ctx.map3(S.FN_MULADD, va, vb, short, vo)
    for h in (va, vb, vc, vo, short):
        h.destroy()
