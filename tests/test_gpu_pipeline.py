"""Smart-container coherence on the GPU and the chained pipeline of
BASELINE.json configs[4] (readings 14 and 15): transfer counts against the protocol's
closed forms, lock-step parity of every call against the CPU oracle, run-to-run determinism, and a
model-based random walk (library vs shadow arrays + the protocol table)."""
import numpy as np
import pytest

import oracle as O
from helpers import assert_map_f32, assert_overlap, assert_reduce_f32
import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu

C32 = float(np.float32(1.0001))


@pytest.fixture()
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


def run_pipeline(ctx, x0, w, iters, verify_at=()):
    """Map(x*1.0001) in place -> MapOverlap1D(r=4, duplicate) -> Reduce(sum); A and B swap roles."""
    n = x0.size
    a, b = ctx.vector_from(x0), ctx.vector(n)
    ctx.reset_stats()
    scalars = []
    for k in range(1, iters + 1):
        check = k in verify_at
        if check:
            a_in = a.numpy().copy()  # the GPU's actual input of this call (a host read: counted below)
        ctx.map(S.FN_MULT, 1.0001, a, None, a)
        if check:
            a_mid = a.numpy().copy()
            assert_map_f32(a_mid, O.map_f32(O.FN_MULT, 1.0001, a_in))
        ctx.mapoverlap_1d(w, 4, S.EDGE_DUPLICATE, 0.0, a, b)
        s = ctx.reduce(S.FN_ADD, b)
        if check:
            b_out = b.numpy().copy()
            ref, ab = O.mapoverlap_1d(w, 4, O.EDGE_DUPLICATE, 0.0, a_mid)
            assert_overlap(b_out, ref, ab)
            r, absum = O.reduce_f32(O.FN_ADD, b_out)
            assert_reduce_f32(s, r, absum)
        scalars.append(s)
        a, b = b, a
    st = ctx.stats()
    final = a.numpy().copy()
    a.destroy()
    b.destroy()
    return scalars, st, final


def test_pipeline_lazy_transfer_counts_lockstep_and_determinism(ctx):
    n, iters = (1 << 20) + 37, 12
    x0 = I.uniform01_f32(I.config_seed(5, 1), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)
    # measurement run: only the scalars are read
    scal, st, final = run_pipeline(ctx, x0, w, iters)
    assert st["h2d_count"] == 1 and st["h2d_bytes"] == 4 * n          # the one upload of A
    assert st["d2h_count"] == 0 and st["d2h_bytes"] == 0              # nothing comes back during the loop
    assert st["scalar_d2h_count"] == iters
    assert st["h2d_elided"] == 3 * iters - 1                           # every other device read reused a valid copy
    assert st["launches"] >= 3 * iters
    # verification run: every call checked in lock-step at iterations 1, 2 and the last
    scal2, st2, final2 = run_pipeline(ctx, x0, w, iters, verify_at=(1, 2, iters))
    assert scal2 == scal, "pipeline scalars are not bit-identical run to run"
    assert np.array_equal(final, final2)
    assert st2["h2d_count"] == 1                                       # host reads never invalidate the device copy
    # three host reads per verified iteration, minus the two that find a valid host copy: A at iteration 1
    # (created from host data) and A at iteration 2 (it is iteration 1's B, already downloaded)
    assert st2["d2h_count"] == 3 * 3 - 2
    # free-running fp64 chain (reported bound, reading 15): drift stays tiny over 12 iterations
    x = x0.astype(np.float64)
    for k in range(iters):
        x = x * C32
        x, _ = O.mapoverlap_1d(w, 4, O.EDGE_DUPLICATE, 0.0, x.astype(np.float32))  # oracle takes fp32 inputs
    assert abs(scal[-1] - x.sum()) <= 1e-4 * np.abs(x).sum()


def test_pipeline_constant_vector_closed_form(ctx):
    # duplicate edges + weights summing to 1 keep a constant vector constant: s_k = n * K * c32^k
    n, iters, K = 300007, 10, 0.75
    w = I.positive_weights_f32(77, 9)
    wsum = float(w.astype(np.float64).sum())
    scal, _, _ = run_pipeline(ctx, np.full(n, K, np.float32), w, iters)
    for k, s in enumerate(scal, start=1):
        expect = n * K * (C32 * wsum) ** k
        assert abs(s - expect) <= 1e-5 * abs(expect), (k, s, expect)


def test_pipeline_eager_moves_five_containers_per_iteration(ctx):
    n, iters = 100003, 4
    x0 = I.uniform01_f32(9001, n)
    w = I.positive_weights_f32(9002, 9)
    lazy, _, lazy_final = run_pipeline(ctx, x0, w, iters)
    ctx.set_coherence(S.EAGER)
    try:
        eager, st, eager_final = run_pipeline(ctx, x0, w, iters)
    finally:
        ctx.set_coherence(S.LAZY)
    assert eager == lazy and np.array_equal(lazy_final, eager_final)   # same kernels, same data
    assert st["h2d_count"] == 3 * iters and st["h2d_bytes"] == 3 * iters * 4 * n
    assert st["d2h_count"] == 2 * iters and st["d2h_bytes"] == 2 * iters * 4 * n
    assert st["h2d_elided"] == 0 and st["d2h_elided"] == 0


# The protocol of SURVEY.md 8(c).7 / DESIGN.md reading 14 written out as a literal table: the model of the random
# walk below is THIS table, not the library's own skel_coherence_step. States: bit 0 = host copy valid, bit 1 = device
# copy valid (0 UNINIT, 1 HOST, 2 DEVICE, 3 SHARED). (state, actor, access) -> (new state, transfer).
_U, _H, _D, _S = 0, 1, 2, 3
_R, _W, _RW = 0, 1, 2   # skel_access values (include/skel.h), restated
MODEL = {
    (_U, "dev", _W): (_D, None), (_U, "host", _W): (_H, None),
    (_H, "dev", _R): (_S, "h2d"), (_H, "dev", _W): (_D, None), (_H, "dev", _RW): (_D, "h2d"),
    (_H, "host", _R): (_H, None), (_H, "host", _W): (_H, None), (_H, "host", _RW): (_H, None),
    (_D, "dev", _R): (_D, None), (_D, "dev", _W): (_D, None), (_D, "dev", _RW): (_D, None),
    (_D, "host", _R): (_S, "d2h"), (_D, "host", _W): (_H, None), (_D, "host", _RW): (_H, "d2h"),
    (_S, "dev", _R): (_S, None), (_S, "dev", _W): (_D, None), (_S, "dev", _RW): (_D, None),
    (_S, "host", _R): (_S, None), (_S, "host", _W): (_H, None), (_S, "host", _RW): (_H, None),
}


def test_coherence_model_based_random_walk(ctx):
    """Random sequences of host writes / host reads / skeleton calls on three containers, applied to
    the library and to shadow host arrays through the oracle + the protocol table."""
    rng = np.random.default_rng(20140529)
    n = 5003
    w = I.positive_weights_f32(31, 5)
    vecs = [ctx.vector(n) for _ in range(3)]
    shadow = [None, None, None]          # fp32 arrays as the GPU holds them (downloaded after each call)
    state = [_U, _U, _U]
    assert (S.READ, S.WRITE, S.READWRITE) == (_R, _W, _RW)
    h2d = d2h = 0
    ctx.reset_stats()

    def dev_access(i, access):
        nonlocal h2d
        new, xfer = MODEL[(state[i], "dev", access)]
        h2d += 1 if xfer == "h2d" else 0
        state[i] = new

    def host_access(i, access):
        nonlocal d2h
        new, xfer = MODEL[(state[i], "host", access)]
        d2h += 1 if xfer == "d2h" else 0
        state[i] = new

    for step in range(120):
        op = rng.integers(0, 5)
        i, j = rng.choice(3, size=2, replace=False)
        if op == 0 or shadow[i] is None:       # host write (whole container)
            data = I.uniform01_f32(1000 + step, n)
            host_access(i, S.WRITE)
            vecs[i].write(data)
            shadow[i] = data.copy()
        elif op == 1:                           # host read
            host_access(i, S.READ)
            got = vecs[i].numpy()
            assert np.array_equal(got, shadow[i]), f"step {step}: stale or wrong data on host read"
        elif op == 2:                           # Map in place
            dev_access(i, S.READWRITE)
            ctx.map(S.FN_MULT, 1.0001, vecs[i], None, vecs[i])
            ref = O.map_f32(O.FN_MULT, 1.0001, shadow[i])
            shadow[i] = ref.astype(np.float32)  # mult of two fp32 values is correctly rounded: 0 ulp
        elif op == 3:                           # MapOverlap i -> j
            dev_access(i, S.READ)
            dev_access(j, S.WRITE)
            ctx.mapoverlap_1d(w, 2, S.EDGE_CONSTANT, 0.0, vecs[i], vecs[j])
            ref, ab = O.mapoverlap_1d(w, 2, O.EDGE_CONSTANT, 0.0, shadow[i])
            host_access(j, S.READ)              # download to resynchronise the shadow with the GPU's fp32 result
            got = vecs[j].numpy()
            assert_overlap(got, ref, ab)
            shadow[j] = got.copy()
        else:                                   # Reduce
            dev_access(i, S.READ)
            s = ctx.reduce(S.FN_ADD, vecs[i])
            r, ab = O.reduce_f32(O.FN_ADD, shadow[i])
            assert_reduce_f32(s, r, ab)
        for k in range(3):
            assert vecs[k].state() == state[k], f"step {step}: container {k} state {vecs[k].state()} != model {state[k]}"
    st = ctx.stats()
    assert st["h2d_count"] == h2d and st["d2h_count"] == d2h, (st, h2d, d2h)
    assert st["h2d_bytes"] == 4 * n * h2d and st["d2h_bytes"] == 4 * n * d2h
    for v in vecs:
        v.destroy()


def test_uninitialised_read_and_alias_errors(ctx):
    a, b = ctx.vector(100), ctx.vector(100)
    with pytest.raises(S.SkelError):
        ctx.map(S.FN_ADD, 1.0, a, None, b)       # a was never written
    a.write(np.ones(100, np.float32))
    with pytest.raises(S.SkelError):
        ctx.mapoverlap_1d(np.ones(3, np.float32), 1, S.EDGE_DUPLICATE, 0.0, a, a)  # output aliases input
    a.destroy()
    b.destroy()


# ------------------------------------------------------------------ per-container events, asynchronous Reduce
def test_host_read_waits_for_its_own_producer_not_for_the_stream(ctx):
    """PAPER.md L116 / L135 (data-dependence tracking, asynchronous calls): a host read of container A returns while
    long-running work on unrelated containers, enqueued AFTER A's producer, is still in flight."""
    import torch
    n_small, n_big = 1000, 1 << 26
    a, a2 = ctx.vector_from(np.arange(n_small, dtype=np.float32)), ctx.vector(n_small)
    big = ctx.vector_from(I.uniform_int_i32(5, n_big, 15))
    out = ctx.vector(n_big, S.I32)
    ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, big, out)   # upload + warm-up
    ctx.sync()
    ctx.map(S.FN_ADD, 1.0, a, None, a2)                 # A's producer: microseconds
    for _ in range(40):                                 # ~4 ms of unrelated device work behind it
        ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, big, out)
    got = a2.numpy()                                    # host READ of a2: waits for the Map's event only
    still_busy = not torch.cuda.current_stream().query()
    assert np.array_equal(got, np.arange(n_small, dtype=np.float32) + 1.0)
    assert still_busy, "the host read drained the whole stream"
    # a host WRITE of `a` (read by the Map) likewise only waits for the Map
    a.write(np.zeros(n_small, np.float32))
    assert not torch.cuda.current_stream().query()
    ctx.sync()
    ref = O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, I.uniform_int_i32(5, n_big, 15))
    assert np.array_equal(out.numpy(), ref)
    for v in (a, a2, big, out):
        v.destroy()


def test_reduce_async_futures(ctx):
    import torch
    n = 300007
    x = I.uniform_pm1_f32(7001, n)
    y = I.uniform_pm1_f32(7002, n)
    v = I.uniform_int_i32(7003, n, 1000)
    vx, vy, vi = ctx.vector_from(x), ctx.vector_from(y), ctx.vector_from(v)
    ctx.reset_stats()
    futs = [ctx.reduce_async(S.FN_ADD, vi), ctx.reduce_async(S.FN_MAX, vi), ctx.reduce_async(S.FN_ADD, vx),
            ctx.mapreduce_async(S.FN_MULT, S.FN_ADD, 0.0, vx, vy), ctx.mapreduce_async(S.FN_MULT, S.FN_ADD, 2.0, vi, None)]
    assert ctx.stats()["scalar_d2h_count"] == 0          # nothing has been read back yet
    assert futs[0].wait() == O.reduce_i32(O.FN_ADD, v)[0]
    assert futs[0].wait() == O.reduce_i32(O.FN_ADD, v)[0]   # may be waited for again
    assert futs[1].wait() == O.reduce_i32(O.FN_MAX, v)[0]
    r, ab = O.reduce_f32(O.FN_ADD, x)
    assert_reduce_f32(futs[2].wait(), r, ab)
    r, ab = O.mapreduce_f32(O.FN_MULT, O.FN_ADD, 0.0, x, y)
    assert_reduce_f32(futs[3].wait(), r, ab)
    assert futs[4].wait() == O.mapreduce_i32(O.FN_MULT, O.FN_ADD, 2, v)
    assert all(f.ready() for f in futs)
    assert ctx.stats()["scalar_d2h_count"] == 6
    # the blocking form still works next to outstanding futures and gives the same bits
    assert ctx.reduce(S.FN_ADD, vx) == futs[2].wait()
    # a context with a live future cannot be destroyed; destroying the future releases its slot
    with pytest.raises(S.SkelError):
        ctx.check(S.lib.skel_ctx_destroy(ctx.h))
    for f in futs:
        f.destroy()
    # the pool: 1024 outstanding futures, the next one is refused with SKEL_ERR_BUSY and leaves no trace
    small = ctx.vector_from(np.ones(64, np.float32))
    many = [ctx.reduce_async(S.FN_ADD, small) for _ in range(1024)]
    with pytest.raises(S.SkelError):
        ctx.reduce_async(S.FN_ADD, small)
    assert all(f.result() == 64.0 for f in many)
    assert ctx.reduce_async(S.FN_ADD, small).result() == 64.0
    # ready() turns true without a wait
    big = ctx.vector_from(I.uniform_int_i32(7004, 1 << 24, 15))
    f = ctx.reduce_async(S.FN_ADD, big)
    torch.cuda.synchronize()
    assert f.ready() and f.result() == O.reduce_i32(O.FN_ADD, I.uniform_int_i32(7004, 1 << 24, 15))[0]
    for c in (vx, vy, vi, small, big):
        c.destroy()


@pytest.mark.parametrize("fusion", [False, True])
def test_pipeline_with_futures_keeps_iterations_in_flight_and_gives_the_same_scalars(ctx, fusion):
    n, iters = (1 << 20) + 37, 12
    x0 = I.uniform01_f32(I.config_seed(5, 1), n)
    w = I.positive_weights_f32(I.config_seed(3, 14), 9)

    def run(use_futures):
        a, b = ctx.vector_from(x0), ctx.vector(n)
        ctx.reset_stats()
        out, futs = [], []
        for _ in range(iters):
            ctx.map(S.FN_MULT, 1.0001, a, None, a)
            ctx.mapoverlap_1d(w, 4, S.EDGE_DUPLICATE, 0.0, a, b)
            if use_futures:
                futs.append(ctx.reduce_async(S.FN_ADD, b))
            else:
                out.append(ctx.reduce(S.FN_ADD, b))
            a, b = b, a
        st_before_wait = ctx.stats()
        out += [f.result() for f in futs]
        st = ctx.stats()
        final = a.numpy().copy()
        a.destroy()
        b.destroy()
        return out, st_before_wait, st, final

    ctx.set_fusion(fusion)
    try:
        blocking, _, st_b, final_b = run(False)
        asynch, st_mid, st_a, final_a = run(True)
    finally:
        ctx.set_fusion(False)
    assert asynch == blocking, "async scalars differ from the blocking ones"
    assert np.array_equal(final_a, final_b)
    assert st_mid["scalar_d2h_count"] == 0 and st_a["scalar_d2h_count"] == iters == st_b["scalar_d2h_count"]
    assert st_a["h2d_count"] == 1 and st_a["d2h_count"] == 0 and st_a["h2d_elided"] == st_b["h2d_elided"]
    assert st_a["launches"] == st_b["launches"] == (iters if fusion else 3 * iters)


def test_replay_hook_runs_the_recorded_calls_both_ways(ctx):
    """skel_replay_* (include/skel.h): the measurement hook behind bench.py's container_layer figure replays recorded
    calls through the container layer or as bare launches; both leave the same results in the containers."""
    n = 200003
    x, v = I.uniform01_f32(8801, n), I.uniform_int_i32(8802, n, 1000)
    w = I.positive_weights_f32(8803, 9)
    vx, vo, vi, vs, res = ctx.vector_from(x), ctx.vector(n), ctx.vector_from(v), ctx.vector(n, S.I32), ctx.vector(4, S.I32)
    ctx.replay_begin()
    ctx.map(S.FN_MULT, 1.0001, vx, None, vo)
    ctx.mapoverlap_1d(w, 4, S.EDGE_DUPLICATE, 0.0, vx, vo)
    ctx.scan(S.FN_ADD, S.SCAN_INCLUSIVE, 0, vi, vs)
    ctx.reduce_to(S.FN_ADD, vi, res, 2)
    assert ctx.replay_end() == 4
    ref, ab = O.mapoverlap_1d(w, 4, O.EDGE_DUPLICATE, 0.0, x)
    for raw in (False, True):
        vo.write(np.zeros(n, np.float32))
        vs.write(np.zeros(n, np.int32))
        ctx.reset_stats()
        host_us, dev_us = ctx.replay_run(raw, 3)
        assert host_us > 0 and dev_us > 0
        st = ctx.stats()
        assert st["launches"] >= 12
        if raw:   # bare launches: the coherence layer saw nothing, the containers still say "host copy valid"
            assert st["h2d_count"] == 0 and vo.state() == S.ST_HOST
            continue
        assert st["h2d_count"] == 0 and st["h2d_elided"] >= 9      # inputs stayed on the device
        assert_overlap(vo.numpy(), ref, ab)
        assert np.array_equal(vs.numpy(), O.scan_i32(O.FN_ADD, O.SCAN_INCLUSIVE, 0, v))
        assert res.numpy()[2] == O.reduce_i32(O.FN_ADD, v)[0]
    with pytest.raises(S.SkelError):
        ctx.replay_begin(), ctx.replay_run(False, 1)   # still recording
    ctx.replay_end()
    for c in (vx, vo, vi, vs, res):
        c.destroy()


def test_adopted_buffers_that_overlap_are_rejected(ctx):
    """alias checks go by device address range, not by handle identity."""
    import torch
    t = torch.rand(3000, device="cuda")
    a = ctx.vector_adopt(t[:2000])
    b = ctx.vector_adopt(t[1000:3000])       # overlaps a
    b2 = ctx.vector_adopt(t[:2000])          # the same memory as a, another handle
    cfree = ctx.vector_adopt(t[2000:3000])   # disjoint from the first 1000 elements only
    a1 = ctx.vector_adopt(t[:1000])
    w = np.ones(3, np.float32)
    for out in (b, b2):
        with pytest.raises(S.SkelError) as ei:
            ctx.mapoverlap_1d(w, 1, S.EDGE_DUPLICATE, 0.0, a, out)
        assert ei.value.status == S.ERR_ALIAS
        with pytest.raises(S.SkelError) as ei:
            ctx.map(S.FN_MULT, 2.0, a, None, out)
        assert ei.value.status == S.ERR_ALIAS
    ctx.map(S.FN_MULT, 2.0, a1, None, cfree)           # disjoint: fine
    ctx.map(S.FN_MULT, 2.0, a, None, a)                # one handle in place: fine
    s1 = ctx.mapreduce(S.FN_MULT, S.FN_ADD, 0.0, a, b2)  # both only read: fine (dot of a with itself)
    assert s1 > 0
    ctx.sync()
    for v in (a, b, b2, cfree, a1):
        v.destroy()
