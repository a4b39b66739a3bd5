"""Range-granular host access on the GPU (include/skel.h skel_vector_host_acquire_range, PAPER.md
L123 "partial copies"): transfer sizes against the closed form, values against shadow arrays (the Map used is
x + 1 in int32: exact), and a model-based random walk mixing whole-container accesses, range accesses and skeleton
calls."""
import numpy as np
import pytest

import skel_inputs as I
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu


@pytest.fixture()
def ctx():
    import torch
    assert torch.cuda.is_available()
    c = S.Context()
    yield c
    c.close()


def test_range_write_uploads_only_the_range(ctx):
    n = 1 << 20
    x = I.uniform_int_i32(1, n, 1000)
    v, o = ctx.vector_from(x), ctx.vector(n, S.I32)
    ctx.map(S.FN_ADD, 1, v, None, o)                      # uploads the whole container once
    assert ctx.stats()["h2d_bytes"] == 4 * n and v.state() == 3
    shadow = x.copy()
    ctx.reset_stats()
    v.write_range(1000, np.arange(500, dtype=np.int32))   # device copy stays valid
    shadow[1000:1500] = np.arange(500)
    v.write_range(1400, np.full(300, 7, np.int32))        # overlaps: the ranges merge
    shadow[1400:1700] = 7
    v.write_range(n - 10, np.full(10, -3, np.int32))
    shadow[n - 10:] = -3
    assert v.state() == 3 and ctx.stats()["h2d_bytes"] == 0
    ctx.map(S.FN_ADD, 1, v, None, o)                      # uploads [1000, 1700) and [n-10, n): two copies
    st = ctx.stats()
    assert st["h2d_bytes"] == 4 * (700 + 10) and st["h2d_count"] == 2
    assert np.array_equal(o.numpy(), shadow + 1)
    ctx.reset_stats()
    ctx.map(S.FN_ADD, 1, v, None, o)                      # nothing left to upload
    assert ctx.stats()["h2d_bytes"] == 0
    assert np.array_equal(v.numpy(), shadow)
    v.destroy(); o.destroy()


def test_range_access_to_a_device_only_container(ctx):
    n = 300007
    x = I.uniform_int_i32(2, n, 1000)
    v, o = ctx.vector_from(x), ctx.vector(n, S.I32)
    ctx.map(S.FN_ADD, 5, v, None, o)                      # o: device valid, host invalid
    shadow = x + 5
    assert o.state() == 2
    ctx.reset_stats()
    assert np.array_equal(o.read_range(12345, 100), shadow[12345:12445])
    st = ctx.stats()
    assert st["d2h_bytes"] == 400 and st["d2h_count"] == 1 and o.state() == 2   # a peek: the state does not change
    o.write_range(50, np.full(20, 9, np.int32))           # host newer in [50, 70); everything else only on the device
    shadow[50:70] = 9
    w = o.host_view_range(S.READWRITE, 60, 20)            # overlaps the written range: it must not be lost
    assert np.array_equal(w, shadow[60:80])
    w += 1
    o.release()
    shadow[60:80] += 1
    ctx.map(S.FN_ADD, 0, o, None, v)                      # reads o: uploads the ranges
    assert np.array_equal(v.numpy(), shadow)
    assert np.array_equal(o.numpy(), shadow)              # whole read: downloads everything, range data intact
    # a whole-container device write discards pending host ranges
    o.write_range(0, np.full(8, 1, np.int32))
    ctx.reset_stats()
    ctx.map(S.FN_ADD, 2, v, None, o)
    assert ctx.stats()["h2d_bytes"] == 0
    assert np.array_equal(o.numpy(), shadow + 2)
    v.destroy(); o.destroy()


def test_matrix_rows_and_errors(ctx):
    rows, cols = 64, 256
    X = I.uniform_int_i32(3, rows * cols, 100).reshape(rows, cols)
    m, out = ctx.matrix_from(X), ctx.vector(rows, S.I32)
    ctx.reduce_rows(S.FN_ADD, m, out)
    ctx.reset_stats()
    view = m.host_view_range(S.WRITE, 3 * cols, 2 * cols)  # rows 3 and 4
    view[...] = 1
    m.release()
    ctx.reduce_rows(S.FN_ADD, m, out)
    assert ctx.stats()["h2d_bytes"] == 4 * 2 * cols
    exp = X.astype(np.int64).sum(axis=1)
    exp[3:5] = cols
    assert np.array_equal(out.numpy(), exp.astype(np.int32))
    fresh = ctx.vector(100, S.I32)
    with pytest.raises(S.SkelError):
        fresh.write_range(0, np.zeros(10, np.int32))       # never written: a partial write is refused
    with pytest.raises(S.SkelError):
        out.read_range(60, 10)                             # out of bounds
    with pytest.raises(S.SkelError):
        out.host_view_range(S.READ, 0, 0)                  # empty range
    for h in (m, out, fresh):
        h.destroy()


def test_random_walk_against_shadow_arrays(ctx):
    n = 70001
    u = I.raw_u64(4, 4000)
    k = 0
    a_sh = I.uniform_int_i32(5, n, 1000)
    b_sh = np.zeros(n, np.int32)
    a, b = ctx.vector_from(a_sh), ctx.vector(n, S.I32)
    ctx.map(S.FN_ADD, 0, a, None, b)
    b_sh = a_sh.copy()
    for step in range(150):
        op = int(u[k] % 7); lo = int(u[k + 1] % n); ln = 1 + int(u[k + 2] % min(5000, n - lo)); k += 3
        if op == 0:                                   # range write on a
            val = (np.arange(ln) + step).astype(np.int32)
            a.write_range(lo, val); a_sh[lo:lo + ln] = val
        elif op == 1:                                 # range read-modify-write on b
            w = b.host_view_range(S.READWRITE, lo, ln); assert np.array_equal(w, b_sh[lo:lo + ln]); w += 3; b.release()
            b_sh[lo:lo + ln] += 3
        elif op == 2:                                 # range read
            assert np.array_equal(a.read_range(lo, ln), a_sh[lo:lo + ln])
        elif op == 3:                                 # skeleton call a -> b
            ctx.map(S.FN_ADD, step, a, None, b); b_sh = a_sh + np.int32(step)
        elif op == 4:                                 # skeleton call b -> a, in place variant afterwards
            ctx.map(S.FN_MAX, 10, b, None, a); a_sh = np.maximum(b_sh, 10)
        elif op == 5:                                 # whole read
            assert np.array_equal(b.numpy(), b_sh)
        else:                                         # whole write
            val = I.uniform_int_i32(100 + step, n, 50); a.write(val); a_sh = val.copy()
    assert np.array_equal(a.numpy(), a_sh) and np.array_equal(b.numpy(), b_sh)
    a.destroy(); b.destroy()


def test_prefetch_host_overlaps_and_stays_coherent(ctx):
    """skel_vector_prefetch_host: the download runs on a copy stream; host accesses wait for it, device writes are
    ordered after it, a stale prefetch is redone."""
    n = 1 << 22
    x = I.uniform_int_i32(11, n, 1000)
    v, o, p = ctx.vector_from(x), ctx.vector(n, S.I32), ctx.vector(n, S.I32)
    ctx.map(S.FN_ADD, 1, v, None, o)
    ctx.reset_stats()
    o.prefetch_host()                                  # async download of x + 1
    assert o.state() == 3 and ctx.stats()["d2h_bytes"] == 4 * n
    ctx.map(S.FN_ADD, 2, o, None, p)                   # reads o while it downloads: no conflict
    ctx.map(S.FN_ADD, 10, v, None, o)                  # OVERWRITES o: must wait for the download to finish reading it
    assert o.state() == 2
    assert np.array_equal(p.numpy(), x + 3)
    ctx.reset_stats()
    assert np.array_equal(o.numpy(), x + 10)           # the prefetched copy was stale: downloaded again
    assert ctx.stats()["d2h_bytes"] == 4 * n
    # prefetch, then a host read finds the data without a second transfer
    ctx.map(S.FN_ADD, 20, v, None, o)
    o.prefetch_host()
    o.prefetch_host()                                  # idempotent
    ctx.reset_stats()
    assert np.array_equal(o.numpy(), x + 20)
    assert ctx.stats()["d2h_bytes"] == 0
    # prefetch of a container with host-written ranges keeps them
    ctx.map(S.FN_ADD, 30, v, None, o)
    o.write_range(5, np.full(4, -1, np.int32))
    o.prefetch_host()
    exp = x + 30
    exp[5:9] = -1
    assert np.array_equal(o.numpy(), exp)
    for h in (v, o, p):
        h.destroy()
