"""skel_reduce_f32_noalloc: the Reduce that allocates nothing (scratch in a static __device__ array).

Collected last on purpose (the suite runs with ``pytest -x``). Checks the new entry point against the EXISTING
Reduce path (skel_reduce through a context) on the same device buffer, within the Reduce tolerance the parity tests
use (helpers.assert_reduce_f32: 1e-5 * sum|x|; MAX exactly), on two calls in a row that share the static scratch,
plus the size limit and that device memory does not move across calls.
"""
import numpy as np
import pytest

import skel_inputs as I
from helpers import assert_reduce_f32
from paper_1405_2915_b200 import skel as S

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def env():
    import torch
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    ctx = S.Context()
    yield torch, ctx
    ctx.close()


def both_paths(torch, ctx, op, t):
    """-> (no-alloc result, existing path's result) for the device tensor t."""
    out = torch.full((1,), float("nan"), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    S.reduce_f32_noalloc(op, t.data_ptr(), t.numel(), out.data_ptr(), 0)
    torch.cuda.synchronize()
    v = ctx.vector_adopt(t)
    ref = ctx.reduce(op, v)
    v.destroy()
    return float(out.item()), float(ref)


@pytest.mark.parametrize("n", [1, 5, 4097, 8192, 8193, 100003, (1 << 22) + 7])
def test_two_calls_in_a_row_match_the_existing_reduce(env, n):
    torch, ctx = env
    x = I.uniform_pm1_f32(9100 + n, n)
    y = I.uniform_pm1_f32(9101 + n, max(1, n // 3))       # second call: another input, a smaller grid, same scratch
    tx, ty = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda()
    for arr, t in ((x, tx), (y, ty), (x, tx)):
        abs_sum = float(np.abs(arr).sum(dtype=np.float64))
        got, ref = both_paths(torch, ctx, S.FN_ADD, t)
        assert_reduce_f32(got, ref, abs_sum)
        got, ref = both_paths(torch, ctx, S.FN_MAX, t)
        assert got == ref == float(arr.max())
    z = (1.0 + x[: min(n, 5000)] * 2.0 ** -12).astype(np.float32)
    got, ref = both_paths(torch, ctx, S.FN_MULT, torch.from_numpy(z).cuda())
    assert abs(got - ref) <= 1e-4 * abs(ref)


def test_maximum_size_unaligned_input_and_determinism(env):
    torch, ctx = env
    nmax = S.noalloc_max_elements()
    assert nmax == 1 << 26 and S.lib.skel_noalloc_scratch_bytes() == 8192 * 4 + 256
    x = I.uniform_pm1_f32(9200, nmax + 1)
    t = torch.from_numpy(x).cuda()
    abs_sum = float(np.abs(x[:nmax]).sum(dtype=np.float64))
    got, ref = both_paths(torch, ctx, S.FN_ADD, t[:nmax])          # 8192 blocks: every partial slot in use
    assert_reduce_f32(got, ref, abs_sum)
    got2, ref2 = both_paths(torch, ctx, S.FN_ADD, t[1:1 + 100003])  # 4-byte aligned only, right after the full grid
    assert_reduce_f32(got2, ref2, float(np.abs(x[1:100004]).sum(dtype=np.float64)))
    assert_reduce_f32(got2, float(x[1:100004].sum(dtype=np.float64)), float(np.abs(x[1:100004]).sum(dtype=np.float64)))
    again, _ = both_paths(torch, ctx, S.FN_ADD, t[:nmax])
    assert again == got                                            # fixed order: bitwise run to run
    with pytest.raises(S.SkelError) as e:                           # one element beyond the static scratch's reach
        S.reduce_f32_noalloc(S.FN_ADD, t.data_ptr(), nmax + 1, t.data_ptr(), 0)
    assert e.value.status == S.ERR_UNSUPPORTED
    assert "exceeds" in str(e.value) and str(nmax) in str(e.value)
    with pytest.raises(S.SkelError):
        S.reduce_f32_noalloc(S.FN_ADD, t.data_ptr(), 0, t.data_ptr(), 0)
    with pytest.raises(S.SkelError):
        S.reduce_f32_noalloc(S.FN_SAXPY, t.data_ptr(), 10, t.data_ptr(), 0)
    with pytest.raises(S.SkelError):
        S.reduce_f32_noalloc(S.FN_ADD, 0, 10, t.data_ptr(), 0)


def test_calls_leave_device_memory_where_it_was(env):
    torch, ctx = env
    n = (1 << 22) + 7
    t = torch.from_numpy(I.uniform_pm1_f32(9300, n)).cuda()
    out = torch.zeros(1, dtype=torch.float32, device="cuda")
    side = torch.cuda.Stream()                                           # torch creates its stream pool here
    for stream in (0, side.cuda_stream):                                 # first calls: set-up, first use of the stream
        S.reduce_f32_noalloc(S.FN_ADD, t.data_ptr(), n, out.data_ptr(), stream)
        torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for k in range(20):
        S.reduce_f32_noalloc(S.FN_ADD, t.data_ptr(), n - k, out.data_ptr(), side.cuda_stream if k % 2 else 0)
        torch.cuda.synchronize()                                         # calls must not overlap: they share the scratch
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
