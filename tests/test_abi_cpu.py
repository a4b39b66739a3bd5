"""CPU-only checks of the C ABI: the library loads, exports every symbol include/skel.h declares,
and its pure host logic (coherence protocol, execution-plan lookup / save / load, argument
validation that precedes any CUDA call) behaves as DESIGN.md states. No compute calls."""
import os
import re

import numpy as np
import pytest

from paper_1405_2915_b200 import skel as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "skel.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(skel_[a-z0-9_]+)\s*\(", text)) - {"skel_alloc_fn", "skel_free_fn"})


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert len(names) >= 40
    for n in names:
        assert hasattr(S.lib, n), f"libskel.so does not export {n}"
    # the binding declares exactly the header's functions
    assert sorted(S.EXPORTS) == names
    assert S.skel_abi_version() == 2


def test_variant_tables():
    for sk in range(S.SK_COUNT):
        names = S.variant_names(sk)
        assert len(names) >= 2 and len(set(names)) == len(names)
    assert S.lib.skel_variant_count(99) == 0
    assert S.lib.skel_variant_name(0, 99) is None


# ---- coherence protocol --------------------------------
U, H, D, SH = S.ST_UNINIT, S.ST_HOST, S.ST_DEVICE, S.ST_SHARED
DEV, HOST = 0, 1
NONE, H2D, D2H = 0, 1, 2
LAZY_TABLE = {
    # (state, actor, access): (new_state, transfer) or None for SKEL_ERR_UNINIT
    (U, DEV, S.READ): None, (U, DEV, S.WRITE): (D, NONE), (U, DEV, S.READWRITE): None,
    (U, HOST, S.READ): None, (U, HOST, S.WRITE): (H, NONE), (U, HOST, S.READWRITE): None,
    (H, DEV, S.READ): (SH, H2D), (H, DEV, S.WRITE): (D, NONE), (H, DEV, S.READWRITE): (D, H2D),
    (H, HOST, S.READ): (H, NONE), (H, HOST, S.WRITE): (H, NONE), (H, HOST, S.READWRITE): (H, NONE),
    (D, DEV, S.READ): (D, NONE), (D, DEV, S.WRITE): (D, NONE), (D, DEV, S.READWRITE): (D, NONE),
    (D, HOST, S.READ): (SH, D2H), (D, HOST, S.WRITE): (H, NONE), (D, HOST, S.READWRITE): (H, D2H),
    (SH, DEV, S.READ): (SH, NONE), (SH, DEV, S.WRITE): (D, NONE), (SH, DEV, S.READWRITE): (D, NONE),
    (SH, HOST, S.READ): (SH, NONE), (SH, HOST, S.WRITE): (H, NONE), (SH, HOST, S.READWRITE): (H, NONE),
}


def test_coherence_lazy_table():
    for (state, actor, access), exp in LAZY_TABLE.items():
        st, ns, tr = S.coherence_step(state, actor, access, S.LAZY)
        if exp is None:
            assert st == S.ERR_UNINIT
        else:
            assert (st, ns, tr) == (S.OK, exp[0], exp[1]), (state, actor, access)


def test_coherence_invariants_random_walk():
    # "stale copies are never accessed": simulate version numbers per copy
    rng = np.random.default_rng(5)
    for mode in (S.LAZY, S.EAGER):
        state, host_ver, dev_ver, latest = U, -1, -1, -1
        for _ in range(5000):
            actor, access = int(rng.integers(2)), int(rng.integers(3))
            st, ns, tr = S.coherence_step(state, actor, access, mode)
            if st != S.OK:
                assert state == U and access != S.WRITE
                continue
            reads, writes = access != S.WRITE, access != S.READ
            if actor == HOST:
                if tr & D2H:
                    assert dev_ver == latest
                    host_ver = dev_ver
                if reads:
                    assert host_ver == latest, "host would read a stale copy"
                if writes:
                    latest += 1
                    host_ver = latest
            else:
                if tr & H2D:
                    assert host_ver == latest
                    dev_ver = host_ver
                if reads:
                    assert dev_ver == latest, "device would read a stale copy"
                if writes:
                    latest += 1
                    dev_ver = latest
                if tr & D2H:
                    host_ver = dev_ver
            state = ns
            assert bool(state & 1) == (host_ver == latest and latest >= 0) or mode == S.EAGER
            if state & 1:
                assert host_ver == latest
            if state & 2:
                assert dev_ver == latest
            assert state != U


def test_coherence_eager_uploads_and_downloads():
    assert S.coherence_step(H, DEV, S.READ, S.EAGER) == (S.OK, H, H2D)
    assert S.coherence_step(SH, DEV, S.READ, S.EAGER) == (S.OK, H, H2D)
    assert S.coherence_step(D, DEV, S.READ, S.EAGER) == (S.OK, D, NONE)
    assert S.coherence_step(H, DEV, S.WRITE, S.EAGER) == (S.OK, H, D2H)
    assert S.coherence_step(U, DEV, S.WRITE, S.EAGER) == (S.OK, H, D2H)
    assert S.coherence_step(H, DEV, S.READWRITE, S.EAGER) == (S.OK, H, H2D | D2H)
    assert S.coherence_step(U, DEV, S.READ, S.EAGER)[0] == S.ERR_UNINIT
    assert S.lib.skel_coherence_step(7, 0, 0, 0, None, None) == S.ERR_INVALID_ARG


# ---- execution plans -----------------------------------------------------------
def test_plan_lookup_set_save_load(tmp_path):
    ctx = S.Context(lazy_cuda=True)
    inst = S.SkelInstance(skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=4, edge=S.EDGE_DUPLICATE)
    other = S.SkelInstance(skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=16, edge=S.EDGE_DUPLICATE)
    default = ctx.plan_lookup(inst, 1 << 20)
    assert 0 <= default < S.lib.skel_variant_count(S.SK_OVERLAP1D)
    ctx.plan_set(inst, 0, 0)
    ctx.plan_set(inst, 1 << 16, 1)
    ctx.plan_set(inst, 1 << 22, 3)
    for n, v in [(0, 0), (1, 0), ((1 << 16) - 1, 0), (1 << 16, 1), ((1 << 22) - 1, 1), (1 << 22, 3), (1 << 30, 3)]:
        assert ctx.plan_lookup(inst, n) == v
    # a radius that was never tuned inherits its nearest tuned neighbour (the dispatch tree, see below);
    # another skeleton / element type is untouched
    assert ctx.plan_lookup(other, 1 << 20) == 1 and ctx.plan_explain(other, 1 << 20) == (1, False, True)
    assert ctx.plan_explain(inst, 1 << 20) == (1, True, True)
    col = S.SkelInstance(skeleton=S.SK_OVERLAP1D_COL, fn=S.FN_WSTENCIL, dtype=S.F32, r0=4, edge=S.EDGE_DUPLICATE)
    assert ctx.plan_explain(col, 1 << 20)[1:] == (False, False)
    ctx.plan_set(inst, 1 << 16, 2)  # overwrite a breakpoint
    assert ctx.plan_lookup(inst, 1 << 17) == 2
    path = str(tmp_path / "b.plan")
    ctx.plan_save(path)
    ctx.plan_clear()
    assert ctx.plan_lookup(inst, 1 << 17) == default
    ctx.plan_load(path)
    assert [ctx.plan_lookup(inst, n) for n in (5, 1 << 17, 1 << 23)] == [0, 2, 3]
    # forcing wins over the plan
    ctx.force_variant(S.SK_OVERLAP1D, 1)
    assert ctx.plan_lookup(inst, 1 << 23) == 1
    ctx.force_variant(S.SK_OVERLAP1D, -1)
    assert ctx.plan_lookup(inst, 1 << 23) == 3
    with pytest.raises(S.SkelError):
        ctx.plan_set(inst, 0, 99)
    with pytest.raises(S.SkelError):
        ctx.plan_load(str(tmp_path / "missing.plan"))
    bad = tmp_path / "bad.plan"
    bad.write_text("not a plan\n")
    with pytest.raises(S.SkelError):
        ctx.plan_load(str(bad))
    assert ctx.plan_lookup(inst, 1 << 23) == 3  # a failed load leaves the plan as it was
    ctx.close()


def test_plan_dispatch_tree_inherits_the_nearest_tuned_neighbour(tmp_path):
    """SURVEY.md 8(f) f3 / PAPER.md L53 "tree-based dispatch structure": skeleton -> dtype -> (fn, fn2) -> shape class ->
    r0 -> r1 -> edge -> size breakpoints. An untuned context takes the nearest tuned child at the first level where it
    has none (radii: nearest in log2(r + 1), ties to the larger radius); skeleton and dtype must match."""
    ctx = S.Context(lazy_cuda=True)
    o1 = lambda r, edge=S.EDGE_DUPLICATE, mode=0, dt=S.F32: S.SkelInstance(  # noqa: E731
        skeleton=S.SK_OVERLAP1D, fn=S.FN_WSTENCIL, dtype=dt, r0=r, edge=edge, mode=mode)
    ctx.plan_set(o1(4), 0, 8)
    ctx.plan_set(o1(4), 1 << 20, 10)
    ctx.plan_set(o1(16), 0, 9)
    ctx.plan_set(o1(1, S.EDGE_CONSTANT), 0, 4)
    n = 1 << 22
    assert ctx.plan_explain(o1(4), n) == (10, True, True) and ctx.plan_explain(o1(4), 5) == (8, True, True)
    # radii: log2(r+1) distance. r=5,6 -> 4; r=8: |log2 9 - log2 5| = 0.848 < |log2 17 - log2 9| = 0.918 -> 4;
    # r=12 -> 16; r=2 -> log2 3: 0.585 from r=1, 0.737 from r=4 -> 1; r=64 -> 16; r=0 -> 1
    expect = {5: 10, 6: 10, 8: 10, 9: 9, 12: 9, 64: 9, 3: 10, 2: 4, 0: 4}
    for r, v in expect.items():
        assert ctx.plan_explain(o1(r), n) == (v, False, True), r
    # the breakpoints of the neighbour are inherited, not just its last variant
    assert ctx.plan_lookup(o1(5), 1000) == 8 and ctx.plan_lookup(o1(5), n) == 10
    # edge policy never tuned for this radius: the first tuned policy of that radius
    assert ctx.plan_explain(o1(4, S.EDGE_CYCLIC), n) == (10, False, True)
    assert ctx.plan_explain(o1(1, S.EDGE_DUPLICATE), n) == (4, False, True)
    # shape class never tuned (rows of a matrix): inherits the vector's subtree; once tuned, it is its own
    assert ctx.plan_explain(o1(4, mode=1), n) == (10, False, True)
    ctx.plan_set(o1(8, mode=1), 0, 7)
    assert ctx.plan_explain(o1(4, mode=1), n) == (7, False, True) and ctx.plan_explain(o1(4), n) == (10, True, True)
    # skeleton and element type must match: nothing is inherited across them
    assert ctx.plan_explain(o1(4, dt=S.I32), n)[2] is False
    red = S.SkelInstance(skeleton=S.SK_REDUCE, fn=S.FN_ADD, dtype=S.F32)
    assert ctx.plan_explain(red, n)[2] is False
    # user function never tuned: the first tuned function of that skeleton and element type
    ctx.plan_set(S.SkelInstance(skeleton=S.SK_REDUCE, fn=S.FN_ADD, dtype=S.I32), 0, 5)
    assert ctx.plan_explain(S.SkelInstance(skeleton=S.SK_REDUCE, fn=S.FN_MAX, dtype=S.I32), n) == (5, False, True)
    # 2D: both radii walk the tree
    o2 = lambda ry, rx: S.SkelInstance(skeleton=S.SK_OVERLAP2D, fn=S.FN_WSTENCIL, dtype=S.F32, r0=ry, r1=rx, edge=S.EDGE_DUPLICATE)  # noqa: E731
    ctx.plan_set(o2(2, 2), 0, 7)
    ctx.plan_set(o2(4, 4), 0, 5)
    assert ctx.plan_lookup(o2(3, 3), n) == 5 and ctx.plan_lookup(o2(1, 1), n) == 7 and ctx.plan_lookup(o2(2, 4), n) == 7
    # save / load round trip keeps the tree; '#' lines (provenance) are comments
    path = tmp_path / "tree.plan"
    ctx.plan_save(str(path))
    text = path.read_text().splitlines()
    path.write_text("\n".join(["# generated by: a test", text[0], "# another comment"] + text[1:]) + "\n")
    ctx.plan_clear()
    assert ctx.plan_explain(o1(5), n)[2] is False
    ctx.plan_load(str(path))
    for r, v in expect.items():
        assert ctx.plan_explain(o1(r), n) == (v, False, True), r
    ctx.close()


def test_plan_file_from_the_environment_reports_a_failed_load(tmp_path):
    import subprocess
    import sys
    code = ("import os, sys; sys.path.insert(0, %r)\n"
            "from paper_1405_2915_b200 import skel as S\n"
            "c = S.Context(lazy_cuda=True)\n"
            "print(S.lib.skel_last_error(c.h).decode())\n" % ROOT)
    bad = tmp_path / "bad.plan"
    bad.write_text("garbage\n")
    out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, SKEL_PLAN_FILE=str(bad)),
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and "SKEL_PLAN_FILE" in out.stdout and "bad.plan" in out.stdout, out.stderr
    good = os.path.join(ROOT, "paper_1405_2915_b200", "plans", "b200.plan")
    out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, SKEL_PLAN_FILE=good),
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0 and "SKEL_PLAN_FILE" not in out.stdout, out.stderr


def test_plan_lookup_is_fast():
    import time
    ctx = S.Context(lazy_cuda=True)
    inst = S.SkelInstance(skeleton=S.SK_MAP, fn=S.FN_ADD, dtype=S.F32, mode=1)
    for k in range(10, 29):
        ctx.plan_set(inst, 1 << k, k % 3)
    import ctypes as C
    v = C.c_int()
    ref = C.byref(inst)
    t = time.perf_counter()
    for _ in range(20000):
        S.lib.skel_plan_lookup(ctx.h, ref, 123456, C.byref(v))
    per = (time.perf_counter() - t) / 20000
    assert per < 20e-6  # includes the ctypes call overhead (~1 us); the lookup itself is O(log)
    ctx.close()


def test_argument_validation_without_cuda():
    ctx = S.Context(lazy_cuda=True)
    import ctypes as C
    h = C.c_void_p()
    assert S.lib.skel_vector_create(None, S.F32, 4, C.byref(h)) == S.ERR_INVALID_ARG
    assert S.lib.skel_vector_create(ctx.h, 7, 4, C.byref(h)) == S.ERR_INVALID_ARG
    a = ctx.vector(8, S.F32)
    b = ctx.vector(9, S.F32)
    i = ctx.vector(8, S.I32)
    m = ctx.matrix(2, 4)
    assert a.state() == S.ST_UNINIT
    res = C.c_float()
    assert S.lib.skel_map(ctx.h, S.FN_ADD, 0.0, a.h, b.h, a.h) == S.ERR_SIZE_MISMATCH
    assert S.lib.skel_map(ctx.h, S.FN_ADD, 0.0, a.h, i.h, a.h) == S.ERR_DTYPE
    assert S.lib.skel_map(ctx.h, S.FN_WSTENCIL, 0.0, a.h, None, a.h) == S.ERR_UNSUPPORTED
    assert S.lib.skel_map(ctx.h, S.FN_SAXPY, 1.0, a.h, None, a.h) == S.ERR_INVALID_ARG
    assert S.lib.skel_map(ctx.h, S.FN_ADD, 0.5, i.h, None, i.h) == S.ERR_INVALID_ARG  # 0.5 is no int32
    assert S.lib.skel_reduce(ctx.h, S.FN_SAXPY, a.h, C.byref(res)) == S.ERR_UNSUPPORTED
    assert S.lib.skel_reduce(ctx.h, S.FN_ADD, None, C.byref(res)) == S.ERR_INVALID_ARG
    e = ctx.vector(0, S.F32)
    assert S.lib.skel_reduce(ctx.h, S.FN_ADD, e.h, C.byref(res)) == S.ERR_EMPTY
    w = (C.c_float * 200)()
    assert S.lib.skel_mapoverlap_1d(ctx.h, w, 65, 0, 0.0, a.h, b.h) == S.ERR_UNSUPPORTED
    assert S.lib.skel_mapoverlap_1d(ctx.h, w, -1, 0, 0.0, a.h, b.h) == S.ERR_UNSUPPORTED
    assert S.lib.skel_mapoverlap_1d(ctx.h, w, 1, 0, 0.0, a.h, b.h) == S.ERR_SIZE_MISMATCH
    assert S.lib.skel_mapoverlap_1d(ctx.h, w, 1, 0, 0.0, a.h, a.h) == S.ERR_ALIAS
    assert S.lib.skel_mapoverlap_1d(ctx.h, w, 1, 0, 0.0, i.h, i.h) == S.ERR_DTYPE
    assert S.lib.skel_mapoverlap_2d(ctx.h, w, 9, 1, 0, 0.0, m.h, m.h) == S.ERR_UNSUPPORTED
    assert S.lib.skel_scan(ctx.h, S.FN_SAXPY, 0, 0.0, a.h, a.h) == S.ERR_UNSUPPORTED
    assert S.lib.skel_scan(ctx.h, S.FN_ADD, 5, 0.0, a.h, a.h) == S.ERR_INVALID_ARG
    assert b"alias" in S.lib.skel_last_error(ctx.h) or True
    assert S.lib.skel_ctx_destroy(ctx.h) == S.ERR_BUSY  # live containers
    for c in (a, b, i, m, e):
        c.destroy()
    ctx.close()


def test_shipped_plan_is_consistent_with_the_variant_tables():
    """plans/b200.plan (the plan bench.py loads): well-formed, loads, every variant id exists for its skeleton,
    breakpoints ascend, and the look-up returns the stored winner at BASELINE.json's full sizes."""
    import os

    path = os.path.join(os.path.dirname(os.path.abspath(S.__file__)), "plans", "b200.plan")
    lines = [ln for ln in open(path).read().split("\n") if not ln.lstrip().startswith("#")]   # '#': provenance comments
    assert lines[0].strip() == "skelplan 1"
    ctx = S.Context(lazy_cuda=True)
    ctx.plan_load(path)
    seen = 0
    for line in lines[1:]:
        f = line.split()
        if not f:
            continue
        key, count, rest = [int(v) for v in f[:8]], int(f[8]), [int(v) for v in f[9:]]
        assert len(rest) == 2 * count and count >= 1
        nmins, variants = rest[0::2], rest[1::2]
        assert nmins == sorted(set(nmins))
        nv = S.lib.skel_variant_count(key[0])
        assert all(0 <= v < nv for v in variants), (line, nv)
        inst = S.SkelInstance(skeleton=key[0], fn=key[1], fn2=key[2], dtype=key[3], r0=key[4], r1=key[5], edge=key[6], mode=key[7])
        for n, v in zip(nmins, variants):
            assert ctx.plan_lookup(inst, max(n, 1)) == v or n == 0
        assert ctx.plan_lookup(inst, 1 << 28) == variants[-1]
        seen += 1
    assert seen >= 20


def test_tuner_instance_selection_and_plan_coverage():
    """tune.py: --only takes comma-separated substrings; every instance the tuner knows (the bench instances and the
    neighbours of the dispatch tree) has its own entry in the shipped plan, found by an exact look-up."""
    import os

    from paper_1405_2915_b200 import tune

    assert tune.selected("reduce_max_i32", None) and tune.selected("reduce_max_i32", "")
    assert tune.selected("reduce_max_i32", "reduce_,dot") and tune.selected("dot_f32", "reduce_,dot")
    assert not tune.selected("scan_add_i32_incl", "reduce_,dot") and not tune.selected("dot_f32", "reduce_,")
    names = [name for name, *_ in tune.instances(S)]
    assert len(names) == len(set(names)) and "overlap2d_5x5_i32" in names and "overlap1d_r4_e1_i32" in names
    path = os.path.join(os.path.dirname(os.path.abspath(S.__file__)), "plans", "b200.plan")
    ctx = S.Context(lazy_cuda=True)
    ctx.plan_load(path)
    for name, inst, lo, hi, cols in tune.instances(S):
        v, exact, from_plan = ctx.plan_explain(inst, 1 << hi)
        assert exact and from_plan, name
        assert 0 <= v < S.lib.skel_variant_count(inst.skeleton), name
    ctx.close()
