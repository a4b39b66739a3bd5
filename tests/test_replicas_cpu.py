"""N > 1 path of bench.py on CPU: world size 2, gloo backend (DESIGN.md §9 "replicas only"): barrier,
max-over-ranks timing and whole-job aggregation. No GPU, no data-path collective."""
import os
import socket
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
from paper_1405_2915_b200.replicas import Replicas
r = Replicas(backend="gloo")
assert r.world == 2
r.barrier()
local_ms = 10.0 if r.rank == 0 else 25.0          # rank 1 is the slow replica
value, ms = r.aggregate_throughput(1000.0, local_ms)
mx = r.max_over_ranks(float(r.rank))
r.barrier()
if r.rank == 0:
    print(json.dumps({{"value": value, "ms": ms, "mx": mx, "world": r.world}}))
r.close()
"""


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_replicas_gloo(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=120) for p in procs]
    for p, (o, e) in zip(procs, outs):
        assert p.returncode == 0, e
    import json
    line = json.loads(outs[0][0].strip().splitlines()[-1])
    assert line["world"] == 2
    assert line["ms"] == 25.0                       # the slowest replica decides
    assert abs(line["value"] - 2 * 1000.0 / 25e-3) < 1e-6   # whole job = both replicas' units in that time
    assert line["mx"] == 1.0
    assert outs[1][0].strip() == ""                 # only rank 0 prints


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_1405_2915_b200.replicas import Replicas
    env = {k: os.environ.pop(k) for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK") if k in os.environ}
    try:
        r = Replicas(backend="gloo")
        assert r.world == 1 and r.max_over_ranks(3.5) == 3.5
        v, ms = r.aggregate_throughput(10.0, 2.0)
        assert ms == 2.0 and abs(v - 5000.0) < 1e-9
    finally:
        os.environ.update(env)
