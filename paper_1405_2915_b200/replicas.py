"""Multi-GPU plumbing of the benchmark: REPLICAS ONLY. The hot path does not shard
(BASELINE.json: one GPU, no collectives), so N GPUs run N independent replicas of the same step.
The only communication is the timing protocol: a barrier on both sides of the timed region and the
MAX over ranks of the device time. Backend "nccl" on GPUs; "gloo" lets the same code run on CPU
(tests/test_replicas_cpu.py, world size 2)."""
from __future__ import annotations

import os


def env_world():
    """(world_size, rank, local_rank) from the torchrun environment; (1, 0, 0) when not launched by it."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


class Replicas:
    def __init__(self, backend: str = "nccl", device=None):
        import torch.distributed as dist
        self.world, self.rank, self.local = env_world()
        self.device = device
        self.dist = dist
        if self.world > 1 and not dist.is_initialized():
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, **kw)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()

    def max_over_ranks(self, x: float) -> float:
        """The slowest replica decides (timing contract: max over ranks)."""
        if self.world == 1:
            return float(x)
        import torch
        t = torch.tensor([x], dtype=torch.float64, device=self.device if self.device is not None else "cpu")
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def aggregate_throughput(self, units_per_replica_step: float, ms_per_step_local: float) -> tuple[float, float]:
        """-> (whole-job units per second, ms per step used): every replica does the same work (weak
        scaling), so the job processed world * units in the time of the slowest replica."""
        ms = self.max_over_ranks(ms_per_step_local)
        return self.world * units_per_replica_step / (ms * 1e-3), ms

    def close(self):
        if self.world > 1 and self.dist.is_initialized():
            self.dist.destroy_process_group()
