"""Host-side plumbing for running N independent replicas of the path, one process per GPU (DESIGN.md "Multi-GPU":
the path does not shard in this build, so there is NO data-path collective).  torch.distributed is used only to
line the replicas up (barrier) and to combine their timings: max over ranks of the elapsed time, sum of the units.
Works with backend "nccl" on GPUs and "gloo" on CPU (tests/test_replicas.py, world_size 2)."""
import os


def env_world():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))


class Replicas:
    def __init__(self, backend=None, device=None):
        self.rank, self.local_rank, self.world = env_world()
        self.dist = None
        self.device = device
        if self.world > 1:
            import torch.distributed as dist
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29511")
            if not dist.is_initialized():
                dist.init_process_group(backend=backend or "nccl", rank=self.rank, world_size=self.world)
            self.dist = dist

    def _tensor(self, value):
        import torch
        return torch.tensor([float(value)], dtype=torch.float64, device=self.device if self.device is not None else "cpu")

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max(self, value):
        if self.dist is None:
            return float(value)
        t = self._tensor(value)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def sum(self, value):
        if self.dist is None:
            return float(value)
        t = self._tensor(value)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        return float(t.item())

    def throughput(self, units_this_rank, elapsed_s_this_rank):
        """Whole-job throughput: units all ranks processed / the slowest rank's time."""
        return self.sum(units_this_rank) / self.max(elapsed_s_this_rank)

    def close(self):
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()
            self.dist = None
