"""Multi-rank plumbing of the bench: "replicas only".

BASELINE.json fixes one GPU for the CFNEB path (no sharding, no collectives): with N ranks every rank runs the same
band on its own GPU.  What crosses ranks is measurement only -- a barrier on both sides of the timed region and the
MAX over ranks of the device-timed duration; value = (units all ranks processed) / (that time).  torch.distributed
is the plumbing (nccl on GPUs; the same code runs on gloo, which is how tests/ cover it on CPU).
"""
import os


class Ranks:
    """world / rank from the torchrun environment; no process group when world == 1."""

    def __init__(self, backend="nccl", device=None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.backend = backend
        self.device = device
        self.dist = None
        if self.world > 1:
            import torch.distributed as dist
            if not dist.is_initialized():
                kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
                dist.init_process_group(backend, **kw)
            self.dist = dist

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def max_over_ranks(self, x):
        """MAX over ranks of a host float (a device-timed duration)."""
        if self.dist is None:
            return float(x)
        import torch
        dev = self.device if self.backend == "nccl" else "cpu"
        t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def throughput(self, units_per_rank, seconds_this_rank):
        """Whole-job units per second: every rank did `units_per_rank`; time = max over ranks."""
        return self.world * units_per_rank / self.max_over_ranks(seconds_this_rank)

    def close(self):
        if self.dist is not None:
            self.dist.barrier()
            self.dist.destroy_process_group()
            self.dist = None
