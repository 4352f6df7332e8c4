"""Multi-GPU plumbing: one process per GPU.

By default `bench.py --gpus N` runs N independent replicas of the workload, one per rank, with no data-path
collective (the slab decomposition of the SPH step, with its neighbour halo exchange, lives in slab.py).  torch.distributed is used only for the barrier around the timed region and for combining the
per-rank results: time = max over ranks, units = sum over ranks.
"""
import os


class Ranks:
    """Rank bookkeeping from the torchrun environment.  backend: "nccl" on GPU boxes, "gloo" in CPU tests."""

    def __init__(self, backend=None):
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.dist = None
        if self.world > 1:
            import torch
            import torch.distributed as dist
            if backend is None:
                backend = "nccl" if torch.cuda.is_available() else "gloo"
            os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
            os.environ.setdefault("MASTER_PORT", "29500")
            if not dist.is_initialized():
                if backend == "nccl":
                    torch.cuda.set_device(self.local_rank)
                    dist.init_process_group(backend, rank=self.rank, world_size=self.world,
                                            device_id=torch.device("cuda", self.local_rank))
                else:
                    dist.init_process_group(backend, rank=self.rank, world_size=self.world)
            self.dist = dist
            self.backend = backend

    def _tensor(self, values):
        import torch
        t = torch.tensor(values, dtype=torch.float64)
        if self.dist is not None and self.backend == "nccl":
            t = t.cuda(self.local_rank)
        return t

    def barrier(self):
        if self.dist is not None:
            self.dist.barrier()

    def combine(self, seconds, units):
        """(max over ranks of seconds, sum over ranks of units); every rank gets the result."""
        if self.dist is None:
            return float(seconds), float(units)
        tmax = self._tensor([seconds])
        usum = self._tensor([units])
        self.dist.all_reduce(tmax, op=self.dist.ReduceOp.MAX)
        self.dist.all_reduce(usum, op=self.dist.ReduceOp.SUM)
        return float(tmax.item()), float(usum.item())

    def reduce_max(self, values):
        if self.dist is None:
            return [float(v) for v in values]
        t = self._tensor(list(values))
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return [float(v) for v in t.tolist()]

    def close(self):
        if self.dist is not None and self.dist.is_initialized():
            self.dist.destroy_process_group()
            self.dist = None


def throughput(seconds_per_rank, units_per_rank):
    """Whole-job throughput of independent replicas: all units / the slowest rank's time."""
    return sum(units_per_rank) / max(seconds_per_rank)
