"""Replica plumbing for N > 1 GPUs ("Multi-GPU": replicas only).

The gauge-fixing path of this library runs on one GPU (BASELINE.json north_star: "there is no
multi-GPU part"); independent configurations -- the usual ensemble workload -- go one per GPU
with no data-path collective.  This module holds the host-side logic around that: which
configuration a rank works on, the barrier that brackets a timed region, the max-over-ranks of a
device time and the whole-job aggregate.  ``torch.distributed`` is used for the barrier and one
scalar all-reduce only (backend "nccl" on GPUs, "gloo" in the CPU tests).  No arithmetic of the
method lives here.
"""
import os

import torch
import torch.distributed as dist


class Replicas:
    """One process per GPU; rank r fixes configuration number r of the ensemble."""

    def __init__(self, backend=None, device=None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.device = device
        self._owns_group = False
        if self.world > 1 and not dist.is_initialized():
            backend = backend or ("nccl" if (device is not None and torch.device(device).type == "cuda") else "gloo")
            kwargs = {}
            if backend == "nccl":
                kwargs["device_id"] = torch.device(device)
            dist.init_process_group(backend, rank=self.rank, world_size=self.world, **kwargs)
            self._owns_group = True

    # ---- which work a rank does
    def config_seed(self, base_seed):
        """Seed of this rank's configuration: distinct per rank, rank 0 keeps the single-GPU seed."""
        return int(base_seed) + self.rank

    def my_items(self, n_items):
        """Indices of an ensemble of n_items configurations this rank fixes (round robin)."""
        return list(range(self.rank, int(n_items), self.world))

    # ---- timing brackets
    def barrier(self):
        if self.world > 1:
            dist.barrier()
        if self.device is not None and torch.device(self.device).type == "cuda":
            torch.cuda.synchronize(self.device)

    def max_over_ranks(self, x):
        """Slowest rank's value (device times are reported as the max over ranks)."""
        if self.world == 1:
            return float(x)
        dev = self.device if (self.device is not None and dist.get_backend() == "nccl") else "cpu"
        t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, x):
        if self.world == 1:
            return float(x)
        dev = self.device if (self.device is not None and dist.get_backend() == "nccl") else "cpu"
        t = torch.tensor([float(x)], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def job_throughput(self, units_this_rank, seconds_this_rank):
        """Whole-job units/s: the units ALL ranks processed divided by the slowest rank's time."""
        return self.sum_over_ranks(units_this_rank) / self.max_over_ranks(seconds_this_rank)

    @property
    def is_root(self):
        return self.rank == 0

    def close(self):
        if self._owns_group and dist.is_initialized():
            dist.destroy_process_group()
            self._owns_group = False
