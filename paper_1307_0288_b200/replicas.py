"""Multi-GPU plumbing: replicas only.

The Chebyshev path of one random vector does not shard (BASELINE.json north_star: "no
sharding, no inter-GPU collectives").  What a multi-GPU user does is what the paper does with
its 10-100 random vectors (eq 18-21; N_r = 10 P:472, 100 P:505, 30 P:553): run
independent vectors, one process per GPU, and average the small moment arrays at the end
(Tr[A] ~ (1/N_r) sum_r <phi_r|A|phi_r>).  That average is the only exchange; it moves a few
KB and is done with one all-reduce (NCCL on GPUs, gloo in the CPU tests).

This module holds no arithmetic of the method: rank bookkeeping, which vector streams a rank
owns, max/mean over ranks.
"""
from __future__ import annotations

import os
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass
class ReplicaContext:
    rank: int
    world: int
    local_rank: int
    initialised_here: bool

    def barrier(self):
        if self.world > 1:
            dist.barrier()

    def _device(self):
        if self.world > 1 and dist.get_backend() == "nccl":
            return torch.device("cuda", torch.cuda.current_device())
        return torch.device("cpu")

    def max_over_ranks(self, value: float) -> float:
        """Max of a per-rank scalar (device-measured time): the job is as slow as its slowest rank."""
        if self.world == 1:
            return float(value)
        t = torch.tensor([float(value)], dtype=torch.float64, device=self._device())
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    def sum_over_ranks(self, value: float) -> float:
        if self.world == 1:
            return float(value)
        t = torch.tensor([float(value)], dtype=torch.float64, device=self._device())
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        return float(t.item())

    def mean_over_ranks(self, mu: torch.Tensor) -> torch.Tensor:
        """Average of per-rank moment arrays (complex128, any shape): the stochastic-trace average
        over the replicas' random vectors (eq 21).  Returns a new tensor on mu's device."""
        if self.world == 1:
            return mu.clone()
        buf = torch.view_as_real(mu.contiguous()).clone().to(self._device())
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
        buf /= self.world
        return torch.view_as_complex(buf).to(mu.device)

    def finalize(self):
        if self.initialised_here and dist.is_initialized():
            dist.destroy_process_group()


def init_from_env(backend: str = "nccl") -> ReplicaContext:
    """Read RANK / LOCAL_RANK / WORLD_SIZE / MASTER_* (torchrun); single process if unset."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world == 1:
        return ReplicaContext(0, 1, local, False)
    started = False
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend == "nccl":
            torch.cuda.set_device(local)
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
        started = True
    return ReplicaContext(rank, world, local, started)


def vector_streams(rank: int, R: int) -> range:
    """Random-vector indices owned by `rank` when every rank evaluates R vectors: rank*R .. rank*R+R-1
    (vector r uses PRNG stream 16 + r of the config's seed)."""
    return range(rank * R, (rank + 1) * R)
