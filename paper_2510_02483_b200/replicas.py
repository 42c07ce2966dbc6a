"""Multi-GPU plumbing for bench.py: "replicas only".

BASELINE.json `north_star` fixes the path to one GPU with no sharding and no collective, so N GPUs run N
independent replicas of the same layer step (one process per GPU).  The only cross-rank traffic is the
measurement itself: a barrier on both sides of the timed region and a MAX over ranks of the device-timed
milliseconds.  This module holds that logic so it can be tested on CPU with the gloo backend (world_size 2).
No arithmetic of the method lives here.
"""
from __future__ import annotations

import os
from dataclasses import dataclass

import torch
import torch.distributed as dist


@dataclass(frozen=True)
class RankEnv:
    rank: int
    local_rank: int
    world_size: int

    @property
    def is_main(self) -> bool:
        return self.rank == 0


def rank_env(env=None) -> RankEnv:
    """RANK / LOCAL_RANK / WORLD_SIZE as torchrun sets them (single process: 0 / 0 / 1)."""
    env = os.environ if env is None else env
    return RankEnv(int(env.get("RANK", 0)), int(env.get("LOCAL_RANK", 0)), int(env.get("WORLD_SIZE", 1)))


def init(backend: str, renv: RankEnv) -> bool:
    """Join the process group when there is more than one rank.  Rendezvous comes from MASTER_ADDR/MASTER_PORT."""
    if renv.world_size <= 1:
        return False
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend, rank=renv.rank, world_size=renv.world_size)
    return True


def barrier(device=None):
    if dist.is_available() and dist.is_initialized():
        if device is not None and device.type == "cuda":
            dist.barrier(device_ids=[device.index])
        else:
            dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """MAX over ranks of a per-rank scalar (the device-timed milliseconds of the timed region)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """SUM over ranks of a per-rank count (units processed, kernels launched)."""
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_throughput(units_this_rank: float, ms_this_rank: float, device=None):
    """(units of all ranks) / (max-over-ranks time): the `value` of bench.py.  Returns (value_per_s, ms_max, units)."""
    ms_max = max_over_ranks(ms_this_rank, device)
    units = sum_over_ranks(units_this_rank, device)
    return units / (ms_max * 1e-3), ms_max, units


def finalize():
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
