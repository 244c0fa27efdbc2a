"""Multi-GPU plumbing for the request-sharded (data-parallel) decode head.

The path shards by request: a CFG pair (or an unpaired row) is an independent unit, the
<= 256 MiB of head weights are replicated on every GPU, and no step of the path exchanges
data between ranks ("replicas only").  torch.distributed is used for the
launch-time barrier and for the max-over-ranks timing only.
"""
from __future__ import annotations

import os
from typing import Tuple

import torch
import torch.distributed as dist


def env_world() -> Tuple[int, int, int]:
    """(rank, local_rank, world_size) from torchrun's environment (1 process => (0, 0, 1))."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str) -> Tuple[int, int, int]:
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29533")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def shard_request_ids(rank: int, world: int, n_req_per_rank: int) -> Tuple[int, int]:
    """Weak scaling: rank r serves global requests [r * n, (r + 1) * n).  Returns (first, count)."""
    if not (0 <= rank < world) or n_req_per_rank < 0:
        raise ValueError("bad rank/world")
    return rank * n_req_per_rank, n_req_per_rank


def barrier(device=None) -> None:
    if dist.is_initialized():
        if device is not None and device.type == "cuda":
            dist.barrier(device_ids=[device.index])
        else:
            dist.barrier()


def max_over_ranks(value: float, device=None) -> float:
    """Device-timed durations are reduced with MAX: the job is as slow as its slowest rank."""
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    if not dist.is_initialized():
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_rate(units_this_rank: float, elapsed_ms_this_rank: float, device=None) -> Tuple[float, float]:
    """(units/s over all ranks, max elapsed ms): total units processed by every rank divided by
    the slowest rank's device time."""
    total = sum_over_ranks(units_this_rank, device)
    worst = max_over_ranks(elapsed_ms_this_rank, device)
    return total / (worst * 1e-3), worst
