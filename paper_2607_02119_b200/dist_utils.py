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


# ---------------------------------------------------------------- stream-sharded heads (W5)
# The alternative sharding for the weight-streaming regime: GPU g holds the head slices of the streams
# {g, g + G, g + 2G, ...} (cfgms_config.stream_base = g, stream_stride = G), every GPU sees all rows, and the
# only exchange per step is an all-gather of n_rows x S_local int32 tokens (<= 32 KB).

def stream_shard(rank: int, world: int, S: int) -> Tuple[int, int, int]:
    """-> (stream_base, stream_stride, S_local) of this rank: streams rank, rank + world, ..."""
    if not (0 <= rank < world) or S < world:
        raise ValueError("need 0 <= rank < world <= S")
    return rank, world, len(range(rank, S, world))


def merge_stream_shards(shards, S: int) -> torch.Tensor:
    """shards[g]: int32 [R][S_local(g)] tokens of rank g (columns = its local streams) -> [R][S]."""
    world = len(shards)
    R = shards[0].shape[0]
    out = torch.empty((R, S), dtype=shards[0].dtype, device=shards[0].device)
    for g, t in enumerate(shards):
        cols = list(range(g, S, world))
        out[:, cols] = t[:, :len(cols)]
    return out


def all_gather_stream_tokens(tokens_local: torch.Tensor, S: int) -> torch.Tensor:
    """The step's one exchange: every rank contributes its [R][S_local] tokens and receives [R][S].
    Ranks with fewer local streams pad to the widest shard (S need not divide the world size)."""
    if not dist.is_initialized():
        return merge_stream_shards([tokens_local], S)
    world, rank = dist.get_world_size(), dist.get_rank()
    widest = len(range(0, S, world))
    R = tokens_local.shape[0]
    mine = torch.full((R, widest), -1, dtype=tokens_local.dtype, device=tokens_local.device)
    mine[:, :tokens_local.shape[1]] = tokens_local
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    return merge_stream_shards(parts, S)


# ---------------------------------------------------------------- device-side token exchange (cfgms_exchange_*)
# The all-gather above is the CPU-testable reference of the exchange; on GPUs the finalize kernel does it itself
# with peer stores into every rank's gather buffer + one flag per destination.  torch.distributed only carries
# the 64-byte CUDA IPC handles at set-up time; no collective runs on the data path.

def exchange_handles(handle: bytes) -> list:
    """Every rank's exchange handle, in rank order (set-up time, any backend)."""
    if len(handle) != 64:
        raise ValueError("a CUDA IPC handle is 64 bytes")
    if not dist.is_initialized():
        return [bytes(handle)]
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, bytes(handle))
    if any(h is None or len(h) != 64 for h in out):
        raise RuntimeError("exchange handle missing from a rank")
    return out


def connect_stream_exchange(ctx, rank: int, world: int) -> None:
    """Create this rank's exchange block and connect it to every peer's (one process per GPU)."""
    handle, base = ctx.exchange_create(world, rank)
    if world == 1:
        ctx.exchange_connect([base])
    else:
        ctx.exchange_connect_ipc(exchange_handles(handle))
