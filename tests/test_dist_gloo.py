"""N > 1 path on CPU: world_size-2 gloo run of the request sharding and the max-over-ranks
timing that bench.py uses (the data path itself has no collective)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2607_02119_b200 import dist_utils
    r, lr, w = dist_utils.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    first, count = dist_utils.shard_request_ids(rank, world, 512)
    dist_utils.barrier()
    # rank 1 is the slow one: the job's time is ITS time, the job's units are the sum
    elapsed = 10.0 if rank == 0 else 25.0
    rate, worst = dist_utils.whole_job_rate(512 * 100.0, elapsed)
    mx = dist_utils.max_over_ranks(float(rank))
    out[rank] = (first, count, rate, worst, mx)
    dist.destroy_process_group()


def test_two_rank_sharding_and_max_over_ranks():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, 29611, out), nprocs=world, join=True)
    assert out[0][0] == 0 and out[1][0] == 512 and out[0][1] == out[1][1] == 512
    for r in range(world):
        _, _, rate, worst, mx = out[r]
        assert worst == 25.0 and mx == 1.0
        assert abs(rate - (2 * 512 * 100.0) / 0.025) < 1e-6


def _shard_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_2607_02119_b200 import dist_utils
    dist_utils.init("gloo")
    S, R = 9, 6                                    # 9 streams over 2 ranks: 5 + 4 local streams
    base, stride, s_local = dist_utils.stream_shard(rank, world, S)
    full = torch.arange(R * S, dtype=torch.int32).reshape(R, S)      # what an unsharded head would emit
    mine = full[:, base::stride].contiguous()
    assert mine.shape == (R, s_local)
    out[rank] = (base, stride, s_local, dist_utils.all_gather_stream_tokens(mine, S).tolist())
    dist.destroy_process_group()


def test_two_rank_stream_sharded_token_all_gather():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_shard_worker, args=(world, 29613, out), nprocs=world, join=True)
    full = torch.arange(6 * 9, dtype=torch.int32).reshape(6, 9).tolist()
    assert out[0][:3] == (0, 2, 5) and out[1][:3] == (1, 2, 4)
    assert out[0][3] == full and out[1][3] == full


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2607_02119_b200 import dist_utils
    assert dist_utils.env_world()[2] >= 1
    if not dist.is_initialized():
        assert dist_utils.max_over_ranks(3.5) == 3.5
        rate, worst = dist_utils.whole_job_rate(1000.0, 10.0)
        assert worst == 10.0 and abs(rate - 1e5) < 1e-9
