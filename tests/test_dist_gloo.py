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


def _exchange_worker(rank, world, port, out):
    """Host logic of the device-side token exchange plus a CPU model of its flag protocol: each rank scatters its
    stream columns of step e into half e & 1 of EVERY rank's gather buffer, then raises flags[q][rank] = e; a rank
    consumes step e once all its flags reached e.  A rank can only start step e + 1 after consuming step e (its
    next input needs everyone's tokens), which is what makes two halves enough — the model checks exactly that
    with skewed ranks over many steps."""
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import time
    from paper_2607_02119_b200 import dist_utils
    dist_utils.init("gloo")
    # 1. set-up: 64-byte handles gathered in rank order
    mine = bytes([rank]) * 64
    handles = dist_utils.exchange_handles(mine)
    assert handles == [bytes([q]) * 64 for q in range(world)]
    try:
        dist_utils.exchange_handles(b"short")
        raise AssertionError("a malformed handle must be refused")
    except ValueError:
        pass
    # 2. the protocol, on shared host memory standing in for the peer-mapped blocks
    bufs, flags = out["bufs"], out["flags"]          # [world][2][R][S] tokens, [world][world] epochs
    S, R = bufs.shape[3], bufs.shape[2]
    base, stride, _ = dist_utils.stream_shard(rank, world, S)
    tok = lambda e, r, s: e * 1000 + r * 16 + s
    ok = True
    for e in range(1, 41):
        if (e * 7 + rank * 3) % 5 == 0:
            time.sleep(0.002)                        # skew the ranks
        for q in range(world):                       # scatter: peer stores
            for s_ in range(base, S, stride):
                for r in range(R):
                    bufs[q, e & 1, r, s_] = tok(e, r, s_)
        for q in range(world):                       # publish (after the stores)
            flags[q, rank] = e
        t0 = time.time()
        while int(flags[rank].min()) < e:            # wait: every rank's step e has landed here
            assert time.time() - t0 < 20
        got = bufs[rank, e & 1].clone()
        want = torch.tensor([[tok(e, r, s_) for s_ in range(S)] for r in range(R)], dtype=got.dtype)
        ok = ok and bool(torch.equal(got, want))
        dist_utils.barrier()                         # stands in for "the next step needs everyone's tokens"
    out[rank] = ok
    dist.destroy_process_group()


def _exchange_worker_entry(rank, world, port, out, bufs, flags):
    box = {"bufs": bufs, "flags": flags}
    _exchange_worker(rank, world, port, box)
    out[rank] = box[rank]


def test_two_rank_exchange_handles_and_flag_protocol():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    # tensors in shared memory travel to the spawned ranks as handles; results come back through the manager
    bufs = torch.zeros((world, 2, 3, 5), dtype=torch.int32).share_memory_()
    flags = torch.zeros((world, world), dtype=torch.int64).share_memory_()
    mp.spawn(_exchange_worker_entry, args=(world, 29617, out, bufs, flags), nprocs=world, join=True)
    assert out[0] is True and out[1] is True


def test_bench_spawns_its_own_ranks_when_asked_for_more_than_one_gpu():
    """`python bench.py --gpus 2` typed WITHOUT torchrun must run two ranks (it re-launches itself the way the driver
    launches it: one process per GPU, rendezvous on 127.0.0.1, a free port) and report n_gpus = 2.  --dry-ranks takes
    the kernels out (gloo, no GPU) and keeps the plumbing: rendezvous, world == --gpus, barrier, the whole-job
    reduction of the timed region (rank r 'serves' 10 requests in 1 + r ms -> 20 requests / 2 ms)."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-ranks"], env=env,
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(l) for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout                                   # rank 0 alone prints
    assert lines[0]["n_gpus"] == 2 and lines[0]["worst_ms"] == 2.0 and lines[0]["value"] == 10000.0
    # a world that does not match --gpus is an error, not a line that claims n_gpus = 1
    bad = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry-ranks"],
                         env=dict(env, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0"), capture_output=True, text=True, timeout=120)
    assert bad.returncode != 0 and "WORLD_SIZE" in (bad.stderr + bad.stdout)


def test_bench_spawn_command_is_the_drivers_launch():
    import importlib.util
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    spec = importlib.util.spec_from_file_location("bench_mod", os.path.join(root, "bench.py"))
    bench = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(bench)
    cmd = bench.spawn_command(4, ["--gpus", "4", "--steps", "7"], 12345)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=4" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "12345"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "7"] and cmd[-5].endswith("bench.py")
    p = bench.free_port()
    assert 1024 < p < 65536
