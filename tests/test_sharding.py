"""`-m "not gpu"`: host logic of the N>1 path -- contiguous point shards, no collective on the data
path; world_size-2 gloo run of the barrier + max-over-ranks timing that bench.py uses."""
import os
import socket

import pytest

from paper_2302_08381_b200.sharding import shard_range


@pytest.mark.parametrize("n", [0, 1, 31, 32, 33, 1000, 100_000, 262_144, 4_000_000])
@pytest.mark.parametrize("world", [1, 2, 3, 4, 8])
def test_shards_partition_the_points(n, world):
    prev = 0
    sizes = []
    for r in range(world):
        a, b = shard_range(n, r, world)
        assert a == prev and a <= b <= n
        if r < world - 1:
            assert b % 32 == 0 or b == n
        prev = b
        sizes.append(b - a)
    assert prev == n
    assert max(sizes) - min(sizes) <= 64      # one tile plus the ragged tail


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = 100_003
    a, b = shard_range(n, rank, world)
    ranges = [None] * world
    dist.all_gather_object(ranges, (a, b))
    dist.barrier()
    t = torch.tensor([10.0 + rank])            # stand-in for this rank's device time
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    cnt = torch.tensor([b - a], dtype=torch.int64)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    q.put((rank, ranges, float(t), int(cnt)))
    dist.destroy_process_group()


def test_two_rank_gloo_run():
    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ranges, tmax, total in res:
        assert ranges[0][0] == 0 and ranges[0][1] == ranges[1][0] and ranges[1][1] == 100_003
        assert tmax == 11.0 and total == 100_003


def test_bench_starts_its_own_ranks():
    """`bench.py --gpus 2` with no launcher in the environment spawns two ranks itself (torch.distributed.run
    on 127.0.0.1); here on the gloo backend with a stub step (--impl stub): one JSON line, from rank 0,
    carrying the max-over-ranks time (rank 1 sleeps twice as long as rank 0)."""
    import json
    import subprocess
    import sys
    from pathlib import Path

    root = Path(__file__).resolve().parent.parent
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, str(root / "bench.py"), "--impl", "stub", "--gpus", "2", "--steps", "20"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["steps"] == 20
    assert line["ms_per_step"] >= 2.0          # rank 1's 2 ms per step, not rank 0's 1 ms
