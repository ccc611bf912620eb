"""N > 1 host logic on CPU: world_size-2 gloo run of the row sharding and the max-over-ranks / sum bookkeeping that
bench.py does under torchrun (the data path itself has no collective)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n, q):
    sys.path.insert(0, ROOT)
    from paper_2606_17065_b200.sharding import shard_rows
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    b, e = shard_rows(n, rank, world)
    rows = torch.tensor([float(e - b)], dtype=torch.float64)
    t = torch.tensor([1.0 + rank], dtype=torch.float64)    # pretend per-rank elapsed ms
    dist.barrier()
    dist.all_reduce(rows, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    q.put((rank, b, e, rows.item(), t.item()))
    dist.destroy_process_group()


def test_two_rank_row_shards_cover_everything():
    n, world = 1_000_003, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, 29531, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
    assert res[0][1] == 0 and res[0][2] == res[1][1] and res[1][2] == n
    assert res[0][1] % 2 == 0 and res[1][1] % 2 == 0
    assert all(r[3] == n for r in res) and all(r[4] == 2.0 for r in res)


def test_shard_rows_properties():
    from paper_2606_17065_b200.sharding import shard_rows
    for n in (0, 1, 2, 7, 1 << 26, (1 << 26) + 5):
        for world in (1, 2, 3, 8):
            cover = 0
            prev = 0
            for r in range(world):
                b, e = shard_rows(n, r, world)
                assert b == prev and e >= b
                prev = e
                cover += e - b
            assert prev == n and cover == n


def test_bench_spawns_its_own_ranks():
    """`python bench.py --gpus 2` without a launcher must start two ranks itself (torch.distributed.run): the CPU self-test
    mode runs the same launcher and shard bookkeeping over gloo and reports what every rank took of ONE array."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    n = 1_000_003
    p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-launch", "--rows", str(n)],
                       env=env, capture_output=True, text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    line = [ln for ln in p.stdout.splitlines() if ln.startswith("{")][-1]
    r = json.loads(line)
    assert r["n_gpus"] == 2 and r["max_ms"] == 2.0            # two ranks really ran (max over ranks of 1 + rank)
    assert r["shards"][0][0] == 0 and r["shards"][0][1] == r["shards"][1][0] and r["shards"][1][1] == n
    assert r["shards"][1][0] % 2 == 0
