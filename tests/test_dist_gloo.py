"""world_size-2 gloo tests (CPU) of the N>1 plumbing: replicas only, no data-path collective."""
import os

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_08446_b200 import dist as D


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, lr, w = D.init("gloo")
    assert (r, w) == (rank, world)
    D.barrier()
    # rank r "processes" 64 sequences per step for 10 steps in (1 + r) seconds
    thr, t = D.whole_job_throughput(64 * 10, 1.0 + rank)
    shard = D.shard_sequences(129, rank, world)
    q.put((rank, thr, t, D.replica_seed(2000, rank), len(shard), shard[0], shard[-1]))
    D.barrier()
    dist.destroy_process_group()


def test_two_rank_replicas_aggregate_over_max_time():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 400
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    res = sorted(q.get(timeout=120) for _ in range(2))
    [p.join(timeout=60) for p in ps]
    assert all(p.exitcode == 0 for p in ps)
    for rank, thr, t, seed, n, lo, hi in res:
        assert t == 2.0 and thr == (640 + 640) / 2.0           # whole-job units / max-over-ranks time
    assert res[0][3] != res[1][3]                               # replicas draw different batches
    assert (res[0][4], res[0][5], res[0][6]) == (65, 0, 64) and (res[1][4], res[1][5], res[1][6]) == (64, 65, 128)


def test_single_process_defaults():
    assert D.env_world()[2] >= 1
    assert D.max_over_ranks(3.5) == 3.5 and D.shard_sequences(10, 0, 1) == list(range(10))


def test_bench_gpus_n_starts_n_ranks_itself():
    """`bench.py --gpus 2` without a torchrun environment must start the two ranks itself (one process per GPU on the
    GPU box; gloo here) and rank 0 must report n_gpus = 2."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    p = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--launch-check"], env=env, capture_output=True,
                       text=True, timeout=300)
    assert p.returncode == 0, p.stderr[-2000:]
    line = [json.loads(ln) for ln in p.stdout.splitlines() if ln.startswith("{")]
    assert len(line) == 1 and line[0] == {"launch_check": True, "n_gpus": 2, "world_size": 2, "requested": 2}
