"""N > 1 path of bench.py on CPU: world size 2, gloo backend (replicas only — no collective on
the data path; the only exchange is the max-over-ranks of the device times)."""
import os
import socket
import sys
from pathlib import Path

import torch.distributed as dist
import torch.multiprocessing as mp

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        local_total_ms = 10.0 * (rank + 1)                     # rank 1 is the slow replica
        total = bench.max_over_ranks(local_total_ms, world, "cpu")
        ms_per_step, value_us = bench.replica_metric(total, steps=5, world=world)
        dist.barrier()
        q.put((rank, total, ms_per_step, value_us, bench.reference_rank_runs(rank)))
    finally:
        dist.destroy_process_group()


def test_replica_bookkeeping_world_size_2_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, total, ms_per_step, value_us, runs_ref in res:
        assert total == 20.0                                   # max over ranks, identical on every rank
        assert ms_per_step == 4.0                              # 20 ms / 5 steps
        assert value_us == 2000.0                              # 2 replicas finish 2 batches per 4 ms step
        assert runs_ref == (rank == 0)                         # reference arm: rank 0 only


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.replica_metric(30.0, 10, 1) == (3.0, 3000.0)


def test_bench_gpus_n_spawns_its_own_ranks():
    """`python bench.py --gpus 2` without torchrun re-executes itself under torch.distributed.run (it used
    to time one replica and print n_gpus 1).  --dry-run keeps the kernels out so this runs on CPU over gloo."""
    import json
    import subprocess
    root = Path(__file__).resolve().parent.parent
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    res = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2", "--dry-run", "--steps", "5"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=root)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, res.stdout                      # rank 0 alone prints
    line = lines[0]
    assert line["n_gpus"] == 2 and line["steps"] == 5
    assert line["ms_per_step"] == 20.0 and line["value"] == 10000.0     # slowest rank: 20 ms per step, 2 replicas
