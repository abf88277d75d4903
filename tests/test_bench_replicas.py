"""bench.py under torchrun (N > 1): replicas only, no data-path collective.  CPU, gloo, world size 2:
the aggregation that turns per-rank measurements into the job's line, and the reference arm's rank discipline."""
import json
import os
import subprocess
import sys

import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times = (1.0 + rank, 5.0 - rank, 0.25 * (rank + 1))           # rank 1 is slower on the first and third
    counts = (1000 + rank, 10 * (rank + 1), 7, 3 + rank, 50)
    t, c = bench.aggregate_replicas(dist, times, counts, "cpu")
    dist.barrier()
    out[rank] = (t, c)
    dist.destroy_process_group()


def test_replica_aggregation_is_max_of_times_and_sum_of_work():
    world, port = 2, 29517
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        t, c = res[rank]
        assert t == (2.0, 5.0, 0.5)
        assert c == (2001, 30, 14, 7, 100)


def test_reference_arm_prints_one_line_from_rank_zero_only():
    env = dict(os.environ, OMP_NUM_THREADS="2")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29519", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0"]
    p = subprocess.run(cmd, capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert p.returncode == 0, p.stderr[-2000:]
    lines = [l for l in p.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["unit"] == "evals/s"
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["n_live"] == 1000 and d["config"]["n_delete"] == 500
