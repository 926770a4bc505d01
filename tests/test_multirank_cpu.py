"""N > 1 host logic on CPU (gloo, world_size 2).  The path is "replicas only" (BASELINE.json north_star says
one GPU; every rank runs an independent replica, no data-path collective), so what there is to test is bench.py's aggregation
(time = max over ranks, work = sum over ranks) and that only rank 0 of a torchrun launch prints the reference arm's line."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    times, counts = bench.aggregate_over_ranks(dist, [10.0 + rank, 5.0 - rank, 0.0], [100 * (rank + 1), 7], torch.device("cpu"))
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        with open(out, "w") as f:
            json.dump({"times": times, "counts": counts}, f)


def test_aggregate_over_ranks_gloo(tmp_path):
    out = str(tmp_path / "agg.json")
    mp.spawn(_worker, args=(2, 29731, out), nprocs=2, join=True)
    r = json.load(open(out))
    assert r["times"] == [11.0, 5.0, 0.0]        # max over ranks
    assert r["counts"] == [300, 14]              # sum over ranks


def test_aggregate_single_rank():
    sys.path.insert(0, ROOT)
    import bench
    t, c = bench.aggregate_over_ranks(None, [1.5, 2.5], [3], torch.device("cpu"))
    assert t == [1.5, 2.5] and c == [3]


def test_reference_arm_under_torchrun_prints_one_line():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29733", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
           "--workload", "plummer_2p13", "--ref-groups", "64"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0 and d["cpu_baseline"]["kind"] == "oracle"
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["config"]["workload"] == "plummer_2p13"
