"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only — the one collective is the max over
ranks of the device times; the reference arm runs on rank 0 alone."""
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
    vals = bench.max_over_ranks([10.0 + rank, 5.0 - rank, 7.0], torch.device("cpu"), world)
    assert bench.replica_seed(rank) != bench.replica_seed(rank + 1)
    if rank == 0:
        json.dump(vals, open(out, "w"))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_gloo(tmp_path):
    out = str(tmp_path / "vals.json")
    mp.spawn(_worker, args=(2, 29653, out), nprocs=2, join=True)
    assert json.load(open(out)) == [11.0, 5.0, 7.0]


def test_reference_arm_runs_on_rank0_only(tmp_path):
    """torchrun --nproc-per-node 2 bench.py --impl reference: rank 0 prints the JSON line, rank 1 exits 0 without work."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29654", os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "cfg1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
