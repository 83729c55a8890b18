"""The N > 1 harness logic of bench.py on CPU: world size 2, gloo, 127.0.0.1 (DESIGN.md section 8:
the path runs as independent replicas, so the only cross-rank steps are the barrier, the MAX of the
timed region over the ranks, and rank 0 printing the one JSON line)."""
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
    dist.barrier()
    got = bench.max_over_ranks(10.0 + rank, dist, "cpu")      # rank r measured 10 + r ms
    out[rank] = got
    dist.destroy_process_group()


def test_max_over_ranks_gloo_world2():
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, 29541, out), nprocs=2, join=True)
        assert dict(out) == {0: 11.0, 1: 11.0}


def test_max_over_ranks_single():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5


def test_reference_arm_under_torchrun_world2():
    """torchrun with two ranks: rank 0 alone times the oracle and prints the line, rank 1 exits 0."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29543", os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1", "--workload", "Tiny"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [json.loads(l) for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = lines[0]
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["unit"] == "particles/s" and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert d["config"]["workload"] == "Tiny"
