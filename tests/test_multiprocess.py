"""N > 1 paths on CPU (gloo, world_size 2): replicas-only sharding of bench.py -- per-rank
seeds, the max-over-ranks timing reduction, and the reference arm under torchrun (rank 0 alone prints)."""
import json
import os
import subprocess
import sys

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    case = bench.make_case("cfg0", rank)
    vals = bench.max_over_ranks([1.0 + rank, 10.0 - rank], "cpu", world)
    out[rank] = (float(case.T.sum()), vals)
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_have_own_seeds_and_times_are_max_over_ranks():
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, 29611, out), nprocs=2, join=True)
    assert out[0][0] != out[1][0]                    # different seeded noise per replica
    assert out[0][1] == out[1][1] == [2.0, 10.0]     # max over ranks, identical on every rank


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", "29612", os.path.join(ROOT, "bench.py"),
           "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "1", "--workload", "cfg0"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0
    assert np.isfinite(d["ms_per_step"])
