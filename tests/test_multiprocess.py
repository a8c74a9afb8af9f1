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


# ------------------------------------------------------------------ x-slab decomposition plumbing
def test_split_grid_and_local_cases_cover_the_grid():
    """PAPER.md:365 split_grid: contiguous, exhaustive, near-equal slabs; exchange faces only between slabs; physical
    boundary kinds kept on the end ranks; periodic grids wrap."""
    from paper_2504_13750_b200 import inputs as I, slab, binding
    import pytest
    assert slab.split_grid(10, 3) == [(0, 4), (4, 7), (7, 10)]
    with pytest.raises(ValueError):
        slab.split_grid(8, 3)
    case = I.config2(nx=50, ny=12)
    seen = np.zeros(50, int)
    for r in range(4):
        lc, (x0, x1), (left, right) = slab.local_case(case, r, 4)
        seen[x0:x1] += 1
        assert np.array_equal(lc.U, case.U[..., x0:x1]) and lc.grid.n[0] == x1 - x0
        assert lc.grid.bc_lo[0] == (I.BC_REFLECT if r == 0 else binding.BC_EXCHANGE)
        assert lc.grid.bc_hi[0] == (I.BC_OUTFLOW if r == 3 else binding.BC_EXCHANGE)
        assert lc.grid.bc_lo[1] == case.grid.bc_lo[1] and (left, right) == (r - 1 if r else None, r + 1 if r < 3 else None)
    assert (seen == 1).all()
    assert slab.neighbours(0, 3, True) == (2, 1) and slab.neighbours(2, 3, True) == (1, 0) and slab.neighbours(0, 1, True) == (None, None)


def _slab_worker(rank, world, port, periodic, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import torch
    from paper_2504_13750_b200 import slab
    comm = slab.DistComm()
    # reduction slots: bit patterns of non-negative doubles; the int64 MAX is the max of the doubles
    vals = torch.tensor([1.5 + rank, 700.25 - 3 * rank, 0.0], dtype=torch.float64)
    slots = vals.view(torch.int64).clone()
    comm.allreduce_max([slots])
    left, right = slab.neighbours(rank, world, periodic)
    mk = lambda v: torch.full((5,), float(v))
    sends, recvs = [(mk(10 * rank + 1), mk(10 * rank + 2))], [(mk(-1), mk(-1))]
    comm.exchange(sends, recvs, [(left, right)])
    out[rank] = (slots.view(torch.float64).tolist(), recvs[0][0].tolist(), recvs[0][1].tolist())
    dist.barrier()
    dist.destroy_process_group()


def test_slab_communicator_over_gloo():
    """DistComm with world_size 2 and 3 on CPU tensors: exact max all-reduce of the slots; a slab's lo ghosts receive its
    left neighbour's hi columns and vice versa, also when both neighbours are the same rank (2 ranks, periodic)."""
    for world, periodic, port in ((2, False, 29621), (2, True, 29622), (3, True, 29623)):
        mgr = mp.Manager()
        out = mgr.dict()
        mp.spawn(_slab_worker, args=(world, port, periodic, out), nprocs=world, join=True)
        for r in range(world):
            slots, rlo, rhi = out[r]
            assert slots == [1.5 + world - 1, 700.25, 0.0]
            left = r - 1 if r > 0 else (world - 1 if periodic else None)
            right = r + 1 if r < world - 1 else (0 if periodic else None)
            assert rlo == [(10 * left + 2) if left is not None else -1.0] * 5, (world, periodic, r, rlo)
            assert rhi == [(10 * right + 1) if right is not None else -1.0] * 5, (world, periodic, r, rhi)
