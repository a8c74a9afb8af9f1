"""x-slab decomposition of a uniform grid over several GPUs (split_grid, exchange_halo,
parallel_boundary_conditions, parallel_rhs, parallel_advance_one_step; :452 "results identical").

Plumbing only: every arithmetic step runs in libjanc's kernels through janc_step_part / janc_halo.  What happens here is
what the paper does with jax.lax.ppermute inside pmap: per RK stage each slab sends the 3 columns next to its interior
x sides to its neighbours, and the max(|u_d| + c) reductions (alpha of eq 4.11, the CFL step) are max-all-reduced so that
every slab uses the values of the undecomposed grid.  The reduction slots hold non-negative doubles as bit patterns,
which order like integers: an int64 MAX all-reduce is exact, so the decomposed run reproduces the single-grid run bit
for bit (tested).

Two communicators with the same interface:
  DistComm   one process per GPU, torch.distributed (NCCL on GPUs; gloo for the CPU test of the plumbing);
  LocalComm  all slabs in one process on one GPU, advanced in lockstep part by part (how the decomposition is tested
             where only one GPU is available; no kernel ever waits on another).
"""
from __future__ import annotations

import numpy as np

from . import binding, inputs as I


def split_grid(nx, world):
    """PAPER.md:365 split_grid: contiguous column ranges [x0, x1) per rank, sizes differing by at most one; every slab
    needs at least 3 columns (the halo depth)."""
    base, extra = divmod(int(nx), int(world))
    if base < I.NG:
        raise ValueError(f"{nx} columns cannot be split into {world} slabs of at least {I.NG} columns")
    out, x = [], 0
    for r in range(world):
        w = base + (1 if r < extra else 0)
        out.append((x, x + w))
        x += w
    return out


def neighbours(rank, world, periodic):
    """(left, right) rank of a slab or None at a physical boundary (physical BCs on the end ranks only)."""
    left = rank - 1 if rank > 0 else (world - 1 if periodic and world > 1 else None)
    right = rank + 1 if rank < world - 1 else (0 if periodic and world > 1 else None)
    return left, right


def local_case(case, rank, world):
    """The slab of `case` (uniform grid) owned by `rank`: its columns, with exchange faces on interior x sides."""
    g = case.grid
    assert g.n_patches == 0, "slab decomposition is for uniform grids"
    x0, x1 = split_grid(g.n[0], world)[rank]
    periodic = g.bc_lo[0] == I.BC_PERIODIC
    left, right = neighbours(rank, world, periodic)
    lo, hi = list(g.bc_lo), list(g.bc_hi)
    if world > 1:
        if left is not None:
            lo[0] = binding.BC_EXCHANGE
        if right is not None:
            hi[0] = binding.BC_EXCHANGE
    n = (x1 - x0,) + tuple(g.n[1:])
    lg = I.Grid(g.ndim, n, g.dx, tuple(lo), tuple(hi))
    U = np.ascontiguousarray(case.U[..., x0:x1])
    T = np.ascontiguousarray(case.T[..., x0:x1])
    return I.Case(f"{case.name}_slab{rank}of{world}", lg, case.mech, U, T, case.cfl, case.nsteps), (x0, x1), (left, right)


class DistComm:
    """torch.distributed communicator: one slab per process."""

    def __init__(self):
        import torch.distributed as dist
        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()

    def allreduce_max(self, slots):
        for t in slots:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)

    def exchange(self, sends, recvs, nbrs):
        """sends / recvs: per local slab (lo, hi) buffers; nbrs: per local slab (left, right) ranks.  My lo columns go
        to my left neighbour's hi ghosts and vice versa.  Messages between one pair of ranks match in posting order, so
        sends are posted lo-then-hi and receives hi-then-lo: with two ranks on a periodic grid (left == right) the
        peer's first message, its lo columns, then lands in my hi ghosts."""
        (send_lo, send_hi), (recv_lo, recv_hi), (left, right) = sends[0], recvs[0], nbrs[0]
        P2P, ops = self.dist.P2POp, []
        if left is not None:
            ops.append(P2P(self.dist.isend, send_lo, left))
        if right is not None:
            ops.append(P2P(self.dist.isend, send_hi, right))
        if right is not None:
            ops.append(P2P(self.dist.irecv, recv_hi, right))
        if left is not None:
            ops.append(P2P(self.dist.irecv, recv_lo, left))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()


class LocalComm:
    """All slabs in this process: reductions and exchanges are tensor operations between them."""

    def __init__(self, world):
        self.rank, self.world = 0, world

    def allreduce_max(self, slots):
        m = slots[0].clone()
        for t in slots[1:]:
            m = m.maximum(t)
        for t in slots:
            t.copy_(m)

    def exchange(self, sends, recvs, nbrs):
        for r, (left, right) in enumerate(nbrs):
            if left is not None:
                recvs[r][0].copy_(sends[left][1])       # my lo ghosts <- left neighbour's hi columns
            if right is not None:
                recvs[r][1].copy_(sends[right][0])      # my hi ghosts <- right neighbour's lo columns


class SlabRun:
    """parallel_advance_one_step over the slabs this process owns (one with DistComm, all with
    LocalComm)."""

    def __init__(self, case, comm, device=0, ranks=None, options=None, local=None):
        """case: the undecomposed case (every owned slab is cut out of it), or None with local = [(slab case with its
        exchange faces set, (x0, x1), (left, right))] when the caller builds its slab directly (weak-scaling runs)."""
        import torch
        self.torch, self.comm, self.case = torch, comm, case
        self.ranks = list(ranks) if ranks is not None else ([comm.rank] if isinstance(comm, DistComm) else list(range(comm.world)))
        self.solvers, self.ranges, self.nbrs, self.bufs = [], [], [], []
        for q, r in enumerate(self.ranks):
            lc, rng, nb = local[q] if local is not None else local_case(case, r, comm.world)
            s = binding.Solver(lc.grid, lc.mech, device=device, options=options)
            s.set_state(lc.U, lc.T)
            n = s.halo_doubles()
            mk = lambda: torch.empty(n, dtype=torch.float64, device=f"cuda:{device}")
            self.solvers.append(s); self.ranges.append(rng); self.nbrs.append(nb)
            self.bufs.append(((mk(), mk()), (mk(), mk())))      # (send lo, send hi), (recv lo, recv hi)
        self.slots = [s.slots_tensor() for s in self.solvers]

    def _all(self, part, stage=0, **kw):
        for s in self.solvers:
            s.step_part(part, stage, **kw)

    def _sync_streams(self):
        # the communicator's copies / collectives run on torch's current stream, the kernels on the solvers' stream:
        # both are torch's current stream here (binding.Solver default), so stream order is program order
        pass

    def step(self, nsteps, cfl=0.0, dt=0.0, chem=True):
        B = binding
        for _ in range(nsteps):
            self._all(B.PART_PRIM, 0)
            self.comm.allreduce_max(self.slots)
            self._all(B.PART_DT, 0, cfl=cfl, dt=dt)
            for stage in range(3):
                if stage > 0:
                    self._all(B.PART_PRIM, stage)
                    self.comm.allreduce_max(self.slots)
                self._all(B.PART_GHOST, stage)
                for s, ((slo, shi), _), (left, right) in zip(self.solvers, self.bufs, self.nbrs):
                    if left is not None:
                        s.halo(stage, 0, slo, unpack=False)
                    if right is not None:
                        s.halo(stage, 1, shi, unpack=False)
                self.comm.exchange([b[0] for b in self.bufs], [b[1] for b in self.bufs], self.nbrs)
                for s, (_, (rlo, rhi)), (left, right) in zip(self.solvers, self.bufs, self.nbrs):
                    if left is not None:
                        s.halo(stage, 0, rlo, unpack=True)
                    if right is not None:
                        s.halo(stage, 1, rhi, unpack=True)
                self._all(B.PART_FLUX, stage)
            self._all(B.PART_SOURCE, 0, chem=chem)

    def last_dt(self):
        return self.solvers[0].last_dt()

    def gather_local(self):
        """[(x0, x1, U_local, T_local)] of the slabs this process owns (host arrays)."""
        out = []
        for s, (x0, x1) in zip(self.solvers, self.ranges):
            U, T = s.get_state()
            assert s.status == 0, "device flag raised"
            out.append((x0, x1, U, T))
        return out

    def assemble(self):
        """The whole grid's state from a LocalComm run."""
        U = np.empty_like(self.case.U); T = np.empty_like(self.case.T)
        for x0, x1, Ul, Tl in self.gather_local():
            U[..., x0:x1] = Ul; T[..., x0:x1] = Tl
        return U, T

    def close(self):
        for s in self.solvers:
            s.close()
