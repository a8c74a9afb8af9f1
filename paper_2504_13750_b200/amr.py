"""Advance / regrid cycles of a two-level block list (JAX-AMR's outer loop: "updating refinement layer" every
few steps, :127-141 Algorithm 1, the dynamic update of N_max).

Plumbing only: the time steps are janc_step, the regridding is janc_regrid_plan / janc_regrid_fill (kernels of
csrc/ghost.cuh + the block-list rebuild in janc.cu); this module keeps the loop, the block list and the memory.

What N_max means here.  In the paper N_{i,max} is the declared number of blocks of layer i: JAX compiles for a fixed
batch size, so redundant blocks exist in memory AND are computed, and Algorithm 1 doubles / halves N_max to limit both
the waste and the recompilations.  The kernels of this library take the number of patches at run time and the
specialised kernels are cached per mechanism, so a regridded list costs neither a compilation nor redundant blocks; what
is worth keeping fixed across regrids is the device memory.  N_max is therefore the CAPACITY of the workspace in level-1
blocks: Algorithm 1 decides when it is re-allocated, every context is created for the valid list only and bound to that
workspace.  Reading B13: the printed second condition, "(N_valid + 1) < 2.5 N_max", holds whenever the first
one fails; it is read as (N_valid + 1) < N_max / 2.5, which gives the hysteresis the text describes.
"""
from __future__ import annotations

import numpy as np

from . import binding, inputs as I


def update_n_max(n_valid, n_max):
    """Algorithm 1 with reading B13; applied until it is stable (one regrid may add many blocks)."""
    n_max = max(1, int(n_max))
    while n_valid + 1 > n_max:
        n_max *= 2
    while n_max > 1 and (n_valid + 1) * 2.5 < n_max:
        n_max //= 2
    return n_max


class AmrRun:
    """case: a two-level block list (inputs.Case with blocks; the level-0 patches first, tiling the domain).
    Every `every` steps the level-1 blocks are rebuilt from the density-jump criterion `thr` with `nbuf` buffer cells
    (PAPER.md:73-75); blocks that survive keep their data, new ones are injected from their parent."""

    def __init__(self, case, thr, nbuf, every, device=0, options=None, n_max=1):
        import torch
        self.torch, self.device, self.options = torch, device, options
        self.mech, self.grid0 = case.mech, case.grid
        self.thr, self.nbuf, self.every = float(thr), int(nbuf), int(every)
        self.n0 = int((np.asarray(case.blocks.level) == 0).sum())
        self.blocks = I.Blocks(np.asarray(case.blocks.level, np.int32).copy(), np.asarray(case.blocks.nbr, np.int32).copy(),
                               np.asarray(case.blocks.parent, np.int32).copy())
        self.n_max = update_n_max(len(self.blocks.level) - self.n0, n_max)
        self.workspace = None
        self.allocations = 0            # how often the workspace was (re-)allocated
        self.regrids = 0
        self.since = 0
        self.solver = None
        self._bind(case.U, case.T)

    def _grid(self, n_patches):
        g = self.grid0
        return I.Grid(g.ndim, g.n, g.dx, g.bc_lo, g.bc_hi, n_patches=n_patches, n_levels=2, ratio=2)

    def _capacity_bytes(self):
        # the workspace of a list with n0 + N_max patches, asked of the library itself
        return binding.workspace_bytes_for(self._grid(self.n0 + self.n_max), self.mech, self.device, self.options)

    def _bind(self, U, T):
        if self.solver is not None:
            self.solver.close()
        need = self._capacity_bytes() + 256
        if self.workspace is None or self.workspace.numel() != need:
            self.workspace = None
            self.workspace = self.torch.empty(need, dtype=self.torch.uint8, device=f"cuda:{self.device}")
            self.allocations += 1
        self.solver = binding.Solver(self._grid(len(self.blocks.level)), self.mech, self.blocks, device=self.device,
                                     options=self.options, workspace=self.workspace)
        self.solver.set_state(U, T)

    @property
    def n_valid(self):
        return len(self.blocks.level) - self.n0

    def regrid(self):
        """updating refinement layer: new list + data on the device, capacity by Algorithm 1, new context on the (possibly
        re-allocated) workspace."""
        level, nbr, parent, U, T = self.solver.regrid(self.thr, self.nbuf, device=True)
        self.blocks = I.Blocks(level, nbr, parent)
        self.n_max = update_n_max(self.n_valid, self.n_max)
        self._bind(U, T)          # U, T are tensors of their own: the old context's workspace may be overwritten
        self.regrids += 1
        self.since = 0

    def step(self, nsteps, cfl, chem=True, crossover=False):
        """Advance nsteps (level-0 steps), regridding after every `every` of them; returns the time advanced."""
        t = 0.0
        for _ in range(int(nsteps)):
            t += self.solver.step(1, cfl=cfl, chem=chem, crossover=crossover)
            assert self.solver.status == 0, "device flag raised"
            self.since += 1
            if self.since >= self.every:
                self.regrid()
        return t

    def state(self):
        return self.solver.get_state()

    def close(self):
        if self.solver is not None:
            self.solver.close()
            self.solver = None
        self.workspace = None
