// ghost.cuh -- batched ghost fill over block lists + average-down.
// PAPER.md:295 (3 ghost layers), :329 (boundary_conditions), :97, :117, :213 (get_ghost_block),
// :215 (update_physical_boundary), :115 (one-to-four injection), :116/:188 (four-to-one mean).
// Readings A14, A15, A19, A21.  Fills U (nvar fields) and the primitives T, p, vel.
#pragma once
#include "common.cuh"

#define GHOST_FPT 4

// grid: (ceil(nf*3*amax / 256), np); only patches with level == lev act (level 0 must be complete
// before level 1 injects from its padded parent).
__global__ void __launch_bounds__(256) k_ghost(Params P, double *__restrict__ U, int lev, int amax) {
  const int patch = blockIdx.y;
  if (P.level[patch] != lev) return;
  const int nf = 2 * P.ndim;
  const int nfield = P.nvar + 2 + P.ndim;          // U components, T, p, u_d
  const int ngrp = (nfield + GHOST_FPT - 1) / GHOST_FPT;   // a thread copies GHOST_FPT fields of one ghost cell
  // 32-bit index arithmetic: one patch has far fewer than 2^31 (ghost cell, field group) items
  unsigned idx = blockIdx.x * blockDim.x + threadIdx.x;
  const unsigned ncellf = (unsigned)(nf * JANC_NG * amax);
  if (idx >= ncellf * (unsigned)ngrp) return;
  const int grp = (int)(idx / ncellf);
  idx -= (unsigned)grp * ncellf;
  const int f = (int)(idx / (unsigned)(amax * JANC_NG));
  const int r_ = (int)(idx - (unsigned)(f * amax * JANC_NG));
  // x faces: the 3 layers are contiguous in memory, so the layer index runs fastest (one 32-byte
  // sector per ghost row instead of three); y / z faces: x runs fastest
  const int t = (f >> 1) == 0 ? r_ / JANC_NG : r_ % amax;
  const int g = ((f >> 1) == 0 ? r_ % JANC_NG : r_ / amax) + 1;
  const int d = f >> 1, side = f & 1;
  const int e1 = d == 0 ? 1 : 0;            // fastest tangential dim
  const int e2 = d == 2 ? 1 : 2;            // slowest tangential dim
  if (t >= P.n[e1] * P.n[e2]) return;
  int dst[3], src[3];
  dst[e1] = t % P.n[e1];
  dst[e2] = t / P.n[e1];
  dst[d] = side == 0 ? -g : P.n[d] - 1 + g;
  src[0] = dst[0]; src[1] = dst[1]; src[2] = dst[2];
  const int kind = P.fkind[patch * nf + f];
  const int bc = side == 0 ? P.bc_lo[d] : P.bc_hi[d];
  if (kind == FK_PHYSICAL && bc == 3) return;      // exchange face: filled by k_halo from the neighbouring slab's buffer
  int q = patch;
  bool flip = false;
  if (kind == FK_NEIGHBOUR || (kind == FK_PHYSICAL && bc == 0 /*periodic*/)) {
    if (kind == FK_NEIGHBOUR) q = P.nbr[patch * nf + f];
    src[d] = side == 0 ? P.n[d] - g : g - 1;
  } else if (kind == FK_PHYSICAL && bc == 1 /*reflect*/) {
    src[d] = side == 0 ? g - 1 : P.n[d] - g;
    flip = true;
  } else if (kind == FK_PHYSICAL) {       /*outflow*/
    src[d] = side == 0 ? 0 : P.n[d] - 1;
  } else {                                  /*coarse parent, piecewise-constant injection*/
    const int *par = P.parent + patch * (1 + P.ndim);
    q = par[0];
    for (int e = 0; e < P.ndim; e++) src[e] = floordiv_i(par[1 + e] * P.n[e] + dst[e], P.ratio);
  }
  const long long di = (long long)patch * P.pc + cell_index(P, dst[0], dst[1], dst[2]);
  const long long si = (long long)q * P.pc + cell_index(P, src[0], src[1], src[2]);
  const long long cd = di - (long long)patch * P.pc, cs = si - (long long)q * P.pc;
  const int f1 = min(nfield, (grp + 1) * GHOST_FPT);
  for (int fld = grp * GHOST_FPT; fld < f1; fld++) {
    if (fld < P.nvar) {
      double val = U[((long long)q * P.nvar + fld) * P.pc + cs];
      if (flip && fld == 1 + d) val = -val;
      U[((long long)patch * P.nvar + fld) * P.pc + cd] = val;
    } else if (fld == P.nvar) {
      P.T[di] = P.T[si];
    } else if (fld == P.nvar + 1) {
      P.p[di] = P.p[si];
    } else {
      const int e = fld - P.nvar - 2;
      double val = P.vel[(long long)e * P.np * P.pc + si];
      if (flip && e == d) val = -val;
      P.vel[(long long)e * P.np * P.pc + di] = val;
    }
  }
}

// Average-down: every level-1 patch writes the mean of its ratio^ndim children cells into the covered
// cells of its parent.  grid: (ceil(nvar*coarse cells per fine patch / 256), np).
__global__ void __launch_bounds__(256) k_average_down(Params P, double *__restrict__ U) {
  const int patch = blockIdx.y;
  if (P.level[patch] == 0) return;
  const int r = P.ratio;
  const int rr[3] = {r, P.ndim > 1 ? r : 1, P.ndim > 2 ? r : 1};
  const int m[3] = {P.n[0] / rr[0], P.n[1] / rr[1], P.n[2] / rr[2]};
  const int nc = m[0] * m[1] * m[2];
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= nc * P.nvar) return;
  const int v = idx / nc;
  int c = idx % nc;
  const int i = c % m[0], j = (c / m[0]) % m[1], k = c / (m[0] * m[1]);
  const int *par = P.parent + patch * (1 + P.ndim);
  const int q = par[0];
  int off[3] = {0, 0, 0};
  for (int e = 0; e < P.ndim; e++) off[e] = par[1 + e] * m[e];
  const double *src = U + ((long long)patch * P.nvar + v) * P.pc;
  double s = 0.0;
  for (int kk = 0; kk < rr[2]; kk++)
    for (int jj = 0; jj < rr[1]; jj++)
      for (int ii = 0; ii < rr[0]; ii++) s += src[cell_index(P, i * rr[0] + ii, j * rr[1] + jj, k * rr[2] + kk)];
  U[((long long)q * P.nvar + v) * P.pc + cell_index(P, off[0] + i, off[1] + j, off[2] + k)] = s * (1.0 / (rr[0] * rr[1] * rr[2]));
}


// x-slab decomposition (split_grid / exchange_halo): the 3 interior columns next to x side `side`
// of every field (U components, T, p, u_d) <-> a contiguous buffer [field][3][nz][ny].  pack: interior -> buffer (what
// the neighbouring slab needs); unpack: buffer -> the ghost columns of that side.  Uniform grid (one patch) only.
__global__ void __launch_bounds__(256) k_halo(Params P, double *__restrict__ U, double *__restrict__ buf, int side, int unpack) {
  const int nfield = P.nvar + 2 + P.ndim;
  const int rows = P.n[1] * P.n[2];
  const long long total = (long long)nfield * JANC_NG * rows;
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= total) return;
  const int r = (int)(idx % rows), g = (int)((idx / rows) % JANC_NG), fld = (int)(idx / ((long long)rows * JANC_NG));
  const int j = r % P.n[1], k = r / P.n[1];
  // pack: lo side sends columns 0..2, hi side columns n-3..n-1; unpack: lo ghosts -3..-1, hi ghosts n..n+2
  const int i = unpack ? (side == 0 ? -JANC_NG + g : P.n[0] + g) : (side == 0 ? g : P.n[0] - JANC_NG + g);
  const long long ci = cell_index(P, i, j, k);
  double *arr = fld < P.nvar ? U + (long long)fld * P.pc : fld == P.nvar ? P.T : fld == P.nvar + 1 ? P.p : P.vel + (long long)(fld - P.nvar - 2) * P.np * P.pc;
  if (unpack) arr[ci] = buf[idx];
  else buf[idx] = arr[ci];
}

// ------------------------------------------------------------------------------------------------ regridding kernels
// PAPER.md:73-75 (criterion mask + buffer cells -> blocks to refine), :175-184; reading B12.
// mark[p][padded cell] (bytes) for the n0 level-0 patches; the ghost layers of rho must be filled (k_ghost, level 0).
__global__ void __launch_bounds__(256) k_regrid_mark(Params P, const double *__restrict__ U, unsigned char *mark, double thr) {
  const int patch = blockIdx.y;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ncell) return;
  const int i = (int)(t % P.n[0]);
  const long long r = t / P.n[0];
  const int j = (int)(r % P.n[1]), k = (int)(r / P.n[1]);
  const long long id = cell_index(P, i, j, k);
  const double *rho = U + (long long)patch * P.nvar * P.pc;
  double g = 0.0;
  for (int d = 0; d < P.ndim; d++) g = fmax(g, fabs(rho[id + P.st[d]] - rho[id - P.st[d]]) / (2.0 * rho[id]));
  mark[(long long)patch * P.pc + id] = g > thr;
}

// the mark of cell (c[0], c[1], c[2]) of level-0 patch p, where each coordinate may lie one cell outside the patch: hop
// through the same-level neighbour lists, highest direction first (periodic sides of a single patch wrap onto itself;
// beyond a wall / outflow side there is nothing to refine)
__device__ __forceinline__ int regrid_mark_at(const Params &P, const unsigned char *mark, int p, int c0, int c1, int c2) {
  int c[3] = {c0, c1, c2};
  for (int d = P.ndim - 1; d >= 0; d--) {
    if (c[d] >= 0 && c[d] < P.n[d]) continue;
    const int side = c[d] < 0 ? 0 : 1;
    int q = P.nbr[p * 2 * P.ndim + 2 * d + side];
    if (q < 0 && (side == 0 ? P.bc_lo[d] : P.bc_hi[d]) == 0) q = p;
    if (q < 0) return 0;
    p = q;
    c[d] = side == 0 ? P.n[d] - 1 : 0;
  }
  return mark[(long long)p * P.pc + cell_index(P, c[0], c[1], c[2])];
}

// one pass of the one-cell box dilation: out = OR of the 3^ndim neighbourhood of in
__global__ void __launch_bounds__(256) k_regrid_dilate(Params P, const unsigned char *in, unsigned char *out) {
  const int patch = blockIdx.y;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ncell) return;
  const int i = (int)(t % P.n[0]);
  const long long r = t / P.n[0];
  const int j = (int)(r % P.n[1]), k = (int)(r / P.n[1]);
  int v = 0;
  for (int dk = (P.ndim > 2 ? -1 : 0); dk <= (P.ndim > 2 ? 1 : 0); dk++)
    for (int dj = (P.ndim > 1 ? -1 : 0); dj <= (P.ndim > 1 ? 1 : 0); dj++)
      for (int di = -1; di <= 1; di++) v |= regrid_mark_at(P, in, patch, i + di, j + dj, k + dk);
  out[(long long)patch * P.pc + cell_index(P, i, j, k)] = (unsigned char)v;
}

// flags[p][sub-region] = 1 if the sub-region holds a marked cell (sub index: x bit 0, y bit 1, z bit 2)
__global__ void __launch_bounds__(256) k_regrid_flags(Params P, const unsigned char *mark, int *flags) {
  const int patch = blockIdx.y;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ncell) return;
  const int i = (int)(t % P.n[0]);
  const long long r = t / P.n[0];
  const int j = (int)(r % P.n[1]), k = (int)(r / P.n[1]);
  if (mark[(long long)patch * P.pc + cell_index(P, i, j, k)]) {
    const int s = (i >= P.n[0] / 2 ? 1 : 0) + (P.ndim > 1 && j >= P.n[1] / 2 ? 2 : 0) + (P.ndim > 2 && k >= P.n[2] / 2 ? 4 : 0);
    flags[patch * (1 << P.ndim) + s] = 1;
  }
}

// data of the regridded list in the interior layout: src[p] >= 0: copy of old patch src[p]; else one-to-four injection
// of sub-region sub[p] of parent par[p]; T likewise.  grid: (cells, new patches)
__global__ void __launch_bounds__(256) k_regrid_fill(Params P, const double *__restrict__ U, const int *src, const int *par, const int *sub,
                                                     double *Unew, double *Tnew) {
  const int p = blockIdx.y;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ncell) return;
  const int i = (int)(t % P.n[0]);
  const long long r = t / P.n[0];
  const int j = (int)(r % P.n[1]), k = (int)(r / P.n[1]);
  int q = src[p];
  long long sid;
  if (q >= 0) sid = cell_index(P, i, j, k);
  else {
    q = par[p];
    const int s = sub[p];
    sid = cell_index(P, ((s & 1) * P.n[0] + i) / 2, P.ndim > 1 ? (((s >> 1) & 1) * P.n[1] + j) / 2 : 0,
                     P.ndim > 2 ? (((s >> 2) & 1) * P.n[2] + k) / 2 : 0);
  }
  for (int v = 0; v < P.nvar; v++) Unew[((long long)p * P.nvar + v) * ncell + t] = U[((long long)q * P.nvar + v) * P.pc + sid];
  Tnew[(long long)p * ncell + t] = P.T[(long long)q * P.pc + sid];
}
