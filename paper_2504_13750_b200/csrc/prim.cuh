// prim.cuh -- fused cons->prim + thermo kernel with the alpha / CFL max-reduction.
// PAPER.md:237-258 (eq 4.2-4.4), :306 (Newton-Raphson from the stored T), :332 (update_aux),
// :337 (cfl), :292 (eq 4.11 alpha).  Readings A3, A6, A16, A17, A20.
#pragma once
#include "common.cuh"

__constant__ MechC c_mech;
static_assert(sizeof(MechC) <= 65536, "MechC must fit constant memory");

// cp_k/R_k and h_k/R_k (eq 4.3, 4.4), Horner form
// coefficient set of species k at T (two-range NASA-7: the upper set from Tmid[k] upwards)
__device__ __forceinline__ const double *nasa_at(int k, double T) {
  return (c_mech.two_range && T >= c_mech.Tmid[k]) ? c_mech.nasa_hi[k] : c_mech.nasa[k];
}
__device__ __forceinline__ double cp_R(int k, double T) {
  const double *a = nasa_at(k, T);
  return a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4])));
}
__device__ __forceinline__ double h_R(int k, double T) {
  const double *a = nasa_at(k, T);
  return a[5] + T * (a[0] + T * (0.5 * a[1] + T * (a[2] * (1.0 / 3.0) + T * (0.25 * a[3] + T * (0.2 * a[4])))));
}
__device__ __forceinline__ double s_R(int k, double T, double lnT) {
  const double *a = nasa_at(k, T);
  return a[0] * lnT + a[6] + T * (a[1] + T * (0.5 * a[2] + T * (a[3] * (1.0 / 3.0) + T * (0.25 * a[4]))));
}

// Newton on e(T) = sum_k Y_k R_k (h_k/R_k - T) = e.  Y[] = mass fractions of all ns species.
// NS > 0: compile-time species count (arrays stay in registers); NS == 0: run-time ns.
template <int NS>
__device__ __forceinline__ bool newton_T(const double *Y, int ns_rt, double e, double &T) {
  const int ns = NS > 0 ? NS : ns_rt;
  bool conv = false;
#pragma unroll 1
  for (int it = 0; it < 50; it++) {
    double f = -e, cv = 0.0;
#pragma unroll
    for (int k = 0; k < ns; k++) {
      double yr = Y[k] * c_mech.Rk[k];
      f = fma(yr, h_R(k, T) - T, f);
      cv = fma(yr, cp_R(k, T) - 1.0, cv);
    }
    double dT = -f / cv;
    T += dT;
    if (fabs(dT) <= 1e-11 * fabs(T)) { conv = true; break; }
  }
  return conv && (T > 0.0) && isfinite(T);
}

// One cell: loads U, returns T, p, c, u[].  Up points at this patch's U block, id = cell index.
template <int NS>
__device__ __forceinline__ bool cons2prim(const Params &P, const double *__restrict__ Up, long long id,
                                          double Tguess, double &T, double &p, double &c, double *u) {
  const int ns = NS > 0 ? NS : P.ns;
  double Y[NS > 0 ? NS : JANC_MAX_NS];
  const double rho = Up[id];
  const double irho = 1.0 / rho;
  double ke = 0.0;
  for (int d = 0; d < P.ndim; d++) {
    u[d] = Up[(long long)(1 + d) * P.pc + id] * irho;
    ke = fma(0.5 * u[d], u[d], ke);
  }
  double ysum = 0.0;
#pragma unroll
  for (int k = 0; k < ns - 1; k++) {
    Y[k] = Up[(long long)(P.ndim + 2 + k) * P.pc + id] * irho;
    ysum += Y[k];
  }
  Y[ns - 1] = 1.0 - ysum;
  const double e = Up[(long long)(P.ndim + 1) * P.pc + id] * irho - ke;
  T = Tguess;
  bool ok = newton_T<NS>(Y, ns, e, T);
  double R = 0.0, cp = 0.0;
#pragma unroll
  for (int k = 0; k < ns; k++) {
    double yr = Y[k] * c_mech.Rk[k];
    R += yr;
    cp = fma(yr, cp_R(k, T), cp);
  }
  p = rho * R * T;
  const double gam = cp / (cp - R);
  c = sqrt(gam * R * T);
  return ok && isfinite(c);
}

// grid: (blocks over the interior cells of one patch, np).  Writes T, p, vel on interior cells and
// (reduce != 0) atomically maxes |u_d|+c into slots[...][level][d].
template <int NS>
__global__ void __launch_bounds__(256) k_prim(Params P, const double *__restrict__ U, int reduce, int slot_base,
                                              double *dbgc) {
  const int patch = blockIdx.y + P.patch0;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double s[3] = {0.0, 0.0, 0.0};
  if (t < ncell) {
    int i = (int)(t % P.n[0]);
    long long r = t / P.n[0];
    int j = (int)(r % P.n[1]);
    int k = (int)(r / P.n[1]);
    long long id = cell_index(P, i, j, k);
    const double *Up = U + (long long)patch * P.nvar * P.pc;
    const long long pid = (long long)patch * P.pc + id;
    double T, p, c, u[3] = {0.0, 0.0, 0.0};
    bool ok = cons2prim<NS>(P, Up, id, P.T[pid], T, p, c, u);
    P.T[pid] = T;
    P.p[pid] = p;
    for (int d = 0; d < P.ndim; d++) {
      P.vel[(long long)d * P.np * P.pc + pid] = u[d];
      s[d] = fabs(u[d]) + c;
    }
    if (dbgc) dbgc[pid] = c;
    if (!ok) *P.flag = 1;
  }
  if (reduce) {
    __shared__ double sh[3][8];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    for (int d = 0; d < P.ndim; d++) {
      double v = s[d];
      if (!(v >= 0.0)) v = 0.0;   // NaN never enters the ordered-int max; the flag reports it
      for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
      if (lane == 0) sh[d][w] = v;
    }
    __syncthreads();
    if (threadIdx.x < P.ndim) {
      double v = 0.0;
      for (int q = 0; q < (int)(blockDim.x >> 5); q++) v = fmax(v, sh[threadIdx.x][q]);
      atomic_max_nonneg(P.slots + slot_base + P.level[patch] * 3 + threadIdx.x, v);
    }
  }
}

// One thread: dt from the step-start maxima (cfl mode) or the fixed value; accumulates t; clears the
// other parity's reduction slots for the next step.
__global__ void k_dt(Params P, int parity, double cfl, double dt_fixed, double dx_factor) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    double dt = dt_fixed;
    if (cfl > 0.0) {
      double smax = 0.0;
      for (int l = 0; l < 2; l++)
        for (int d = 0; d < P.ndim; d++) smax = fmax(smax, slot_value(P.slots + SLOT(parity, 0, l, d)));
      dt = cfl * (P.dxmin * dx_factor) / smax;     // dx_factor = ratio for the crossover advance (the level-0 step)
    }
    P.scal[0] = dt;
    P.scal[1] += dt;
    for (int q = 0; q < JANC_NSLOT / 2; q++) P.slots[SLOT(1 - parity, 0, 0, 0) + q] = 0ull;
  }
}
