// static_scratch.cuh -- janc_cfl_dt_static (include/janc.h): the CFL time step of a state with no workspace and no
// allocation, for callers that cannot call cudaMalloc (graph capture, serving loops).  PAPER.md:337 (cfl), :292 (the
// max(|u_d| + c) of eq 4.11), :237-258 / :306 (cons->prim, Newton from a starting T).
// Included at the end of janc.cu: cudaGetSymbolAddress has to sit in the translation unit that defines the array.
//
// The scratch of the reduction is a file-scope array: every GPU that loads the library holds its 1.5 MiB until exit.
//   [0, 32)                      header; word 0 (as int) = error flag, cleared at the start of every call
//   [32, 32 + 3 * MAX_BLOCKS)    per-CTA partial maxima [block][direction], every used entry rewritten by every call
// One array per device and process, shared by every call: calls that overlap on the GPU race (see include/janc.h).
#pragma once

#define JANC_STATIC_THREADS 256
#define JANC_STATIC_MAX_BLOCKS (JANC_STATIC_MAX_CELLS / JANC_STATIC_THREADS)      // 65536
#define JANC_STATIC_HEADER 32
static __device__ __align__(256) double g_static_scratch[JANC_STATIC_HEADER + 3 * JANC_STATIC_MAX_BLOCKS];

// In host code g_static_scratch is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current.
static std::mutex g_static_mutex;
static double *g_static_ptr[JANC_MAX_DEVICES] = {nullptr};

// The variant of k_prim for a state in the interior layout: no T / p / vel written, the CTA's maxima go to its own row
// of the scratch instead of the atomic slots of a workspace.  Q: Params with pc = cells per patch (no ghosts).
__global__ void __launch_bounds__(JANC_STATIC_THREADS) k_speed_static(Params Q, const double *__restrict__ U,
                                                                      const double *__restrict__ Tg, long long total,
                                                                      double *__restrict__ scratch) {
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  double s[3] = {0.0, 0.0, 0.0};
  if (t < total) {
    const long long patch = t / Q.pc, id = t - patch * Q.pc;
    double T, p, c, u[3] = {0.0, 0.0, 0.0};
    const bool ok = cons2prim<0>(Q, U + patch * Q.nvar * Q.pc, id, Tg ? Tg[t] : 1000.0, T, p, c, u);
    for (int d = 0; d < Q.ndim; d++) s[d] = fabs(u[d]) + c;
    if (!ok) *(int *)scratch = 1;
  }
  __shared__ double sh[3][JANC_STATIC_THREADS / 32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int d = 0; d < 3; d++) {
    double v = s[d];
    if (!(v >= 0.0)) v = 0.0;      // as k_prim: NaN never enters a maximum; the flag reports it
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) sh[d][w] = v;
  }
  __syncthreads();
  if (threadIdx.x < 3) {
    double v = 0.0;
    for (int q = 0; q < JANC_STATIC_THREADS / 32; q++) v = fmax(v, sh[threadIdx.x][q]);
    scratch[JANC_STATIC_HEADER + 3LL * blockIdx.x + threadIdx.x] = v;
  }
}

// One CTA: the maxima over the partial rows and dt as k_dt forms it (cfl * dx_min / max over the directions).
__global__ void __launch_bounds__(1024) k_dt_static(const double *__restrict__ scratch, int nblocks, int ndim, double cfl,
                                                    double dxmin, double *__restrict__ out) {
  __shared__ double sh[3][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  double s[3] = {0.0, 0.0, 0.0};
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x)
    for (int d = 0; d < 3; d++) s[d] = fmax(s[d], scratch[JANC_STATIC_HEADER + 3LL * b + d]);
  for (int d = 0; d < 3; d++) {
    double v = s[d];
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) sh[d][w] = v;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double smax = 0.0;
    for (int d = 0; d < 3; d++) {
      double v = 0.0;
      for (int q = 0; q < (int)(blockDim.x >> 5); q++) v = fmax(v, sh[d][q]);
      out[1 + d] = v;
      if (d < ndim) smax = fmax(smax, v);
    }
    const double dt = cfl * (dxmin * 1.0) / smax;
    out[0] = *(const int *)scratch ? nan("") : dt;
  }
}

extern "C" int janc_cfl_dt_static(janc_ctx *c, const double *U_dev, const double *T_dev, double cfl, double *out_dev) {
  if (!c || !U_dev || !out_dev) return JANC_EINVAL;
  if (!c->have_mech) { c->err = "set a mechanism first"; return JANC_ESTATE; }
  if (!(cfl > 0.0)) { c->err = "janc_cfl_dt_static: cfl must be positive"; return JANC_EINVAL; }
  const long long total = (long long)c->np * c->ncell;
  if (total > JANC_STATIC_MAX_CELLS) {
    c->err = "janc_cfl_dt_static: " + std::to_string(total) + " cells exceed the static scratch (JANC_STATIC_MAX_CELLS = " +
             std::to_string((long long)JANC_STATIC_MAX_CELLS) + "); use janc_step / janc_step_part with a workspace";
    return JANC_EINVAL;
  }
  CK(cudaSetDevice(c->device));
  double *scratch = nullptr;
  {
    std::lock_guard<std::mutex> lk(g_static_mutex);
    if (!g_static_ptr[c->device]) {
      void *q = nullptr;
      CK(cudaGetSymbolAddress(&q, g_static_scratch));
      g_static_ptr[c->device] = (double *)q;
    }
    scratch = g_static_ptr[c->device];
  }
  // the kernel reads the species tables from c_mech whatever kernels the context's own step runs
  std::unique_lock<std::mutex> mech_lock(g_mech_mutex);
  if (g_mech_owner[c->device] != c->id) {
    CK(cudaDeviceSynchronize());
    CK(cudaMemcpyToSymbol(c_mech, &c->mech, sizeof(MechC), 0, cudaMemcpyHostToDevice));
    g_mech_owner[c->device] = c->id;
  }
  Params Q = c->P;
  Q.pc = c->ncell;
  const int nblocks = (int)((total + JANC_STATIC_THREADS - 1) / JANC_STATIC_THREADS);
  CK(cudaMemsetAsync(scratch, 0, JANC_STATIC_HEADER * sizeof(double), c->stream));
  k_speed_static<<<nblocks, JANC_STATIC_THREADS, 0, c->stream>>>(Q, U_dev, T_dev, total, scratch);
  note_launch(c, cudaGetLastError());
  k_dt_static<<<1, 1024, 0, c->stream>>>(scratch, nblocks, c->g.ndim, cfl, c->P.dxmin, out_dev);
  note_launch(c, cudaGetLastError());
  return take_launch_error(c);
}
