// janc.cu -- host side of libjanc (C ABI declared in include/janc.h) + small utility kernels.
// No CPU fallback: every step of the path runs in the kernels of prim/ghost/flux/chem.cuh.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <string>
#include <vector>

#include <dlfcn.h>
#include <map>
#include <mutex>
#include <nvrtc.h>
#include <set>

#include "../../include/janc.h"
#include "chem.cuh"
#include "chemgen.h"
#include "chemgen_roles.h"
#include "flux.cuh"
#include "ghost.cuh"
#include "mechfile.h"
#include "prim.cuh"

// janc_set_option keys (include/janc.h); defaults are what the product runs
struct Options {
  bool graph = true;                    // "graph": replay one captured CUDA graph per step
  bool jit = true;                      // "jit": run-time specialised kernels (NVRTC)
  int jit_max_unknowns = JANC_JIT_MAX_N1;   // "jit_max_unknowns": largest system of the one-thread-per-cell kernel
  bool jit_big_smem = false;            // "jit_big" = "smem": the shared-memory kernel instead of the role-warp kernel
  int roles = 8;                        // "roles": 8 or 16 role-warps
  bool roles_lu_rows = true;            // "roles_lu" = "rows": LU with one row per lane | "columns": Gauss-Jordan across the role warps
  bool roles_newton_prim = true;        // "roles_newton" = "prim": T* from a cons->prim launch before the role-warp kernel | "kernel"
  bool tma = true;                      // "tma": 2-D tiles through cp.async.bulk.tensor (TMA) where the layout allows | cp.async
  bool halo_in_kernel = true;           // "halo" = "auto": 2-D patches <= 16 x 16 / small grids gather their halo in the
                                        //   flux kernel; "ghost": always materialise ghosts with k_ghost
};

struct janc_ctx {
  Options opt;
  std::set<const void *> attr_done;     // kernels whose dynamic shared-memory attribute is set on THIS context's device
  cudaError_t launch_err = cudaSuccess; // first failed kernel launch since the last check
  bool uses_cmech = false;              // table-driven kernels (c_mech in constant memory) are on this context's path
  CUtensorMap mapU[3], mapP, mapV;      // 2-D TMA path: {Px, Py, fields} over the RK registers A, B, C, over p and over vel
  bool have_tma = false;
  Flux3Maps map3[3];                    // 3-D TMA path: per RK register, the three box shapes over the register, vel and p
  bool have_tma3 = false;
  janc_grid g;
  int device;
  cudaStream_t stream;
  int np, nvar, ns, nr;
  bool have_mech, have_ws, have_state, have_blocks;
  MechC mech;
  Params P;
  long long ncell;       // interior cells per patch
  // workspace carve-up
  size_t ws_bytes;
  double *A, *B, *C;     // RK registers (A holds the state between steps)
  double *dbgc, *stageU, *stageT;
  int *d_level, *d_nbr, *d_parent, *d_fkind;
  std::vector<int> level, nbr, parent, fkind;
  int parity;
  int lvl_first[2] = {0, 0}, lvl_count[2] = {0, 0};   // patches of each level if they are contiguous (by_level)
  bool by_level = true;
  int act0 = 0, actn = 0;                             // patches the kernels of the current launches act on
  std::vector<int> rg_src, rg_par, rg_sub;            // regrid plan: where the data of every new patch comes from
  long long launches;
  int num_sms;
  // One step = 11..12 small launches; a step of each slot parity is captured once into a CUDA graph and replayed
  // (launch-bound grids: cfg 0 / cfg 1).  Captured on an internal stream (the caller's may be the legacy default
  // stream, which cannot be captured), launched on the caller's.
  struct StepGraph { cudaGraphExec_t exec = nullptr; double cfl = 0.0, dt = 0.0; int flags = 0; long long launches = 0; } graph[2];
  cudaStream_t cap_stream = nullptr;
  bool use_graph = true, warmed = false;
  int jit_chem_nt, jit_chem_cells, jit_chem_mode;   // threads per CTA, cells per CTA, see jit_chem_mode()
  size_t jit_chem_smem;
  cudaKernel_t jit_prim;     // mechanism-specialised cons->prim kernel, null if not in use
  cudaKernel_t jit_src = nullptr;   // explicit-variant source kernel (chemgen::generate_source), compiled on first use
  bool jit_src_tried = false;
  cudaKernel_t jit_kernel;   // mechanism-specialised chemistry kernel (chemgen.h), null if not in use
  std::string jit_log;
  unsigned long long id;
  std::string err;
};

static unsigned long long g_next_id = 1;
// The table-driven fallback kernels read the mechanism from __constant__ c_mech, one copy per device, shared by all
// contexts of the process.  g_mech_mutex serialises every call that launches such kernels (held for the whole call);
// g_mech_owner[device] = which context's mechanism sits in that device's c_mech.  A re-upload first drains the device.
static std::mutex g_mech_mutex;
static std::mutex g_jit_mutex;                // the per-process caches of compiled kernels
#define JANC_MAX_DEVICES 64
static unsigned long long g_mech_owner[JANC_MAX_DEVICES] = {0};

#define CK(call)                                                                         \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess) {                                                             \
      c->err = std::string(#call) + ": " + cudaGetErrorString(e_);                       \
      return JANC_ECUDA;                                                                 \
    }                                                                                    \
  } while (0)

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ------------------------------------------------------------------ utility kernels
// interior layout [np][nf][ncell]  <->  padded layout [np][nf][pc]
__global__ void __launch_bounds__(256) k_pack(Params P, const double *__restrict__ src, double *__restrict__ dst,
                                              int nf, int unpack, double fill) {
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const unsigned nbx = (unsigned)((ncell + blockDim.x - 1) / blockDim.x);   // grid.x = nbx * np * nf (grid.y is limited to 65535)
  const long long t = (long long)(blockIdx.x % nbx) * blockDim.x + threadIdx.x;
  if (t >= ncell) return;
  const int fp = blockIdx.x / nbx;
  const int f = fp % nf, patch = fp / nf;
  const int i = (int)(t % P.n[0]);
  const long long r = t / P.n[0];
  const int j = (int)(r % P.n[1]), k = (int)(r / P.n[1]);
  const long long pi = ((long long)patch * nf + f) * P.pc + cell_index(P, i, j, k);
  const long long ii = ((long long)patch * nf + f) * ncell + t;
  if (unpack) dst[ii] = src[pi];
  else dst[pi] = src ? src[ii] : fill;
}

__global__ void k_dfma(double *out, int iters) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 1.0000001, b = 1e-9;
#pragma unroll 1
  for (int i = 0; i < iters; i++) {
#pragma unroll
    for (int u = 0; u < 8; u++) {
      a0 = fma(a0, m, b); a1 = fma(a1, m, b); a2 = fma(a2, m, b); a3 = fma(a3, m, b);
      a4 = fma(a4, m, b); a5 = fma(a5, m, b); a6 = fma(a6, m, b); a7 = fma(a7, m, b);
    }
  }
  double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
  if (s == 123.456) out[0] = s;
}

// ------------------------------------------------------------------ create / destroy
extern "C" int janc_create(const janc_grid *grid, int device, void *cuda_stream, janc_ctx **out) {
  if (!grid || !out) return JANC_EINVAL;
  if (grid->ndim < 1 || grid->ndim > 3) return JANC_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return JANC_ECUDA;
  if (cudaSetDevice(device) != cudaSuccess) return JANC_ECUDA;
  janc_ctx *c = new (std::nothrow) janc_ctx();
  if (!c) return JANC_ENOMEM;
  c->g = *grid;
  c->device = device;
  c->num_sms = 148;
  if (device >= JANC_MAX_DEVICES) { delete c; return JANC_EINVAL; }
  cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
  c->stream = (cudaStream_t)cuda_stream;
  c->np = grid->n_patches > 0 ? grid->n_patches : 1;
  if (c->np > 65535) { delete c; return JANC_EINVAL; }   // patches ride on gridDim.y
  if (grid->n_patches <= 0) { c->g.n_levels = 1; c->g.ratio = 2; }
  if (c->g.n_levels < 1 || c->g.n_levels > 2 || (c->g.n_levels == 2 && c->g.ratio != 2)) { delete c; return JANC_EINVAL; }
  Params &P = c->P;
  memset(&P, 0, sizeof P);
  P.ndim = grid->ndim; P.np = c->np; P.nlev = c->g.n_levels; P.ratio = c->g.ratio;
  P.patch0 = 0; P.dt_scale = 1.0; c->act0 = 0; c->actn = c->np;
  c->lvl_first[0] = 0; c->lvl_count[0] = c->np;
  P.pc = 1; c->ncell = 1;
  double dxmin = 1e300;
  for (int d = 0; d < 3; d++) {
    if (d < grid->ndim) {
      if (grid->n[d] < 1 || !(grid->dx[d] > 0.0)) { delete c; return JANC_EINVAL; }
      if (c->g.n_levels == 2 && grid->n[d] % 2) { delete c; return JANC_EINVAL; }
      P.n[d] = grid->n[d]; P.G[d] = JANC_NG; P.P[d] = grid->n[d] + 2 * JANC_NG;
      double dx = grid->dx[d];
      P.invdx[0][d] = 1.0 / dx; P.invdx[1][d] = 1.0 / (dx / c->g.ratio);
      double dxf = c->g.n_levels == 2 ? dx / c->g.ratio : dx;
      if (dxf < dxmin) dxmin = dxf;
      P.bc_lo[d] = grid->bc_lo[d]; P.bc_hi[d] = grid->bc_hi[d];
      if (P.bc_lo[d] < 0 || P.bc_lo[d] > 3 || P.bc_hi[d] < 0 || P.bc_hi[d] > 3) { delete c; return JANC_EINVAL; }
      // exchange faces (x-slab decomposition): x sides of a uniform grid only
      if ((P.bc_lo[d] == JANC_BC_EXCHANGE || P.bc_hi[d] == JANC_BC_EXCHANGE) && (d != 0 || grid->n_patches > 0)) { delete c; return JANC_EINVAL; }
      // 3 ghost layers are copied from 3 distinct interior cells by the periodic / mirror / neighbour rules;
      // only zero-gradient sides work on thinner grids (e.g. the one-cell 0-D reactor)
      const bool thin_ok = grid->n_patches <= 0 && P.bc_lo[d] == 2 && P.bc_hi[d] == 2;
      if (grid->n[d] < JANC_NG && !thin_ok) { delete c; return JANC_EINVAL; }
    } else {
      c->g.n[d] = 1; P.n[d] = 1; P.G[d] = 0; P.P[d] = 1; P.invdx[0][d] = P.invdx[1][d] = 0.0;
    }
    P.st[d] = P.pc; P.pc *= P.P[d]; c->ncell *= P.n[d];
  }
  if (P.pc >= (1LL << 31)) { delete c; return JANC_EINVAL; }   // per-patch cell indices are 32-bit in the generated kernels
  P.dxmin = dxmin;
  int nf = 2 * grid->ndim;
  c->level.assign(c->np, 0);
  c->nbr.assign((size_t)c->np * nf, -1);
  c->parent.assign((size_t)c->np * (1 + grid->ndim), -1);
  c->fkind.assign((size_t)c->np * nf, FK_PHYSICAL);
  c->id = g_next_id++;
  c->jit_kernel = nullptr;
  c->jit_prim = nullptr;
  *out = c;
  return JANC_OK;
}

static void invalidate_graphs(janc_ctx *c);

extern "C" void janc_destroy(janc_ctx *c) {
  if (!c) return;
  { std::lock_guard<std::mutex> lk(g_mech_mutex); if (g_mech_owner[c->device] == c->id) g_mech_owner[c->device] = 0; }
  invalidate_graphs(c);
  if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
  delete c;
}

extern "C" const char *janc_last_error(const janc_ctx *c) { return c ? c->err.c_str() : "null context"; }
extern "C" long long janc_launch_count(const janc_ctx *c) { return c ? c->launches : 0; }

// ------------------------------------------------------------------ mechanism
// janc_mech (host arrays) -> MechC tables; err receives a text on failure
static int fill_mech(const janc_mech *m, MechC &M, std::string &err) {
  if (!m) return JANC_EINVAL;
  if (m->ns < 1 || m->ns > JANC_MAX_NS || m->nr < 0 || m->nr > JANC_MAX_NR) { err = "ns/nr out of range"; return JANC_EINVAL; }
  if (!m->W || !m->nasa) return JANC_EINVAL;
  if (m->nr > 0 && (!m->nu_f || !m->nu_b || !m->A || !m->b || !m->Ta)) return JANC_EINVAL;
  memset(&M, 0, sizeof M);
  M.ns = m->ns; M.nr = m->nr;
  for (int k = 0; k < m->ns; k++) {
    if (!(m->W[k] > 0.0)) return JANC_EINVAL;
    M.W[k] = m->W[k]; M.invW[k] = 1.0 / m->W[k]; M.Rk[k] = JANC_RU / m->W[k];
    for (int q = 0; q < 7; q++) M.nasa[k][q] = m->nasa[k * 7 + q];
    if (m->nasa_hi && m->T_mid) {
      for (int q = 0; q < 7; q++) M.nasa_hi[k][q] = m->nasa_hi[k * 7 + q];
      M.Tmid[k] = m->T_mid[k];
      M.two_range = 1;
    }
  }
  for (int i = 0; i < m->nr; i++) {
    if (!(m->A[i] > 0.0)) { err = "A must be > 0"; return JANC_EINVAL; }
    M.lnA[i] = log(m->A[i]); M.b[i] = m->b[i]; M.Ta[i] = m->Ta[i]; M.Asign[i] = 1.0;
    M.rev[i] = m->reversible ? (m->reversible[i] != 0) : 1;
    M.tb[i] = m->third_body ? (m->third_body[i] != 0) : 0;
    int nre = 0, npr = 0, dn = 0;
    for (int k = 0; k < m->ns; k++) {
      int f = m->nu_f[i * m->ns + k], b = m->nu_b[i * m->ns + k];
      if (f < 0 || b < 0) return JANC_EINVAL;
      if (nre + f > JANC_MAX_ORDER || npr + b > JANC_MAX_ORDER) { err = "reaction order too large"; return JANC_EINVAL; }
      for (int q = 0; q < f; q++) M.reac[i][nre++] = (unsigned char)k;
      for (int q = 0; q < b; q++) M.prod[i][npr++] = (unsigned char)k;
      dn += b - f;
    }
    M.nreac[i] = (unsigned char)nre; M.nprod[i] = (unsigned char)npr; M.dn[i] = (signed char)dn;
    if (M.tb[i]) {
      if (M.ntb >= JANC_MAX_TB) { err = "too many third-body reactions"; return JANC_EINVAL; }
      M.tbi[i] = (unsigned char)M.ntb;
      for (int k = 0; k < m->ns; k++) M.eff[M.ntb][k] = m->eff ? m->eff[i * m->ns + k] : 1.0;
      M.ntb++;
    }
    for (int k = 0; k < m->ns; k++) M.dnu[i][k] = (double)(m->nu_b[i * m->ns + k] - m->nu_f[i * m->ns + k]);
  }
  // derivative entries of eq 4.7 grouped by the species (column) they differentiate
  M.nent = 0;
  for (int j = 0; j < m->ns; j++) {
    M.col_start[j] = M.nent;
    for (int i = 0; i < m->nr; i++)
      for (int side = 0; side < 2; side++) {
        if (side == 1 && !M.rev[i]) continue;
        const unsigned char *lst = side == 0 ? M.reac[i] : M.prod[i];
        const int cnt = side == 0 ? M.nreac[i] : M.nprod[i];
        for (int e = 0; e < cnt; e++) {
          if (lst[e] != j) continue;
          if (M.nent >= JANC_MAX_ENT) { err = "mechanism has too many derivative entries"; return JANC_EINVAL; }
          DqEntry &E = M.ent[M.nent++];
          E.rx = (unsigned char)i; E.side = (unsigned char)side; E.nother = 0;
          for (int e2 = 0; e2 < cnt; e2++) if (e2 != e) E.other[E.nother++] = lst[e2];
        }
      }
  }
  for (int j = m->ns; j <= JANC_MAX_NS; j++) M.col_start[j] = M.nent;
  return JANC_OK;
}

// ------------------------------------------------------------------ run-time specialised chemistry
// NVRTC is reached through dlopen so that libjanc.so loads (and the generic kernels run) where it is
// absent; the cubin is loaded with the runtime's cudaLibrary API (no link against libcuda).
struct ChemArgs { double *U; double *T; const double *scal; int *flag; int n0, n1, n2, G0, G1, G2; long long st0, st1, st2, pc; int np, patch0; double dts; };

struct NvrtcApi {
  void *h = nullptr;
  nvrtcResult (*create)(nvrtcProgram *, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
  nvrtcResult (*compile)(nvrtcProgram, int, const char *const *) = nullptr;
  nvrtcResult (*cubin_size)(nvrtcProgram, size_t *) = nullptr;
  nvrtcResult (*cubin)(nvrtcProgram, char *) = nullptr;
  nvrtcResult (*log_size)(nvrtcProgram, size_t *) = nullptr;
  nvrtcResult (*log)(nvrtcProgram, char *) = nullptr;
  nvrtcResult (*destroy)(nvrtcProgram *) = nullptr;
  bool ok = false;
};

static NvrtcApi &nvrtc_api() {
  static NvrtcApi a;
  static bool tried = false;
  if (tried) return a;
  tried = true;
  const char *names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"};
  for (const char *n : names) { a.h = dlopen(n, RTLD_NOW | RTLD_LOCAL); if (a.h) break; }
  if (!a.h) return a;
  a.create = (decltype(a.create))dlsym(a.h, "nvrtcCreateProgram");
  a.compile = (decltype(a.compile))dlsym(a.h, "nvrtcCompileProgram");
  a.cubin_size = (decltype(a.cubin_size))dlsym(a.h, "nvrtcGetCUBINSize");
  a.cubin = (decltype(a.cubin))dlsym(a.h, "nvrtcGetCUBIN");
  a.log_size = (decltype(a.log_size))dlsym(a.h, "nvrtcGetProgramLogSize");
  a.log = (decltype(a.log))dlsym(a.h, "nvrtcGetProgramLog");
  a.destroy = (decltype(a.destroy))dlsym(a.h, "nvrtcDestroyProgram");
  a.ok = a.create && a.compile && a.cubin_size && a.cubin && a.log_size && a.log && a.destroy;
  return a;
}

// CUDA C -> sm_100a cubin.  Needs no device.
static bool jit_compile(const std::string &src, std::vector<char> &cubin, std::string &log) {
  NvrtcApi &a = nvrtc_api();
  if (!a.ok) { log = "NVRTC not available (dlopen libnvrtc.so.12 failed)"; return false; }
  nvrtcProgram prog;
  if (a.create(&prog, src.c_str(), "k_chem_jit.cu", 0, nullptr, nullptr) != NVRTC_SUCCESS) { log = "nvrtcCreateProgram failed"; return false; }
  const char *opts[] = {"--gpu-architecture=sm_100a", "--std=c++17", "-lineinfo"};
  const nvrtcResult r = a.compile(prog, 3, opts);
  size_t ls = 0;
  a.log_size(prog, &ls);
  if (ls > 1) { log.resize(ls); a.log(prog, &log[0]); }
  bool ok = r == NVRTC_SUCCESS;
  if (ok) {
    size_t n = 0;
    ok = a.cubin_size(prog, &n) == NVRTC_SUCCESS && n > 0;
    if (ok) { cubin.resize(n); ok = a.cubin(prog, cubin.data()) == NVRTC_SUCCESS; }
  }
  a.destroy(&prog);
  return ok;
}

struct PrimArgs { const double *U; double *T; double *p; double *vel; double *dbgc; unsigned long long *slots;
                  const int *level; int *flag; int n0, n1, n2, G0, G1, G2; long long st0, st1, st2, pc; int np, reduce, slot_base, patch0; };
struct SrcArgs { const double *Uk; double *Uout; const double *T; const double *scal; int n0, n1, n2, G0, G1, G2; long long st0, st1, st2, pc; double coef; int patch0; };
struct JitKernels { cudaKernel_t chem = nullptr, prim = nullptr, src = nullptr; };

// 0: table-driven kernel, 1: register-resident specialised kernel (one thread per cell), 2: one thread per cell
// with the matrix in smem, 3: 8 role-warps per 32 cells with the matrix columns in registers (chemgen_roles.h)
static int jit_chem_mode(const MechC &M, const Options &opt) {
  if (M.ns < 2 || M.nr < 1) return 0;
  if (M.ns - 1 <= opt.jit_max_unknowns) return 1;
  if (chemgen::roles_applicable(M) && !opt.jit_big_smem) return 3;
  const size_t smem = (size_t)(M.ns - 1) * M.ns * JANC_JIT_NT_BIG * sizeof(double);
  return smem <= 200 * 1024 ? 2 : 0;
}

// Generate + compile + load the kernels specialised for c->mech (cons->prim for any mechanism, chemistry
// for <= JANC_JIT_MAX_N1 unknowns); on any failure the table-driven kernels stay.
static void jit_setup(janc_ctx *c) {
  c->jit_kernel = nullptr;
  c->jit_prim = nullptr;
  c->jit_src = nullptr;
  c->jit_src_tried = false;
  c->jit_log.clear();
  const MechC &M = c->mech;
  c->jit_chem_mode = 0;
  if (!c->opt.jit) { c->jit_log = "disabled by janc_set_option(\"jit\", \"0\")"; return; }
  chemgen::roles_nr_ref() = c->opt.roles;
  chemgen::roles_lu_rows_ref() = c->opt.roles_lu_rows;
  chemgen::roles_newton_ref() = !c->opt.roles_newton_prim;
  const int mode = jit_chem_mode(M, c->opt);
  const bool chem = mode != 0;
  c->jit_chem_mode = mode;
  c->jit_chem_nt = mode == 3 ? chemgen::roles_nr() * 32 : mode == 2 ? JANC_JIT_NT_BIG : JANC_JIT_NT;
  c->jit_chem_cells = mode == 3 ? 32 : c->jit_chem_nt;
  c->jit_chem_smem = mode == 3 ? chemgen::roles_layout(M, c->g.ndim).smem() : mode == 2 ? (size_t)(M.ns - 1) * M.ns * JANC_JIT_NT_BIG * sizeof(double) : 0;
  std::string src = chemgen::generate_prim(M, c->g.ndim);
  if (mode == 3) src += chemgen::generate_roles(M, c->g.ndim);
  else if (chem) src += chemgen::generate(M, c->g.ndim, mode == 2);
  else c->jit_log = "chemistry: mechanism outside the specialised range; ";
  static std::map<std::string, JitKernels> cache;          // per process, keyed by device + source
  std::lock_guard<std::mutex> lk(g_jit_mutex);
  const std::string key = std::to_string(c->device) + "\n" + src;
  auto it = cache.find(key);
  if (it != cache.end()) { c->jit_kernel = it->second.chem; c->jit_prim = it->second.prim; return; }
  std::vector<char> cubin;
  std::string log;
  if (!jit_compile(src, cubin, log)) { c->jit_log += log; return; }
  cudaLibrary_t lib;
  cudaError_t e = cudaLibraryLoadData(&lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
  if (e != cudaSuccess) { c->jit_log += std::string("cudaLibraryLoadData: ") + cudaGetErrorString(e); cudaGetLastError(); return; }
  JitKernels k;
  e = cudaLibraryGetKernel(&k.prim, lib, "k_prim_jit");
  if (e == cudaSuccess && chem) e = cudaLibraryGetKernel(&k.chem, lib, "k_chem_jit");
  if (e == cudaSuccess && c->jit_chem_smem > 48 * 1024)
    e = cudaKernelSetAttributeForDevice(k.chem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->jit_chem_smem, c->device);
  if (e != cudaSuccess) { c->jit_log += std::string("cudaLibraryGetKernel: ") + cudaGetErrorString(e); cudaGetLastError(); return; }
  cache[key] = k;
  c->jit_kernel = k.chem;
  c->jit_prim = k.prim;
}

// The explicit-variant source kernel is compiled on first use (janc_step with flags bit 1): a 100-reaction mechanism
// costs ~5 s of NVRTC time that the default path should not pay.
static void jit_setup_source(janc_ctx *c) {
  if (c->jit_src || c->jit_src_tried) return;
  c->jit_src_tried = true;
  const MechC &M = c->mech;
  if (!c->opt.jit) { c->jit_log += " source kernel: disabled by janc_set_option(\"jit\", \"0\")"; return; }
  if (M.ns < 2 || M.nr < 1) return;
  const std::string src = chemgen::generate_source(M, c->g.ndim, true);
  static std::map<std::string, cudaKernel_t> cache;
  std::lock_guard<std::mutex> lk(g_jit_mutex);
  const std::string key = std::to_string(c->device) + "\n" + src;
  auto it = cache.find(key);
  if (it != cache.end()) { c->jit_src = it->second; return; }
  std::vector<char> cubin;
  std::string log;
  if (!jit_compile(src, cubin, log)) { c->jit_log += log; return; }
  cudaLibrary_t lib;
  cudaKernel_t k = nullptr;
  cudaError_t e = cudaLibraryLoadData(&lib, cubin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
  if (e == cudaSuccess) e = cudaLibraryGetKernel(&k, lib, "k_src_jit");
  if (e != cudaSuccess) { c->jit_log += std::string("source kernel: ") + cudaGetErrorString(e); cudaGetLastError(); return; }
  cache[key] = k;
  c->jit_src = k;
}

extern "C" const char *janc_chem_kernel(const janc_ctx *c) {
  if (!c || !c->have_mech) return "none";
  if (c->jit_kernel) return c->jit_chem_mode == 3 ? "jit-roles" : c->jit_chem_mode == 2 ? "jit-smem" : "jit";
  return (c->ns == 2 || c->ns == 9) ? "reg" : "generic";
}
extern "C" const char *janc_jit_log(const janc_ctx *c) { return c ? c->jit_log.c_str() : ""; }

// Diagnostic, needs no device: emit the specialised source for a mechanism and compile it for sm_100a.
extern "C" int janc_jit_probe(const janc_mech *m, int ndim, char *src_out, size_t cap, size_t *src_len, size_t *cubin_bytes) {
  if (!m || ndim < 1 || ndim > 3) return JANC_EINVAL;
  std::unique_ptr<MechC> Mp(new (std::nothrow) MechC);
  if (!Mp) return JANC_ENOMEM;
  MechC &M = *Mp;
  std::string err;
  int rc = fill_mech(m, M, err);
  if (rc) return rc;
  const Options opt;
  chemgen::roles_nr_ref() = opt.roles;
  chemgen::roles_lu_rows_ref() = opt.roles_lu_rows;
  chemgen::roles_newton_ref() = !opt.roles_newton_prim;
  const int mode = jit_chem_mode(M, opt);
  std::string src = chemgen::generate_prim(M, ndim);
  if (mode == 3) src += chemgen::generate_roles(M, ndim);
  else if (mode) src += chemgen::generate(M, ndim, mode == 2);
  if (M.ns >= 2 && M.nr >= 1) src += chemgen::generate_source(M, ndim, mode == 0);   // same translation unit here: helpers once
  if (src_len) *src_len = src.size();
  if (src_out && cap > 0) { size_t n = src.size() < cap - 1 ? src.size() : cap - 1; memcpy(src_out, src.data(), n); src_out[n] = 0; }
  if (cubin_bytes) {
    std::vector<char> cubin;
    std::string log;
    *cubin_bytes = 0;
    if (!jit_compile(src, cubin, log)) { fprintf(stderr, "janc_jit_probe: %s\n", log.c_str()); return JANC_ESTATE; }
    *cubin_bytes = cubin.size();
  }
  return JANC_OK;
}

// ------------------------------------------------------------------ Chemkin-format reader (mechfile.h; host only)
extern "C" int janc_mech_parse(const char *mech_text, const char *thermo_text, janc_mech_file **out, char *err, size_t errcap) {
  if (!mech_text || !out) return JANC_EINVAL;
  janc_mech_file *F = new (std::nothrow) janc_mech_file();
  if (!F) return JANC_ENOMEM;
  bool ok = false;
  try { ok = mechfile::parse(mech_text, thermo_text, *F); } catch (...) { F->err = "internal error while parsing"; }
  if (!ok) {
    if (err && errcap) { strncpy(err, F->err.c_str(), errcap - 1); err[errcap - 1] = 0; }
    delete F;
    return JANC_EINVAL;
  }
  *out = F;
  return JANC_OK;
}

extern "C" int janc_mech_file_view(const janc_mech_file *F, janc_mech *v) {
  if (!F || !v) return JANC_EINVAL;
  v->ns = (int)F->species.size(); v->nr = (int)F->A.size();
  v->W = F->W.data(); v->nasa = F->nasa.data(); v->nu_f = F->nu_f.data(); v->nu_b = F->nu_b.data();
  v->A = F->A.data(); v->b = F->b.data(); v->Ta = F->Ta.data(); v->reversible = F->reversible.data();
  v->third_body = F->third_body.data(); v->eff = F->eff.data(); v->nasa_hi = F->nasa_hi.data(); v->T_mid = F->T_mid.data();
  return JANC_OK;
}

extern "C" const char *janc_mech_file_species(const janc_mech_file *F, int k) {
  return (F && k >= 0 && k < (int)F->species.size()) ? F->species[k].c_str() : "";
}

extern "C" void janc_mech_file_free(janc_mech_file *F) { delete F; }

extern "C" int janc_set_mechanism(janc_ctx *c, const janc_mech *m) {
  if (!c || !m) return JANC_EINVAL;
  // fill a temporary table and commit it only on success: a rejected mechanism leaves the context as it was
  std::unique_ptr<MechC> tmp(new (std::nothrow) MechC);
  if (!tmp) return JANC_ENOMEM;
  std::string err;
  int rc = fill_mech(m, *tmp, err);
  if (rc) { c->err = err.empty() ? "malformed mechanism" : err; return rc; }
  if (cudaSetDevice(c->device) != cudaSuccess) return JANC_ECUDA;
  c->mech = *tmp;
  invalidate_graphs(c);
  jit_setup(c);
  c->ns = m->ns; c->nr = m->nr;
  c->nvar = c->g.ndim + 2 + m->ns - 1;
  c->P.nvar = c->nvar; c->P.ns = m->ns;
  c->have_mech = true; c->have_ws = false; c->have_state = false;
  // which kernels of the path read c_mech: the table-driven cons->prim and / or chemistry
  c->uses_cmech = !c->jit_prim || (m->ns > 1 && m->nr > 0 && !c->jit_kernel);
  { std::lock_guard<std::mutex> lk(g_mech_mutex); if (g_mech_owner[c->device] == c->id) g_mech_owner[c->device] = 0; }
  return JANC_OK;
}

// Contexts on the table-driven path hold g_mech_mutex for the whole launching call (MechLock) and make sure their
// mechanism is the one in the device's c_mech; a re-upload drains the device first, so no kernel of another context
// that still reads the old table is in flight.
struct MechLock {
  std::unique_lock<std::mutex> lk;
  explicit MechLock(janc_ctx *c) { if (c->uses_cmech) lk = std::unique_lock<std::mutex>(g_mech_mutex); }
};

static int upload_mech(janc_ctx *c) {
  if (!c->uses_cmech || g_mech_owner[c->device] == c->id) return JANC_OK;
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpyToSymbol(c_mech, &c->mech, sizeof(MechC), 0, cudaMemcpyHostToDevice));
  g_mech_owner[c->device] = c->id;
  return JANC_OK;
}

extern "C" int janc_set_option(janc_ctx *c, const char *key, const char *value) {
  if (!c || !key || !value) return JANC_EINVAL;
  const std::string k = key, v = value;
  const bool on = !(v == "0" || v == "off" || v == "false");
  if (k == "graph") { c->opt.graph = on; c->use_graph = on; if (!on) invalidate_graphs(c); return JANC_OK; }
  if (k == "tma") { c->opt.tma = on; invalidate_graphs(c); return JANC_OK; }
  if (k == "halo") {
    if (v != "auto" && v != "ghost") { c->err = "halo: auto | ghost"; return JANC_EINVAL; }
    c->opt.halo_in_kernel = v == "auto"; invalidate_graphs(c); return JANC_OK;
  }
  // the remaining keys select kernels at janc_set_mechanism time
  if (c->have_mech) { c->err = "option '" + k + "' must be set before janc_set_mechanism"; return JANC_ESTATE; }
  if (k == "jit") { c->opt.jit = on; return JANC_OK; }
  if (k == "jit_max_unknowns") { c->opt.jit_max_unknowns = atoi(value); return JANC_OK; }
  if (k == "jit_big") {
    if (v != "roles" && v != "smem") { c->err = "jit_big: roles | smem"; return JANC_EINVAL; }
    c->opt.jit_big_smem = v == "smem"; return JANC_OK;
  }
  if (k == "roles") {
    if (v != "8" && v != "16") { c->err = "roles: 8 | 16"; return JANC_EINVAL; }
    c->opt.roles = atoi(value); return JANC_OK;
  }
  if (k == "roles_lu") {
    if (v != "rows" && v != "columns") { c->err = "roles_lu: rows | columns"; return JANC_EINVAL; }
    c->opt.roles_lu_rows = v == "rows"; return JANC_OK;
  }
  if (k == "roles_newton") {
    if (v != "prim" && v != "kernel") { c->err = "roles_newton: prim | kernel"; return JANC_EINVAL; }
    c->opt.roles_newton_prim = v == "prim"; return JANC_OK;
  }
  c->err = "unknown option '" + k + "'";
  return JANC_EINVAL;
}

// ------------------------------------------------------------------ workspace
struct Carve { size_t off; size_t take(size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; } };

static void carve(janc_ctx *c, char *base, size_t *total) {
  Carve cv{0};
  const size_t cells = (size_t)c->np * c->P.pc, nf = 2 * c->g.ndim;
  size_t oA = cv.take(cells * c->nvar * 8), oB = cv.take(cells * c->nvar * 8), oC = cv.take(cells * c->nvar * 8);
  size_t oT = cv.take(cells * 8), op = cv.take(cells * 8), ov = cv.take(cells * c->g.ndim * 8), oc = cv.take(cells * 8);
  size_t osU = cv.take((size_t)c->np * c->ncell * c->nvar * 8), osT = cv.take((size_t)c->np * c->ncell * 8);
  size_t oslots = cv.take(JANC_NSLOT * 8), oscal = cv.take(4 * 8), oflag = cv.take(16);
  size_t olev = cv.take(c->np * 4), onbr = cv.take(c->np * nf * 4), opar = cv.take(c->np * (1 + c->g.ndim) * 4), ofk = cv.take(c->np * nf * 4);
  if (total) *total = cv.off;
  if (base) {
    c->A = (double *)(base + oA); c->B = (double *)(base + oB); c->C = (double *)(base + oC);
    c->P.T = (double *)(base + oT); c->P.p = (double *)(base + op); c->P.vel = (double *)(base + ov);
    c->dbgc = (double *)(base + oc); c->stageU = (double *)(base + osU); c->stageT = (double *)(base + osT);
    c->P.slots = (unsigned long long *)(base + oslots); c->P.scal = (double *)(base + oscal); c->P.flag = (int *)(base + oflag);
    c->d_level = (int *)(base + olev); c->d_nbr = (int *)(base + onbr); c->d_parent = (int *)(base + opar); c->d_fkind = (int *)(base + ofk);
    c->P.level = c->d_level; c->P.nbr = c->d_nbr; c->P.parent = c->d_parent; c->P.fkind = c->d_fkind;
  }
}

extern "C" size_t janc_workspace_bytes(const janc_ctx *c) {
  if (!c || !c->have_mech) return 0;
  size_t total = 0;
  carve(const_cast<janc_ctx *>(c), nullptr, &total);
  return total;
}

static int upload_lists(janc_ctx *c) {
  CK(cudaMemcpyAsync(c->d_level, c->level.data(), c->level.size() * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->d_nbr, c->nbr.data(), c->nbr.size() * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->d_parent, c->parent.data(), c->parent.size() * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(c->d_fkind, c->fkind.data(), c->fkind.size() * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return JANC_OK;
}

// Tensor maps of the 2-D TMA path: a 3-D view {Px, Py, fields} of an array of padded fields, box = one 64 x 16 tile
// with its 3 ghost layers.  cuTensorMapEncodeTiled is reached through the runtime (no link against libcuda).
static bool make_map(CUtensorMap *m, void *base, int Px, int Py, long long nfields, int bx, int by) {
  typedef CUresult (*encode_t)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                               const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static encode_t enc = nullptr;
  if (!enc) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) {
      cudaGetLastError();
      return false;
    }
    enc = (encode_t)fn;
  }
  const cuuint64_t dims[3] = {(cuuint64_t)Px, (cuuint64_t)Py, (cuuint64_t)nfields};
  const cuuint64_t strides[2] = {(cuuint64_t)Px * 8, (cuuint64_t)Px * Py * 8};
  const cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// 4-D view {Px, Py, Pz, fields} for the 3-D TMA path: one map per box shape
static bool make_map4(CUtensorMap *m, void *base, const int *Pd, long long nfields, int bx, int by, int bz) {
  typedef CUresult (*encode_t)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                               const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void *fn = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || !fn) {
    cudaGetLastError();
    return false;
  }
  const cuuint64_t dims[4] = {(cuuint64_t)Pd[0], (cuuint64_t)Pd[1], (cuuint64_t)Pd[2], (cuuint64_t)nfields};
  const cuuint64_t strides[3] = {(cuuint64_t)Pd[0] * 8, (cuuint64_t)Pd[0] * Pd[1] * 8, (cuuint64_t)Pd[0] * Pd[1] * Pd[2] * 8};
  const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz, 1};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  return ((encode_t)fn)(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                        CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// which tile the non-gathering 2-D path uses: 0 = 64 x 16 (8-cell pencils), 1 = 32 x 16, 2 = 16 x 16 (4-cell pencils)
static int tile2d(const janc_ctx *c) { return c->P.n[0] <= 16 && c->P.n[1] <= 16 ? 2 : c->P.n[0] <= 32 ? 1 : 0; }

#define JANC_F3T 16, 8, 8, 8      // tile and pencil length of the 3-D TMA flux kernel

static void setup_tma3(janc_ctx *c) {
  c->have_tma3 = false;
  const Params &P = c->P;
  if (c->g.ndim != 3 || (P.P[0] & 1)) return;      // global strides must be multiples of 16 bytes
  constexpr int T[4] = {JANC_F3T};
  double *regs[3] = {c->A, c->B, c->C};
  bool ok = true;
  for (int d = 0; d < 3; d++) {
    const int bx = T[0] + (d == 0 ? 6 : 2), by = T[1] + (d == 1 ? 6 : 0), bz = T[2] + (d == 2 ? 6 : 0);   // y / z boxes start at an even x
    for (int q = 0; q < 3; q++) {
      ok = ok && make_map4(&c->map3[q].U[d], regs[q], P.P, (long long)c->np * c->nvar, bx, by, bz);
      ok = ok && make_map4(&c->map3[q].V[d], P.vel, P.P, (long long)c->np * 3, bx, by, bz);
      ok = ok && make_map4(&c->map3[q].P[d], P.p, P.P, c->np, bx, by, bz);
    }
  }
  c->have_tma3 = ok;
}

template <int TX, int TY, int TZ, int SEG>
static void launch_flux3_tma(janc_ctx *c, const double *Uk, const double *U0, double *Uout, int slot_base, double coef) {
  using C = Flux3TmaCfg<TX, TY, TZ, SEG>;
  const Params &P = c->P;
  smem_attr(c, (const void *)k_flux_rk3_tma<TX, TY, TZ, SEG>, C::SMEM);
  const unsigned tiles = (unsigned)(((P.n[0] + TX - 1) / TX) * ((P.n[1] + TY - 1) / TY) * ((P.n[2] + TZ - 1) / TZ));
  const int which = Uk == c->A ? 0 : Uk == c->B ? 1 : 2;
  k_flux_rk3_tma<TX, TY, TZ, SEG><<<dim3(tiles, (unsigned)c->actn, 1), C::NT, C::SMEM, c->stream>>>(P, U0, Uout, slot_base, coef, Uk == U0 ? 1 : 0,
                                                                                          c->map3[which]);
}

static void setup_tma(janc_ctx *c) {
  c->have_tma = false;
  setup_tma3(c);
  const Params &P = c->P;
  if (c->g.ndim != 2 || (P.P[0] & 1) || ((long long)P.P[0] * P.P[1] & 1)) return;   // strides must be multiples of 16 bytes
  const int t = tile2d(c), bx = (t == 0 ? 64 : t == 1 ? 32 : 16) + 6, by = 16 + 6;
  double *regs[3] = {c->A, c->B, c->C};
  bool ok = true;
  for (int q = 0; q < 3; q++) ok = ok && make_map(&c->mapU[q], regs[q], P.P[0], P.P[1], (long long)c->np * c->nvar, bx, by);
  ok = ok && make_map(&c->mapP, P.p, P.P[0], P.P[1], c->np, bx, by);
  ok = ok && make_map(&c->mapV, P.vel, P.P[0], P.P[1], (long long)c->np * 2, bx, by);
  c->have_tma = ok;
}

template <int TX, int TY, int SEG>
static void launch_flux2_tma(janc_ctx *c, const double *Uk, const double *U0, double *Uout, int slot_base, double coef) {
  using C = Flux2TmaCfg<TX, TY, SEG>;
  const Params &P = c->P;
  smem_attr(c, (const void *)k_flux_rk2_tma<TX, TY, SEG>, C::SMEM);
  const unsigned tiles = (unsigned)(((P.n[0] + TX - 1) / TX) * ((P.n[1] + TY - 1) / TY));
  const int which = Uk == c->A ? 0 : Uk == c->B ? 1 : 2;
  k_flux_rk2_tma<TX, TY, SEG><<<dim3(tiles, (unsigned)c->actn, 1), C::NT, C::SMEM, c->stream>>>(P, U0, Uout, slot_base, coef, Uk == U0 ? 1 : 0,
                                                                                      c->mapU[which], c->mapP, c->mapV);
}

extern "C" int janc_bind_workspace(janc_ctx *c, void *dev_ptr, size_t bytes) {
  if (!c || !c->have_mech || !dev_ptr) return JANC_EINVAL;
  size_t need = janc_workspace_bytes(c);
  if (bytes < need || ((uintptr_t)dev_ptr & 255)) { c->err = "workspace too small or misaligned"; return JANC_EINVAL; }
  CK(cudaSetDevice(c->device));
  invalidate_graphs(c);
  carve(c, (char *)dev_ptr, nullptr);
  c->ws_bytes = need;
  CK(cudaMemsetAsync(dev_ptr, 0, need, c->stream));
  c->have_ws = true; c->have_state = false; c->parity = 0;
  setup_tma(c);
  return upload_lists(c);
}

// ------------------------------------------------------------------ block lists
extern "C" int janc_set_blocks(janc_ctx *c, const int32_t *level, const int32_t *nbr, const int32_t *parent) {
  if (!c || c->g.n_patches <= 0 || !level || !nbr) return JANC_EINVAL;
  invalidate_graphs(c);
  const int nd = c->g.ndim, nf = 2 * nd, np = c->np;
  for (int p = 0; p < np; p++) {
    if (level[p] < 0 || level[p] >= c->g.n_levels) { c->err = "level out of range"; return JANC_EINVAL; }
    for (int f = 0; f < nf; f++) {
      int q = nbr[p * nf + f];
      if (q >= np || (q >= 0 && level[q] != level[p])) { c->err = "bad neighbour id"; return JANC_EINVAL; }
    }
    if (level[p] > 0) {
      if (!parent) return JANC_EINVAL;
      int k = parent[p * (1 + nd)];
      if (k < 0 || k >= np || level[k] != level[p] - 1) { c->err = "bad parent id"; return JANC_EINVAL; }
      for (int e = 0; e < nd; e++) {
        int s = parent[p * (1 + nd) + 1 + e];
        if (s < 0 || s >= c->g.ratio) { c->err = "bad sub-region index"; return JANC_EINVAL; }
      }
    }
  }
  for (int p = 0; p < np; p++) {
    c->level[p] = level[p];
    for (int f = 0; f < nf; f++) c->nbr[p * nf + f] = nbr[p * nf + f];
    for (int e = 0; e <= nd; e++) c->parent[p * (1 + nd) + e] = parent ? parent[p * (1 + nd) + e] : -1;
  }
  // which source fills each face: neighbour, physical BC, or the coarse parent
  for (int p = 0; p < np; p++)
    for (int f = 0; f < nf; f++) {
      int kind;
      if (c->nbr[p * nf + f] >= 0) kind = FK_NEIGHBOUR;
      else if (c->level[p] == 0) kind = FK_PHYSICAL;
      else {
        const int k = c->parent[p * (1 + nd)], d = f / 2, side = f % 2;
        const int s = c->parent[p * (1 + nd) + 1 + d];
        const bool at_parent_edge = side == 0 ? (s == 0) : (s == c->g.ratio - 1);
        kind = (at_parent_edge && c->nbr[k * nf + f] < 0) ? FK_PHYSICAL : FK_COARSE;
      }
      c->fkind[p * nf + f] = kind;
    }
  // patches of a level contiguous (levels in non-decreasing order)?  The crossover advance launches one level at a time.
  c->by_level = true;
  c->lvl_first[0] = c->lvl_first[1] = 0; c->lvl_count[0] = c->lvl_count[1] = 0;
  for (int p = 0; p < np; p++) {
    if (p > 0 && c->level[p] < c->level[p - 1]) c->by_level = false;
    if (c->lvl_count[c->level[p]]++ == 0) c->lvl_first[c->level[p]] = p;
  }
  c->have_blocks = true;
  if (c->have_ws) return upload_lists(c);
  return JANC_OK;
}

// ------------------------------------------------------------------ state in / out
static dim3 cell_grid(const janc_ctx *c, int threads, int ny) {
  return dim3((unsigned)((c->ncell + threads - 1) / threads), (unsigned)ny, 1);
}

static dim3 pack_grid(const janc_ctx *c, int nfields_total) {
  return dim3((unsigned)((c->ncell + 255) / 256) * (unsigned)nfields_total, 1, 1);
}

extern "C" int janc_set_state(janc_ctx *c, const double *U, const double *Tg, int on_device) {
  if (!c || !U) return JANC_EINVAL;
  if (!c->have_ws) { c->err = "bind a workspace first"; return JANC_ESTATE; }
  CK(cudaSetDevice(c->device));
  const size_t nU = (size_t)c->np * c->nvar * c->ncell, nT = (size_t)c->np * c->ncell;
  const double *dU = U, *dT = Tg;
  if (!on_device) {
    CK(cudaMemcpyAsync(c->stageU, U, nU * 8, cudaMemcpyHostToDevice, c->stream));
    dU = c->stageU;
    if (Tg) { CK(cudaMemcpyAsync(c->stageT, Tg, nT * 8, cudaMemcpyHostToDevice, c->stream)); dT = c->stageT; }
  }
  k_pack<<<pack_grid(c, c->np * c->nvar), 256, 0, c->stream>>>(c->P, dU, c->A, c->nvar, 0, 0.0);
  k_pack<<<pack_grid(c, c->np), 256, 0, c->stream>>>(c->P, dT, c->P.T, 1, 0, 1000.0);
  c->launches += 2;
  CK(cudaMemsetAsync(c->P.flag, 0, 4, c->stream));
  CK(cudaMemsetAsync(c->P.slots, 0, JANC_NSLOT * 8, c->stream));
  CK(cudaMemsetAsync(c->P.scal, 0, 4 * 8, c->stream));
  c->parity = 0;
  CK(cudaGetLastError());
  if (!on_device) CK(cudaStreamSynchronize(c->stream));   // host buffers may be reused by the caller
  c->have_state = true;
  return JANC_OK;
}

static int read_flag(janc_ctx *c) {
  int flag = 0;
  CK(cudaMemcpyAsync(&flag, c->P.flag, 4, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  CK(cudaGetLastError());
  return flag ? JANC_ENONFINITE : JANC_OK;
}

extern "C" int janc_status(janc_ctx *c) {
  if (!c) return JANC_EINVAL;
  if (!c->have_ws) return JANC_ESTATE;
  return read_flag(c);
}

extern "C" int janc_get_state(janc_ctx *c, double *U, double *T, int on_device) {
  if (!c) return JANC_EINVAL;
  if (!c->have_state) { c->err = "no state"; return JANC_ESTATE; }
  CK(cudaSetDevice(c->device));
  const size_t nU = (size_t)c->np * c->nvar * c->ncell, nT = (size_t)c->np * c->ncell;
  if (U) {
    double *dst = on_device ? U : c->stageU;
    k_pack<<<pack_grid(c, c->np * c->nvar), 256, 0, c->stream>>>(c->P, c->A, dst, c->nvar, 1, 0.0);
    c->launches++;
    if (!on_device) CK(cudaMemcpyAsync(U, c->stageU, nU * 8, cudaMemcpyDeviceToHost, c->stream));
  }
  if (T) {
    double *dst = on_device ? T : c->stageT;
    k_pack<<<pack_grid(c, c->np), 256, 0, c->stream>>>(c->P, c->P.T, dst, 1, 1, 0.0);
    c->launches++;
    if (!on_device) CK(cudaMemcpyAsync(T, c->stageT, nT * 8, cudaMemcpyDeviceToHost, c->stream));
  }
  return read_flag(c);
}

// ------------------------------------------------------------------ the step
struct Prof {                       // optional per-phase timing of one step (CUDA events on the stream)
  std::vector<cudaEvent_t> ev;
  std::vector<int> phase;
};

static void prof_mark(janc_ctx *c, Prof *pf, int phase) {
  if (!pf) return;
  cudaEvent_t e;
  cudaEventCreate(&e);
  cudaEventRecord(e, c->stream);
  pf->ev.push_back(e);
  pf->phase.push_back(phase);
}

// every kernel launch of the step goes through here: counts it and keeps the first failure for the calling ABI function
static void note_launch(janc_ctx *c, cudaError_t e) {
  if (e != cudaSuccess && c->launch_err == cudaSuccess) c->launch_err = e;
  c->launches++;
}
static int take_launch_error(janc_ctx *c) {
  if (c->launch_err == cudaSuccess) return JANC_OK;
  c->err = std::string("kernel launch failed: ") + cudaGetErrorString(c->launch_err);
  c->launch_err = cudaSuccess;
  cudaGetLastError();
  return JANC_ECUDA;
}
// dynamic shared-memory limit of a kernel, once per context (= per device)
static void smem_attr(janc_ctx *c, const void *fn, size_t bytes) {
  if (c->attr_done.count(fn)) return;
  const cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e != cudaSuccess && c->launch_err == cudaSuccess) c->launch_err = e;
  c->attr_done.insert(fn);
}

template <int NS>
static void launch_prim(janc_ctx *c, const double *U, int reduce, int slot_base, double *dbgc) {
  k_prim<NS><<<cell_grid(c, 256, c->actn), 256, 0, c->stream>>>(c->P, U, reduce, slot_base, dbgc);
}
static void do_prim(janc_ctx *c, const double *U, int reduce, int slot_base, double *dbgc, Prof *pf) {
  if (c->jit_prim) {
    const Params &P = c->P;
    PrimArgs a{U, P.T, P.p, P.vel, dbgc, P.slots, P.level, P.flag, P.n[0], P.n[1], P.n[2], P.G[0], P.G[1], P.G[2],
               P.st[0], P.st[1], P.st[2], P.pc, P.np, reduce, slot_base, c->act0};
    void *args[] = {&a};
    note_launch(c, cudaLaunchKernel((const void *)c->jit_prim, cell_grid(c, 256, c->actn), dim3(256, 1, 1), args, 0, c->stream));
    prof_mark(c, pf, 0);
    return;
  }
  switch (c->ns) {
    case 1: launch_prim<1>(c, U, reduce, slot_base, dbgc); break;
    case 2: launch_prim<2>(c, U, reduce, slot_base, dbgc); break;
    case 9: launch_prim<9>(c, U, reduce, slot_base, dbgc); break;
    case 20: launch_prim<20>(c, U, reduce, slot_base, dbgc); break;
    default: launch_prim<0>(c, U, reduce, slot_base, dbgc); break;
  }
  note_launch(c, cudaGetLastError());
  prof_mark(c, pf, 0);
}

// 2-D patches of at most 16 x 16 cells, and small 2-D grids (launch-bound): the flux kernel gathers its halo itself
// (flux.cuh, GATHER); no ghost fill
static bool small_grid(const janc_ctx *c) { return (long long)c->np * c->ncell < 600000; }
static bool gather_mode(const janc_ctx *c) {
  if (c->P.bc_lo[0] == JANC_BC_EXCHANGE || c->P.bc_hi[0] == JANC_BC_EXCHANGE) return false;   // halos arrive in the ghost cells
  return c->opt.halo_in_kernel && c->g.ndim == 2 && ((c->P.n[0] <= 16 && c->P.n[1] <= 16) || small_grid(c));
}

// only_lev < 0: every level, coarse first (level 1 injects from its padded parent); else just that level
static void do_ghost(janc_ctx *c, double *U, Prof *pf, int only_lev = -1) {
  if (gather_mode(c)) return;
  const int nd = c->g.ndim;
  int amax = 1;
  for (int d = 0; d < nd; d++) {
    int a = 1;
    for (int e = 0; e < nd; e++) if (e != d) a *= c->P.n[e];
    if (a > amax) amax = a;
  }
  const long long total = (long long)2 * nd * JANC_NG * amax * ((c->nvar + 2 + nd + GHOST_FPT - 1) / GHOST_FPT);
  dim3 grid((unsigned)((total + 255) / 256), (unsigned)c->np, 1);
  for (int lev = 0; lev < c->g.n_levels; lev++) {
    if (only_lev >= 0 && lev != only_lev) continue;
    k_ghost<<<grid, 256, 0, c->stream>>>(c->P, U, lev, amax);
    note_launch(c, cudaGetLastError());
  }
  prof_mark(c, pf, 1);
}

template <int NDIM, int TX, int TY, int TZ, int SEG>
static void launch_flux(janc_ctx *c, const double *Uk, const double *U0, double *Uout, int slot_base, double coef) {
  using C = FluxCfg<NDIM, TX, TY, TZ, SEG>;
  const Params &P = c->P;
  smem_attr(c, (const void *)k_flux_rk<NDIM, TX, TY, TZ, SEG>, C::SMEM);
  const unsigned tiles = (unsigned)(((P.n[0] + TX - 1) / TX) * ((P.n[1] + TY - 1) / TY) * ((P.n[2] + TZ - 1) / TZ));
  k_flux_rk<NDIM, TX, TY, TZ, SEG><<<dim3(tiles, (unsigned)c->actn, 1), C::NT, C::SMEM, c->stream>>>(P, Uk, U0, Uout, slot_base, coef);
}

template <int TX, int TY, int SEG, bool GATHER = false>
static void launch_flux2(janc_ctx *c, const double *Uk, const double *U0, double *Uout, int slot_base, double coef) {
  using C = Flux2Cfg<TX, TY, SEG, GATHER>;
  const Params &P = c->P;
  smem_attr(c, (const void *)k_flux_rk2<TX, TY, SEG, GATHER>, C::SMEM);
  const unsigned tiles = (unsigned)(((P.n[0] + TX - 1) / TX) * ((P.n[1] + TY - 1) / TY));
  k_flux_rk2<TX, TY, SEG, GATHER><<<dim3(tiles, (unsigned)c->actn, 1), C::NT, C::SMEM, c->stream>>>(P, Uk, U0, Uout, slot_base, coef);
}

static void do_flux(janc_ctx *c, const double *Uk, const double *U0, double *Uout, int slot_base, double coef, Prof *pf) {
  const Params &P = c->P;
  if (c->g.ndim == 1) launch_flux<1, 128, 1, 1, 4>(c, Uk, U0, Uout, slot_base, coef);
  else if (c->g.ndim == 2) {
    const bool tiny = c->P.n[0] <= 16 && c->P.n[1] <= 16;
    if (gather_mode(c) && tiny) launch_flux2<16, 16, 4, true>(c, Uk, U0, Uout, slot_base, coef);   // AMR patches: halo gathered in-kernel; 2 warps per patch
    else if (gather_mode(c)) launch_flux2<32, 16, 4, true>(c, Uk, U0, Uout, slot_base, coef);   // small grids: 4x the CTAs, no ghost launches
    else if (c->opt.tma && c->have_tma) {     // materialised ghosts: one TMA box per field
      const int t = tile2d(c);
      if (t == 2) launch_flux2_tma<16, 16, 4>(c, Uk, U0, Uout, slot_base, coef);
      else if (t == 1) launch_flux2_tma<32, 16, 4>(c, Uk, U0, Uout, slot_base, coef);
      else launch_flux2_tma<64, 16, 8>(c, Uk, U0, Uout, slot_base, coef);
    }
    else if (c->P.n[0] <= 32) launch_flux2<32, 16, 4, false>(c, Uk, U0, Uout, slot_base, coef);   // patches of <= 32 columns with materialised ghosts
    else launch_flux2<64, 16, 8>(c, Uk, U0, Uout, slot_base, coef);
  } else if (c->opt.tma && c->have_tma3) launch_flux3_tma<JANC_F3T>(c, Uk, U0, Uout, slot_base, coef);   // boxes by TMA, two units ahead
  else launch_flux<3, 16, 8, 8, 8>(c, Uk, U0, Uout, slot_base, coef);   // 128 threads, 39 KB: 4 independent CTAs per SM overlap stage / walk
  note_launch(c, cudaGetLastError());
  prof_mark(c, pf, 2);
}

template <int NS>
static void launch_chem(janc_ctx *c, double *U) {
  k_chem<NS><<<cell_grid(c, 128, c->actn), 128, 0, c->stream>>>(c->P, U);
}
template <int NS>
static void launch_chem_reg(janc_ctx *c, double *U) {
  constexpr int NT = 64;
  const size_t smem = (size_t)(NS + 2 * c->nr + c->mech.ntb) * NT * sizeof(double);
  smem_attr(c, (const void *)k_chem_reg<NS, NT>, 227 * 1024);
  k_chem_reg<NS, NT><<<cell_grid(c, NT, c->actn), NT, smem, c->stream>>>(c->P, U);
}
static void do_chem(janc_ctx *c, double *U, Prof *pf) {
  if (c->jit_kernel) {
    const Params &P = c->P;
    // role-warp kernel: T* = T(U*) from the bandwidth-bound cons->prim kernel (chemgen_roles.h, roles_newton_ref)
    if (c->jit_chem_mode == 3 && c->opt.roles_newton_prim) do_prim(c, U, 0, 0, nullptr, pf);   // timed as cons->prim (phase 0)
    ChemArgs a{U, P.T, P.scal, P.flag, P.n[0], P.n[1], P.n[2], P.G[0], P.G[1], P.G[2], P.st[0], P.st[1], P.st[2], P.pc, c->actn, c->act0, P.dt_scale};
    void *args[] = {&a};
    dim3 grid = cell_grid(c, c->jit_chem_cells, c->actn);
    if (c->jit_chem_mode == 3) {      // persistent CTAs, one per SM, each takes 32-cell turns
      const long long turns = (long long)grid.x * grid.y;
      grid = dim3((unsigned)(turns < c->num_sms ? turns : c->num_sms), 1, 1);
    }
    note_launch(c, cudaLaunchKernel((const void *)c->jit_kernel, grid, dim3(c->jit_chem_nt, 1, 1), args, c->jit_chem_smem, c->stream));
    prof_mark(c, pf, 3);
    return;
  }
  switch (c->ns) {
    case 2: launch_chem_reg<2>(c, U); break;
    case 9: launch_chem_reg<9>(c, U); break;
    case 20: launch_chem<20>(c, U); break;
    default: launch_chem<0>(c, U); break;
  }
  note_launch(c, cudaGetLastError());
  prof_mark(c, pf, 3);
}

// explicit variant: add coef dt S(Uk) to the stage result on the species rows
static void do_src(janc_ctx *c, const double *Uk, double *Uout, double coef, Prof *pf) {
  const Params &P = c->P;
  SrcArgs a{Uk, Uout, P.T, P.scal, P.n[0], P.n[1], P.n[2], P.G[0], P.G[1], P.G[2], P.st[0], P.st[1], P.st[2], P.pc, coef * P.dt_scale, c->act0};
  void *args[] = {&a};
  note_launch(c, cudaLaunchKernel((const void *)c->jit_src, cell_grid(c, 128, c->actn), dim3(128, 1, 1), args, 0, c->stream));
  prof_mark(c, pf, 3);
}

static void set_active(janc_ctx *c, int first, int count, double dt_scale) {
  c->act0 = first; c->actn = count;
  c->P.patch0 = first; c->P.dt_scale = dt_scale;
}

// advance_flux (TVD-RK3 over rhs) + advance_source_term of the active patches, A -> A.
// sub: which reduction-slot set the stages use; first_prim: evaluate update_aux of A (false: the caller's evaluation at
// the start of the step is still valid for these patches); glev: ghost-fill level (-1: all levels, coarse first)
static void advance_active(janc_ctx *c, int par, int sub, bool first_prim, int glev, int flags, Prof *pf) {
  const bool esrc = (flags & 2) && c->jit_src && c->ns > 1 && c->nr > 0;   // source inside every stage
  if (first_prim) do_prim(c, c->A, 1, SLOTX(par, sub, 0, 0, 0), nullptr, pf);
  do_ghost(c, c->A, pf, glev);
  do_flux(c, c->A, c->A, c->B, SLOTX(par, sub, 0, 0, 0), 1.0, pf);
  if (esrc) do_src(c, c->A, c->B, 1.0, pf);
  do_prim(c, c->B, 1, SLOTX(par, sub, 1, 0, 0), nullptr, pf);
  do_ghost(c, c->B, pf, glev);
  do_flux(c, c->B, c->A, c->C, SLOTX(par, sub, 1, 0, 0), 0.25, pf);
  if (esrc) do_src(c, c->B, c->C, 0.25, pf);
  // stage 3 writes U* over U^n in place: each cell reads its own U^n before writing
  do_prim(c, c->C, 1, SLOTX(par, sub, 2, 0, 0), nullptr, pf);
  do_ghost(c, c->C, pf, glev);
  do_flux(c, c->C, c->A, c->A, SLOTX(par, sub, 2, 0, 0), 2.0 / 3.0, pf);
  if (esrc) do_src(c, c->C, c->A, 2.0 / 3.0, pf);
  // advance_source_term: T* inside the chemistry kernel; explicit variant: only refresh aux
  const bool chem = !(flags & 3) && c->ns > 1 && c->nr > 0;
  if (chem) do_chem(c, c->A, pf);
  else do_prim(c, c->A, 0, 0, nullptr, pf);
}

// advance_one_step: cfl -> advance_flux (RK3 over rhs) -> advance_source_term.
// flags bit 2: crossover advance of a two-level block list (Fig 2a, reading B9): two half steps of level 1
// with its coarse-fine ghosts taken from the level-0 state at the start of the step, then one step of level 0.
static void step_once(janc_ctx *c, double cfl, double dt_fixed, int flags, Prof *pf) {
  const int par = c->parity;
  const bool crossover = (flags & 4) && c->g.n_levels == 2 && c->lvl_count[1] > 0;
  prof_mark(c, pf, -1);
  // update_aux on U^n of every patch (also the cfl() evaluation), then dt
  set_active(c, 0, c->np, 1.0);
  do_prim(c, c->A, 1, SLOTX(par, 0, 0, 0, 0), nullptr, pf);
  k_dt<<<1, 32, 0, c->stream>>>(c->P, par, cfl, dt_fixed, crossover ? (double)c->g.ratio : 1.0);
  note_launch(c, cudaGetLastError());
  prof_mark(c, pf, 0);
  if (!crossover) {
    advance_active(c, par, 0, false, -1, flags, pf);
  } else {
    // level 0 keeps its state at t^n in all three RK registers while level 1 runs: stages 2 and 3 of level 1 read
    // their coarse-fine ghosts from B and C
    do_ghost(c, c->A, pf, 0);
    const size_t off = (size_t)c->lvl_first[0] * c->nvar * c->P.pc, cnt = (size_t)c->lvl_count[0] * c->nvar * c->P.pc * sizeof(double);
    cudaMemcpyAsync(c->B + off, c->A + off, cnt, cudaMemcpyDeviceToDevice, c->stream);
    cudaMemcpyAsync(c->C + off, c->A + off, cnt, cudaMemcpyDeviceToDevice, c->stream);
    prof_mark(c, pf, 1);
    set_active(c, c->lvl_first[1], c->lvl_count[1], 0.5);
    advance_active(c, par, 0, false, 1, flags, pf);
    advance_active(c, par, 1, true, 1, flags, pf);
    set_active(c, c->lvl_first[0], c->lvl_count[0], 1.0);
    advance_active(c, par, 0, false, 0, flags, pf);
    set_active(c, 0, c->np, 1.0);
  }
  if (c->g.n_levels > 1) {
    const int r = c->g.ratio, nd = c->g.ndim;
    long long nc = c->ncell;
    for (int d = 0; d < nd; d++) nc /= r;
    dim3 grid((unsigned)((nc * c->nvar + 255) / 256), (unsigned)c->np, 1);
    k_average_down<<<grid, 256, 0, c->stream>>>(c->P, c->A);
    note_launch(c, cudaGetLastError());
    prof_mark(c, pf, 4);
  }
  c->parity = 1 - par;
}

static void invalidate_graphs(janc_ctx *c) {
  for (auto &G : c->graph) { if (G.exec) cudaGraphExecDestroy(G.exec); G.exec = nullptr; }
  c->warmed = false;
}

// One step through the cached graph of the current parity; the first step after any (re)configuration runs eagerly
// (it also sets the kernels' shared-memory attributes), and any capture problem switches the context to eager launches.
static void run_step(janc_ctx *c, double cfl, double dt_fixed, int flags) {
  if (!c->use_graph || !c->warmed) { step_once(c, cfl, dt_fixed, flags, nullptr); c->warmed = true; return; }
  const int par = c->parity;
  janc_ctx::StepGraph &G = c->graph[par];
  if (!G.exec || G.cfl != cfl || G.dt != dt_fixed || G.flags != flags) {
    if (G.exec) { cudaGraphExecDestroy(G.exec); G.exec = nullptr; }
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) c->cap_stream = nullptr;
    bool ok = c->cap_stream != nullptr;
    const cudaStream_t user = c->stream;
    const long long l0 = c->launches;
    cudaGraph_t g = nullptr;
    if (ok) ok = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed) == cudaSuccess;
    if (ok) {
      c->stream = c->cap_stream;
      step_once(c, cfl, dt_fixed, flags, nullptr);
      c->stream = user;
      ok = cudaStreamEndCapture(c->cap_stream, &g) == cudaSuccess && g != nullptr;
      G.launches = c->launches - l0;
      c->launches = l0;
      c->parity = par;
    }
    if (ok) ok = cudaGraphInstantiate(&G.exec, g, 0) == cudaSuccess;
    if (g) cudaGraphDestroy(g);
    if (!ok) {
      const cudaError_t e = cudaGetLastError();
      G.exec = nullptr;
      c->use_graph = false;
      c->jit_log += std::string(" [step graph: capture / instantiate failed (") + cudaGetErrorString(e) + "), eager launches from here on]";
      step_once(c, cfl, dt_fixed, flags, nullptr);
      return;
    }
    G.cfl = cfl; G.dt = dt_fixed; G.flags = flags;
  }
  if (const cudaError_t e = cudaGraphLaunch(G.exec, c->stream); e != cudaSuccess) {
    cudaGetLastError();
    c->use_graph = false;
    c->jit_log += std::string(" [step graph: launch failed (") + cudaGetErrorString(e) + "), eager launches from here on]";
    step_once(c, cfl, dt_fixed, flags, nullptr);
    return;
  }
  c->launches += G.launches;
  c->parity = 1 - par;
}

static int check_ready(janc_ctx *c) {
  if (!c) return JANC_EINVAL;
  if (!c->have_state) { c->err = "no state"; return JANC_ESTATE; }
  if (c->g.n_patches > 0 && !c->have_blocks) { c->err = "block mode needs janc_set_blocks"; return JANC_ESTATE; }
  return JANC_OK;
}

extern "C" int janc_step(janc_ctx *c, int nsteps, double cfl, double dt_fixed, int flags, double *t_advanced) {
  int rc = check_ready(c);
  if (rc) return rc;
  if (nsteps < 0 || (!(cfl > 0.0) && !(dt_fixed > 0.0))) { c->err = "need cfl > 0 or dt_fixed > 0"; return JANC_EINVAL; }
  if ((flags & 4) && c->g.n_levels == 2 && !c->by_level) {
    c->err = "the crossover advance needs the patches ordered by level (all level-0 patches first)";
    return JANC_EINVAL;
  }
  if ((flags & 2) && c->ns > 1 && c->nr > 0) jit_setup_source(c);
  if ((flags & 2) && c->ns > 1 && c->nr > 0 && !c->jit_src) {
    c->err = "explicit source variant needs the run-time specialised kernel (NVRTC): " + c->jit_log;
    return JANC_ESTATE;
  }
  CK(cudaSetDevice(c->device));
  MechLock mech_lock(c);
  rc = upload_mech(c);
  if (rc) return rc;
  double t0 = 0.0;
  if (t_advanced) {
    CK(cudaMemcpyAsync(&t0, c->P.scal + 1, 8, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
  }
  for (int s = 0; s < nsteps; s++) run_step(c, cfl, dt_fixed, flags);
  if ((rc = take_launch_error(c)) != JANC_OK) return rc;
  CK(cudaGetLastError());
  if (t_advanced) {
    double t1 = 0.0;
    CK(cudaMemcpyAsync(&t1, c->P.scal + 1, 8, cudaMemcpyDeviceToHost, c->stream));
    rc = read_flag(c);
    *t_advanced = t1 - t0;
    return rc;
  }
  return JANC_OK;
}

// ------------------------------------------------------------------ x-slab decomposition
// One step cut into the parts between which the slabs of a decomposed grid talk to each other; the caller (binding /
// slab.py: torch.distributed plumbing) supplies the max all-reduce of the reduction slots and the halo exchange.
static double *rk_register(janc_ctx *c, int which) { return which == 0 ? c->A : which == 1 ? c->B : c->C; }

extern "C" int janc_step_part(janc_ctx *c, int part, int stage, double cfl, double dt_fixed, int flags) {
  int rc = check_ready(c);
  if (rc) return rc;
  if (c->g.n_patches > 0 || stage < 0 || stage > 2 || (flags & ~1)) { c->err = "janc_step_part: uniform grid, stage 0..2, flags 0 or 1"; return JANC_EINVAL; }
  CK(cudaSetDevice(c->device));
  MechLock mech_lock(c);
  rc = upload_mech(c);
  if (rc) return rc;
  const int par = c->parity;
  set_active(c, 0, c->np, 1.0);
  double *Uk = rk_register(c, stage);
  static const double coef[3] = {1.0, 0.25, 2.0 / 3.0};
  switch (part) {
    case JANC_PART_PRIM:    // update_aux of the stage state + its max(|u_d| + c) into the reduction slots
      do_prim(c, Uk, 1, SLOTX(par, 0, stage, 0, 0), nullptr, nullptr);
      break;
    case JANC_PART_DT:      // cfl() from the (all-reduced) slots of stage 0
      if (!(cfl > 0.0) && !(dt_fixed > 0.0)) { c->err = "need cfl > 0 or dt_fixed > 0"; return JANC_EINVAL; }
      k_dt<<<1, 32, 0, c->stream>>>(c->P, par, cfl, dt_fixed, 1.0);
      note_launch(c, cudaGetLastError());
      break;
    case JANC_PART_GHOST:   // physical boundaries of the stage state (exchange faces are left to janc_halo)
      do_ghost(c, Uk, nullptr);
      break;
    case JANC_PART_FLUX:    // fluxes + divergence + RK stage: A -> B, B -> C, C -> A
      do_flux(c, Uk, c->A, stage == 0 ? c->B : stage == 1 ? c->C : c->A, SLOTX(par, 0, stage, 0, 0), coef[stage], nullptr);
      break;
    case JANC_PART_SOURCE:  // advance_source_term (or only update_aux with flags bit 0), end of the step
      if (!(flags & 1) && c->ns > 1 && c->nr > 0) do_chem(c, c->A, nullptr);
      else do_prim(c, c->A, 0, 0, nullptr, nullptr);
      c->parity = 1 - par;
      break;
    default: c->err = "janc_step_part: unknown part"; return JANC_EINVAL;
  }
  if ((rc = take_launch_error(c)) != JANC_OK) return rc;
  CK(cudaGetLastError());
  return JANC_OK;
}

extern "C" size_t janc_halo_doubles(const janc_ctx *c) {
  if (!c || !c->have_mech) return 0;
  return (size_t)(c->nvar + 2 + c->g.ndim) * JANC_NG * c->P.n[1] * c->P.n[2];
}

extern "C" int janc_halo(janc_ctx *c, int stage, int side, double *buf_dev, int unpack) {
  int rc = check_ready(c);
  if (rc) return rc;
  if (c->g.n_patches > 0 || stage < 0 || stage > 2 || side < 0 || side > 1 || !buf_dev) return JANC_EINVAL;
  CK(cudaSetDevice(c->device));
  const size_t n = janc_halo_doubles(c);
  set_active(c, 0, c->np, 1.0);
  k_halo<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->P, rk_register(c, stage), buf_dev, side, unpack);
  note_launch(c, cudaGetLastError());
  return take_launch_error(c);
}

extern "C" int janc_reduction_slots(const janc_ctx *c, size_t *byte_offset, size_t *count) {
  if (!c || !c->have_ws || !byte_offset || !count) return JANC_EINVAL;
  *byte_offset = (size_t)((const char *)c->P.slots - (const char *)c->A);     // A is the first piece of the workspace
  *count = JANC_NSLOT;
  return JANC_OK;
}

// ------------------------------------------------------------------ regridding (B12)
extern "C" int janc_regrid_plan(janc_ctx *c, double thr, int nbuf, int32_t *np_new, int32_t *level, int32_t *nbr, int32_t *parent) {
  int rc = check_ready(c);
  if (rc) return rc;
  if (!np_new || !level || !nbr || !parent || nbuf < 0 || nbuf > 64) return JANC_EINVAL;
  const int nd = c->g.ndim, nf = 2 * nd, nsub = 1 << nd, np = c->np;
  int n0 = 0;
  while (n0 < np && c->level[n0] == 0) n0++;
  if (c->g.n_patches <= 0 || c->g.n_levels != 2 || !c->by_level || n0 == 0) {
    c->err = "janc_regrid_plan: a two-level block list with the level-0 patches first";
    return JANC_EINVAL;
  }
  CK(cudaSetDevice(c->device));
  // 1. criterion on the level-0 state with its ghosts filled; 2. nbuf box dilations (B holds the marks: free between steps)
  set_active(c, 0, np, 1.0);
  {
    int amax = 1;
    for (int d = 0; d < nd; d++) { int a = 1; for (int e = 0; e < nd; e++) if (e != d) a *= c->P.n[e]; if (a > amax) amax = a; }
    const long long total = (long long)2 * nd * JANC_NG * amax * ((c->nvar + 2 + nd + GHOST_FPT - 1) / GHOST_FPT);
    k_ghost<<<dim3((unsigned)((total + 255) / 256), (unsigned)np, 1), 256, 0, c->stream>>>(c->P, c->A, 0, amax);
    note_launch(c, cudaGetLastError());
  }
  unsigned char *m0 = (unsigned char *)c->B, *m1 = m0 + align_up((size_t)n0 * c->P.pc, 256);
  int *d_flags = (int *)(m1 + align_up((size_t)n0 * c->P.pc, 256));
  const dim3 grid = cell_grid(c, 256, n0);
  CK(cudaMemsetAsync(m0, 0, 2 * align_up((size_t)n0 * c->P.pc, 256) + (size_t)n0 * nsub * 4, c->stream));
  k_regrid_mark<<<grid, 256, 0, c->stream>>>(c->P, c->A, m0, thr);
  note_launch(c, cudaGetLastError());
  for (int pass = 0; pass < nbuf; pass++) {
    k_regrid_dilate<<<grid, 256, 0, c->stream>>>(c->P, m0, m1);
    note_launch(c, cudaGetLastError());
    unsigned char *t_ = m0; m0 = m1; m1 = t_;
  }
  k_regrid_flags<<<grid, 256, 0, c->stream>>>(c->P, m0, d_flags);
  note_launch(c, cudaGetLastError());
  std::vector<int> flags((size_t)n0 * nsub);
  CK(cudaMemcpyAsync(flags.data(), d_flags, flags.size() * 4, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  if ((rc = take_launch_error(c)) != JANC_OK) return rc;
  // 3. - 5. the new list (host): refined sub-regions in the order (parent, sub-index), neighbours through the parents
  std::vector<int> newid((size_t)n0 * nsub, -1), oldid((size_t)n0 * nsub, -1);
  for (int p = n0; p < np; p++) {
    const int *par = &c->parent[(size_t)p * (1 + nd)];
    int sidx = 0;
    for (int e = 0; e < nd; e++) sidx |= par[1 + e] << e;
    oldid[(size_t)par[0] * nsub + sidx] = p;
  }
  int np2 = n0;
  for (int q = 0; q < n0 * nsub; q++) if (flags[q]) newid[q] = np2++;
  c->rg_src.assign(np2, -1); c->rg_par.assign(np2, -1); c->rg_sub.assign(np2, 0);
  for (int p = 0; p < n0; p++) {
    level[p] = 0; c->rg_src[p] = p;
    for (int f = 0; f < nf; f++) nbr[p * nf + f] = c->nbr[(size_t)p * nf + f];
    for (int e = 0; e <= nd; e++) parent[p * (1 + nd) + e] = -1;
  }
  for (int p = 0; p < n0; p++)
    for (int sidx = 0; sidx < nsub; sidx++) {
      const int id = newid[(size_t)p * nsub + sidx];
      if (id < 0) continue;
      level[id] = 1;
      parent[id * (1 + nd)] = p;
      for (int e = 0; e < nd; e++) parent[id * (1 + nd) + 1 + e] = (sidx >> e) & 1;
      for (int d = 0; d < nd; d++)
        for (int side = 0; side < 2; side++) {
          const int bit = (sidx >> d) & 1;
          const bool inside = (side == 0) == (bit == 1);                 // the sibling across this face lies in the same parent
          const int k2 = inside ? p : c->nbr[(size_t)p * nf + 2 * d + side];
          nbr[id * nf + 2 * d + side] = k2 >= 0 ? newid[(size_t)k2 * nsub + (sidx ^ (1 << d))] : -1;
        }
      c->rg_src[id] = oldid[(size_t)p * nsub + sidx];
      c->rg_par[id] = p; c->rg_sub[id] = sidx;
    }
  *np_new = np2;
  return JANC_OK;
}

extern "C" int janc_regrid_fill(janc_ctx *c, double *U_new, double *T_new, int on_device) {
  int rc = check_ready(c);
  if (rc) return rc;
  if (!U_new || !T_new) return JANC_EINVAL;
  if (c->rg_src.empty()) { c->err = "janc_regrid_fill: no plan (call janc_regrid_plan first)"; return JANC_ESTATE; }
  CK(cudaSetDevice(c->device));
  const int np2 = (int)c->rg_src.size();
  const size_t nU = (size_t)np2 * c->nvar * c->ncell, nT = (size_t)np2 * c->ncell;
  // device scratch in B: the three int lists, then (host output only) the new arrays
  int *d_src = (int *)c->B, *d_par = d_src + np2, *d_sub = d_par + np2;
  double *dU = U_new, *dT = T_new;
  if (!on_device) {
    dU = (double *)((char *)c->B + align_up((size_t)3 * np2 * 4, 256));
    dT = dU + nU;
    const size_t need = align_up((size_t)3 * np2 * 4, 256) + (nU + nT) * 8, have = (size_t)c->np * c->nvar * c->P.pc * 8 * 2;   // B and C are contiguous
    if (need > have) { c->err = "janc_regrid_fill: the new list does not fit the scratch registers; pass device buffers"; return JANC_ENOMEM; }
  }
  CK(cudaMemcpyAsync(d_src, c->rg_src.data(), (size_t)np2 * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(d_par, c->rg_par.data(), (size_t)np2 * 4, cudaMemcpyHostToDevice, c->stream));
  CK(cudaMemcpyAsync(d_sub, c->rg_sub.data(), (size_t)np2 * 4, cudaMemcpyHostToDevice, c->stream));
  set_active(c, 0, c->np, 1.0);
  k_regrid_fill<<<cell_grid(c, 256, np2), 256, 0, c->stream>>>(c->P, c->A, d_src, d_par, d_sub, dU, dT);
  note_launch(c, cudaGetLastError());
  if (!on_device) {
    CK(cudaMemcpyAsync(U_new, dU, nU * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemcpyAsync(T_new, dT, nT * 8, cudaMemcpyDeviceToHost, c->stream));
  }
  CK(cudaStreamSynchronize(c->stream));
  return take_launch_error(c);
}

extern "C" int janc_last_dt(janc_ctx *c, double *dt) {
  if (!c || !dt) return JANC_EINVAL;
  if (!c->have_ws) return JANC_ESTATE;
  CK(cudaMemcpyAsync(dt, c->P.scal, 8, cudaMemcpyDeviceToHost, c->stream));
  CK(cudaStreamSynchronize(c->stream));
  return JANC_OK;
}

extern "C" int janc_profile_step(janc_ctx *c, double cfl, double dt_fixed, float *ms_out, int *n_out) {
  int rc = check_ready(c);
  if (rc) return rc;
  if (!ms_out) return JANC_EINVAL;
  CK(cudaSetDevice(c->device));
  MechLock mech_lock(c);
  rc = upload_mech(c);
  if (rc) return rc;
  Prof pf;
  step_once(c, cfl, dt_fixed, 0, &pf);
  if ((rc = take_launch_error(c)) != JANC_OK) { for (auto e : pf.ev) cudaEventDestroy(e); return rc; }
  CK(cudaStreamSynchronize(c->stream));
  for (int q = 0; q < 6; q++) { ms_out[q] = 0.f; if (n_out) n_out[q] = 0; }
  for (size_t e = 1; e < pf.ev.size(); e++) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, pf.ev[e - 1], pf.ev[e]);
    ms_out[pf.phase[e]] += ms;
    if (n_out) n_out[pf.phase[e]]++;
  }
  float tot = 0.f;
  cudaEventElapsedTime(&tot, pf.ev.front(), pf.ev.back());
  ms_out[5] = tot;
  if (n_out) n_out[5] = (int)pf.ev.size() - 1;
  for (auto e : pf.ev) cudaEventDestroy(e);
  return read_flag(c);
}

extern "C" int janc_debug_cons2prim(janc_ctx *c, double *T, double *p, double *cs, int on_device) {
  int rc = check_ready(c);
  if (rc) return rc;
  CK(cudaSetDevice(c->device));
  MechLock mech_lock(c);
  rc = upload_mech(c);
  if (rc) return rc;
  do_prim(c, c->A, 0, 0, c->dbgc, nullptr);
  if ((rc = take_launch_error(c)) != JANC_OK) return rc;
  const size_t nT = (size_t)c->np * c->ncell;
  double *srcs[3] = {c->P.T, c->P.p, c->dbgc};
  double *dsts[3] = {T, p, cs};
  for (int q = 0; q < 3; q++) {
    if (!dsts[q]) continue;
    double *dst = on_device ? dsts[q] : c->stageT;
    k_pack<<<pack_grid(c, c->np), 256, 0, c->stream>>>(c->P, srcs[q], dst, 1, 1, 0.0);
    c->launches++;
    if (!on_device) {
      CK(cudaMemcpyAsync(dsts[q], c->stageT, nT * 8, cudaMemcpyDeviceToHost, c->stream));
      CK(cudaStreamSynchronize(c->stream));
    }
  }
  return read_flag(c);
}

extern "C" int janc_measure_dfma_peak(int device, void *cuda_stream, double *dfma_per_s) {
  if (!dfma_per_s) return JANC_EINVAL;
  if (cudaSetDevice(device) != cudaSuccess) return JANC_ECUDA;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return JANC_ECUDA;
  double *d = nullptr;
  if (cudaMalloc(&d, 64) != cudaSuccess) return JANC_ECUDA;
  const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 4096;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  double best = 0.0;
  for (int rep = 0; rep < 6; rep++) {
    cudaEventRecord(e0, st);
    k_dfma<<<blocks, threads, 0, st>>>(d, iters);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(d); return JANC_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    double rate = (double)blocks * threads * iters * 64.0 / (ms * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  *dfma_per_s = best;
  return JANC_OK;
}

#include "static_scratch.cuh"   // janc_cfl_dt_static: the entry point that allocates nothing
