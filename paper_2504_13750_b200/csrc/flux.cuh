// flux.cuh -- x/y/z reconstruction + flux sweeps fused with the divergence and the RK stage.
// PAPER.md:288-295 (eq 4.11 Lax-Friedrichs splitting, WENO5 on 6 template points, 3 ghosts),
// :283-286 (eq 4.10 conservative difference), :297/:339 (TVD-RK3), :232 (F, G).
// Readings A1 (WENO5-JS, eps 1e-6, p 2), A2 (component-wise), A3/A20 (alpha per direction per
// level, from the stage state), A4 (increment form of SSP-RK3), A24 (x, y, z order).
//
// Work decomposition ("pencil walk"): a CTA owns a TX x TY x TZ tile of one patch and loops over the
// nvar components.  For each direction every thread walks a pencil of SEG consecutive cells along
// that direction and produces the SEG+1 face fluxes of the pencil from the SEG+6 cells it touches;
// first and second differences of the split fluxes are shared between neighbouring faces, so one
// face costs ~2 x 38 fp64 instructions and each split flux is evaluated once per pencil.
//   x: the tile rows (+3 ghosts each side) of 2f+- = F +- alpha U are staged once in shared memory
//      with coalesced loads; pencils then read them row-wise (odd pitch, conflict-free).
//   y, z: the tile extended by 3 cells along the sweep direction is staged the same way ([z][y][x], odd x pitch);
//      lanes run along x, so pencil reads are conflict-free.
// Pencil results (-dF/dx_d) are summed per cell in shared memory; a coalesced pass applies the RK stage (2-D kernel: the
// thread that walks a y pencil adds its result to the x part and applies the RK stage of its own cells, lanes along x).
// No flux array ever goes to HBM: per stage the kernel reads U^(k) (+ U^n) and writes U^(k+1).
//
// WENO5 in difference form.  With D_k = v_{k+1} - v_k (k = 0..3 over v_{-2..+2}):
//   beta_0 = 13/12 (D1-D0)^2 + 1/4 (3 D1 - D0)^2,  beta_1 = 13/12 (D2-D1)^2 + 1/4 (D1+D2)^2,
//   beta_2 = 13/12 (D3-D2)^2 + 1/4 (D3 - 3 D2)^2,
//   q_0 = v_0 + (5 D1 - 2 D0)/6,  q_1 = v_0 + (D1 + 2 D2)/6,  q_2 = v_0 + (4 D2 - D3)/6
// which is the Jiang-Shu formula of SURVEY 8(c) step 5 re-grouped (identical in exact arithmetic).
// The kernel reconstructs 2f+- (not f+-): beta scales by 4, so eps -> 4 eps keeps the weights those of f+-; beta is
// further carried as 4 beta, i.e. B_k = 16 eps + 13/3 (D_{k+1}-D_k)^2 + t_k^2 with t_0 = 3 D1 - D0, t_1 = D1 + D2,
// t_2 = D3 - 3 D2; the 1/2 is folded into 1/dx.  a_k = d_k/(eps+beta_k)^2 is evaluated as 10 d_k prod_{l!=k} B_l^2 over
// the common denominator (one reciprocal per reconstruction), and the q_k numerators re-use t_k:
//   5 D1 - 2 D0 = 2 t_0 - D1,   D1 + 2 D2 = t_1 + D2,   4 D2 - D3 = D2 - t_2.
// One reconstruction is 30 fp64 instructions (4 for its share of the differences, 21 below, half of the 10 that join
// the two reconstructions of a face over one reciprocal).
#pragma once
#include "common.cuh"
#include <type_traits>

#define JANC_WENO_EPS16 1.6e-5   // 16 * 1e-6, see above

// 1/x for normal, finite x > 0: MUFU seed (>= 20 bits) + one cubic step r (1 + e + e^2), e = 1 - x r  (error e^3 < 2^-60
// before rounding; no slow path).
__device__ __forceinline__ double rcp_pos(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  return fma(fma(e, e, e), r, r);
}

// 6 (q - v) = num / den of the reconstruction with differences D0..D3 about the centre value v (den >= 1e-18: the
// two reconstructions of a face share one reciprocal, of the product of their denominators);  S_k = 16 eps + 13/3 (D_{k+1}-D_k)^2
__device__ __forceinline__ void weno5_diff(double D0, double D1, double D2, double D3, double S0, double S1, double S2,
                                           double &num, double &den) {
  const double t0 = fma(3.0, D1, -D0), t1 = D1 + D2, t2 = fma(-3.0, D2, D3);
  double b0 = fma(t0, t0, S0), b1 = fma(t1, t1, S1), b2 = fma(t2, t2, S2);
  b0 *= b0; b1 *= b1; b2 *= b2;
  // 10 a_k = (b1 b2, 6 b0 b2, 3 b0 b1):  num = b1 b2 c0 + 3 b0 (2 b2 c1 + b1 c2),  den = b1 b2 + 3 b0 (2 b2 + b1)
  const double c0 = fma(2.0, t0, -D1), c1 = t1 + D2, c2 = D2 - t2;
  const double a0 = b1 * b2, h = 3.0 * b0, w = b2 + b2;
  num = fma(a0, c0, h * fma(w, c1, b1 * c2));
  den = fma(h, w + b1, a0);
}

// Face fluxes of one pencil, streamed: ld(k, fp2, fm2) returns 2f+ and 2f- of pencil cell k-3
// (k = 0..SEG+5); Fh[q], q = 0..SEG, is twice the numerical flux at the face between cells q-1 and q.
// Cell k is fetched just before the first face that needs it, so only a 6-cell window is live.
template <int SEG, class Load>
__device__ __forceinline__ void weno_faces(Load &&ld, double (&Fh)[SEG + 1]) {
  constexpr double K = 13.0 / 3.0;
  double P[SEG + 6], M[SEG + 6], dP[SEG + 5], dM[SEG + 5], sP[SEG + 4], sM[SEG + 4];
#pragma unroll
  for (int k = 0; k < 5; k++) ld(k, P[k], M[k]);
#pragma unroll
  for (int k = 0; k < 4; k++) { dP[k] = P[k + 1] - P[k]; dM[k] = M[k + 1] - M[k]; }
#pragma unroll
  for (int k = 0; k < 3; k++) {
    const double s = dP[k + 1] - dP[k], r = dM[k + 1] - dM[k];
    sP[k] = fma(K * s, s, JANC_WENO_EPS16);
    sM[k] = fma(K * r, r, JANC_WENO_EPS16);
  }
#pragma unroll
  for (int q = 0; q <= SEG; q++) {
    ld(q + 5, P[q + 5], M[q + 5]);
    dP[q + 4] = P[q + 5] - P[q + 4]; dM[q + 4] = M[q + 5] - M[q + 4];
    const double s = dP[q + 4] - dP[q + 3], r = dM[q + 4] - dM[q + 3];
    sP[q + 3] = fma(K * s, s, JANC_WENO_EPS16);
    sM[q + 3] = fma(K * r, r, JANC_WENO_EPS16);
    double np, dp, nm, dm;
    // plus part: stencil cells q-3..q+1 (array q..q+4), upwind centre = array q+2
    weno5_diff(dP[q], dP[q + 1], dP[q + 2], dP[q + 3], sP[q], sP[q + 1], sP[q + 2], np, dp);
    // minus part: mirror image, cells q+2..q-2 (array q+5..q+1), centre = array q+3
    weno5_diff(-dM[q + 4], -dM[q + 3], -dM[q + 2], -dM[q + 1], sM[q + 3], sM[q + 2], sM[q + 1], nm, dm);
    Fh[q] = fma(fma(nm, dp, np * dm) * rcp_pos(dp * dm), 1.0 / 6.0, P[q + 2] + M[q + 3]);
  }
}

// physical flux component m of direction d from (U_m, u_d, p):  F = (U_m + cE p) u_d + cM p  with
// (cE, cM) = (0,1) for the normal momentum, (1,0) for the energy, (0,0) otherwise.
__device__ __forceinline__ void split2(double Um, double ud, double p, double cE, double cM, double alpha,
                                       double &fp2, double &fm2) {
  const double F = fma(fma(cE, p, Um), ud, cM * p);
  fp2 = fma(alpha, Um, F);
  fm2 = fma(-alpha, Um, F);
}

// the same for a component without a pressure term (cE = cM = 0): bit-for-bit split2's result
__device__ __forceinline__ void split_adv(double Um, double ud, double alpha, double &fp2, double &fm2) {
  const double F = Um * ud;
  fp2 = fma(alpha, Um, F);
  fm2 = fma(-alpha, Um, F);
}

template <int NDIM, int TX, int TY, int TZ, int SEG>
struct FluxCfg {
  static constexpr int NT = TX * TY * TZ / SEG;          // threads per CTA = pencils per direction
  static constexpr int ROWS = TY * TZ;
  static constexpr int XP = ((TX + 6) | 1);              // odd pitch of the staged x rows
  static constexpr int LP = TX | 1;                      // odd pitch of the per-cell accumulator and of the y / z stages
  static constexpr int NOUT = TX * TY * TZ;
  static constexpr int SX = ROWS * XP;                                    // staged cells, x sweep
  static constexpr int SY = NDIM > 1 ? TZ * (TY + 6) * LP : 0;            //               y sweep: [TZ][TY+6][LP]
  static constexpr int SZ = NDIM > 2 ? (TZ + 6) * TY * LP : 0;            //               z sweep: [TZ+6][TY][LP]
  static constexpr int STAGE = SX > SY ? (SX > SZ ? SX : SZ) : (SY > SZ ? SY : SZ);
  static constexpr size_t SMEM = (size_t)(2 * STAGE + ROWS * LP) * sizeof(double);
  static_assert(TX % SEG == 0 && (NDIM < 2 || TY % SEG == 0) && (NDIM < 3 || TZ % SEG == 0), "tile % SEG");
  static_assert(NT >= 32 && NT <= 1024, "threads");
};

// grid: (tiles of one patch, np).  Uout = U0 + coef * ((Uk - U0) + dt * L(Uk)).
template <int NDIM, int TX, int TY, int TZ, int SEG>
__global__ void __launch_bounds__(TX * TY * TZ / SEG, 512 / (TX * TY * TZ / SEG) > 0 ? 512 / (TX * TY * TZ / SEG) : 1)
k_flux_rk(Params P, const double *__restrict__ Uk, const double *U0, double *Uout, int slot_base, double coef) {
  using C = FluxCfg<NDIM, TX, TY, TZ, SEG>;
  constexpr int NT = C::NT;
  extern __shared__ double flux_smem[];
  double *sFp = flux_smem, *sFm = sFp + C::STAGE, *sL = sFm + C::STAGE;

  const int tid = threadIdx.x;
  const int patch = blockIdx.y + P.patch0;
  const int lev = P.level[patch];
  const int ntx = (P.n[0] + TX - 1) / TX, nty = (P.n[1] + TY - 1) / TY;
  const int o0 = (blockIdx.x % ntx) * TX, o1 = ((blockIdx.x / ntx) % nty) * TY, o2 = (blockIdx.x / (ntx * nty)) * TZ;
  const double dt = P.scal[0] * P.dt_scale;
  const long long pbase = (long long)patch * P.pc;
  const double *Ukp = Uk + pbase * P.nvar;
  const double *U0p = U0 + pbase * P.nvar;
  double *Uop = Uout + pbase * P.nvar;
  const double *pp = P.p + pbase;
  double alpha[3], hidx[3];
#pragma unroll
  for (int d = 0; d < NDIM; d++) {
    alpha[d] = slot_value(P.slots + slot_base + lev * 3 + d);
    hidx[d] = 0.5 * P.invdx[lev][d];
  }
  // last loadable index along each dim (keeps ragged tiles inside the padded array)
  const int mx0 = P.n[0] + 2, mx1 = NDIM > 1 ? P.n[1] + 2 : 0, mx2 = NDIM > 2 ? P.n[2] + 2 : 0;
  const int in1 = NDIM > 1 ? P.n[1] - 1 : 0, in2 = NDIM > 2 ? P.n[2] - 1 : 0;
  // 32-bit offsets within a field (a patch holds < 2^31 padded cells, janc_create)
  const int s1 = NDIM > 1 ? (int)P.st[1] : 0, s2 = NDIM > 2 ? (int)P.st[2] : 0;
  const int goff = P.G[0] + P.G[1] * s1 + P.G[2] * s2;

#pragma unroll 1
  for (int m = 0; m < P.nvar; m++) {
    const double *Um = Ukp + (long long)m * P.pc;
    const double *U0m = U0p + (long long)m * P.pc;
    double *Uom = Uop + (long long)m * P.pc;
    const double cEn = m == NDIM + 1 ? 1.0 : 0.0;
    // ---------------- x: stage 2f+- rows, then walk
    {
      const double cM = m == 1 ? 1.0 : 0.0;
      const double *ux = P.vel + pbase;
      // advected components (no pressure term) are staged by their own loop: no p load, 3-instruction split flux
      auto stage_x = [&](auto gen) {
#pragma unroll 12
        for (int it = tid; it < C::ROWS * (TX + 6); it += NT) {
          const int xi = it % (TX + 6), r = it / (TX + 6);
          const int gx = min(o0 + xi - 3, mx0), gy = min(o1 + r % TY, in1), gz = min(o2 + r / TY, in2);
          const int id = goff + gx + gy * s1 + gz * s2;
          double a, b;
          if (decltype(gen)::value) split2(Um[id], ux[id], pp[id], cEn, cM, alpha[0], a, b);
          else split_adv(Um[id], ux[id], alpha[0], a, b);
          sFp[r * C::XP + xi] = a;
          sFm[r * C::XP + xi] = b;
        }
      };
      if (m == 1 || m == NDIM + 1) stage_x(std::true_type{}); else stage_x(std::false_type{});
      __syncthreads();
      const int r = tid % C::ROWS, xs = (tid / C::ROWS) * SEG;
      double Fh[SEG + 1];
      const double *rp = sFp + r * C::XP + xs, *rm = sFm + r * C::XP + xs;
      weno_faces<SEG>([&](int k, double &a, double &b) { a = rp[k]; b = rm[k]; }, Fh);
#pragma unroll
      for (int i = 0; i < SEG; i++) sL[r * C::LP + xs + i] = (Fh[i] - Fh[i + 1]) * hidx[0];
      __syncthreads();
    }
    // ---------------- y and z: the tile extended by 3 cells along d is staged as 2f+- (coalesced along x, all
    //                  loads of a thread independent), pencils then read shared memory (lanes along x: conflict-free)
#pragma unroll
    for (int d = 1; d < NDIM; d++) {
      const double cM = m == 1 + d ? 1.0 : 0.0;
      const double *ud = P.vel + (long long)d * P.np * P.pc + pbase;
      const double al = alpha[d];
      const int EY = d == 1 ? TY + 6 : TY, EZ = d == 2 ? TZ + 6 : TZ;     // staged extent
      auto stage_d = [&](auto gen) {
#pragma unroll 12
        for (int it = tid; it < TX * EY * EZ; it += NT) {
          const int x = it % TX, yy = (it / TX) % EY, zz = it / (TX * EY);
          const int gx = min(o0 + x, P.n[0] - 1);
          const int gy = d == 1 ? min(o1 + yy - 3, mx1) : min(o1 + yy, in1);
          const int gz = d == 2 ? min(o2 + zz - 3, mx2) : min(o2 + zz, in2);
          const int id = goff + gx + gy * s1 + gz * s2;
          double a, b;
          if (decltype(gen)::value) split2(Um[id], ud[id], pp[id], cEn, cM, al, a, b);
          else split_adv(Um[id], ud[id], al, a, b);
          sFp[(zz * EY + yy) * C::LP + x] = a;
          sFm[(zz * EY + yy) * C::LP + x] = b;
        }
      };
      if (m == 1 + d || m == NDIM + 1) stage_d(std::true_type{}); else stage_d(std::false_type{});
      __syncthreads();
      const int x = tid % TX, rest = tid / TX;
      // d == 1: pencils along y, the other index is z;  d == 2: pencils along z, the other index is y
      const int other = d == 1 ? rest % TZ : rest % TY;
      const int seg = (d == 1 ? rest / TZ : rest / TY) * SEG;
      const int ly = d == 1 ? seg : other, lz = d == 1 ? other : seg;
      const int base = (lz * EY + ly) * C::LP + x;
      const int sk = d == 1 ? C::LP : EY * C::LP;                          // stride of one pencil step in the stage
      double Fh[SEG + 1];
      weno_faces<SEG>([&](int k, double &a, double &b) { a = sFp[base + k * sk]; b = sFm[base + k * sk]; }, Fh);
      double *acc = sL + (lz * TY + ly) * C::LP + x;
      const int sa = d == 1 ? C::LP : TY * C::LP;
#pragma unroll
      for (int i = 0; i < SEG; i++) acc[i * sa] += (Fh[i] - Fh[i + 1]) * hidx[d];
      __syncthreads();
    }
    // ---------------- RK stage (increment form), coalesced
#pragma unroll
    for (int o = tid; o < C::NOUT; o += NT) {
      const int lx = o % TX, ly = (o / TX) % TY, lz = o / (TX * TY);
      const int g0 = o0 + lx, g1 = o1 + ly, g2 = o2 + lz;
      if (g0 < P.n[0] && g1 < P.n[1] && g2 < P.n[2]) {
        const int id = goff + g0 + g1 * s1 + g2 * s2;
        const double u0 = U0m[id];
        Uom[id] = u0 + coef * ((Um[id] - u0) + dt * sL[(lz * TY + ly) * C::LP + lx]);
      }
    }
    // the next component's x pencils overwrite sL only after its staging barrier
  }
}

// ------------------------------------------------------------------------------------------------
// 2-D variant with the tile resident in shared memory.  p, u, v of the tile + 3 ghost layers are
// copied once per CTA and U_m (same box) is double-buffered with cp.async: the copy of component
// m+1 runs while the pencils of component m are computed, so the walks only ever wait on shared
// memory.  Odd row pitch: x pencils (lanes = rows) and y pencils (lanes = columns) are both
// conflict-free, so no transposed staging pass is needed.
__device__ __forceinline__ void cp_async8(double *dst_smem, const double *src) {
  const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// Where the value of cell (i, j) of `patch` (interior coordinates, ghosts at -3..-1 and n..n+2) comes from:
// the rule of k_ghost (ghost.cuh) followed to an interior cell -- same-level neighbour, physical BC
// (periodic / reflect / outflow), or piecewise-constant injection from the coarse parent, whose own ghost
// is then resolved once more (reading A19).  flip bit d: the normal momentum / velocity of direction d
// changes sign (slip wall, A15).  Corner ghosts are never read by the sweeps (A21).
__device__ __forceinline__ void ghost_source2d(const Params &P, int patch, int i, int j, int &q, int &ci, int &cj, int &flip) {
  q = patch; ci = i; cj = j; flip = 0;
#pragma unroll 1
  for (int pass = 0; pass < 2; pass++) {
    const bool ox = ci < 0 || ci >= P.n[0], oy = cj < 0 || cj >= P.n[1];
    if (!ox && !oy) return;
    if (ox && oy) { ci = min(max(ci, 0), P.n[0] - 1); cj = min(max(cj, 0), P.n[1] - 1); return; }
    const int d = ox ? 0 : 1;
    const int cd = ox ? ci : cj;
    const int side = cd < 0 ? 0 : 1;
    const int g = side == 0 ? -cd : cd - P.n[d] + 1;
    const int f = 2 * d + side;
    const int kind = P.fkind[q * 4 + f];
    const int bc = side == 0 ? P.bc_lo[d] : P.bc_hi[d];
    int nd_ = cd;
    bool done = true;
    if (kind == FK_NEIGHBOUR || (kind == FK_PHYSICAL && bc == 0)) {
      if (kind == FK_NEIGHBOUR) q = P.nbr[q * 4 + f];
      nd_ = side == 0 ? P.n[d] - g : g - 1;
    } else if (kind == FK_PHYSICAL && bc == 1) {
      nd_ = side == 0 ? g - 1 : P.n[d] - g;
      flip |= 1 << d;
    } else if (kind == FK_PHYSICAL) {
      nd_ = side == 0 ? 0 : P.n[d] - 1;
    } else {
      const int *par = P.parent + q * 3;
      ci = floordiv_i(par[1] * P.n[0] + ci, P.ratio);
      cj = floordiv_i(par[2] * P.n[1] + cj, P.ratio);
      q = par[0];
      done = false;
    }
    if (done) { if (ox) ci = nd_; else cj = nd_; return; }
  }
}

// GATHER: the halo of the box is fetched straight from the cells the ghost rule points at -- the ghost layers are
// never written to HBM and k_ghost is not launched (AMR patches of <= 16 x 16, one tile per patch; small uniform
// grids, where three extra launches per step are a tenth of the step).
template <int TX, int TY, int SEG, bool GATHER = false>
struct Flux2Cfg {
  static constexpr int NT = TX * TY / SEG;
  static constexpr int BX = TX + 6, BY = TY + 6;
  static constexpr int PIT = BX | 1;
  static constexpr int BOX = PIT * BY;
  static constexpr int LP = TX | 1;
  static constexpr size_t SMEM = (size_t)(5 * BOX + TY * LP) * sizeof(double) + (GATHER ? (size_t)BX * BY * 12 : 0);
  // resident CTAs the register allocation aims at: the 64 x 16 tile is limited to 3 per SM by its 71 KB of shared
  // memory, so it may use 168 registers (1 % faster than 128); the others keep <= 128 registers for 4+ CTAs
  static constexpr int MINB = (TX == 64 && TY == 16 && SEG == 8 && !GATHER) ? 3 : (512 / NT > 0 ? 512 / NT : 1);
  static_assert(TX % SEG == 0 && TY % SEG == 0, "tile % SEG");
};

template <int TX, int TY, int SEG, bool GATHER>
__global__ void __launch_bounds__(Flux2Cfg<TX, TY, SEG, GATHER>::NT, Flux2Cfg<TX, TY, SEG, GATHER>::MINB)
k_flux_rk2(Params P, const double *__restrict__ Uk, const double *U0, double *Uout, int slot_base, double coef) {
  using C = Flux2Cfg<TX, TY, SEG, GATHER>;
  constexpr int NT = C::NT, PIT = C::PIT;
  extern __shared__ double flux_smem[];
  double *sp = flux_smem, *su = sp + C::BOX, *sv = su + C::BOX, *sU = sv + C::BOX, *sL = sU + 2 * C::BOX;
  int *sq = (int *)(sL + TY * C::LP), *sc = sq + C::BX * C::BY;           // GATHER: source patch / cell
  unsigned char *sfl = (unsigned char *)(sc + C::BX * C::BY);             //         flip bits

  const int tid = threadIdx.x;
  const int patch = blockIdx.y + P.patch0;
  const int lev = P.level[patch];
  const int ntx = (P.n[0] + TX - 1) / TX;
  const int o0 = (blockIdx.x % ntx) * TX, o1 = (blockIdx.x / ntx) * TY;
  const double dt = P.scal[0] * P.dt_scale;
  const long long pbase = (long long)patch * P.pc;
  const double *Ukp = Uk + pbase * P.nvar;
  const double *U0p = U0 + pbase * P.nvar;
  double *Uop = Uout + pbase * P.nvar;
  const int st1i = (int)P.st[1];
  const int goff = P.G[1] * st1i + P.G[0];              // offset of interior cell (0, 0) within a field
  const double ax = slot_value(P.slots + slot_base + lev * 3 + 0), ay = slot_value(P.slots + slot_base + lev * 3 + 1);
  const double hx = 0.5 * P.invdx[lev][0], hy = 0.5 * P.invdx[lev][1];
  const int mxp = P.P[0] - 1, myp = P.P[1] - 1;     // last padded index (ragged tiles stay in the array)
  const bool same = Uk == U0;                        // stage 0: U^n is the stage state, already in smem

  if (GATHER) {
    for (int it = tid; it < C::BX * C::BY; it += NT) {
      int q, ci, cj, fl;
      // patch coordinates of this box cell (ragged tiles stay within the 3 ghost layers)
      ghost_source2d(P, patch, min(o0 + it % C::BX - 3, P.n[0] + 2), min(o1 + it / C::BX - 3, P.n[1] + 2), q, ci, cj, fl);
      sq[it] = q;
      sc[it] = (int)cell_index(P, ci, cj, 0);
      sfl[it] = (unsigned char)fl;
    }
    __syncthreads();
  }
  // copy field `fld` of an array with `fpp` fields per patch into a box
  auto load_box = [&](double *dst, const double *base, int fpp, int fld) {
    const double *fb = base + ((long long)patch * fpp + fld) * P.pc;
    const double *fbg = base + (long long)fld * P.pc;
    const int fppc = fpp * (int)P.pc;                   // GATHER: patches / small grids, fields of one patch < 2^31 cells
#pragma unroll 4
    for (int it = tid; it < C::BX * C::BY; it += NT) {
      const int bx = it % C::BX, by = it / C::BX;
      if (GATHER) {
        cp_async8(dst + by * PIT + bx, fbg + ((long long)sq[it] * fppc + sc[it]));      // one 32 x 32 -> 64 multiply
      } else {   // 32-bit offsets within a field (a patch holds < 2^31 padded cells, janc_create)
        const int gx = min(o0 + bx, mxp), gy = min(o1 + by, myp);
        cp_async8(dst + by * PIT + bx, fb + (gy * st1i + gx));
      }
    }
  };
  // slip walls: negate the mirrored normal momentum / velocity (bit = 1 << direction)
  auto fix_flips = [&](double *box, int bit) {
    for (int it = tid; it < C::BX * C::BY; it += NT)
      if (sfl[it] & bit) { double *e = box + (it / C::BX) * PIT + it % C::BX; *e = -*e; }
  };
  load_box(sp, P.p, 1, 0);
  load_box(su, P.vel, 1, 0);
  load_box(sv, P.vel + (long long)P.np * P.pc, 1, 0);
  load_box(sU, Uk, P.nvar, 0);
  cp_async_commit();
  if (P.nvar > 1) load_box(sU + C::BOX, Uk, P.nvar, 1);
  cp_async_commit();

#pragma unroll 1
  for (int m = 0; m < P.nvar; m++) {
    const double *sUm = sU + (m & 1) * C::BOX;
    const double cEn = m == 3 ? 1.0 : 0.0;
    cp_async_wait<1>();
    __syncthreads();
    if (GATHER && m <= 2) {
      if (m == 0) { fix_flips(su, 1); fix_flips(sv, 2); }
      else fix_flips(sU + (m & 1) * C::BOX, m);                 // m = 1: x momentum (bit 1), m = 2: y momentum (bit 2)
      __syncthreads();
    }
    {  // x pencils: lanes run over rows
      const double cM = m == 1 ? 1.0 : 0.0;
      const int r = tid % TY, xs = (tid / TY) * SEG;
      const int base = (r + 3) * PIT + xs;
      double Fh[SEG + 1];
      if (m == 1 || m == 3)
        weno_faces<SEG>([&](int k, double &a, double &b) { split2(sUm[base + k], su[base + k], sp[base + k], cEn, cM, ax, a, b); }, Fh);
      else   // advected components (rho, transverse momentum, rho Y_k): F = U_m u, no pressure read
        weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sUm[base + k], su[base + k], ax, a, b); }, Fh);
#pragma unroll
      for (int i = 0; i < SEG; i++) sL[r * C::LP + xs + i] = (Fh[i] - Fh[i + 1]) * hx;
    }
    __syncthreads();
    {  // y pencils: lanes run over columns.  The thread that walks cells (x, ys..ys+SEG-1) also applies their RK stage
       // (increment form): U^n is requested before the walk and consumed after it; loads and stores are coalesced along x.
      const double cM = m == 2 ? 1.0 : 0.0;
      const int x = tid % TX, ys = (tid / TX) * SEG;
      const int g0 = o0 + x, gc0 = min(g0, P.n[0] - 1);
      const double *U0m = U0p + (long long)m * P.pc;
      double *Uom = Uop + (long long)m * P.pc;
      double u0v[SEG];
      if (!same) {
#pragma unroll
        for (int i = 0; i < SEG; i++)
          u0v[i] = U0m[goff + min(o1 + ys + i, P.n[1] - 1) * st1i + gc0];
      }
      const int base = ys * PIT + x + 3;
      double Fh[SEG + 1];
      if (m == 2 || m == 3)
        weno_faces<SEG>([&](int k, double &a, double &b) { split2(sUm[base + k * PIT], sv[base + k * PIT], sp[base + k * PIT], cEn, cM, ay, a, b); }, Fh);
      else
        weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sUm[base + k * PIT], sv[base + k * PIT], ay, a, b); }, Fh);
#pragma unroll
      for (int i = 0; i < SEG; i++) {
        const int g1 = o1 + ys + i;
        if (g0 < P.n[0] && g1 < P.n[1]) {
          const double L = sL[(ys + i) * C::LP + x] + (Fh[i] - Fh[i + 1]) * hy;
          const double uk = sUm[(ys + i + 3) * PIT + x + 3];
          const double u0 = same ? uk : u0v[i];
          Uom[goff + g1 * st1i + g0] = u0 + coef * ((uk - u0) + dt * L);
        }
      }
    }
    __syncthreads();   // everyone is done with sU[m & 1] and sL
    if (m + 2 < P.nvar) load_box(sU + (m & 1) * C::BOX, Uk, P.nvar, m + 2);
    cp_async_commit();
  }
}

// ------------------------------------------------------------------------------------------------
// TMA variant of the 2-D kernel (uniform grids and patches with materialised ghosts): the tile + 3 ghost layers of
// p, u, v and of every component U_m arrive as ONE cp.async.bulk.tensor box each (a 3-D tensor map {Px, Py, fields}
// over the padded arrays; a box that sticks out of the array is zero-filled, and only cells outside the grid ever see
// those zeros), signalled through an mbarrier.  The box is dense (pitch = TX + 6 doubles): the per-element index math
// of the cp.async loads (a fifth of the kernel's instructions) disappears, in exchange x pencils (lanes = rows) read
// with a 2-way bank conflict.  Requires an even padded width (global strides are multiples of 16 bytes).
#include <cuda.h>

__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count) {
  asm volatile("mbarrier.init.shared.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long *bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
  asm volatile(
      "{\n .reg .pred p;\n WAIT_%=:\n mbarrier.try_wait.parity.shared.b64 p, [%0], %1;\n @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}\n" ::"r"(
          (unsigned)__cvta_generic_to_shared(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(double *dst, const CUtensorMap *map, unsigned long long *bar, int x, int y, int z) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(
                   (unsigned)__cvta_generic_to_shared(dst)),
               "l"(map), "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(x), "r"(y), "r"(z)
               : "memory");
}

template <int TX, int TY, int SEG>
struct Flux2TmaCfg {
  static constexpr int NT = TX * TY / SEG;
  static constexpr int BX = TX + 6, BY = TY + 6;
  static constexpr int PIT = BX;                                          // dense box
  static constexpr int BOX = (BX * BY * 8 + 127) / 128 * 16;              // doubles, padded to 128 bytes
  static constexpr int LP = TX | 1;
  static constexpr unsigned BOX_BYTES = BX * BY * 8;
  static constexpr size_t SMEM = (size_t)(5 * BOX + TY * LP) * sizeof(double) + 64;
  static constexpr int MINB = NT >= 128 ? 3 : 512 / NT;                   // resident CTAs the register allocation aims at
  static_assert(TX % SEG == 0 && TY % SEG == 0 && (BX * 8) % 16 == 0, "tile");
};

template <int TX, int TY, int SEG>
__global__ void __launch_bounds__(TX * TY / SEG, Flux2TmaCfg<TX, TY, SEG>::MINB)
k_flux_rk2_tma(Params P, const double *U0, double *Uout, int slot_base, double coef, int same_i,
               const __grid_constant__ CUtensorMap mapU, const __grid_constant__ CUtensorMap mapP,
               const __grid_constant__ CUtensorMap mapV) {
  using C = Flux2TmaCfg<TX, TY, SEG>;
  constexpr int NT = C::NT, PIT = C::PIT;
  extern __shared__ __align__(128) double flux_smem[];
  double *sp = flux_smem, *su = sp + C::BOX, *sv = su + C::BOX, *sU = sv + C::BOX, *sL = sU + 2 * C::BOX;
  unsigned long long *bars = (unsigned long long *)(sL + TY * C::LP);     // [0], [1]: U buffers (the first also p, u, v)

  const int tid = threadIdx.x;
  const int patch = blockIdx.y + P.patch0;
  const int lev = P.level[patch];
  const int ntx = (P.n[0] + TX - 1) / TX;
  const int o0 = (blockIdx.x % ntx) * TX, o1 = (blockIdx.x / ntx) * TY;
  const double dt = P.scal[0] * P.dt_scale;
  const long long pbase = (long long)patch * P.pc;
  const double *U0p = U0 + pbase * P.nvar;
  double *Uop = Uout + pbase * P.nvar;
  const int st1i = (int)P.st[1];
  const int goff = P.G[1] * st1i + P.G[0];
  const double ax = slot_value(P.slots + slot_base + lev * 3 + 0), ay = slot_value(P.slots + slot_base + lev * 3 + 1);
  const double hx = 0.5 * P.invdx[lev][0], hy = 0.5 * P.invdx[lev][1];
  const bool same = same_i != 0;

  if (tid == 0) {
    mbar_init(bars, 1);
    mbar_init(bars + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    mbar_expect_tx(bars, 4 * C::BOX_BYTES);
    tma_load_3d(sp, &mapP, bars, o0, o1, patch);
    tma_load_3d(su, &mapV, bars, o0, o1, patch);
    tma_load_3d(sv, &mapV, bars, o0, o1, P.np + patch);
    tma_load_3d(sU, &mapU, bars, o0, o1, patch * P.nvar);
    if (P.nvar > 1) {
      mbar_expect_tx(bars + 1, C::BOX_BYTES);
      tma_load_3d(sU + C::BOX, &mapU, bars + 1, o0, o1, patch * P.nvar + 1);
    }
  }

#pragma unroll 1
  for (int m = 0; m < P.nvar; m++) {
    const double *sUm = sU + (m & 1) * C::BOX;
    const double cEn = m == 3 ? 1.0 : 0.0;
    mbar_wait(bars + (m & 1), (m >> 1) & 1);
    {  // x pencils: lanes run over rows
      const double cM = m == 1 ? 1.0 : 0.0;
      const int r = tid % TY, xs = (tid / TY) * SEG;
      const int base = (r + 3) * PIT + xs;
      double Fh[SEG + 1];
      if (m == 1 || m == 3)
        weno_faces<SEG>([&](int k, double &a, double &b) { split2(sUm[base + k], su[base + k], sp[base + k], cEn, cM, ax, a, b); }, Fh);
      else
        weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sUm[base + k], su[base + k], ax, a, b); }, Fh);
#pragma unroll
      for (int i = 0; i < SEG; i++) sL[r * C::LP + xs + i] = (Fh[i] - Fh[i + 1]) * hx;
    }
    __syncthreads();
    {  // y pencils: lanes run over columns; the thread applies the RK stage of its own cells
      const double cM = m == 2 ? 1.0 : 0.0;
      const int x = tid % TX, ys = (tid / TX) * SEG;
      const int g0 = o0 + x, gc0 = min(g0, P.n[0] - 1);
      const double *U0m = U0p + (long long)m * P.pc;
      double *Uom = Uop + (long long)m * P.pc;
      double u0v[SEG];
      if (!same) {
#pragma unroll
        for (int i = 0; i < SEG; i++) u0v[i] = U0m[goff + min(o1 + ys + i, P.n[1] - 1) * st1i + gc0];
      }
      const int base = ys * PIT + x + 3;
      double Fh[SEG + 1];
      if (m == 2 || m == 3)
        weno_faces<SEG>([&](int k, double &a, double &b) { split2(sUm[base + k * PIT], sv[base + k * PIT], sp[base + k * PIT], cEn, cM, ay, a, b); }, Fh);
      else
        weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sUm[base + k * PIT], sv[base + k * PIT], ay, a, b); }, Fh);
#pragma unroll
      for (int i = 0; i < SEG; i++) {
        const int g1 = o1 + ys + i;
        if (g0 < P.n[0] && g1 < P.n[1]) {
          const double L = sL[(ys + i) * C::LP + x] + (Fh[i] - Fh[i + 1]) * hy;
          const double uk = sUm[(ys + i + 3) * PIT + x + 3];
          const double u0 = same ? uk : u0v[i];
          Uom[goff + g1 * st1i + g0] = u0 + coef * ((uk - u0) + dt * L);
        }
      }
    }
    __syncthreads();   // everyone is done with sU[m & 1] and sL
    if (tid == 0 && m + 2 < P.nvar) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy reads before the async-proxy write
      mbar_expect_tx(bars + (m & 1), C::BOX_BYTES);
      tma_load_3d(sU + (m & 1) * C::BOX, &mapU, bars + (m & 1), o0, o1, patch * P.nvar + m + 2);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// TMA variant of the 3-D kernel (materialised ghosts, even padded width).  The work of a tile is cut into units
// (component m, direction d); a unit needs the tile extended by 3 cells along d only -- one dense box
// {TX (+6), TY (+6), TZ (+6)} of U_m, one of u_d and, for the normal momentum and the energy, one of p -- which arrive
// as cp.async.bulk.tensor boxes of a 4-D tensor map {Px, Py, Pz, fields} (one map per box shape), two units ahead of
// the walk: while the pencils of unit u are walked, the boxes of unit u + 1 are in flight or landed.  No thread
// executes a staging loop: the split fluxes 2f+- = F +- alpha U are formed by the walk from the raw boxes (as in the
// 2-D kernel), the x and y contributions wait in the per-cell accumulator, and the thread that walks a z pencil
// (lanes along x: coalesced) adds its own and applies the RK stage of its cells.  Same arithmetic, in the same order,
// as k_flux_rk<3, ...>: results are bit-identical.
__device__ __forceinline__ void tma_load_4d(double *dst, const CUtensorMap *map, unsigned long long *bar, int x, int y, int z, int f) {
  asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(
                   (unsigned)__cvta_generic_to_shared(dst)),
               "l"(map), "r"((unsigned)__cvta_generic_to_shared(bar)), "r"(x), "r"(y), "r"(z), "r"(f)
               : "memory");
}

struct Flux3Maps { CUtensorMap U[3], V[3], P[3]; };       // [d]: the box shape of direction d over the stage state, vel, p

template <int TX, int TY, int TZ, int SEG>
struct Flux3TmaCfg {
  static constexpr int NT = TX * TY * TZ / SEG;
  static constexpr int TXB = TX + 2;                                      // x extent of the y / z boxes: a TMA box starts at a 16-byte aligned
                                                                         // address, i.e. at an even padded x; interior cell 0 sits at x = 3
  static constexpr int NB0 = (TX + 6) * TY * TZ, NB1 = TXB * (TY + 6) * TZ, NB2 = TXB * TY * (TZ + 6);   // doubles per box
  static constexpr int NBMAX = NB0 > NB1 ? (NB0 > NB2 ? NB0 : NB2) : (NB1 > NB2 ? NB1 : NB2);
  static constexpr int BOX = (NBMAX + 15) / 16 * 16;                      // 128-byte aligned slots
  static constexpr int LP = TX | 1;
  static constexpr int ROWS = TY * TZ;
  static constexpr size_t SMEM = (size_t)(6 * BOX + ROWS * LP) * sizeof(double) + 64;
  static_assert(TX % SEG == 0 && TY % SEG == 0 && TZ % SEG == 0 && (TX * 8) % 16 == 0, "tile");
  static_assert(NT % TX == 0 && NT % ROWS == 0, "thread maps");
};

template <int TX, int TY, int TZ, int SEG>
__global__ void __launch_bounds__(TX * TY * TZ / SEG, 2)
k_flux_rk3_tma(Params P, const double *U0, double *Uout, int slot_base, double coef, int same_i,
               const __grid_constant__ Flux3Maps M) {
  using C = Flux3TmaCfg<TX, TY, TZ, SEG>;
  constexpr int NT = C::NT;
  extern __shared__ __align__(128) double flux_smem[];
  double *sL = flux_smem + 6 * C::BOX;
  unsigned long long *bars = (unsigned long long *)(sL + C::ROWS * C::LP);

  const int tid = threadIdx.x;
  const int patch = blockIdx.y + P.patch0;
  const int lev = P.level[patch];
  const int ntx = (P.n[0] + TX - 1) / TX, nty = (P.n[1] + TY - 1) / TY;
  const int o0 = (blockIdx.x % ntx) * TX, o1 = ((blockIdx.x / ntx) % nty) * TY, o2 = (blockIdx.x / (ntx * nty)) * TZ;
  const double dt = P.scal[0] * P.dt_scale;
  const long long pbase = (long long)patch * P.pc;
  const double *U0p = U0 + pbase * P.nvar;
  double *Uop = Uout + pbase * P.nvar;
  const int s1 = (int)P.st[1], s2 = (int)P.st[2];
  const int goff = P.G[0] + P.G[1] * s1 + P.G[2] * s2;
  double alpha[3], hidx[3];
#pragma unroll
  for (int d = 0; d < 3; d++) {
    alpha[d] = slot_value(P.slots + slot_base + lev * 3 + d);
    hidx[d] = 0.5 * P.invdx[lev][d];
  }
  const bool same = same_i != 0;
  const int nunits = 3 * P.nvar;

  // unit u = 3 m + d goes to slot u & 1: boxes U, u_d, p at (3 slot + 0 / 1 / 2) * BOX.  d is a compile-time constant
  // (the tensor maps are addressed statically in the kernel's parameter space).
  auto issue = [&](int m, auto dc) {
    constexpr int d = decltype(dc)::value;
    const int s = (3 * m + d) & 1;
    const bool needp = m == 1 + d || m == 4;
    constexpr unsigned nb = (d == 0 ? C::NB0 : d == 1 ? C::NB1 : C::NB2) * 8u;
    double *b = flux_smem + 3 * s * C::BOX;
    const int cx = o0 + (d == 0 ? 0 : 2), cy = o1 + (d == 1 ? 0 : 3), cz = o2 + (d == 2 ? 0 : 3);     // padded coordinates (x even)
    mbar_expect_tx(bars + s, needp ? 3 * nb : 2 * nb);
    tma_load_4d(b, &M.U[d], bars + s, cx, cy, cz, patch * P.nvar + m);
    tma_load_4d(b + C::BOX, &M.V[d], bars + s, cx, cy, cz, d * P.np + patch);
    if (needp) tma_load_4d(b + 2 * C::BOX, &M.P[d], bars + s, cx, cy, cz, patch);
  };
  if (tid == 0) {
    mbar_init(bars, 1);
    mbar_init(bars + 1, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) { issue(0, std::integral_constant<int, 0>{}); issue(0, std::integral_constant<int, 1>{}); }

  // one unit: wait for its boxes, walk, hand the slot to unit u + 2
  auto unit = [&](int m, auto dc) {
    constexpr int d = decltype(dc)::value;
    const double cEn = m == 4 ? 1.0 : 0.0;
    const bool en = m == 4;
    {
      const int u = 3 * m + d, s = u & 1;
      const double *sU = flux_smem + 3 * s * C::BOX, *sV = sU + C::BOX, *sP = sV + C::BOX;
      const double cM = m == 1 + d ? 1.0 : 0.0;
      const bool withp = en || m == 1 + d;
      const double al = alpha[d];
      double Fh[SEG + 1];
      if (d == 0) {           // x pencils: lanes run over the rows (y, z) of the box [z][y][TX + 6]
        const int r = tid % C::ROWS, xs = (tid / C::ROWS) * SEG;
        const int base = r * (TX + 6) + xs;
        mbar_wait(bars + s, (u >> 1) & 1);
        if (withp) weno_faces<SEG>([&](int k, double &a, double &b) { split2(sU[base + k], sV[base + k], sP[base + k], cEn, cM, al, a, b); }, Fh);
        else weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sU[base + k], sV[base + k], al, a, b); }, Fh);
#pragma unroll
        for (int i = 0; i < SEG; i++) sL[r * C::LP + xs + i] = (Fh[i] - Fh[i + 1]) * hidx[0];
      } else if (d == 1) {    // y pencils: lanes along x, box [z][TY + 6][TX + 2], cell x at column x + 1
        constexpr int TXB = C::TXB;
        const int x = tid % TX, rest = tid / TX;
        const int lz = rest % TZ, seg = (rest / TZ) * SEG;
        const int base = (lz * (TY + 6) + seg) * TXB + x + 1;
        mbar_wait(bars + s, (u >> 1) & 1);
        if (withp) weno_faces<SEG>([&](int k, double &a, double &b) { split2(sU[base + k * TXB], sV[base + k * TXB], sP[base + k * TXB], cEn, cM, al, a, b); }, Fh);
        else weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sU[base + k * TXB], sV[base + k * TXB], al, a, b); }, Fh);
        double *acc = sL + (lz * TY + seg) * C::LP + x;
#pragma unroll
        for (int i = 0; i < SEG; i++) acc[i * C::LP] += (Fh[i] - Fh[i + 1]) * hidx[1];
      } else {                // z pencils: lanes along x, box [TZ + 6][y][TX + 2]; RK stage of the pencil's own cells
        const int x = tid % TX, rest = tid / TX;
        const int ly = rest % TY, seg = (rest / TY) * SEG;
        const int base = (seg * TY + ly) * C::TXB + x + 1;
        constexpr int SK = TY * C::TXB;
        const int g0 = o0 + x, g1 = o1 + ly;
        const int idc = goff + min(g0, P.n[0] - 1) + min(g1, P.n[1] - 1) * s1;
        const double *U0m = U0p + (long long)m * P.pc;
        double *Uom = Uop + (long long)m * P.pc;
        double u0v[SEG];
        if (!same) {
#pragma unroll
          for (int i = 0; i < SEG; i++) u0v[i] = U0m[idc + min(o2 + seg + i, P.n[2] - 1) * s2];
        }
        mbar_wait(bars + s, (u >> 1) & 1);
        if (withp) weno_faces<SEG>([&](int k, double &a, double &b) { split2(sU[base + k * SK], sV[base + k * SK], sP[base + k * SK], cEn, cM, al, a, b); }, Fh);
        else weno_faces<SEG>([&](int k, double &a, double &b) { split_adv(sU[base + k * SK], sV[base + k * SK], al, a, b); }, Fh);
#pragma unroll
        for (int i = 0; i < SEG; i++) {
          const int g2 = o2 + seg + i;
          if (g0 < P.n[0] && g1 < P.n[1] && g2 < P.n[2]) {
            const double L = sL[((seg + i) * TY + ly) * C::LP + x] + (Fh[i] - Fh[i + 1]) * hidx[2];
            const double uk = sU[base + (i + 3) * SK];
            const double u0 = same ? uk : u0v[i];
            Uom[goff + g0 + g1 * s1 + g2 * s2] = u0 + coef * ((uk - u0) + dt * L);
          }
        }
      }
      __syncthreads();   // everyone is done with slot s; sL is ordered between the directions
      if (tid == 0 && u + 2 < nunits) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy reads before the async-proxy write
        issue(d == 0 ? m : m + 1, std::integral_constant<int, (d + 2) % 3>{});
      }
    }
  };
#pragma unroll 1
  for (int m = 0; m < P.nvar; m++) {
    unit(m, std::integral_constant<int, 0>{});
    unit(m, std::integral_constant<int, 1>{});
    unit(m, std::integral_constant<int, 2>{});
  }
}
