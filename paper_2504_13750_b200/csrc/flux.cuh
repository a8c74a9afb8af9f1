// flux.cuh -- x/y/z reconstruction + flux sweeps fused with the divergence and the RK stage.
// PAPER.md:288-295 (eq 4.11 Lax-Friedrichs splitting, WENO5 on 6 template points, 3 ghosts),
// :283-286 (eq 4.10 conservative difference), :297/:339 (TVD-RK3), :232 (F, G).
// Readings A1 (WENO5-JS, eps 1e-6, p 2), A2 (component-wise), A3/A20 (alpha per direction per
// level, from the stage state), A4 (increment form of SSP-RK3), A24 (x, y, z order).
//
// Work decomposition ("pair" form): the thread at cell c forms, for one component and one direction,
// the split fluxes f+ and f- on the window c-2..c+2 ONCE and reconstructs from it both
//     G(c) = Fhat+_{c+1/2}   (WENO5 on f+_{c-2..c+2})
//     H(c) = Fhat-_{c-1/2}   (WENO5 on f-_{c+2..c-2}, the mirror image)
// so that  Fhat_{c+1/2} = G(c) + H(c+1).  G and H go through shared memory; the divergence of cell c
// is  -(G(c) + H(c+1) - G(c-1) - H(c)) / dx.  Per tile and direction the items are the tile cells
// plus one rim cell at each end: every face is reconstructed exactly once, no flux array in HBM.
#pragma once
#include "common.cuh"

// WENO5-JS value at +1/2 from v_{-2..+2}, one division:
//   a_k = d_k / (eps + beta_k)^2  ==  d_k * prod_{l != k} (eps + beta_l)^2 / prod_l (eps+beta_l)^2
__device__ __forceinline__ double weno5_js(double v0, double v1, double v2, double v3, double v4) {
  const double eps = 1e-6, c1312 = 13.0 / 12.0;
  double t1, t2;
  t1 = (v0 - 2.0 * v1) + v2; t2 = (v0 - 4.0 * v1) + 3.0 * v2;
  double b0 = fma(c1312 * t1, t1, fma(0.25 * t2, t2, eps));
  t1 = (v1 - 2.0 * v2) + v3; t2 = v1 - v3;
  double b1 = fma(c1312 * t1, t1, fma(0.25 * t2, t2, eps));
  t1 = (v2 - 2.0 * v3) + v4; t2 = (3.0 * v2 - 4.0 * v3) + v4;
  double b2 = fma(c1312 * t1, t1, fma(0.25 * t2, t2, eps));
  b0 *= b0; b1 *= b1; b2 *= b2;
  const double a0 = 0.1 * (b1 * b2), a1 = 0.6 * (b0 * b2), a2 = 0.3 * (b0 * b1);
  const double q0 = fma(2.0, v0, fma(-7.0, v1, 11.0 * v2));
  const double q1 = fma(5.0, v2, fma(2.0, v3, -v1));
  const double q2 = fma(2.0, v2, fma(5.0, v3, -v4));
  const double num = fma(a0, q0, fma(a1, q1, a2 * q2));
  const double den = 6.0 * ((a0 + a1) + a2);
  return num / den;
}

template <int NDIM, int TX, int TY, int TZ, int NT>
__global__ void __launch_bounds__(NT)
k_flux_rk(Params P, const double *__restrict__ Uk, const double *U0, double *Uout, int slot_base, double coef) {
  constexpr int T_[3] = {TX, TY, TZ};
  constexpr int NOUT = TX * TY * TZ;
  constexpr int OPT = (NOUT + NT - 1) / NT;                 // outputs per thread
  constexpr int MAXI = NDIM == 1 ? (TX + 2) * TY * TZ
                     : NDIM == 2 ? ((TX + 2) * TY > TX * (TY + 2) ? (TX + 2) * TY : TX * (TY + 2)) * TZ
                     : ((TX + 2) * TY * TZ > TX * (TY + 2) * TZ
                            ? ((TX + 2) * TY * TZ > TX * TY * (TZ + 2) ? (TX + 2) * TY * TZ : TX * TY * (TZ + 2))
                            : (TX * (TY + 2) * TZ > TX * TY * (TZ + 2) ? TX * (TY + 2) * TZ : TX * TY * (TZ + 2)));
  __shared__ double sG[2][MAXI], sH[2][MAXI];

  const int patch = blockIdx.y;
  const int lev = P.level[patch];
  const int ntx = (P.n[0] + TX - 1) / TX, nty = (P.n[1] + TY - 1) / TY;
  const int bx = blockIdx.x % ntx, by = (blockIdx.x / ntx) % nty, bz = blockIdx.x / (ntx * nty);
  const int o0[3] = {bx * TX, by * TY, bz * TZ};
  const double dt = P.scal[0];
  const double *Ukp = Uk + (long long)patch * P.nvar * P.pc;
  const double *U0p = U0 + (long long)patch * P.nvar * P.pc;
  double *Uop = Uout + (long long)patch * P.nvar * P.pc;
  const double *pp = P.p + (long long)patch * P.pc;

  int q = 0;
#pragma unroll 1
  for (int m = 0; m < P.nvar; m++) {
    const double *Um = Ukp + (long long)m * P.pc;
    double Lacc[OPT];
#pragma unroll
    for (int r = 0; r < OPT; r++) Lacc[r] = 0.0;
#pragma unroll
    for (int d = 0; d < NDIM; d++, q++) {
      const int buf = q & 1;
      const int B0 = TX + (d == 0 ? 2 : 0), B1 = TY + (d == 1 ? 2 : 0), B2 = TZ + (d == 2 ? 2 : 0);
      const int nitems = B0 * B1 * B2;
      const long long sd = P.st[d];
      const double alpha = slot_value(P.slots + slot_base + lev * 3 + d);
      const double *ud = P.vel + ((long long)d * P.np + patch) * P.pc;
      const double *Umom = Ukp + (long long)(1 + d) * P.pc;
      const int kindm = m == 0 ? 0 : (m == 1 + d ? 1 : (m == NDIM + 1 ? 2 : 3));
#pragma unroll 1
      for (int it = threadIdx.x; it < nitems; it += NT) {
        int l[3] = {it % B0, (it / B0) % B1, it / (B0 * B1)};
        l[d] -= 1;
        const int g0 = o0[0] + l[0], g1 = o0[1] + l[1], g2 = o0[2] + l[2];
        const int gd = d == 0 ? g0 : (d == 1 ? g1 : g2);
        bool valid = gd <= P.n[d];
        if (d != 0) valid = valid && g0 < P.n[0];
        if (d != 1) valid = valid && g1 < P.n[1];
        if (d != 2) valid = valid && g2 < P.n[2];
        double G = 0.0, H = 0.0;
        if (valid) {
          const long long id = cell_index(P, g0, g1, g2);
          double fp[5], fm[5];
#pragma unroll
          for (int s = 0; s < 5; s++) {
            const long long c = id + (long long)(s - 2) * sd;
            const double Uv = Um[c];
            double F;
            if (kindm == 0) F = Umom[c];                       // rho u_d
            else if (kindm == 1) F = fma(Uv, ud[c], pp[c]);    // rho u_d u_d + p
            else if (kindm == 2) F = ud[c] * (Uv + pp[c]);     // u_d (E + p)
            else F = Uv * ud[c];                               // rho u_j u_d, rho Y_k u_d
            const double aU = alpha * Uv;
            fp[s] = 0.5 * (F + aU);
            fm[s] = 0.5 * (F - aU);
          }
          G = weno5_js(fp[0], fp[1], fp[2], fp[3], fp[4]);
          H = weno5_js(fm[4], fm[3], fm[2], fm[1], fm[0]);
        }
        sG[buf][it] = G;
        sH[buf][it] = H;
      }
      __syncthreads();
      const double idx = P.invdx[lev][d];
#pragma unroll
      for (int r = 0; r < OPT; r++) {
        const int o = threadIdx.x + r * NT;
        if (o < NOUT) {
          int l[3] = {o % TX, (o / TX) % TY, o / (TX * TY)};
          l[d] += 1;
          const int c = (l[2] * B1 + l[1]) * B0 + l[0];
          const int sI = d == 0 ? 1 : (d == 1 ? B0 : B0 * B1);
          const double Fr = sG[buf][c] + sH[buf][c + sI];
          const double Fl = sG[buf][c - sI] + sH[buf][c];
          Lacc[r] -= (Fr - Fl) * idx;
        }
      }
    }
    // RK stage (increment form): Uout = U0 + coef * ((Uk - U0) + dt * L)
#pragma unroll
    for (int r = 0; r < OPT; r++) {
      const int o = threadIdx.x + r * NT;
      if (o < NOUT) {
        const int g0 = o0[0] + o % TX, g1 = o0[1] + (o / TX) % TY, g2 = o0[2] + o / (TX * TY);
        if (g0 < P.n[0] && g1 < P.n[1] && g2 < P.n[2]) {
          const long long id = cell_index(P, g0, g1, g2) + (long long)m * P.pc;
          const double u0 = U0p[id];
          Uop[id] = u0 + coef * ((Ukp[id] - u0) + dt * Lacc[r]);
        }
      }
    }
  }
  (void)T_;
}
