// chem.cuh -- point-implicit chemistry kernel (advance_source_term).
// PAPER.md:260-277 (eq 4.6-4.9 rates, K_eq), :297-304 (eq 4.12-4.13), :333.
// Readings A9 (third body only where flagged), A10 (irreversible), A11 (Jacobian w.r.t.
// rho*Y_1..Ns-1 at frozen T and rho, Y_Ns through rho), A12 (no clipping).
// One thread per cell: T* by Newton (fused cons->prim), rates, analytic Jacobian, (I - dt J) d = dt w
// by Gaussian elimination with partial pivoting, rhoY += d.
#pragma once
#include <type_traits>
#include "prim.cuh"

template <int I, int E, class F>
__device__ __forceinline__ void static_for(F &&f) {
  if constexpr (I < E) {
    f(std::integral_constant<int, I>{});
    static_for<I + 1, E>(f);
  }
}

template <int NS>
__global__ void __launch_bounds__(128) k_chem(Params P, double *__restrict__ U) {
  constexpr int NSM = NS > 0 ? NS : JANC_MAX_NS;
  constexpr int N1M = NSM - 1;
  const int ns = NS > 0 ? NS : P.ns;
  const int n1 = ns - 1;
  const int nr = c_mech.nr;
  const int patch = blockIdx.y + P.patch0;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ncell) return;
  const int i = (int)(t % P.n[0]);
  const long long r_ = t / P.n[0];
  const int j = (int)(r_ % P.n[1]);
  const int k = (int)(r_ / P.n[1]);
  const long long id = cell_index(P, i, j, k);
  double *Up = U + (long long)patch * P.nvar * P.pc;
  const long long pid = (long long)patch * P.pc + id;

  // ---- T* = T(U*)  (update_aux)
  double T, pr, cs, u[3];
  bool ok = cons2prim<NS>(P, Up, id, P.T[pid], T, pr, cs, u);
  P.T[pid] = T;

  // ---- molar concentrations X_k = rho Y_k / W_k, Y_Ns by difference
  const double rho = Up[id];
  double X[NSM], ry[N1M > 0 ? N1M : 1];
  double s = 0.0;
#pragma unroll
  for (int a = 0; a < n1; a++) {
    ry[a] = Up[(long long)(P.ndim + 2 + a) * P.pc + id];
    X[a] = ry[a] * c_mech.invW[a];
    s += ry[a];
  }
  X[n1] = (rho - s) * c_mech.invW[n1];

  // ---- g_j = s_j/R_j - h_j/(R_j T)
  const double lnT = log(T), iT = 1.0 / T;
  double g[NSM];
#pragma unroll
  for (int a = 0; a < ns; a++) g[a] = s_R(a, T, lnT) - h_R(a, T) * iT;
  const double lnC0 = log(JANC_PATM / (JANC_RU * T));

  // ---- omega (mol-based, all species) and D[k][j] = sum_i dnu_ik dq_i/dX_j
  double wdot[NSM];
  double D[N1M > 0 ? N1M : 1][NSM];
#pragma unroll
  for (int a = 0; a < ns; a++) wdot[a] = 0.0;
  for (int a = 0; a < n1; a++)
    for (int b = 0; b < ns; b++) D[a][b] = 0.0;

  for (int rx = 0; rx < nr; rx++) {
    const int nre = c_mech.nreac[rx], npr = c_mech.nprod[rx];
    const double lnkf = c_mech.lnA[rx] + c_mech.b[rx] * lnT - c_mech.Ta[rx] * iT;
    const double kf = exp(lnkf);
    double kb = 0.0;
    if (c_mech.rev[rx]) {
      double sum = 0.0;
      for (int e = 0; e < npr; e++) sum += g[c_mech.prod[rx][e]];
      for (int e = 0; e < nre; e++) sum -= g[c_mech.reac[rx][e]];
      kb = exp(lnkf - sum - (double)c_mech.dn[rx] * lnC0);
    }
    double pf = kf, pb = kb;
    for (int e = 0; e < nre; e++) pf *= X[c_mech.reac[rx][e]];
    for (int e = 0; e < npr; e++) pb *= X[c_mech.prod[rx][e]];
    double M = 1.0;
    const bool tb = c_mech.tb[rx] != 0;
    if (tb) {
      M = 0.0;
      for (int a = 0; a < ns; a++) M = fma(c_mech.eff[c_mech.tbi[rx]][a], X[a], M);
    }
    const double rnet = pf - pb;
    const double q = M * rnet;
    // stoichiometric scatter of q and of dq/dX
    for (int e = 0; e < npr; e++) wdot[c_mech.prod[rx][e]] += q;
    for (int e = 0; e < nre; e++) wdot[c_mech.reac[rx][e]] -= q;
    // dq/dX_j: forward part: for each reactant entry e, M kf prod_{e' != e} X
    for (int side = 0; side < 2; side++) {
      const unsigned char *lst = side == 0 ? c_mech.reac[rx] : c_mech.prod[rx];
      const int cnt = side == 0 ? nre : npr;
      const double kk = side == 0 ? M * kf : -M * kb;
      if (kk == 0.0) continue;
      for (int e = 0; e < cnt; e++) {
        double dq = kk;
        for (int e2 = 0; e2 < cnt; e2++)
          if (e2 != e) dq *= X[lst[e2]];
        const int jcol = lst[e];
        for (int e3 = 0; e3 < npr; e3++) { int kr = c_mech.prod[rx][e3]; if (kr < n1) D[kr][jcol] += dq; }
        for (int e3 = 0; e3 < nre; e3++) { int kr = c_mech.reac[rx][e3]; if (kr < n1) D[kr][jcol] -= dq; }
      }
    }
    if (tb) {
      for (int e3 = 0; e3 < npr; e3++) {
        int kr = c_mech.prod[rx][e3];
        if (kr < n1) for (int a = 0; a < ns; a++) D[kr][a] = fma(c_mech.eff[c_mech.tbi[rx]][a], rnet, D[kr][a]);
      }
      for (int e3 = 0; e3 < nre; e3++) {
        int kr = c_mech.reac[rx][e3];
        if (kr < n1) for (int a = 0; a < ns; a++) D[kr][a] = fma(-c_mech.eff[c_mech.tbi[rx]][a], rnet, D[kr][a]);
      }
    }
  }

  if (n1 > 0 && nr > 0) {
    // ---- A = I - dt J,  J_kl = W_k (D[k][l]/W_l - D[k][Ns]/W_Ns);  rhs = dt W_k wdot_k
    const double dt = P.scal[0] * P.dt_scale;
    double rhs[N1M > 0 ? N1M : 1];
    const double iWn = c_mech.invW[n1];
    for (int a = 0; a < n1; a++) {
      const double wk = c_mech.W[a];
      const double dl = D[a][n1] * iWn;
      for (int b = 0; b < n1; b++) {
        const double J = wk * (D[a][b] * c_mech.invW[b] - dl);
        D[a][b] = (a == b ? 1.0 : 0.0) - dt * J;
      }
      rhs[a] = dt * wk * wdot[a];
    }
    // ---- Gaussian elimination with partial pivoting
    for (int c = 0; c < n1; c++) {
      int piv = c;
      double best = fabs(D[c][c]);
      for (int r = c + 1; r < n1; r++) {
        double v = fabs(D[r][c]);
        if (v > best) { best = v; piv = r; }
      }
      if (!(best > 0.0)) ok = false;
      if (piv != c) {
        for (int b = c; b < n1; b++) { double tmp = D[c][b]; D[c][b] = D[piv][b]; D[piv][b] = tmp; }
        double tmp = rhs[c]; rhs[c] = rhs[piv]; rhs[piv] = tmp;
      }
      const double ipv = 1.0 / D[c][c];
      for (int r = c + 1; r < n1; r++) {
        const double f = D[r][c] * ipv;
        for (int b = c + 1; b < n1; b++) D[r][b] = fma(-f, D[c][b], D[r][b]);
        rhs[r] = fma(-f, rhs[c], rhs[r]);
      }
    }
    for (int r = n1 - 1; r >= 0; r--) {
      double sum = rhs[r];
      for (int b = r + 1; b < n1; b++) sum = fma(-D[r][b], rhs[b], sum);
      rhs[r] = sum / D[r][r];
    }
    for (int a = 0; a < n1; a++) {
      if (!isfinite(rhs[a])) ok = false;
      Up[(long long)(P.ndim + 2 + a) * P.pc + id] = ry[a] + rhs[a];
    }
  }
  if (!ok) *P.flag = 1;
}

// ------------------------------------------------------------------------------------------------
// k_chem_reg: register-resident variant for small species counts (NS <= 12), one thread per cell.
// Every per-cell array indexed by a *static* (unrolled) index lives in registers: Y, g, wdot, the
// (NS-1) x NS matrix D and the linear system.  The mechanism tables are uniform across the warp, so
// the few arrays that must be indexed by a run-time species / reaction id (X_j for the rate products,
// M k_f and M k_b per reaction for the derivative terms) sit in shared memory as [slot][thread]:
// conflict-free, uniform address arithmetic.  D is gathered column by column (static column j, run-time
// list of the derivative terms of that column, dense static rows weighted by dnu_ik), which replaces
// the dynamically indexed scatter of k_chem (local memory: 16 GB of spill traffic per launch on cfg2).
// Partial pivoting uses predicated row swaps so that the matrix never leaves registers.
template <int NS, int NT>
__global__ void __launch_bounds__(NT) k_chem_reg(Params P, double *__restrict__ U) {
  constexpr int N1 = NS - 1;
  extern __shared__ double sm[];
  const int nr = c_mech.nr;
  double *sX = sm + threadIdx.x;                  // [NS]
  double *scf = sX + NS * NT;                     // [nr]  M k_f
  double *scb = scf + nr * NT;                    // [nr]  -M k_b
  double *srn = scb + nr * NT;                    // [ntb] k_f prod X - k_b prod X of third-body reactions
  const int patch = blockIdx.y + P.patch0;
  const long long ncell = (long long)P.n[0] * P.n[1] * P.n[2];
  long long t = (long long)blockIdx.x * NT + threadIdx.x;
  const bool live = t < ncell;
  if (!live) t = ncell - 1;                       // idle lanes recompute the last cell, store nothing
  const int i = (int)(t % P.n[0]);
  const long long r_ = t / P.n[0];
  const int j_ = (int)(r_ % P.n[1]);
  const int k_ = (int)(r_ / P.n[1]);
  const long long id = cell_index(P, i, j_, k_);
  double *Up = U + (long long)patch * P.nvar * P.pc;
  const long long pid = (long long)patch * P.pc + id;

  // ---- T* = T(U*)  (update_aux), X_k = rho Y_k / W_k
  const double rho = Up[id];
  const double irho = 1.0 / rho;
  double ke = 0.0;
  for (int d = 0; d < P.ndim; d++) {
    const double ud = Up[(long long)(1 + d) * P.pc + id] * irho;
    ke = fma(0.5 * ud, ud, ke);
  }
  double ry[N1 > 0 ? N1 : 1], Y[NS], X[NS];
  double ysum = 0.0, rsum = 0.0;
#pragma unroll
  for (int a = 0; a < N1; a++) {
    ry[a] = Up[(long long)(P.ndim + 2 + a) * P.pc + id];
    Y[a] = ry[a] * irho;
    ysum += Y[a];
    rsum += ry[a];
    X[a] = ry[a] * c_mech.invW[a];
  }
  Y[N1] = 1.0 - ysum;
  X[N1] = (rho - rsum) * c_mech.invW[N1];
  const double e = Up[(long long)(P.ndim + 1) * P.pc + id] * irho - ke;
  double T = P.T[pid];
  bool ok = newton_T<NS>(Y, NS, e, T);
  if (live) P.T[pid] = T;
#pragma unroll
  for (int a = 0; a < NS; a++) sX[a * NT] = X[a];

  // ---- g_j = s_j/R_j - h_j/(R_j T)
  const double lnT = log(T), iT = 1.0 / T;
  double g[NS];
#pragma unroll
  for (int a = 0; a < NS; a++) g[a] = s_R(a, T, lnT) - h_R(a, T) * iT;
  const double lnC0 = log(JANC_PATM / (JANC_RU * T));

  // ---- rates of progress (eq 4.7-4.9); wdot_k = sum_i dnu_ik q_i (mol-based)
  double wdot[NS];
#pragma unroll
  for (int a = 0; a < NS; a++) wdot[a] = 0.0;
#pragma unroll 2
  for (int rx = 0; rx < nr; rx++) {
    const int nre = c_mech.nreac[rx], npr = c_mech.nprod[rx];
    const double lnkf = fma(c_mech.b[rx], lnT, c_mech.lnA[rx]) - c_mech.Ta[rx] * iT;
    double dg = (double)c_mech.dn[rx] * lnC0;
#pragma unroll
    for (int a = 0; a < NS; a++) dg = fma(c_mech.dnu[rx][a], g[a], dg);
    const double kf = exp(lnkf);
    const double kb = c_mech.rev[rx] ? exp(lnkf - dg) : 0.0;
    double pf = kf, pb = kb;
    for (int e2 = 0; e2 < nre; e2++) pf *= sX[c_mech.reac[rx][e2] * NT];
    for (int e2 = 0; e2 < npr; e2++) pb *= sX[c_mech.prod[rx][e2] * NT];
    const double rnet = pf - pb;
    double M = 1.0;
    if (c_mech.tb[rx]) {
      const int tq = c_mech.tbi[rx];
      M = 0.0;
#pragma unroll
      for (int a = 0; a < NS; a++) M = fma(c_mech.eff[tq][a], X[a], M);
      srn[tq * NT] = rnet;
    }
    scf[rx * NT] = M * kf;
    scb[rx * NT] = -(M * kb);
    const double q = M * rnet;
#pragma unroll
    for (int a = 0; a < NS; a++) wdot[a] = fma(c_mech.dnu[rx][a], q, wdot[a]);
  }

  if (N1 > 0 && nr > 0) {
    // ---- D[k][j] = sum_i dnu_ik dq_i/dX_j, column by column
    double D[N1 > 0 ? N1 : 1][NS];
#pragma unroll
    for (int j = 0; j < NS; j++) {
      double col[N1 > 0 ? N1 : 1];
#pragma unroll
      for (int k = 0; k < N1; k++) col[k] = 0.0;
      const int e0 = c_mech.col_start[j], e1 = c_mech.col_start[j + 1];
      for (int en = e0; en < e1; en++) {
        const int erx = c_mech.ent[en].rx, nother = c_mech.ent[en].nother;
        double dq = c_mech.ent[en].side ? scb[erx * NT] : scf[erx * NT];
        for (int o = 0; o < nother; o++) dq *= sX[c_mech.ent[en].other[o] * NT];
#pragma unroll
        for (int k = 0; k < N1; k++) col[k] = fma(c_mech.dnu[erx][k], dq, col[k]);
      }
      for (int rx = 0; rx < nr; rx++) {            // third-body factor: dM_i/dX_j = a_ij
        if (!c_mech.tb[rx]) continue;
        const int tq = c_mech.tbi[rx];
        const double v = c_mech.eff[tq][j] * srn[tq * NT];
#pragma unroll
        for (int k = 0; k < N1; k++) col[k] = fma(c_mech.dnu[rx][k], v, col[k]);
      }
#pragma unroll
      for (int k = 0; k < N1; k++) D[k][j] = col[k];
    }
    // ---- A = I - dt J,  J_kl = W_k (D[k][l]/W_l - D[k][Ns]/W_Ns);  rhs = dt W_k wdot_k
    const double dt = P.scal[0] * P.dt_scale;
    double rhs[N1 > 0 ? N1 : 1];
    const double iWn = c_mech.invW[N1];
#pragma unroll
    for (int a = 0; a < N1; a++) {
      const double wk = -dt * c_mech.W[a];
      const double dl = D[a][N1] * iWn;
#pragma unroll
      for (int b = 0; b < N1; b++) D[a][b] = fma(wk, fma(D[a][b], c_mech.invW[b], -dl), a == b ? 1.0 : 0.0);
      rhs[a] = -wk * wdot[a];
    }
    // ---- Gaussian elimination, partial pivoting by predicated row swaps.  static_for (template
    // recursion) rather than "#pragma unroll": nvcc leaves the swap loop rolled otherwise and the
    // matrix falls into local memory.
    static_for<0, N1>([&](auto c_) {
      constexpr int c = decltype(c_)::value;
      int piv = c;
      double best = fabs(D[c][c]);
      static_for<c + 1, N1>([&](auto r_) {
        constexpr int r = decltype(r_)::value;
        const double v = fabs(D[r][c]);
        if (v > best) { best = v; piv = r; }
      });
      if (!(best > 0.0)) ok = false;
      static_for<c + 1, N1>([&](auto r_) {
        constexpr int r = decltype(r_)::value;
        const bool sw = piv == r;
        static_for<c, N1>([&](auto b_) {
          constexpr int b = decltype(b_)::value;
          const double x = D[c][b], y = D[r][b];
          D[c][b] = sw ? y : x;
          D[r][b] = sw ? x : y;
        });
        const double x = rhs[c], y = rhs[r];
        rhs[c] = sw ? y : x;
        rhs[r] = sw ? x : y;
      });
      const double ipv = 1.0 / D[c][c];
      static_for<c + 1, N1>([&](auto r_) {
        constexpr int r = decltype(r_)::value;
        const double f = D[r][c] * ipv;
        static_for<c + 1, N1>([&](auto b_) {
          constexpr int b = decltype(b_)::value;
          D[r][b] = fma(-f, D[c][b], D[r][b]);
        });
        rhs[r] = fma(-f, rhs[c], rhs[r]);
      });
      D[c][c] = ipv;
    });
    static_for<0, N1>([&](auto q_) {
      constexpr int r = N1 - 1 - decltype(q_)::value;
      double sum = rhs[r];
      static_for<r + 1, N1>([&](auto b_) {
        constexpr int b = decltype(b_)::value;
        sum = fma(-D[r][b], rhs[b], sum);
      });
      rhs[r] = sum * D[r][r];
    });
#pragma unroll
    for (int a = 0; a < N1; a++) {
      if (!isfinite(rhs[a])) ok = false;
      if (live) Up[(long long)(P.ndim + 2 + a) * P.pc + id] = ry[a] + rhs[a];
    }
  }
  if (!ok && live) *P.flag = 1;
}
