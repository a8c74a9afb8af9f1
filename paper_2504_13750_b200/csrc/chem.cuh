// chem.cuh -- point-implicit chemistry kernel (advance_source_term).
// PAPER.md:260-277 (eq 4.6-4.9 rates, K_eq), :297-304 (eq 4.12-4.13), :333.
// Readings A9 (third body only where flagged), A10 (irreversible), A11 (Jacobian w.r.t.
// rho*Y_1..Ns-1 at frozen T and rho, Y_Ns through rho), A12 (no clipping).
// One thread per cell: T* by Newton (fused cons->prim), rates, analytic Jacobian, (I - dt J) d = dt w
// by Gaussian elimination with partial pivoting, rhoY += d.
#pragma once
#include "prim.cuh"

template <int NS>
__global__ void __launch_bounds__(128) k_chem(Params P, double *__restrict__ U) {
  constexpr int NSM = NS > 0 ? NS : JANC_MAX_NS;
  constexpr int N1M = NSM - 1;
  const int ns = NS > 0 ? NS : P.ns;
  const int n1 = ns - 1;
  const int nr = c_mech.nr;
  const int patch = blockIdx.y;
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
      for (int a = 0; a < ns; a++) M = fma(c_mech.eff[rx][a], X[a], M);
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
        if (kr < n1) for (int a = 0; a < ns; a++) D[kr][a] = fma(c_mech.eff[rx][a], rnet, D[kr][a]);
      }
      for (int e3 = 0; e3 < nre; e3++) {
        int kr = c_mech.reac[rx][e3];
        if (kr < n1) for (int a = 0; a < ns; a++) D[kr][a] = fma(-c_mech.eff[rx][a], rnet, D[kr][a]);
      }
    }
  }

  if (n1 > 0 && nr > 0) {
    // ---- A = I - dt J,  J_kl = W_k (D[k][l]/W_l - D[k][Ns]/W_Ns);  rhs = dt W_k wdot_k
    const double dt = P.scal[0];
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
