// chemgen_roles.h -- run-time specialised point-implicit chemistry for LARGE mechanisms ("jit-roles").
// PAPER.md:260-277 (eq 4.6-4.9), :297-304 (eq 4.12-4.13), :333 (solve_implicit_rate), :340; readings A9-A12.
//
// Why another kernel: with one thread per cell (chemgen.h) the (Ns-1) x Ns system of a 20-species mechanism
// (3 KB per cell) has to live in shared memory, which leaves room for ~2 warps per SM and the kernel crawls
// on latency.  Here a CTA of 8 warps advances 32 cells: lane = cell, warp = ROLE.  Role w owns
//   * species  k = w, w+8, w+16      (Newton partial sums for T, the final rho Y_k update),
//   * reactions dealt round-robin    (Arrhenius / equilibrium exponentials, rates of progress; shared
//                                     table-driven code, tables in __constant__ memory indexed by the
//                                     warp-uniform role: no divergence, no per-lane table traffic),
//   * columns  j = w, w+8, w+16 of the system [I - dt J | rhs], held in REGISTERS (57 doubles for Ns = 20).
// The Jacobian columns are assembled by role-specific literal code (switch on the warp index: every
// species / reaction index a literal, every update one register FMA, structural zeros never touched),
// reading the 2 Nr rate coefficients the roles exchanged through shared memory ([row][cell], conflict-free).
// Gaussian elimination with partial pivoting is column-distributed: the owner of column c finds the pivot
// and publishes the multipliers (double-buffered: one CTA barrier per column), every role swaps / updates
// its own columns in registers.  The upper triangle then goes to shared memory and the role holding the
// right-hand side back-substitutes.  All 8 roles of a cell see bit-identical T (same sums, same order).
#pragma once
#include <algorithm>

#include "chemgen.h"

#define JANC_ROLES 8
#define JANC_ROLES_MAXSLOT 3      // columns per role held in registers => Ns <= 24

namespace chemgen {

struct RolesLayout {
  int oX, oP, oN, oRN, oDL, oRHS, oF, oPIV, oXS, oR, rows;   // offsets in rows of 32 doubles
  size_t smem() const { return (size_t)rows * 32 * sizeof(double); }
};

inline bool roles_applicable(const MechC &M) {
  return M.ns >= 3 && M.ns <= JANC_ROLES * JANC_ROLES_MAXSLOT && M.nr >= 1;
}

inline RolesLayout roles_layout(const MechC &M) {
  const int ns = M.ns, n1 = ns - 1, nr = M.nr;
  RolesLayout L;
  int o = 0;
  L.oX = o; o += ns + 1;                     // X_k, plus a dummy species with X = 1
  L.oP = o; o += 16;                         // partial sums of rho Y_k and Y_k per role
  L.oN = o; o += 16;                         // Newton partial sums per role
  L.oRN = o; o += M.ntb > 0 ? M.ntb : 1;     // net rate without the third-body factor (third-body reactions)
  L.oDL = o; o += n1;                        // D_kN / W_N
  L.oRHS = o; o += n1;                       // dt W_k wdot_k
  L.oF = o; o += 2 * n1;                     // elimination multipliers, double-buffered
  L.oPIV = o; o += 2;                        // pivot row (int), double-buffered
  L.oXS = o; o += n1;                        // solution
  L.oR = o; o += std::max(3 * nr, n1 * (n1 + 1) / 2);   // M k_f, M k_b, q per reaction; later the upper triangle
  L.rows = o;
  return L;
}

inline std::string generate_roles(const MechC &M, int ndim) {
  const int ns = M.ns, nr = M.nr, n1 = ns - 1, nvar = ndim + 2 + n1, NR = JANC_ROLES;
  const int NSL = (ns + NR - 1) / NR;                  // column slots per role (columns 0..n1)
  const int wN = n1 % NR, sN = n1 / NR;                // role / slot of column N (later the right-hand side)
  const RolesLayout L = roles_layout(M);
  Emitter E;
  std::string &src = E.s;
  auto row = [](int r) { return "SM(" + I(r) + ")"; };
  auto A = [](int s, int k) { return "A" + I(s) + "_" + I(k); };

  // ---- per-reaction stoichiometry
  std::vector<std::vector<int>> cf(nr, std::vector<int>(ns, 0)), cb(nr, std::vector<int>(ns, 0)), dnu(nr, std::vector<int>(ns, 0));
  int maxof = 1, maxob = 1;
  bool any_rev = false;
  for (int i = 0; i < nr; i++) {
    for (int e = 0; e < M.nreac[i]; e++) cf[i][M.reac[i][e]]++;
    for (int e = 0; e < M.nprod[i]; e++) cb[i][M.prod[i][e]]++;
    for (int k = 0; k < ns; k++) dnu[i][k] = cb[i][k] - cf[i][k];
    maxof = std::max(maxof, (int)M.nreac[i]);
    if (M.rev[i]) { maxob = std::max(maxob, (int)M.nprod[i]); any_rev = true; }
  }
  // ---- Newton polynomials (h_k/R_k - T, c_p,k/R_k - 1) truncated at the highest degree any species uses
  int degh = 1, degc = 0;
  for (int k = 0; k < ns; k++)
    for (int q = 1; q <= 4; q++)
      if (M.nasa[k][q] != 0.0) { degh = std::max(degh, q + 1); degc = std::max(degc, q); }
  // ---- reverse rate: ln k_b = ln k_f - dn ln(p_atm / (R_u T)) - sum_k dnu_k g_k(T) collected per reaction as
  //      d0 + d1 ln T + d2 / T + T (d3 + T (d4 + T (d5 + T d6)))   (eq 4.8-4.9; g_k = s_k/R - h_k/(R T))
  const int NKB = 3 + degc;
  std::vector<double> kbc((size_t)nr * 7, 0.0);
  for (int i = 0; i < nr; i++) {
    double *d = &kbc[(size_t)i * 7];
    d[0] = M.lnA[i] - (double)M.dn[i] * log(JANC_PATM / JANC_RU);
    d[1] = M.b[i] + (double)M.dn[i];
    d[2] = -M.Ta[i];
    for (int k = 0; k < ns; k++) {
      if (dnu[i][k] == 0) continue;
      const double v = (double)dnu[i][k];
      const double *c = M.nasa[k];
      d[0] -= v * (c[6] - c[0]);
      d[1] -= v * c[0];
      d[2] += v * c[5];
      d[3] -= v * c[1] * 0.5;
      d[4] -= v * c[2] / 6.0;
      d[5] -= v * c[3] / 12.0;
      d[6] -= v * c[4] / 20.0;
    }
  }
  // ---- reactions dealt to roles: third-body reactions first (their efficiency sums are the long ones)
  std::vector<int> order;
  for (int i = 0; i < nr; i++) if (M.tb[i]) order.push_back(i);
  for (int i = 0; i < nr; i++) if (!M.tb[i]) order.push_back(i);
  const int NSLOT = (nr + NR - 1) / NR;
  std::vector<int> ri((size_t)NR * NSLOT, -1);
  for (int q = 0; q < nr; q++) ri[(size_t)(q % NR) * NSLOT + q / NR] = order[q];

  // =========================================================================== tables
  src += "// generated by chemgen_roles.h for ns=" + I(ns) + " nr=" + I(nr) + " ndim=" + I(ndim) + "\n";
  src += "struct ChemArgs { double *U; double *T; const double *scal; int *flag; int n0, n1, n2, G0, G1, G2;"
         " long long st0, st1, st2, pc; };\n";
  auto table = [&](const std::string &decl, const std::vector<std::string> &v) {
    src += "__constant__ " + decl + " = {";
    for (size_t q = 0; q < v.size(); q++) src += (q ? ", " : "") + v[q];
    src += "};\n";
  };
  std::vector<std::string> t;
  t.clear(); for (int k = 0; k < ns; k++) t.push_back(num(M.invW[k]));
  table("double c_iW[" + I(ns) + "]", t);
  t.clear(); for (int k = 0; k < ns; k++) t.push_back(num(M.Rk[k]));
  table("double c_Rk[" + I(ns) + "]", t);
  t.clear();
  for (int k = 0; k < ns; k++) {
    const double *c = M.nasa[k];
    const double hc[6] = {c[5], c[0] - 1.0, 0.5 * c[1], c[2] / 3.0, 0.25 * c[3], 0.2 * c[4]};
    for (int q = 0; q <= degh; q++) t.push_back(num(hc[q]));
  }
  table("double c_hc[" + I(ns * (degh + 1)) + "]", t);
  t.clear();
  for (int k = 0; k < ns; k++) {
    const double *c = M.nasa[k];
    const double cc[5] = {c[0] - 1.0, c[1], c[2], c[3], c[4]};
    for (int q = 0; q <= degc; q++) t.push_back(num(cc[q]));
  }
  table("double c_cc[" + I(ns * (degc + 1)) + "]", t);
  t.clear(); for (int i = 0; i < nr; i++) { t.push_back(num(M.lnA[i])); t.push_back(num(M.b[i])); t.push_back(num(-M.Ta[i])); }
  table("double c_kf[" + I(nr * 3) + "]", t);
  t.clear(); for (int i = 0; i < nr; i++) for (int q = 0; q < NKB; q++) t.push_back(num(kbc[(size_t)i * 7 + q]));
  table("double c_kb[" + I(nr * NKB) + "]", t);
  t.clear();
  for (int q = 0; q < (M.ntb > 0 ? M.ntb : 1); q++) for (int k = 0; k < ns; k++) t.push_back(num(M.ntb > 0 ? M.eff[q][k] : 0.0));
  table("double c_eff[" + I((M.ntb > 0 ? M.ntb : 1) * ns) + "]", t);
  t.clear(); for (int v : ri) t.push_back(I(v));
  table("int c_ri[" + I(NR * NSLOT) + "]", t);
  t.clear(); for (int i = 0; i < nr; i++) t.push_back(I((M.rev[i] ? 1 : 0) | ((M.tb[i] ? M.tbi[i] + 1 : 0) << 1)));
  table("int c_fl[" + I(nr) + "]", t);
  t.clear(); for (int i = 0; i < nr; i++) for (int q = 0; q < maxof; q++) t.push_back(I(q < M.nreac[i] ? M.reac[i][q] : ns));
  table("unsigned char c_re[" + I(nr * maxof) + "]", t);
  t.clear(); for (int i = 0; i < nr; i++) for (int q = 0; q < maxob; q++) t.push_back(I(q < M.nprod[i] ? M.prod[i][q] : ns));
  table("unsigned char c_pr[" + I(nr * maxob) + "]", t);

  // =========================================================================== kernel
  src += "#define SM(r) sm_[(r) * 32 + lane]\n";
  src += "#define BAR() asm volatile(\"bar.sync 0;\" ::: \"memory\")\n";
  src += "extern \"C\" __global__ void __launch_bounds__(" + I(NR * 32) + ", 1) k_chem_jit(ChemArgs a) {\n";
  E.line("extern __shared__ double sm_[];");
  E.line("const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;");
  E.line("int *s_piv = (int *)(sm_ + " + I(L.oPIV * 32) + ");");
  E.line("const long long ncell = (long long)a.n0 * a.n1 * a.n2;");
  E.line("long long t = (long long)blockIdx.x * 32 + lane;");
  E.line("const bool live = t < ncell;");
  E.line("if (!live) t = ncell - 1;   // idle lanes recompute the last cell and store nothing");
  E.line("const int ci = (int)(t % a.n0); const long long r_ = t / a.n0;");
  E.line("const int cj = (int)(r_ % a.n1), ck = (int)(r_ / a.n1);");
  E.line("const long long id = (ci + a.G0) * a.st0 + (cj + a.G1) * a.st1 + (ck + a.G2) * a.st2;");
  E.line("double *Up = a.U + (long long)blockIdx.y * " + I(nvar) + " * a.pc + id;");
  E.line("const long long pid = (long long)blockIdx.y * a.pc + id;");
  E.line("const double dt = a.scal[0];");
  // ---- cons -> prim pieces (eq 4.2); species k = w + 8 s belong to this role
  E.line("const double rho = Up[0], irho = 1.0 / rho;");
  E.line("double ke = 0.0;");
  for (int d = 0; d < ndim; d++)
    E.line("{ const double ud = Up[" + I(1 + d) + " * a.pc] * irho; ke = fma(0.5 * ud, ud, ke); }");
  E.line("const double e = Up[" + I(ndim + 1) + " * a.pc] * irho - ke;");
  E.line("double pr_ = 0.0, py_ = 0.0;");
  for (int s = 0; s < NSL; s++) {
    const std::string ss = I(s);
    E.line("const int k" + ss + " = w + " + I(NR * s) + ";");
    E.line("double ry" + ss + " = k" + ss + " < " + I(n1) + " ? Up[(long long)(" + I(ndim + 2) + " + k" + ss + ") * a.pc] : 0.0;");
    E.line("double Y" + ss + " = ry" + ss + " * irho;");
    E.line("pr_ += ry" + ss + "; py_ += Y" + ss + ";");
    E.line("if (k" + ss + " < " + I(n1) + ") SM(" + I(L.oX) + " + k" + ss + ") = ry" + ss + " * c_iW[k" + ss + "];");
  }
  E.line("SM(" + I(L.oP) + " + w) = pr_; SM(" + I(L.oP + 8) + " + w) = py_;");
  E.line("if (w == 0) SM(" + I(L.oX + ns) + ") = 1.0;");
  E.line("BAR();");
  E.line("{ double rsum = 0.0, ysum = 0.0;");
  E.line("  #pragma unroll");
  E.line("  for (int q = 0; q < 8; q++) { rsum += SM(" + I(L.oP) + " + q); ysum += SM(" + I(L.oP + 8) + " + q); }");
  E.line("  if (w == " + I(wN) + ") { ry" + I(sN) + " = rho - rsum; Y" + I(sN) + " = 1.0 - ysum; SM(" + I(L.oX + n1) + ") = ry" + I(sN) + " * " + num(M.invW[n1]) + "; } }");
  for (int s = 0; s < NSL; s++)
    E.line("const double yr" + I(s) + " = k" + I(s) + " < " + I(ns) + " ? Y" + I(s) + " * c_Rk[k" + I(s) + " < " + I(ns) + " ? k" + I(s) + " : 0] : 0.0;");
  // ---- Newton on e(T) (eq 4.3-4.4, reading A6): partial sums per role, summed in the same order by everyone
  E.line("double T = a.T[pid];");
  E.line("bool conv = false;");
  E.line("#pragma unroll 1");
  E.line("for (int it = 0; it < 50; it++) {");
  E.line("  double f = 0.0, cv = 0.0;");
  for (int s = 0; s < NSL; s++) {
    const std::string ks = "k" + I(s);
    std::string h = "h_[" + I(degh) + "]", c = "c_[" + I(degc) + "]";
    for (int q = degh - 1; q >= 0; q--) h = "fma(T, " + h + ", h_[" + I(q) + "])";
    for (int q = degc - 1; q >= 0; q--) c = "fma(T, " + c + ", c_[" + I(q) + "])";
    E.line("  if (" + ks + " < " + I(ns) + ") { const double *h_ = c_hc + " + ks + " * " + I(degh + 1) + ", *c_ = c_cc + " + ks + " * " + I(degc + 1) + ";");
    E.line("    f = fma(yr" + I(s) + ", " + h + ", f); cv = fma(yr" + I(s) + ", " + c + ", cv); }");
  }
  E.line("  SM(" + I(L.oN) + " + w) = f; SM(" + I(L.oN + 8) + " + w) = cv;");
  E.line("  BAR();");
  E.line("  f = -e; cv = 0.0;");
  E.line("  #pragma unroll");
  E.line("  for (int q = 0; q < 8; q++) { f += SM(" + I(L.oN) + " + q); cv += SM(" + I(L.oN + 8) + " + q); }");
  E.line("  const double dT = -f / cv;");
  E.line("  if (!conv) { T += dT; if (fabs(dT) <= 1e-11 * fabs(T)) conv = true; }");
  E.line("  if (__syncthreads_and(conv)) break;");
  E.line("}");
  E.line("bool ok = conv && (T > 0.0) && isfinite(T);");
  E.line("if (live && w == 0) a.T[pid] = T;");
  // ---- rates of progress (eq 4.7-4.9): shared code, tables indexed by the warp-uniform role
  E.line("{ const double lnT = log(T), iT = 1.0 / T;");
  E.line("  #pragma unroll 1");
  E.line("  for (int r = 0; r < " + I(NSLOT) + "; r++) {");
  E.line("    const int i = c_ri[w * " + I(NSLOT) + " + r];");
  E.line("    if (i < 0) break;");
  E.line("    const double *f_ = c_kf + 3 * i;");
  E.line("    const double lkf = fma(f_[2], iT, fma(f_[1], lnT, f_[0]));");
  E.line("    const double kf = exp(lkf);");
  E.line("    const int fl = c_fl[i];");
  E.line("    double kb = 0.0;");
  if (any_rev) {
    E.line("    if (fl & 1) { const double *d_ = c_kb + " + I(NKB) + " * i;");
    std::string lk = "fma(d_[2], iT, fma(d_[1], lnT, d_[0]))";
    if (degc > 0) {
      std::string pol = "d_[" + I(NKB - 1) + "]";
      for (int q = NKB - 2; q >= 3; q--) pol = "fma(T, " + pol + ", d_[" + I(q) + "])";
      lk = "fma(T, " + pol + ", " + lk + ")";
    }
    E.line("      kb = exp(" + lk + "); }");
  }
  E.line("    double pf = kf, pb = kb;");
  for (int q = 0; q < maxof; q++) E.line("    pf *= SM(" + I(L.oX) + " + c_re[i * " + I(maxof) + " + " + I(q) + "]);");
  if (any_rev) for (int q = 0; q < maxob; q++) E.line("    pb *= SM(" + I(L.oX) + " + c_pr[i * " + I(maxob) + " + " + I(q) + "]);");
  E.line("    const double rn = pf - pb;");
  E.line("    double Mi = 1.0;");
  if (M.ntb > 0) {
    E.line("    const int tb_ = (fl >> 1) - 1;");
    E.line("    if (tb_ >= 0) { const double *ef = c_eff + tb_ * " + I(ns) + ";");
    E.line("      Mi = ef[0] * SM(" + I(L.oX) + ");");
    E.line("      #pragma unroll");
    E.line("      for (int j = 1; j < " + I(ns) + "; j++) Mi = fma(ef[j], SM(" + I(L.oX) + " + j), Mi);");
    E.line("      SM(" + I(L.oRN) + " + tb_) = rn; }");
  }
  E.line("    SM(" + I(L.oR) + " + i) = Mi * kf; SM(" + I(L.oR + nr) + " + i) = Mi * kb; SM(" + I(L.oR + 2 * nr) + " + i) = Mi * rn;");
  E.line("  }");
  E.line("}");
  E.line("BAR();");
  // ---- role-specific literal code: right-hand-side rows and Jacobian columns of this role
  {
    std::string decl = "double ";
    for (int s = 0; s < NSL; s++)
      for (int k = 0; k < n1; k++) decl += A(s, k) + " = 0.0" + (s == NSL - 1 && k == n1 - 1 ? ";" : ", ");
    E.line(decl);
  }
  E.line("switch (w) {");
  for (int w = 0; w < NR; w++) {
    E.line("case " + I(w) + ": {");
    // wdot_k = sum_i dnu_ik q_i for the rows of this role; rhs_k = dt W_k wdot_k
    for (int s = 0; s < NSL; s++) {
      const int k = w + NR * s;
      if (k >= n1) continue;
      std::string sum;
      for (int i = 0; i < nr; i++) {
        if (dnu[i][k] == 0) continue;
        const std::string q = row(L.oR + 2 * nr + i);
        if (sum.empty()) sum = dnu[i][k] == 1 ? q : dnu[i][k] == -1 ? "-" + q : num((double)dnu[i][k]) + " * " + q;
        else if (dnu[i][k] == 1) sum = "(" + sum + " + " + q + ")";
        else if (dnu[i][k] == -1) sum = "(" + sum + " - " + q + ")";
        else sum = "fma(" + num((double)dnu[i][k]) + ", " + q + ", " + sum + ")";
      }
      E.line("  " + row(L.oRHS + k) + " = " + (sum.empty() ? std::string("0.0") : "(dt * " + num(M.W[k]) + ") * " + sum) + ";");
    }
    // columns: D_kj = sum_i dnu_ik dq_i/dX_j accumulated straight into the registers of column j
    std::vector<char> needX(ns, 0);
    for (int s = 0; s < NSL; s++) {
      const int j = w + NR * s;
      if (j > n1) continue;
      for (int i = 0; i < nr; i++) {
        if (cf[i][j] > 0) for (int k = 0; k < ns; k++) if (cf[i][k] - (k == j ? 1 : 0) > 0) needX[k] = 1;
        if (M.rev[i] && cb[i][j] > 0) for (int k = 0; k < ns; k++) if (cb[i][k] - (k == j ? 1 : 0) > 0) needX[k] = 1;
      }
    }
    for (int k = 0; k < ns; k++) if (needX[k]) E.line("  const double X" + I(k) + " = " + row(L.oX + k) + ";");
    for (int s = 0; s < NSL; s++) {
      const int j = w + NR * s;
      if (j > n1) continue;
      E.line("  // column " + I(j));
      Acc acc(n1);
      for (int i = 0; i < nr; i++) {
        const bool rev = M.rev[i] != 0, tb = M.tb[i] != 0;
        const std::string si = I(i);
        std::string dq;
        const std::string cfs = row(L.oR + i), cbs = row(L.oR + nr + i);
        if (cf[i][j] > 0) dq = (cf[i][j] > 1 ? num((double)cf[i][j]) + " * " : std::string("")) + xprod(cfs, cf[i].data(), ns, j);
        if (rev && cb[i][j] > 0) dq += (dq.empty() ? "-" : " - ") + (cb[i][j] > 1 ? num((double)cb[i][j]) + " * " : std::string("")) + xprod(cbs, cb[i].data(), ns, j);
        if (tb) {
          const double a = M.eff[M.tbi[i]][j];
          const std::string rn = row(L.oRN + M.tbi[i]);
          if (a != 0.0) dq = dq.empty() ? num(a) + " * " + rn : "fma(" + num(a) + ", " + rn + ", " + dq + ")";
        }
        if (dq.empty()) continue;
        bool any = false;
        for (int k = 0; k < n1; k++) any = any || dnu[i][k] != 0;
        if (!any) continue;
        E.line("  { const double dq = " + dq + ";");
        for (int k = 0; k < n1; k++) {
          if (dnu[i][k] == 0) continue;
          acc.set[k] = 1;
          if (dnu[i][k] == 1) E.line("    " + A(s, k) + " += dq;");
          else if (dnu[i][k] == -1) E.line("    " + A(s, k) + " -= dq;");
          else E.line("    " + A(s, k) + " = fma(" + num((double)dnu[i][k]) + ", dq, " + A(s, k) + ");");
        }
        E.line("  }");
      }
      if (j == n1)
        for (int k = 0; k < n1; k++) E.line("  " + row(L.oDL + k) + " = " + A(s, k) + " * " + num(M.invW[n1]) + ";");
    }
    E.line("} break;");
  }
  E.line("}");
  E.line("BAR();");
  // ---- A = I - dt J,  J_kl = W_k (D_kl / W_l - D_kN / W_N);  column N becomes rhs = dt W_k wdot_k  (eq 4.12-4.13, A11)
  E.line("{");
  for (int k = 0; k < n1; k++) E.line("  const double mw" + I(k) + " = -dt * " + num(M.W[k]) + ", dl" + I(k) + " = " + row(L.oDL + k) + ";");
  for (int s = 0; s < NSL; s++) {
    const std::string js = "k" + I(s);
    E.line("  if (" + js + " < " + I(n1) + ") { const double iw = c_iW[" + js + "];");
    for (int k = 0; k < n1; k++)
      E.line("    " + A(s, k) + " = fma(mw" + I(k) + ", fma(" + A(s, k) + ", iw, -dl" + I(k) + "), " + js + " == " + I(k) + " ? 1.0 : 0.0);");
    E.line("  }");
    if (s == sN) {
      E.line("  else if (" + js + " == " + I(n1) + ") {");
      for (int k = 0; k < n1; k++) E.line("    " + A(s, k) + " = " + row(L.oRHS + k) + ";");
      E.line("  }");
    }
  }
  E.line("}");
  // ---- Gaussian elimination with partial pivoting, column-distributed (the oracle's pivot choice: first row of
  //      maximal |a_rc|); L is not kept: the right-hand side is a column of the system
  auto swap_chain = [&](int s, int c, const std::string &ind) {
    for (int r = c + 1; r < n1; r++)
      E.line(ind + "{ const bool sw = piv == " + I(r) + "; const double x_ = " + A(s, c) + ", y_ = " + A(s, r) + "; " +
             A(s, c) + " = sw ? y_ : x_; " + A(s, r) + " = sw ? x_ : y_; }");
  };
  for (int c = 0; c < n1; c++) {
    const int oc = c % NR, sc = c / NR, pb = c & 1;
    const bool last = c + 1 == n1;
    E.line("{ // column " + I(c));
    E.line("  if (w == " + I(oc) + ") {");
    if (!last) {
      E.line("    int piv = " + I(c) + "; double best = fabs(" + A(sc, c) + "), v;");
      for (int r = c + 1; r < n1; r++)
        E.line("    v = fabs(" + A(sc, r) + "); if (v > best) { best = v; piv = " + I(r) + "; }");
      E.line("    if (!(best > 0.0)) ok = false;");
      E.line("    if (__any_sync(0xffffffffu, piv != " + I(c) + ")) {");
      swap_chain(sc, c, "      ");
      E.line("    }");
      E.line("    s_piv[" + I(pb * 32) + " + lane] = piv;");
    } else {
      E.line("    if (!(fabs(" + A(sc, c) + ") > 0.0)) ok = false;");
    }
    E.line("    const double ip = 1.0 / " + A(sc, c) + ";");
    for (int r = c + 1; r < n1; r++) E.line("    " + row(L.oF + pb * n1 + r) + " = " + A(sc, r) + " * ip;");
    E.line("    " + A(sc, c) + " = ip;");
    E.line("  }");
    if (!last) {
      E.line("  BAR();");
      E.line("  const int piv = s_piv[" + I(pb * 32) + " + lane];");
      E.line("  if (__any_sync(0xffffffffu, piv != " + I(c) + ")) {");
      E.line("    if (w != " + I(oc) + ") {");
      swap_chain(sc, c, "      ");
      E.line("    }");
      for (int s = sc + 1; s < NSL; s++) swap_chain(s, c, "    ");
      E.line("  }");
      for (int r = c + 1; r < n1; r++) E.line("  const double f" + I(r) + " = " + row(L.oF + pb * n1 + r) + ";");
      E.line("  if (w > " + I(oc) + ") {");
      for (int r = c + 1; r < n1; r++) E.line("    " + A(sc, r) + " = fma(-f" + I(r) + ", " + A(sc, c) + ", " + A(sc, r) + ");");
      E.line("  }");
      for (int s = sc + 1; s < NSL; s++)
        for (int r = c + 1; r < n1; r++) E.line("  " + A(s, r) + " = fma(-f" + I(r) + ", " + A(s, c) + ", " + A(s, r) + ");");
    }
    E.line("}");
  }
  // ---- upper triangle (reciprocal pivots on the diagonal) -> shared memory; the role holding the rhs solves
  // (the rate arrays are dead since the barrier after the assembly: the triangle takes their place)
  auto tri = [&](int k) { return L.oR + k * n1 - k * (k - 1) / 2 - k; };   // + j
  for (int s = 0; s < NSL; s++) {
    const std::string js = "k" + I(s);
    E.line("if (" + js + " < " + I(n1) + ") {");
    for (int k = 0; k < n1; k++) {
      if (k > NR * s + NR - 1) break;
      E.line("  if (" + I(k) + " <= " + js + ") SM(" + I(tri(k)) + " + " + js + ") = " + A(s, k) + ";");
    }
    E.line("}");
  }
  E.line("BAR();");
  E.line("if (w == " + I(wN) + ") {");
  for (int r = n1 - 1; r >= 0; r--) {
    E.line("  " + A(sN, r) + " *= " + row(tri(r) + r) + ";");
    for (int k = 0; k < r; k++) E.line("  " + A(sN, k) + " = fma(-" + row(tri(k) + r) + ", " + A(sN, r) + ", " + A(sN, k) + ");");
  }
  for (int k = 0; k < n1; k++) {
    E.line("  if (!isfinite(" + A(sN, k) + ")) ok = false;");
    E.line("  " + row(L.oXS + k) + " = " + A(sN, k) + ";");
  }
  E.line("}");
  E.line("BAR();");
  for (int s = 0; s < NSL; s++)
    E.line("if (live && k" + I(s) + " < " + I(n1) + ") Up[(long long)(" + I(ndim + 2) + " + k" + I(s) + ") * a.pc] = ry" + I(s) +
           " + SM(" + I(L.oXS) + " + k" + I(s) + ");");
  E.line("if (!ok && live) *a.flag = 1;");
  src += "}\n#undef SM\n#undef BAR\n";
  return src;
}

}  // namespace chemgen
