// chemgen.h -- run-time specialisation of the point-implicit chemistry kernel (host side).
// PAPER.md:260-277 (eq 4.6-4.9), :297-304 (eq 4.12-4.13), :333 (solve_implicit_rate), :340.
//
// The paper's solver is JIT-compiled by XLA with the mechanism baked in as constants
// (PAPER.md:24, :39).  The B200 counterpart: janc_set_mechanism() emits CUDA C for *this*
// mechanism -- every species / reaction index a literal, every coefficient an immediate, structural
// zeros of the Jacobian never touched -- and compiles it with NVRTC for sm_100a.  All per-cell
// arrays (X, g, wdot, the (Ns-1) x Ns derivative matrix, the linear system) become named scalars,
// i.e. registers; there is no table lookup, no shared memory and no local memory in the kernel.
// One thread per cell; partial pivoting keeps the oracle's pivot choice (predicated row swaps,
// skipped warp-wide when no lane needs one).
//
// The generic kernels of chem.cuh remain the path for mechanisms with more than JANC_JIT_MAX_N1
// unknowns or when NVRTC is not available (janc_chem_kernel() reports which one runs).
#pragma once
#include <cstdio>
#include <cstdlib>
#include <string>
#include <vector>

#include "common.cuh"

#define JANC_JIT_MAX_N1 12
#define JANC_JIT_NT 64
#define JANC_JIT_NT_BIG 32

namespace chemgen {

inline std::string num(double v) {
  char buf[64];
  snprintf(buf, sizeof buf, "%.17g", v);
  std::string s(buf);
  if (s.find_first_of(".eEn") == std::string::npos) s += ".0";
  if (v < 0) s = "(" + s + ")";
  return s;
}
inline std::string I(int v) { return std::to_string(v); }

// Horner form of c[0] + c[1] T + ... truncated at the highest non-zero coefficient
inline std::string horner(const double *c, int n) {
  int deg = n - 1;
  while (deg > 0 && c[deg] == 0.0) deg--;
  std::string s = num(c[deg]);
  for (int k = deg - 1; k >= 0; k--) s = "fma(T, " + s + ", " + num(c[k]) + ")";
  return s;
}

// The same polynomial for two-range NASA-7 data: every coefficient is a select on hi<k> (T >= T_mid of species k,
// declared by emit_range_flags next to each temperature the polynomials are evaluated at)
inline std::string horner2(const double *lo, const double *hi, int n, int k) {
  int deg = n - 1;
  while (deg > 0 && lo[deg] == 0.0 && hi[deg] == 0.0) deg--;
  auto co = [&](int q) { return lo[q] == hi[q] ? num(lo[q]) : "(hi" + std::to_string(k) + " ? " + num(hi[q]) + " : " + num(lo[q]) + ")"; };
  std::string s = co(deg);
  for (int q = deg - 1; q >= 0; q--) s = "fma(T, " + s + ", " + co(q) + ")";
  return s;
}
// polynomial in T of species k built from its 7 NASA coefficients by `build` (fills out[n])
template <class F>
inline std::string nasa_poly(const MechC &M, int k, int n, F build) {
  double lo[8], hi[8];
  build(M.nasa[k], lo);
  if (!M.two_range) return horner(lo, n);
  build(M.nasa_hi[k], hi);
  return horner2(lo, hi, n, k);
}

struct Emitter {
  std::string s;
  void line(const std::string &l) { s += "  " + l + "\n"; }
};

// accumulate  name (+|-)= coef * expr  keeping track of first assignment (structural zeros)
struct Acc {
  std::vector<char> set;
  explicit Acc(int n) : set(n, 0) {}
};
inline void accum(Emitter &E, Acc &A, int idx, const std::string &name, int coef, const std::string &expr) {
  if (coef == 0) return;
  if (!A.set[idx]) {
    A.set[idx] = 1;
    if (coef == 1) E.line("double " + name + " = " + expr + ";");
    else if (coef == -1) E.line("double " + name + " = -" + expr + ";");
    else E.line("double " + name + " = " + num((double)coef) + " * " + expr + ";");
  } else {
    if (coef == 1) E.line(name + " += " + expr + ";");
    else if (coef == -1) E.line(name + " -= " + expr + ";");
    else E.line(name + " = fma(" + num((double)coef) + ", " + expr + ", " + name + ");");
  }
}

// product  pre * X_a^na * X_b^nb ...  with one power of species `skip` removed (skip < 0: none)
inline std::string xprod(const std::string &pre, const int *cnt, int ns, int skip) {
  std::string s = pre;
  for (int j = 0; j < ns; j++) {
    int n = cnt[j] - (j == skip ? 1 : 0);
    for (int q = 0; q < n; q++) s += " * X" + I(j);
  }
  return s;
}

// Device helpers shared by the generated kernels.
//   exp_nb: branch-free exp (Cody-Waite reduction, degree-13 Taylor polynomial on |r| <= ln2/2 in Estrin form: < 2 ulp), argument
//           clamped to the finite range; half the instructions of the library exp and no slow-path branch, so the
//           exponentials of neighbouring reactions interleave.
//   rcp_nb: 1/x from the MUFU seed + 2 Newton steps (full fp64 precision for normal x of either sign; a zero or
//           denormal pivot gives inf / nan, which the callers' isfinite checks flag).
// form: 0 = Horner with literal coefficients, 1 = Estrin, 2 = Horner with the coefficients in __constant__ memory (the
// FMAs then take them as constant-bank operands; literals that do not fit a 32-bit immediate are re-materialised with
// two moves each time they are used)
inline void emit_math(std::string &src, int form = 0) {
  const bool estrin = form == 1;
  if (form == 2)
    src += "__constant__ double c_exp[14] = {1.6059043836821613e-10, 2.08767569878681e-09, 2.505210838544172e-08, 2.755731922398589e-07,\n"
           "  2.7557319223985893e-06, 2.48015873015873e-05, 1.984126984126984e-04, 1.388888888888889e-03, 8.333333333333333e-03,\n"
           "  4.1666666666666664e-02, 1.6666666666666666e-01, 0.5, 1.0, 1.0};\n";
  src += "__device__ __forceinline__ double exp_nb(double x) {\n"
         "  x = x < -708.0 ? -708.0 : (x > 709.0 ? 709.0 : x);     // two compares + selects (fmin / fmax carry NaN handling)\n"
         "  const double t = fma(x, 1.4426950408889634, 6755399441055744.0);\n"
         "  const int n = __double2loint(t);\n"
         "  const double nf = t - 6755399441055744.0;\n"
         "  double r = fma(nf, -6.93147180369123816490e-01, x);\n"
         "  r = fma(nf, -1.90821492927058770002e-10, r);\n";
  // Horner (13 FMAs) where many threads hide the chain (one thread per cell; literal coefficients measured 0.7 % faster
  // than the constant-bank form there, Estrin 4.5 % slower).  The role-warp kernel interleaves the eight exponentials of
  // a trip, which hides the chain as well: Horner from the constant bank (form 2) is 1.2 % faster there than Estrin
  // (16 operations, depth 5, its second constant of every FMA re-materialised with two moves)
  if (estrin)
    src +=
         "  const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;            // Estrin: dependency depth 5 instead of 13\n"
         "  const double q0 = r + 1.0, q1 = fma(1.6666666666666666e-01, r, 0.5), q2 = fma(8.333333333333333e-03, r, 4.1666666666666664e-02);\n"
         "  const double q3 = fma(1.984126984126984e-04, r, 1.388888888888889e-03), q4 = fma(2.7557319223985893e-06, r, 2.48015873015873e-05);\n"
         "  const double q5 = fma(2.505210838544172e-08, r, 2.755731922398589e-07), q6 = fma(1.6059043836821613e-10, r, 2.08767569878681e-09);\n"
         "  const double s0 = fma(q1, r2, q0), s1 = fma(q3, r2, q2), s2 = fma(q5, r2, q4);\n"
         "  const double t0 = fma(s1, r4, s0), t1 = fma(q6, r4, s2);\n"
         "  const double p = fma(t1, r8, t0);\n";
  else if (form == 2)
    src +=
         "  double p = c_exp[0];\n"
         "  #pragma unroll\n"
         "  for (int k = 1; k < 14; k++) p = fma(p, r, c_exp[k]);\n";
  else
    src +=
         "  double p = 1.6059043836821613e-10;\n"
         "  p = fma(p, r, 2.08767569878681e-09); p = fma(p, r, 2.505210838544172e-08); p = fma(p, r, 2.755731922398589e-07);\n"
         "  p = fma(p, r, 2.7557319223985893e-06); p = fma(p, r, 2.48015873015873e-05); p = fma(p, r, 1.984126984126984e-04);\n"
         "  p = fma(p, r, 1.388888888888889e-03); p = fma(p, r, 8.333333333333333e-03); p = fma(p, r, 4.1666666666666664e-02);\n"
         "  p = fma(p, r, 1.6666666666666666e-01); p = fma(p, r, 0.5); p = fma(p, r, 1.0); p = fma(p, r, 1.0);\n";
  src +=
         "  // 2^n goes straight into the exponent field: p is in [0.70, 1.42] and n in [-1021, 1023] after the clamp, so the\n"
         "  // biased exponent stays within [1, 2046] (no fp64 instruction, no intermediate overflow)\n"
         "  return __hiloint2double(__double2hiint(p) + (n << 20), __double2loint(p));\n"
         "}\n"
         "__device__ __forceinline__ double rcp_nb(double x) {\n"
         "  double r;\n"
         "  asm(\"rcp.approx.ftz.f64 %0, %1;\" : \"=d\"(r) : \"d\"(x));\n"
         "  r = fma(fma(-x, r, 1.0), r, r);\n"
         "  r = fma(fma(-x, r, 1.0), r, r);\n"
         "  return r;\n"
         "}\n";
}

// Newton on e(T) = sum_k Y_k R_k (h_k/R_k - T) (eq 4.3-4.4; reading A6): expects yr<k>, e, T; sets ok
// two-range data: which coefficient set every species uses at the current T (reading A7 -> SURVEY NEXT-3)
inline void emit_range_flags(Emitter &E, const MechC &M, const std::string &ind, const std::vector<char> *need = nullptr) {
  if (!M.two_range) return;
  for (int k = 0; k < M.ns; k++)
    if (!need || (*need)[k]) E.line(ind + "const bool hi" + I(k) + " = T >= " + num(M.Tmid[k]) + ";");
}

inline void emit_newton(Emitter &E, const MechC &M) {
  const int ns = M.ns;
  E.line("bool ok = false;");
  E.line("#pragma unroll 1");
  E.line("for (int it = 0; it < 50; it++) {");
  E.line("  double f = -e, cv = 0.0;");
  emit_range_flags(E, M, "  ");
  for (int k = 0; k < ns; k++) {
    // h_k/R_k - T = a5 + (a0-1) T + a1/2 T^2 + ... ;  cp_k/R_k - 1 = (a0-1) + a1 T + ...
    const std::string h = nasa_poly(M, k, 6, [](const double *c, double *o) { o[0] = c[5]; o[1] = c[0] - 1.0; o[2] = 0.5 * c[1]; o[3] = c[2] / 3.0; o[4] = 0.25 * c[3]; o[5] = 0.2 * c[4]; });
    const std::string cv = nasa_poly(M, k, 5, [](const double *c, double *o) { o[0] = c[0] - 1.0; o[1] = c[1]; o[2] = c[2]; o[3] = c[3]; o[4] = c[4]; });
    E.line("  f = fma(yr" + I(k) + ", " + h + ", f);");
    E.line("  cv = fma(yr" + I(k) + ", " + cv + ", cv);");
  }
  E.line("  const double dT = -f / cv;");
  E.line("  T += dT;");
  E.line("  if (fabs(dT) <= 1e-11 * fabs(T)) { ok = true; break; }");
  E.line("}");
  E.line("ok = ok && (T > 0.0) && isfinite(T);");
}

// Shared-memory tail of the big-mechanism kernel: A = I - dt J in place (column Ns-1 becomes the
// right-hand side), Gaussian elimination with partial pivoting, back substitution, store.
inline void emit_big_solve(Emitter &E, const MechC &M, int ndim, const Acc &accW) {
  const int ns = M.ns, n1 = ns - 1, NT = JANC_JIT_NT_BIG;
  const std::string sNT = I(NT), sNS = I(ns), sN1 = I(n1);
  std::string iw = "const double iW_[" + sN1 + "] = {";
  for (int l = 0; l < n1; l++) iw += num(M.invW[l]) + (l + 1 < n1 ? ", " : "};");
  E.line(iw);
  E.line("#define EL(r, c) S[((r) * " + sNS + " + (c)) * " + sNT + "]");
  for (int k = 0; k < n1; k++) {
    const std::string sk = I(k);
    E.line("{ const double dl = EL(" + sk + ", " + sN1 + ") * " + num(M.invW[n1]) + ", mw = -dt * " + num(M.W[k]) + ";");
    E.line("  #pragma unroll 1");
    E.line("  for (int l = 0; l < " + sN1 + "; l++) EL(" + sk + ", l) = fma(mw, fma(EL(" + sk + ", l), iW_[l], -dl), l == " + sk + " ? 1.0 : 0.0);");
    E.line("  EL(" + sk + ", " + sN1 + ") = " + (accW.set[k] ? "-mw * w" + sk : std::string("0.0")) + "; }");
  }
  E.line("#pragma unroll 1");
  E.line("for (int c = 0; c < " + sN1 + "; c++) {");
  E.line("  int piv = c; double best = fabs(EL(c, c));");
  E.line("  for (int r = c + 1; r < " + sN1 + "; r++) { const double v = fabs(EL(r, c)); if (v > best) { best = v; piv = r; } }");
  E.line("  if (!(best > 0.0)) ok = false;");
  E.line("  if (piv != c) for (int b = c; b <= " + sN1 + "; b++) { const double x_ = EL(c, b); EL(c, b) = EL(piv, b); EL(piv, b) = x_; }");
  E.line("  const double ip = 1.0 / EL(c, c);");
  E.line("  for (int r = c + 1; r < " + sN1 + "; r++) {");
  E.line("    const double f = EL(r, c) * ip;");
  E.line("    #pragma unroll 4");
  E.line("    for (int b = c + 1; b <= " + sN1 + "; b++) EL(r, b) = fma(-f, EL(c, b), EL(r, b));");
  E.line("  }");
  E.line("  EL(c, c) = ip;");
  E.line("}");
  E.line("#pragma unroll 1");
  E.line("for (int r = " + I(n1 - 1) + "; r >= 0; r--) {");
  E.line("  double sum = EL(r, " + sN1 + ");");
  E.line("  for (int b = r + 1; b < " + sN1 + "; b++) sum = fma(-EL(r, b), EL(b, " + sN1 + "), sum);");
  E.line("  EL(r, " + sN1 + ") = sum * EL(r, r);");
  E.line("}");
  E.line("#pragma unroll 1");
  E.line("for (int k = 0; k < " + sN1 + "; k++) {");
  E.line("  const double d_ = EL(k, " + sN1 + ");");
  E.line("  if (!isfinite(d_)) ok = false;");
  E.line("  if (live) Up[(" + I(ndim + 2) + " + k) * a.pc] += d_;");
  E.line("}");
  E.line("if (!ok && live) *a.flag = 1;");
  E.line("#undef EL");
}

// big == false: everything in registers (N1 <= JANC_JIT_MAX_N1).
// big == true : the (Ns-1) x Ns derivative matrix / linear system lives in shared memory as [entry][lane]
//               (32 threads per CTA, conflict-free); rates and the sparse Jacobian scatter are still
//               specialised (literal addresses), the dense elimination is a loop over shared memory.
inline std::string generate(const MechC &M, int ndim, bool big = false) {
  const int NT = big ? JANC_JIT_NT_BIG : JANC_JIT_NT;
  const int ns = M.ns, nr = M.nr, n1 = ns - 1, nvar = ndim + 2 + n1;
  Emitter E;
  std::string &src = E.s;
  src += "// generated by chemgen.h for ns=" + I(ns) + " nr=" + I(nr) + " ndim=" + I(ndim) + "\n";
  src += "struct ChemArgs { double *U; double *T; const double *scal; int *flag; int n0, n1, n2, G0, G1, G2;"
         " long long st0, st1, st2, pc; int np, patch0; double dts; };\n";
  emit_math(src);
  src += "extern \"C\" __global__ void __launch_bounds__(" + I(NT) + ") k_chem_jit(ChemArgs a) {\n";
  E.line("const long long ncell = (long long)a.n0 * a.n1 * a.n2;");
  if (big) {
    E.line("extern __shared__ double sm_[];");
    E.line("double *S = sm_ + threadIdx.x;          // entry i of this cell's matrix: S[i * " + I(NT) + "]");
    E.line("#pragma unroll 1");
    E.line("for (int i_ = 0; i_ < " + I(n1 * ns) + "; i_++) S[i_ * " + I(NT) + "] = 0.0;");
  }
  E.line("long long t = (long long)blockIdx.x * " + I(NT) + " + threadIdx.x;");
  E.line("const bool live = t < ncell;");
  E.line("if (!live) t = ncell - 1;   // idle lanes recompute the last cell and store nothing");
  // a patch holds fewer than 2^31 cells (janc_create): 32-bit divisions instead of the 64-bit software routine
  E.line("const unsigned t32 = (unsigned)t, r_ = t32 / (unsigned)a.n0; const int ci = (int)(t32 - r_ * (unsigned)a.n0);");
  E.line("const unsigned k_ = r_ / (unsigned)a.n1; const int cj = (int)(r_ - k_ * (unsigned)a.n1), ck = (int)k_;");
  E.line("const long long id = (ci + a.G0) * a.st0 + (cj + a.G1) * a.st1 + (ck + a.G2) * a.st2;");
  E.line("double *Up = a.U + (long long)(blockIdx.y + a.patch0) * " + I(nvar) + " * a.pc + id;");
  E.line("const long long pid = (long long)(blockIdx.y + a.patch0) * a.pc + id;");
  // ---- cons -> prim pieces (eq 4.2), X_k = rho Y_k / W_k
  E.line("const double rho = Up[0], irho = 1.0 / rho;");
  E.line("double ke = 0.0;");
  for (int d = 0; d < ndim; d++)
    E.line("{ const double ud = Up[" + I(1 + d) + " * a.pc] * irho; ke = fma(0.5 * ud, ud, ke); }");
  E.line("double ysum = 0.0, rsum = 0.0;");
  for (int k = 0; k < n1; k++) {
    E.line("const double ry" + I(k) + " = Up[" + I(ndim + 2 + k) + " * a.pc];");
    E.line("const double Y" + I(k) + " = ry" + I(k) + " * irho, X" + I(k) + " = ry" + I(k) + " * " + num(M.invW[k]) + ";");
    E.line("ysum += Y" + I(k) + "; rsum += ry" + I(k) + ";");
  }
  E.line("const double Y" + I(n1) + " = 1.0 - ysum, X" + I(n1) + " = (rho - rsum) * " + num(M.invW[n1]) + ";");
  E.line("const double e = Up[" + I(ndim + 1) + " * a.pc] * irho - ke;");
  for (int k = 0; k < ns; k++) E.line("const double yr" + I(k) + " = Y" + I(k) + " * " + num(M.Rk[k]) + ";");
  E.line("double T = a.T[pid];");
  emit_newton(E, M);
  E.line("if (live) a.T[pid] = T;");
  // ---- g_j = s_j/R_j - h_j/(R_j T) for species of reversible reactions (eq 4.4-4.5, 4.9)
  std::vector<char> need_g(ns, 0);
  bool any_rev = false;
  for (int i = 0; i < nr; i++)
    if (M.rev[i]) {
      any_rev = true;
      for (int k = 0; k < ns; k++) if (M.dnu[i][k] != 0.0) need_g[k] = 1;
    }
  E.line("const double lnT = log(T), iT = 1.0 / T;");
  emit_range_flags(E, M, "", &need_g);
  for (int k = 0; k < ns; k++) {
    if (!need_g[k]) continue;
    const std::string sp = nasa_poly(M, k, 5, [](const double *c, double *o) { o[0] = c[6]; o[1] = c[1]; o[2] = 0.5 * c[2]; o[3] = c[3] / 3.0; o[4] = 0.25 * c[4]; });   // + a0 ln T
    const std::string hp = nasa_poly(M, k, 6, [](const double *c, double *o) { o[0] = c[5]; o[1] = c[0]; o[2] = 0.5 * c[1]; o[3] = c[2] / 3.0; o[4] = 0.25 * c[3]; o[5] = 0.2 * c[4]; });
    const std::string a0 = nasa_poly(M, k, 1, [](const double *c, double *o) { o[0] = c[0]; });
    E.line("const double g" + I(k) + " = fma(" + a0 + ", lnT, " + sp + ") - (" + hp + ") * iT;");
  }
  if (any_rev) E.line("const double lnC0 = " + num(std::log(JANC_PATM / JANC_RU)) + " - lnT;   // ln(p0 / (Ru T))");
  E.line("const double dt = a.scal[0] * a.dts;");
  // ---- rates of progress (eq 4.7-4.9), wdot_k = sum_i dnu_ik q_i, D_k_j = sum_i dnu_ik dq_i/dX_j
  Acc accW(ns), accD(n1 * ns);
  for (int i = 0; i < nr; i++) {
    const std::string si = I(i);
    int cf[JANC_MAX_NS] = {0}, cb[JANC_MAX_NS] = {0}, dnu[JANC_MAX_NS];
    for (int e = 0; e < M.nreac[i]; e++) cf[M.reac[i][e]]++;
    for (int e = 0; e < M.nprod[i]; e++) cb[M.prod[i][e]]++;
    for (int k = 0; k < ns; k++) dnu[k] = cb[k] - cf[k];
    E.line("// reaction " + si);
    std::string lnk = num(M.lnA[i]);
    if (M.b[i] != 0.0) lnk = "fma(" + num(M.b[i]) + ", lnT, " + lnk + ")";
    if (M.Ta[i] != 0.0) lnk = "fma(" + num(-M.Ta[i]) + ", iT, " + lnk + ")";
    E.line("const double lk" + si + " = " + lnk + ";");
    E.line("const double kf" + si + " = exp_nb(lk" + si + ");");
    const bool rev = M.rev[i] != 0, tb = M.tb[i] != 0;
    if (rev) {
      std::string dg = M.dn[i] != 0 ? num((double)M.dn[i]) + " * lnC0" : std::string("0.0");
      for (int k = 0; k < ns; k++) {
        if (dnu[k] == 0) continue;
        dg = "fma(" + num((double)dnu[k]) + ", g" + I(k) + ", " + dg + ")";
      }
      E.line("const double kb" + si + " = exp_nb(lk" + si + " - " + dg + ");");
    }
    std::string rn = xprod("kf" + si, cf, ns, -1);
    if (rev) rn += " - " + xprod("kb" + si, cb, ns, -1);
    E.line("const double rn" + si + " = " + rn + ";");
    std::string cfs = "kf" + si, cbs = "kb" + si, qs = "rn" + si;
    if (tb) {
      const double *ef = M.eff[M.tbi[i]];
      std::string m = num(ef[0]) + " * X0";
      for (int k = 1; k < ns; k++) m = "fma(" + num(ef[k]) + ", X" + I(k) + ", " + m + ")";
      E.line("const double M" + si + " = " + m + ";");
      E.line("const double q" + si + " = M" + si + " * rn" + si + ", cf" + si + " = M" + si + " * kf" + si +
             (rev ? ", cb" + si + " = M" + si + " * kb" + si : std::string("")) + ";");
      cfs = "cf" + si; cbs = "cb" + si; qs = "q" + si;
    }
    for (int k = 0; k < ns; k++) accum(E, accW, k, "w" + I(k), dnu[k], qs);
    // dq_i/dX_j
    for (int j = 0; j < ns; j++) {
      std::string dq;
      if (cf[j] > 0) dq = (cf[j] > 1 ? num((double)cf[j]) + " * " : std::string("")) + xprod(cfs, cf, ns, j);
      if (rev && cb[j] > 0) dq += (dq.empty() ? "-" : " - ") + (cb[j] > 1 ? num((double)cb[j]) + " * " : std::string("")) + xprod(cbs, cb, ns, j);
      if (tb) {
        const double a = M.eff[M.tbi[i]][j];
        if (a != 0.0) dq = dq.empty() ? num(a) + " * rn" + si : "fma(" + num(a) + ", rn" + si + ", " + dq + ")";
      }
      if (dq.empty()) continue;
      const std::string dn = "dq" + si + "_" + I(j);
      E.line("const double " + dn + " = " + dq + ";");
      for (int k = 0; k < n1; k++) {
        if (!big) { accum(E, accD, k * ns + j, "D" + I(k) + "_" + I(j), dnu[k], dn); continue; }
        if (dnu[k] == 0) continue;
        const std::string el = "S[" + I((k * ns + j) * NT) + "]";
        if (dnu[k] == 1) E.line(el + " += " + dn + ";");
        else if (dnu[k] == -1) E.line(el + " -= " + dn + ";");
        else E.line(el + " = fma(" + num((double)dnu[k]) + ", " + dn + ", " + el + ");");
      }
    }
  }
  if (big) {
    emit_big_solve(E, M, ndim, accW);
    src += "}\n";
    return src;
  }
  // ---- A = I - dt J,  J_kl = W_k (D_kl / W_l - D_kNs / W_Ns);  rhs = dt W_k wdot_k   (eq 4.12-4.13, A11)
  for (int k = 0; k < n1; k++) {
    const std::string sk = I(k);
    const bool hasN = accD.set[k * ns + n1] != 0;
    if (hasN) E.line("const double dl" + sk + " = D" + sk + "_" + I(n1) + " * " + num(M.invW[n1]) + ";");
    E.line("const double mw" + sk + " = -dt * " + num(M.W[k]) + ";");
    for (int l = 0; l < n1; l++) {
      const std::string one = k == l ? "1.0" : "0.0";
      const bool has = accD.set[k * ns + l] != 0;
      std::string inner;
      if (has && hasN) inner = "fma(D" + sk + "_" + I(l) + ", " + num(M.invW[l]) + ", -dl" + sk + ")";
      else if (has) inner = "D" + sk + "_" + I(l) + " * " + num(M.invW[l]);
      else if (hasN) inner = "-dl" + sk;
      if (inner.empty()) E.line("double A" + sk + "_" + I(l) + " = " + one + ";");
      else E.line("double A" + sk + "_" + I(l) + " = fma(mw" + sk + ", " + inner + ", " + one + ");");
    }
    if (accW.set[k]) E.line("double b" + sk + " = -mw" + sk + " * w" + sk + ";");
    else E.line("double b" + sk + " = 0.0;");
  }
  // ---- Gaussian elimination with partial pivoting (row swaps predicated per lane, skipped when no
  //      lane of the warp needs one), back substitution
  auto A = [](int r, int c) { return "A" + I(r) + "_" + I(c); };
  for (int c = 0; c < n1; c++) {
    E.line("{ // column " + I(c));
    if (c + 1 < n1) {
      E.line("  int piv = " + I(c) + "; double best = fabs(" + A(c, c) + "), v;");
      for (int r = c + 1; r < n1; r++)
        E.line("  v = fabs(" + A(r, c) + "); if (v > best) { best = v; piv = " + I(r) + "; }");
      E.line("  if (!(best > 0.0)) ok = false;");
      E.line("  if (__any_sync(0xffffffffu, piv != " + I(c) + ")) {");
      E.line("    double x_, y_;");
      for (int r = c + 1; r < n1; r++) {
        E.line("    { const bool sw = piv == " + I(r) + ";");
        for (int b = c; b < n1; b++)
          E.line("      x_ = " + A(c, b) + "; y_ = " + A(r, b) + "; " + A(c, b) + " = sw ? y_ : x_; " + A(r, b) + " = sw ? x_ : y_;");
        E.line("      x_ = b" + I(c) + "; y_ = b" + I(r) + "; b" + I(c) + " = sw ? y_ : x_; b" + I(r) + " = sw ? x_ : y_; }");
      }
      E.line("  }");
    } else {
      E.line("  if (!(fabs(" + A(c, c) + ") > 0.0)) ok = false;");
    }
    E.line("  const double ip = rcp_nb(" + A(c, c) + ");");
    for (int r = c + 1; r < n1; r++) {
      E.line("  { const double f = " + A(r, c) + " * ip;");
      for (int b = c + 1; b < n1; b++) E.line("    " + A(r, b) + " = fma(-f, " + A(c, b) + ", " + A(r, b) + ");");
      E.line("    b" + I(r) + " = fma(-f, b" + I(c) + ", b" + I(r) + "); }");
    }
    E.line("  " + A(c, c) + " = ip;");
    E.line("}");
  }
  for (int r = n1 - 1; r >= 0; r--) {
    std::string sum = "b" + I(r);
    for (int b = r + 1; b < n1; b++) sum = "fma(-" + A(r, b) + ", b" + I(b) + ", " + sum + ")";
    E.line("b" + I(r) + " = (" + sum + ") * " + A(r, r) + ";");
  }
  for (int k = 0; k < n1; k++) {
    E.line("if (!isfinite(b" + I(k) + ")) ok = false;");
    E.line("if (live) Up[" + I(ndim + 2 + k) + " * a.pc] = ry" + I(k) + " + b" + I(k) + ";");
  }
  E.line("if (!ok && live) *a.flag = 1;");
  src += "}\n";
  return src;
}

// Explicit source variant: S_k = W_k omega_k(T, X) of the stage state is part of the
// right-hand side of every RK stage.  The flux kernel has already written Uout = U0 + coef ((Uk - U0) + dt L(Uk)); this
// kernel adds coef dt S(Uk) on the species rows, with the temperature cons->prim recovered for Uk.  One thread per cell,
// rates fully specialised (literal indices, immediate coefficients); emits helpers only if `with_math`.
inline std::string generate_source(const MechC &M, int ndim, bool with_math) {
  const int ns = M.ns, nr = M.nr, n1 = ns - 1, nvar = ndim + 2 + n1;
  Emitter E;
  std::string &src = E.s;
  src += "struct SrcArgs { const double *Uk; double *Uout; const double *T; const double *scal; int n0, n1, n2, G0, G1, G2;"
         " long long st0, st1, st2, pc; double coef; int patch0; };\n";
  if (with_math) emit_math(src);
  src += "extern \"C\" __global__ void __launch_bounds__(128) k_src_jit(SrcArgs a) {\n";
  E.line("const long long ncell = (long long)a.n0 * a.n1 * a.n2;");
  E.line("const long long t = (long long)blockIdx.x * 128 + threadIdx.x;");
  E.line("if (t >= ncell) return;");
  // a patch holds fewer than 2^31 cells (janc_create): 32-bit divisions instead of the 64-bit software routine
  E.line("const unsigned t32 = (unsigned)t, r_ = t32 / (unsigned)a.n0; const int ci = (int)(t32 - r_ * (unsigned)a.n0);");
  E.line("const unsigned k_ = r_ / (unsigned)a.n1; const int cj = (int)(r_ - k_ * (unsigned)a.n1), ck = (int)k_;");
  E.line("const long long id = (ci + a.G0) * a.st0 + (cj + a.G1) * a.st1 + (ck + a.G2) * a.st2;");
  E.line("const double *Up = a.Uk + (long long)(blockIdx.y + a.patch0) * " + I(nvar) + " * a.pc + id;");
  E.line("double *Uo = a.Uout + (long long)(blockIdx.y + a.patch0) * " + I(nvar) + " * a.pc + id;");
  E.line("const double T = a.T[(long long)(blockIdx.y + a.patch0) * a.pc + id];");
  E.line("const double rho = Up[0];");
  E.line("double rsum = 0.0;");
  for (int k = 0; k < n1; k++) {
    E.line("const double ry" + I(k) + " = Up[" + I(ndim + 2 + k) + " * a.pc], X" + I(k) + " = ry" + I(k) + " * " + num(M.invW[k]) + ";");
    E.line("rsum += ry" + I(k) + ";");
  }
  E.line("const double X" + I(n1) + " = (rho - rsum) * " + num(M.invW[n1]) + ";");
  std::vector<char> need_g(ns, 0);
  bool any_rev = false;
  for (int i = 0; i < nr; i++)
    if (M.rev[i]) {
      any_rev = true;
      for (int k = 0; k < ns; k++) if (M.dnu[i][k] != 0.0) need_g[k] = 1;
    }
  E.line("const double lnT = log(T), iT = 1.0 / T;");
  emit_range_flags(E, M, "", &need_g);
  for (int k = 0; k < ns; k++) {
    if (!need_g[k]) continue;
    const std::string sp = nasa_poly(M, k, 5, [](const double *c, double *o) { o[0] = c[6]; o[1] = c[1]; o[2] = 0.5 * c[2]; o[3] = c[3] / 3.0; o[4] = 0.25 * c[4]; });   // + a0 ln T
    const std::string hp = nasa_poly(M, k, 6, [](const double *c, double *o) { o[0] = c[5]; o[1] = c[0]; o[2] = 0.5 * c[1]; o[3] = c[2] / 3.0; o[4] = 0.25 * c[3]; o[5] = 0.2 * c[4]; });
    const std::string a0 = nasa_poly(M, k, 1, [](const double *c, double *o) { o[0] = c[0]; });
    E.line("const double g" + I(k) + " = fma(" + a0 + ", lnT, " + sp + ") - (" + hp + ") * iT;");
  }
  if (any_rev) E.line("const double lnC0 = " + num(std::log(JANC_PATM / JANC_RU)) + " - lnT;   // ln(p0 / (Ru T))");
  Acc accW(ns);
  for (int i = 0; i < nr; i++) {
    const std::string si = I(i);
    int cf[JANC_MAX_NS] = {0}, cb[JANC_MAX_NS] = {0}, dnu[JANC_MAX_NS];
    for (int e = 0; e < M.nreac[i]; e++) cf[M.reac[i][e]]++;
    for (int e = 0; e < M.nprod[i]; e++) cb[M.prod[i][e]]++;
    for (int k = 0; k < ns; k++) dnu[k] = cb[k] - cf[k];
    std::string lnk = num(M.lnA[i]);
    if (M.b[i] != 0.0) lnk = "fma(" + num(M.b[i]) + ", lnT, " + lnk + ")";
    if (M.Ta[i] != 0.0) lnk = "fma(" + num(-M.Ta[i]) + ", iT, " + lnk + ")";
    E.line("const double lk" + si + " = " + lnk + ";");
    std::string rn = xprod("exp_nb(lk" + si + ")", cf, ns, -1);
    if (M.rev[i]) {
      std::string dg = M.dn[i] != 0 ? num((double)M.dn[i]) + " * lnC0" : std::string("0.0");
      for (int k = 0; k < ns; k++) {
        if (dnu[k] == 0) continue;
        dg = "fma(" + num((double)dnu[k]) + ", g" + I(k) + ", " + dg + ")";
      }
      rn += " - " + xprod("exp_nb(lk" + si + " - " + dg + ")", cb, ns, -1);
    }
    std::string q = "(" + rn + ")";
    if (M.tb[i]) {
      const double *ef = M.eff[M.tbi[i]];
      std::string m = num(ef[0]) + " * X0";
      for (int k = 1; k < ns; k++) m = "fma(" + num(ef[k]) + ", X" + I(k) + ", " + m + ")";
      q = "(" + m + ") * " + q;
    }
    E.line("const double q" + si + " = " + q + ";");
    for (int k = 0; k < n1; k++) accum(E, accW, k, "w" + I(k), dnu[k], "q" + si);
  }
  E.line("const double cdt = a.coef * a.scal[0];");
  for (int k = 0; k < n1; k++)
    if (accW.set[k]) E.line("Uo[" + I(ndim + 2 + k) + " * a.pc] = fma(cdt * " + num(M.W[k]) + ", w" + I(k) + ", Uo[" + I(ndim + 2 + k) + " * a.pc]);");
  src += "}\n";
  return src;
}

// Specialised fused cons->prim + thermo kernel with the alpha / CFL max-reduction (same contract as
// k_prim of prim.cuh).  256 threads per CTA.
inline std::string generate_prim(const MechC &M, int ndim) {
  const int ns = M.ns, n1 = ns - 1, nvar = ndim + 2 + n1;
  Emitter E;
  std::string &src = E.s;
  src += "struct PrimArgs { const double *U; double *T; double *p; double *vel; double *dbgc; unsigned long long *slots;"
         " const int *level; int *flag; int n0, n1, n2, G0, G1, G2; long long st0, st1, st2, pc; int np, reduce, slot_base, patch0; };\n";
  src += "extern \"C\" __global__ void __launch_bounds__(256) k_prim_jit(PrimArgs a) {\n";
  E.line("const long long ncell = (long long)a.n0 * a.n1 * a.n2;");
  E.line("const long long t = (long long)blockIdx.x * 256 + threadIdx.x;");
  for (int d = 0; d < ndim; d++) E.line("double s" + I(d) + " = 0.0;");
  E.line("if (t < ncell) {");
  // a patch holds fewer than 2^31 cells (janc_create): 32-bit divisions instead of the 64-bit software routine
  E.line("const unsigned t32 = (unsigned)t, r_ = t32 / (unsigned)a.n0; const int ci = (int)(t32 - r_ * (unsigned)a.n0);");
  E.line("const unsigned k_ = r_ / (unsigned)a.n1; const int cj = (int)(r_ - k_ * (unsigned)a.n1), ck = (int)k_;");
  E.line("const long long id = (ci + a.G0) * a.st0 + (cj + a.G1) * a.st1 + (ck + a.G2) * a.st2;");
  E.line("const double *Up = a.U + (long long)(blockIdx.y + a.patch0) * " + I(nvar) + " * a.pc + id;");
  E.line("const long long pid = (long long)(blockIdx.y + a.patch0) * a.pc + id;");
  E.line("const double rho = Up[0], irho = 1.0 / rho;");
  E.line("double ke = 0.0;");
  for (int d = 0; d < ndim; d++)
    E.line("const double u" + I(d) + " = Up[" + I(1 + d) + " * a.pc] * irho; ke = fma(0.5 * u" + I(d) + ", u" + I(d) + ", ke);");
  E.line("double ysum = 0.0;");
  for (int k = 0; k < n1; k++) {
    E.line("const double Y" + I(k) + " = Up[" + I(ndim + 2 + k) + " * a.pc] * irho;");
    E.line("ysum += Y" + I(k) + ";");
  }
  E.line("const double Y" + I(n1) + " = 1.0 - ysum;");
  E.line("const double e = Up[" + I(ndim + 1) + " * a.pc] * irho - ke;");
  for (int k = 0; k < ns; k++) E.line("const double yr" + I(k) + " = Y" + I(k) + " * " + num(M.Rk[k]) + ";");
  E.line("double T = a.T[pid];");
  emit_newton(E, M);
  E.line("double R = 0.0, cp = 0.0;");
  emit_range_flags(E, M, "");
  for (int k = 0; k < ns; k++) {
    const std::string cc = nasa_poly(M, k, 5, [](const double *c, double *o) { o[0] = c[0]; o[1] = c[1]; o[2] = c[2]; o[3] = c[3]; o[4] = c[4]; });
    E.line("R += yr" + I(k) + "; cp = fma(yr" + I(k) + ", " + cc + ", cp);");
  }
  E.line("const double p = rho * R * T;");
  E.line("const double c = sqrt(cp / (cp - R) * R * T);");
  E.line("a.T[pid] = T; a.p[pid] = p;");
  for (int d = 0; d < ndim; d++) {
    E.line("a.vel[" + I(d) + "LL * a.np * a.pc + pid] = u" + I(d) + ";");
    E.line("s" + I(d) + " = fabs(u" + I(d) + ") + c;");
  }
  E.line("if (a.dbgc) a.dbgc[pid] = c;");
  E.line("if (!(ok && isfinite(c))) *a.flag = 1;");
  E.line("}");
  E.line("if (a.reduce) {");
  E.line("  __shared__ double sh[" + I(ndim) + "][8];");
  E.line("  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;");
  for (int d = 0; d < ndim; d++) {
    E.line("  { double v = s" + I(d) + "; if (!(v >= 0.0)) v = 0.0;");
    E.line("    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));");
    E.line("    if (lane == 0) sh[" + I(d) + "][w] = v; }");
  }
  E.line("  __syncthreads();");
  E.line("  if (threadIdx.x < " + I(ndim) + ") {");
  E.line("    double v = 0.0;");
  E.line("    for (int q = 0; q < 8; q++) v = fmax(v, sh[threadIdx.x][q]);");
  E.line("    atomicMax(a.slots + a.slot_base + a.level[blockIdx.y + a.patch0] * 3 + threadIdx.x, (unsigned long long)__double_as_longlong(v));");
  E.line("  }");
  E.line("}");
  src += "}\n";
  return src;
}

}  // namespace chemgen
