// chemgen_roles.h -- run-time specialised point-implicit chemistry for LARGE mechanisms ("jit-roles").
// PAPER.md:260-277 (eq 4.6-4.9), :297-304 (eq 4.12-4.13), :333 (solve_implicit_rate), :340; readings A9-A12.
//
// Why another kernel: with one thread per cell (chemgen.h) the (Ns-1) x Ns system of a 20-species mechanism
// (3 KB per cell) has to live in shared memory, which leaves room for ~2 warps per SM and the kernel crawls
// on latency.  Here a persistent CTA of 8 warps (one per SM) advances 32 cells per turn: lane = cell,
// warp = ROLE.  Role w owns
//   * species  k = w, w+8, w+16      (X_k, the final rho Y_k update; T* = T(U*) comes from a cons->prim launch in front of
//                                     this kernel, or -- option roles_newton = kernel -- from Newton partial sums per role),
//   * reactions dealt round-robin    (Arrhenius / equilibrium exponentials, rates of progress: shared table-driven code;
//                                     one packed record per (role, slot), copied once per CTA into shared memory and read
//                                     with warp-uniform addresses: broadcast loads, no divergence; four reactions per
//                                     trip, emitted as loads / arithmetic / stores so that their exponential chains overlap),
//   * columns  j = w, w+8, w+16 of the system [I - dt J | rhs], assembled in REGISTERS (57 doubles for Ns = 20).
// The Jacobian columns are assembled by role-specific literal code (switch on the warp index: every
// species / reaction index a literal, every update one register FMA, structural zeros never touched),
// reading the 2 Nr rate coefficients the roles exchanged through shared memory ([row][cell], conflict-free); the
// third-body efficiency terms, which touch every column, are code shared by all roles.
// Linear solve (default, roles_lu = rows): the columns are transposed through shared memory and factorised with one
// ROW per lane inside a warp -- 8 lanes per cell, no inter-warp synchronisation, pivot rows broadcast through a per-cell
// U store in shared memory, rolled and software-pipelined column loop (see the emitter below).  Kept as roles_lu =
// columns: column-distributed Gauss-Jordan across the role warps with producer / consumer named barriers.
// Neither fast path swaps rows: the owner checks that the diagonal entry IS the partial-pivoting choice
// (first row of maximal |a_rc|, r >= c); if any of the 32 cells needs a swap the CTA solves the system in
// shared memory with a generic, loop-based pivoted elimination (same pivot rule as the oracle).
#pragma once
#include <algorithm>

#include "chemgen.h"

#define JANC_ROLES_MAXCOLS 24      // columns of [I - dt J | rhs] incl. the temporary N column => Ns <= 24

namespace chemgen {

// roles (warps) per CTA: 8 roles x 3 column slots (255 registers; the default) or 16 roles x 2 slots (128 registers).
// Measured on cfg 4: 59 ms with 8 roles, 81 ms with 16 -- the per-column publish -> consume chain, not the number of
// resident warps, bounds the elimination, and it is longer with 16 participants.
// The count is a per-thread setting of the generator, set by janc.cu from the context's options (janc_set_option "roles")
// before any function of this header is called.
inline int &roles_nr_ref() { static thread_local int v = 8; return v; }
inline int roles_nr() { return roles_nr_ref(); }
// elimination variant (janc_set_option "roles_lu"): true = the system is transposed through shared memory and
// factorised with one ROW per lane inside a warp (no inter-warp synchronisation), false = the column-distributed
// Gauss-Jordan across the role warps
inline bool &roles_lu_rows_ref() { static thread_local bool v = true; return v; }
// where T* = T(U*) comes from (janc_set_option "roles_newton"): false = the cons->prim kernel is run on U* just before this
// kernel and T* is read from the T array (default: in this kernel the Newton iteration is a chain of barriers and
// dependent operations on 8 warps per SM, 2.1 k cycles per turn; the bandwidth-bound cons->prim kernel does it for the
// whole grid in 0.6 ms at full occupancy), true = the Newton iteration runs inside this kernel
inline bool &roles_newton_ref() { static thread_local bool v = false; return v; }

struct RolesLayout {
  int oX, oP, oN, oRN, oDL, oRHS, oF, oPIV, oIP, oXS, oNX, oR, oPB, rows;   // offsets in rows of 32 doubles
  int rstr, pbs;                                                   // row-LU: row stride of the transposed system, pivot-row buffer stride per cell (doubles)
  size_t ntd, nti;                                                 // table sizes (doubles, ints) behind the rows
  size_t smem() const { return (size_t)rows * 32 * sizeof(double) + ntd * sizeof(double) + nti * sizeof(int); }
};

// sizes that depend on the mechanism only: polynomial degrees, reaction orders, table lengths
struct RolesDims { int degh, degc, nkb, maxof, maxob, nslot; };
// Reactions are dealt to the roles round-robin, third-body reactions first; a role's list is its third-body reactions
// followed by the others padded to a multiple of four with the dummy reaction `nr` (k_f = 1, no species, results
// stored to rows of their own), so that the rate loop only has a four-reactions-per-trip body.
inline int roles_slots(const MechC &M) {
  const int NR = roles_nr();
  int ntb = 0;
  for (int i = 0; i < M.nr; i++) ntb += M.tb[i] ? 1 : 0;
  int best = 1;
  for (int w = 0; w < NR; w++) {
    int tb = 0, other = 0;
    for (int q = w; q < M.nr; q += NR) (q < ntb ? tb : other)++;
    best = std::max(best, tb + (other + 3) / 4 * 4);
  }
  return best;
}
inline RolesDims roles_dims(const MechC &M) {
  RolesDims D{1, 0, 3, 1, 1, roles_slots(M)};
  for (int k = 0; k < M.ns; k++)
    for (int q = 1; q <= 4; q++)
      if (M.nasa[k][q] != 0.0) { D.degh = std::max(D.degh, q + 1); D.degc = std::max(D.degc, q); }
  D.nkb = 3 + D.degc;
  for (int i = 0; i < M.nr; i++) {
    D.maxof = std::max(D.maxof, (int)M.nreac[i]);
    if (M.rev[i]) D.maxob = std::max(D.maxob, (int)M.nprod[i]);
  }
  return D;
}
// The rate loop reads one packed record per (role, slot) instead of tables indexed by the reaction number: the addresses
// depend on the loop counter only (no load -> index -> load chain) and the record comes in 16-byte loads.
//   doubles (RC, even): ln A, b, -Ta, the NKB reverse-rate coefficients, 1.0 / 0.0 = reversible
//   ints    (RX, multiple of 4): reaction index (nr = dummy, -1 = end of list), third-body row + 1, reactants, products
inline int roles_rc(const MechC &M) { return (3 + roles_dims(M).nkb + 1 + 1) / 2 * 2; }
inline int roles_rx(const MechC &M) { const RolesDims D = roles_dims(M); return (2 + D.maxof + D.maxob + 3) / 4 * 4; }
inline size_t roles_table_doubles(const MechC &M) {
  const RolesDims D = roles_dims(M);
  const size_t n = (size_t)roles_nr() * D.nslot * roles_rc(M) + (size_t)2 * M.ns + (size_t)M.ns * (D.degh + 1) + (size_t)M.ns * (D.degc + 1) + (size_t)M.ntb * M.ns;
  return (n + 1) / 2 * 2;        // the int table behind it stays 16-byte aligned
}
inline size_t roles_table_ints(const MechC &M) {
  const RolesDims D = roles_dims(M);
  return (size_t)roles_nr() * D.nslot * roles_rx(M) + (size_t)roles_nr() * 2;      // records + per-role trip counts
}

inline bool roles_applicable(const MechC &M) {
  if (M.two_range) return false;     // the reverse-rate polynomial collected per reaction on the host assumes one coefficient set
  return M.ns >= 3 && M.ns <= JANC_ROLES_MAXCOLS && M.nr >= 1;
}

inline RolesLayout roles_layout(const MechC &M, int ndim) {
  const int ns = M.ns, n1 = ns - 1, nr = M.nr;
  RolesLayout L;
  int o = 0;
  L.oX = o; o += ns + 1;                     // X_k, plus a dummy species with X = 1
  L.oP = o; o += 2 * roles_nr();             // partial sums of rho Y_k and Y_k per role
  L.oN = o; o += 2 * roles_nr();             // Newton partial sums per role
  L.oRN = o; o += M.ntb > 0 ? M.ntb : 1;     // net rate without the third-body factor (third-body reactions)
  L.oDL = o; o += n1;                        // D_kN / W_N
  L.oRHS = o; o += n1;                       // dt W_k wdot_k
  L.oPIV = o; o += n1;                       // "this cell needs a row swap" (int, first half of each row), per column
  L.oIP = o; o += n1;                        // reciprocal pivots
  L.oXS = o; o += n1;                        // solution
  L.oNX = o; o += ndim + 2 + n1 + 1;         // U (nvar rows) and T of the NEXT turn's cells, prefetched with cp.async
  // one region, three lives: M k_f, M k_b, q per reaction (until the assembly barrier); the multipliers of every
  // column (elimination: nothing is reused, so the roles may run several columns apart); the whole system (slow path)
  // row-LU: the system transposed to [row][column][cell] with the row stride padded by the cells per warp, so that the
  // lanes of a warp (lane = row group x cells per warp + cell) read 32 consecutive doubles
  L.rstr = (n1 + 1) * 32 + 32 / roles_nr();
  { int usz = 0; for (int c = 0; c < n1; c++) usz += (n1 + 1 - c + 1) / 2 * 2;   // triangular U store per cell, even row lengths,
    L.pbs = usz + (n1 + 2) / 2 * 2 + 4; }                                          // + the overrun of fixed-length row writes

  L.oR = o; o += std::max(std::max(3 * (nr + 1), n1 * (n1 + 1)), roles_lu_rows_ref() ? (n1 * L.rstr + 31) / 32 : 0);
  L.oF = L.oR;
  L.oPB = o; if (roles_lu_rows_ref()) o += L.pbs;                        // U store: pbs doubles per cell x 32 cells
  L.rows = o;
  L.ntd = roles_table_doubles(M);
  L.nti = roles_table_ints(M);
  return L;
}

inline std::string generate_roles(const MechC &M, int ndim) {
  const int ns = M.ns, nr = M.nr, n1 = ns - 1, nvar = ndim + 2 + n1, NR = roles_nr();
  const int NSL = (ns + NR - 1) / NR;                  // column slots per role (columns 0..n1)
  const int wN = n1 % NR, sN = n1 / NR;                // role / slot of column N (later the right-hand side)
  const RolesLayout L = roles_layout(M, ndim);
  Emitter E;
  std::string &src = E.s;
  auto row = [](int r) { return "SM(" + I(r) + ")"; };
  auto A = [](int s, int k) { return "A" + I(s) + "_" + I(k); };

  // ---- per-reaction stoichiometry
  std::vector<std::vector<int>> cf(nr, std::vector<int>(ns, 0)), cb(nr, std::vector<int>(ns, 0)), dnu(nr, std::vector<int>(ns, 0));
  const RolesDims DM = roles_dims(M);
  const int maxof = DM.maxof, maxob = DM.maxob;
  bool any_rev = false, all_rev = true;
  for (int i = 0; i < nr; i++) {
    if (!M.rev[i]) all_rev = false;
    for (int e = 0; e < M.nreac[i]; e++) cf[i][M.reac[i][e]]++;
    for (int e = 0; e < M.nprod[i]; e++) cb[i][M.prod[i][e]]++;
    for (int k = 0; k < ns; k++) dnu[i][k] = cb[i][k] - cf[i][k];
    if (M.rev[i]) any_rev = true;
  }
  // ---- Newton polynomials (h_k/R_k - T, c_p,k/R_k - 1) truncated at the highest degree any species uses
  const int degh = DM.degh, degc = DM.degc;
  // ---- reverse rate: ln k_b = ln k_f - dn ln(p_atm / (R_u T)) - sum_k dnu_k g_k(T) collected per reaction as
  //      d0 + d1 ln T + d2 / T + T (d3 + T (d4 + T (d5 + T d6)))   (eq 4.8-4.9; g_k = s_k/R - h_k/(R T))
  const int NKB = DM.nkb;
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
  const int NSLOT = DM.nslot;
  std::vector<int> ri((size_t)NR * NSLOT, -1);
  const int nrs = nr + 1;                              // row stride of the k_f / k_b / q rows: the dummy reaction has rows too
  for (int w = 0; w < NR; w++) {
    int n = 0, other = 0;
    for (int q = w; q < nr; q += NR) { ri[(size_t)w * NSLOT + n++] = order[q]; if (!M.tb[order[q]]) other++; }
    for (; other % 4; other++) ri[(size_t)w * NSLOT + n++] = nr;
  }

  // =========================================================================== tables
  src += "// generated by chemgen_roles.h for ns=" + I(ns) + " nr=" + I(nr) + " ndim=" + I(ndim) + "\n";
  src += "struct ChemArgs { double *U; double *T; const double *scal; int *flag; int n0, n1, n2, G0, G1, G2;"
         " long long st0, st1, st2, pc; int np, patch0; double dts; };\n";
  // Tables: emitted as two __constant__ arrays, copied once per (persistent) CTA into shared memory, where the
  // warp-uniform, run-time indexed reads of the rate loop are plain broadcast loads.
  std::vector<std::string> td, ti;
  auto addd = [&](const std::string &name, int &off) { off = (int)td.size(); (void)name; };
  int oiW, oRk, ohc, occ, oeff;
  const int RC = roles_rc(M), RX = roles_rx(M);
  // packed records first (16-byte aligned: the tables start on a 256-byte boundary)
  for (int w = 0; w < NR; w++)
    for (int q = 0; q < NSLOT; q++) {
      const int i = ri[(size_t)w * NSLOT + q];
      const bool real = i >= 0 && i < nr;
      std::vector<std::string> rec;
      rec.push_back(num(real ? M.lnA[i] : 0.0)); rec.push_back(num(real ? M.b[i] : 0.0)); rec.push_back(num(real ? -M.Ta[i] : 0.0));
      for (int e = 0; e < NKB; e++) rec.push_back(num(real ? kbc[(size_t)i * 7 + e] : 0.0));
      rec.push_back(num(real && M.rev[i] ? 1.0 : 0.0));
      while ((int)rec.size() < RC) rec.push_back(num(0.0));
      for (auto &v : rec) td.push_back(v);
      std::vector<int> rx;
      rx.push_back(i); rx.push_back(real && M.tb[i] ? M.tbi[i] + 1 : 0);
      for (int e = 0; e < maxof; e++) rx.push_back(real && e < M.nreac[i] ? M.reac[i][e] : ns);
      for (int e = 0; e < maxob; e++) rx.push_back(real && e < M.nprod[i] ? M.prod[i][e] : ns);
      while ((int)rx.size() < RX) rx.push_back(0);
      for (int v : rx) ti.push_back(I(v));
    }
  addd("iW", oiW); for (int k = 0; k < ns; k++) td.push_back(num(M.invW[k]));
  addd("Rk", oRk); for (int k = 0; k < ns; k++) td.push_back(num(M.Rk[k]));
  addd("hc", ohc);
  for (int k = 0; k < ns; k++) {
    const double *c = M.nasa[k];
    const double hc[6] = {c[5], c[0] - 1.0, 0.5 * c[1], c[2] / 3.0, 0.25 * c[3], 0.2 * c[4]};
    for (int q = 0; q <= degh; q++) td.push_back(num(hc[q]));
  }
  addd("cc", occ);
  for (int k = 0; k < ns; k++) {
    const double *c = M.nasa[k];
    const double cc[5] = {c[0] - 1.0, c[1], c[2], c[3], c[4]};
    for (int q = 0; q <= degc; q++) td.push_back(num(cc[q]));
  }
  addd("eff", oeff); for (int q = 0; q < M.ntb; q++) for (int k = 0; k < ns; k++) td.push_back(num(M.eff[q][k]));
  if (td.size() % 2) td.push_back(num(0.0));
  // per role: where its third-body reactions end and where its (padded) list ends -- the loops run on these counts
  // instead of testing a table entry they have just loaded
  const int ocnt = (int)ti.size();
  for (int w = 0; w < NR; w++) {
    int ntb_w = 0, nend = 0;
    for (int q = 0; q < NSLOT; q++) {
      const int i = ri[(size_t)w * NSLOT + q];
      if (i < 0) break;
      nend = q + 1;
      if (i < nr && M.tb[i]) ntb_w = q + 1;
    }
    ti.push_back(I(ntb_w)); ti.push_back(I(nend));
  }
  const int NTD = (int)td.size(), NTI = (int)ti.size();
  if ((size_t)NTD != roles_table_doubles(M) || (size_t)NTI != roles_table_ints(M)) return std::string("#error roles table size\n");
  src += "__constant__ double g_td[" + I(NTD) + "] = {";
  for (int q = 0; q < NTD; q++) src += (q ? ", " : "") + td[q];
  src += "};\n__constant__ int g_ti[" + I(NTI) + "] = {";
  for (int q = 0; q < NTI; q++) src += (q ? ", " : "") + ti[q];
  src += "};\n";
  emit_math(src, 2);
  // =========================================================================== kernel
  src += "#define SM(r) sm_[(r) * 32 + lane]\n";
  src += "#define BAR() asm volatile(\"bar.sync 0;\" ::: \"memory\")\n";
  src += "#define PST2(p, a, x, y) asm volatile(\"{ .reg .pred q; setp.ne.s32 q, %0, 0; @q st.shared.v2.f64 [%1], {%2, %3}; }\" :: \"r\"(p), \"r\"(a), \"d\"(x), \"d\"(y) : \"memory\")\n";
  src += "#define PST1(p, a, x) asm volatile(\"{ .reg .pred q; setp.ne.s32 q, %0, 0; @q st.shared.f64 [%1], %2; }\" :: \"r\"(p), \"r\"(a), \"d\"(x) : \"memory\")\n";
  src += "#define AWAIT(id) asm volatile(\"barrier.sync %0, " + I(NR * 32) + ";\" :: \"r\"(id) : \"memory\")\n";
  src += "#define PUBLISH(id) do { asm volatile(\"barrier.arrive %0, " + I(NR * 32) + ";\" :: \"r\"(id) : \"memory\"); } while (0)\n";
  // the next turn's inputs: (nvar + 1) x 32 doubles, one 8-byte cp.async each, spread over the CTA
  // (32-bit index arithmetic, once per thread: a patch holds fewer than 2^31 cells; the 64-bit divisions this replaces
  //  were ~1500 instructions per thread and turn)
  src += "__device__ __forceinline__ void prefetch_turn(const ChemArgs &a, double *sm_, int prel, unsigned lt, unsigned ncell) {\n"
         "  const int l = threadIdx.x & 31;\n"
         "  unsigned t = lt * 32u + l;\n"
         "  if (t >= ncell) t = ncell - 1u;\n"
         "  const unsigned ci = t % (unsigned)a.n0, r_ = t / (unsigned)a.n0;\n"
         "  const unsigned cj = r_ % (unsigned)a.n1, ck = r_ / (unsigned)a.n1;\n"
         "  const long long id = (ci + a.G0) * a.st0 + (cj + a.G1) * a.st1 + (ck + a.G2) * a.st2;\n"
         "  const long long pb = prel + a.patch0;      // prel: patch relative to a.patch0, lt: turn within the patch\n"
         "  for (int v = threadIdx.x >> 5; v < " + I(nvar + 1) + "; v += " + I(NR) + ") {\n"
         "    const double *src = v < " + I(nvar) + " ? a.U + (pb * " + I(nvar) + " + v) * a.pc + id : a.T + pb * a.pc + id;\n"
         "    const unsigned dst = (unsigned)__cvta_generic_to_shared(sm_ + (" + I(L.oNX) + " + v) * 32 + l);\n"
         "    asm volatile(\"cp.async.ca.shared.global [%0], [%1], 8;\" :: \"r\"(dst), \"l\"(src) : \"memory\");\n"
         "  }\n"
         "  asm volatile(\"cp.async.commit_group;\" ::: \"memory\");\n"
         "}\n";
  src += "extern \"C\" __global__ void __launch_bounds__(" + I(NR * 32) + ", 1) k_chem_jit(ChemArgs a) {\n";
  E.line("extern __shared__ double sm_[];");
  E.line("const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;");
  E.line("double *s_td = sm_ + " + I(L.rows * 32) + ";");
  E.line("int *s_ti = (int *)(s_td + " + I(NTD) + ");");
  E.line("for (int q = threadIdx.x; q < " + I(NTD) + "; q += " + I(NR * 32) + ") s_td[q] = g_td[q];");
  E.line("for (int q = threadIdx.x; q < " + I(NTI) + "; q += " + I(NR * 32) + ") s_ti[q] = g_ti[q];");
  E.line("const double *c_iW = s_td + " + I(oiW) + ", *c_Rk = s_td + " + I(oRk) + ", *c_hc = s_td + " + I(ohc) + ", *c_cc = s_td + " + I(occ) +
         ", *c_eff = s_td + " + I(oeff) + ";");
  E.line("const double2 *c_rc = (const double2 *)s_td + w * " + I(NSLOT * RC / 2) + ";     // this role's records");
  E.line("const int4 *c_rx = (const int4 *)s_ti + w * " + I(NSLOT * RX / 4) + ";");
  E.line("int *s_flag = (int *)(sm_ + " + I(L.oPIV * 32) + ");");
  E.line("const unsigned ncell = (unsigned)a.n0 * (unsigned)a.n1 * (unsigned)a.n2, nbp = (ncell + 31u) / 32u;");
  E.line("const long long nbt = (long long)nbp * a.np;");
  E.line("const double dt = a.scal[0] * a.dts;");
  E.line("int prel = (int)(blockIdx.x / nbp); unsigned lt = blockIdx.x % nbp;     // patch (relative) and turn within it, advanced without divisions");
  E.line("if ((long long)blockIdx.x < nbt) prefetch_turn(a, sm_, prel, lt, ncell);");
  E.line("asm volatile(\"cp.async.wait_all;\" ::: \"memory\");");
  E.line("BAR();");
  E.line("const int r_tb = s_ti[" + I(ocnt) + " + 2 * w], r_end = s_ti[" + I(ocnt) + " + 2 * w + 1];     // this role's trip counts");
  E.line("#pragma unroll 1");
  E.line("for (long long bt = blockIdx.x; bt < nbt; bt += gridDim.x) {   // persistent CTA: 32 cells per turn");
  E.line("const int patch = prel + a.patch0;");
  E.line("unsigned t = lt * 32u + lane;");
  E.line("const bool live = t < ncell;");
  E.line("if (!live) t = ncell - 1u;   // idle lanes recompute the last cell and store nothing");
  E.line("const unsigned ci = t % (unsigned)a.n0, r_ = t / (unsigned)a.n0;");
  E.line("const unsigned cj = r_ % (unsigned)a.n1, ck = r_ / (unsigned)a.n1;");
  E.line("const long long id = (ci + a.G0) * a.st0 + (cj + a.G1) * a.st1 + (ck + a.G2) * a.st2;");
  E.line("double *Up = a.U + (long long)patch * " + I(nvar) + " * a.pc + id;");
  E.line("const long long pid = (long long)patch * a.pc + id;");
  // ---- cons -> prim pieces (eq 4.2); species k = w + 8 s belong to this role
  E.line("const double rho = SM(" + I(L.oNX) + "), irho = 1.0 / rho;");
  E.line("double ke = 0.0;");
  for (int d = 0; d < ndim; d++)
    E.line("{ const double ud = SM(" + I(L.oNX + 1 + d) + ") * irho; ke = fma(0.5 * ud, ud, ke); }");
  E.line("const double e = SM(" + I(L.oNX + ndim + 1) + ") * irho - ke;");
  E.line("double T = SM(" + I(L.oNX + nvar) + ");");
  E.line("double pr_ = 0.0, py_ = 0.0;");
  for (int s = 0; s < NSL; s++) {
    const std::string ss = I(s);
    E.line("const int k" + ss + " = w + " + I(NR * s) + ";");
    E.line("double ry" + ss + " = k" + ss + " < " + I(n1) + " ? SM(" + I(L.oNX + ndim + 2) + " + k" + ss + ") : 0.0;");
    E.line("double Y" + ss + " = ry" + ss + " * irho;");
    E.line("pr_ += ry" + ss + "; py_ += Y" + ss + ";");
    E.line("if (k" + ss + " < " + I(n1) + ") SM(" + I(L.oX) + " + k" + ss + ") = ry" + ss + " * c_iW[k" + ss + "];");
  }
  E.line("SM(" + I(L.oP) + " + w) = pr_; SM(" + I(L.oP + NR) + " + w) = py_;");
  E.line("if (w == 0) SM(" + I(L.oX + ns) + ") = 1.0;");
  E.line("BAR();");
  E.line("unsigned nlt = lt + gridDim.x; int nprel = prel;");
  E.line("while (nlt >= nbp) { nlt -= nbp; nprel++; }");
  E.line("if (bt + gridDim.x < nbt) prefetch_turn(a, sm_, nprel, nlt, ncell);   // lands during this turn");
  E.line("{ double rsum = 0.0, ysum = 0.0;");
  E.line("  #pragma unroll");
  E.line("  for (int q = 0; q < " + I(NR) + "; q++) { rsum += SM(" + I(L.oP) + " + q); ysum += SM(" + I(L.oP + NR) + " + q); }");
  // X of the last species: every role forms the same value (same sums, same order) and stores it itself before its own
  // reads in the rate loop -- no barrier is needed between this store and those reads (with T* from the cons->prim
  // launch there is no Newton loop, whose barriers used to separate them)
  E.line("  SM(" + I(L.oX + n1) + ") = (rho - rsum) * " + num(M.invW[n1]) + ";");
  E.line("  if (w == " + I(wN) + ") { ry" + I(sN) + " = rho - rsum; Y" + I(sN) + " = 1.0 - ysum; } }");
  for (int s = 0; s < NSL; s++)
    E.line("const double yr" + I(s) + " = k" + I(s) + " < " + I(ns) + " ? Y" + I(s) + " * c_Rk[k" + I(s) + " < " + I(ns) + " ? k" + I(s) + " : 0] : 0.0;");
  // ---- Newton on e(T) (eq 4.3-4.4, reading A6): partial sums per role, summed in the same order by everyone
  if (roles_newton_ref()) {
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
  E.line("  SM(" + I(L.oN) + " + w) = f; SM(" + I(L.oN + NR) + " + w) = cv;");
  E.line("  BAR();");
  E.line("  f = -e; cv = 0.0;");
  E.line("  #pragma unroll");
  E.line("  for (int q = 0; q < " + I(NR) + "; q++) { f += SM(" + I(L.oN) + " + q); cv += SM(" + I(L.oN + NR) + " + q); }");
  E.line("  const double dT = -f / cv;");
  E.line("  if (!conv) { T += dT; if (fabs(dT) <= 1e-11 * fabs(T)) conv = true; }");
  E.line("  if (__syncthreads_and(conv)) break;");
  E.line("}");
  E.line("bool ok = conv && (T > 0.0) && isfinite(T);");
  E.line("if (live && w == 0) a.T[pid] = T;");
  } else {
  E.line("bool ok = (T > 0.0) && isfinite(T);     // T* was computed by the cons->prim kernel launched before this one");
  }
  // ---- rates of progress (eq 4.7-4.9): shared code, tables indexed by the warp-uniform role.  Third-body
  //      reactions come first in every role's list; the others are taken two at a time (branch-free body,
  //      so the two exponential chains interleave).
  // One reaction in three parts, so that a trip through the loop can be emitted as  loads of all its reactions / arithmetic
  // / stores: everything lives in one shared-memory array, so the compiler may not move the loads of the next reaction
  // above the stores of the previous one, and a body written reaction by reaction executes them one after the other
  // (two exponential chains in flight instead of eight).
  auto rate_loads = [&](const std::string &S, const std::string &slot) {
    const int ND2 = RC / 2, NI4 = RX / 4;
    auto dv = [&](int e) { return "rc" + I(e / 2) + S + (e % 2 ? ".y" : ".x"); };
    auto iv = [&](int e) { static const char *c[4] = {".x", ".y", ".z", ".w"}; return "rx" + I(e / 4) + S + c[e % 4]; };
    std::string l = "    const double2 ";
    for (int e = 0; e < ND2; e++) l += "rc" + I(e) + S + " = c_rc[(" + slot + ") * " + I(ND2) + " + " + I(e) + "]" + (e + 1 < ND2 ? ", " : ";");
    E.line(l);
    l = "    const int4 ";
    for (int e = 0; e < NI4; e++) l += "rx" + I(e) + S + " = c_rx[(" + slot + ") * " + I(NI4) + " + " + I(e) + "]" + (e + 1 < NI4 ? ", " : ";");
    E.line(l);
    E.line("    const int i" + S + " = " + iv(0) + ";");
    E.line("    const double f0" + S + " = " + dv(0) + ", f1" + S + " = " + dv(1) + ", f2" + S + " = " + dv(2) + ";");
    if (any_rev) {
      l = "    const double ";
      for (int q = 0; q < NKB; q++) l += "d" + I(q) + S + " = " + dv(3 + q) + (q + 1 < NKB ? ", " : ";");
      E.line(l);
      if (!all_rev) E.line("    const double rv" + S + " = " + dv(3 + NKB) + ";");
    }
    for (int q = 0; q < maxof; q++) E.line("    const double xf" + I(q) + S + " = SM(" + I(L.oX) + " + " + iv(2 + q) + ");");
    if (any_rev) for (int q = 0; q < maxob; q++) E.line("    const double xb" + I(q) + S + " = SM(" + I(L.oX) + " + " + iv(2 + maxof + q) + ");");
  };
  auto rate_math = [&](const std::string &S) {
    E.line("    const double kf" + S + " = exp_nb(fma(f2" + S + ", iT, fma(f1" + S + ", lnT, f0" + S + ")));");
    if (any_rev) {
      std::string lk = "fma(d2" + S + ", iT, fma(d1" + S + ", lnT, d0" + S + "))";
      if (degc > 0) {
        std::string pol = "d" + I(NKB - 1) + S;
        for (int q = NKB - 2; q >= 3; q--) pol = "fma(T, " + pol + ", d" + I(q) + S + ")";
        lk = "fma(T, " + pol + ", " + lk + ")";
      }
      // branch-free: irreversible reactions multiply a finite exponential by zero
      if (all_rev) E.line("    const double kb" + S + " = exp_nb(" + lk + ");");
      else E.line("    const double kb" + S + " = exp_nb(" + lk + ") * rv" + S + ";");
    } else {
      E.line("    const double kb" + S + " = 0.0;");
    }
    E.line("    double pf" + S + " = kf" + S + ", pb" + S + " = kb" + S + ";");
    for (int q = 0; q < maxof; q++) E.line("    pf" + S + " *= xf" + I(q) + S + ";");
    if (any_rev) for (int q = 0; q < maxob; q++) E.line("    pb" + S + " *= xb" + I(q) + S + ";");
    E.line("    const double rn" + S + " = pf" + S + " - pb" + S + ";");
  };
  auto rate_stores = [&](const std::string &S) {
    E.line("    SM(" + I(L.oR) + " + i" + S + ") = kf" + S + "; SM(" + I(L.oR + nrs) + " + i" + S + ") = kb" + S + "; SM(" + I(L.oR + 2 * nrs) + " + i" + S + ") = rn" + S + ";");
  };
  const std::string RI = "c_rx[r * " + I(RX / 4) + "].x", RTB = "c_rx[r * " + I(RX / 4) + "].y";
  E.line("{ const double lnT = log(T), iT = 1.0 / T;");
  E.line("  int r = 0;");
  if (M.ntb > 0) {
    E.line("  #pragma unroll 1");
    E.line("  for (; r < r_tb; r++) {");
    rate_loads("", "r");
    E.line("    const int tb_ = rx0.y - 1;");
    E.line("    const double *ef = c_eff + tb_ * " + I(ns) + ";");
    // four partial sums: the ns-term chain of dependent FMAs would be the longest path of the trip
    E.line("    double Mi, Mi1 = 0.0, Mi2 = 0.0, Mi3 = 0.0;");
    E.line("    Mi = ef[0] * SM(" + I(L.oX) + ");");
    for (int j = 1; j < ns; j++) {
      const std::string acc = (j % 4 == 0) ? "Mi" : "Mi" + I(j % 4);
      E.line("    " + acc + " = fma(ef[" + I(j) + "], SM(" + I(L.oX + j) + "), " + acc + ");");
    }
    E.line("    Mi = (Mi + Mi1) + (Mi2 + Mi3);");
    rate_math("");
    E.line("    SM(" + I(L.oRN) + " + tb_) = rn;");
    E.line("    SM(" + I(L.oR) + " + i) = Mi * kf; SM(" + I(L.oR + nrs) + " + i) = Mi * kb; SM(" + I(L.oR + 2 * nrs) + " + i) = Mi * rn;");
    E.line("  }");
  }
  E.line("  #pragma unroll 1");
  E.line("  for (; r < r_end; r += 4) {");
  for (int q = 0; q < 4; q++) rate_loads(std::string(1, (char)('a' + q)), "r + " + I(q));
  for (int q = 0; q < 4; q++) rate_math(std::string(1, (char)('a' + q)));
  for (int q = 0; q < 4; q++) rate_stores(std::string(1, (char)('a' + q)));
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
        const std::string q = row(L.oR + 2 * nrs + i);
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
        const std::string cfs = row(L.oR + i), cbs = row(L.oR + nrs + i);
        if (cf[i][j] > 0) dq = (cf[i][j] > 1 ? num((double)cf[i][j]) + " * " : std::string("")) + xprod(cfs, cf[i].data(), ns, j);
        if (rev && cb[i][j] > 0) dq += (dq.empty() ? "-" : " - ") + (cb[i][j] > 1 ? num((double)cb[i][j]) + " * " : std::string("")) + xprod(cbs, cb[i].data(), ns, j);
        (void)tb;     // the efficiency term a_ij r_i of a third-body reaction touches every column: shared code below
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
    }
    E.line("} break;");
  }
  E.line("}");
  // ---- third-body efficiencies (eq 4.7): D_kj += dnu_ik a_ij r_i for EVERY column j.  The same code for every role
  //      (a_ij comes from the table, indexed by the role's columns), so its instructions are fetched once for the
  //      eight warps: role-specific straight-line code streams from L2 at well under one instruction per clock.
  if (M.ntb > 0) {
    E.line("{");
    for (int s = 0; s < NSL; s++)
      E.line("  const double *ef" + I(s) + " = c_eff + (k" + I(s) + " <= " + I(n1) + " ? k" + I(s) + " : 0);");
    for (int i = 0; i < nr; i++) {
      if (!M.tb[i]) continue;
      bool any = false;
      for (int k = 0; k < n1; k++) any = any || dnu[i][k] != 0;
      if (!any) continue;
      const int q = M.tbi[i];
      E.line("  { const double rn = " + row(L.oRN + q) + ";");
      for (int s = 0; s < NSL; s++) E.line("    const double t" + I(s) + " = ef" + I(s) + "[" + I(q * ns) + "] * rn;");
      for (int k = 0; k < n1; k++) {
        if (dnu[i][k] == 0) continue;
        for (int s = 0; s < NSL; s++) {
          if (dnu[i][k] == 1) E.line("    " + A(s, k) + " += t" + I(s) + ";");
          else if (dnu[i][k] == -1) E.line("    " + A(s, k) + " -= t" + I(s) + ";");
          else E.line("    " + A(s, k) + " = fma(" + num((double)dnu[i][k]) + ", t" + I(s) + ", " + A(s, k) + ");");
        }
      }
      E.line("  }");
    }
    E.line("}");
  }
  E.line("if (w == " + I(wN) + ") {");
  for (int k = 0; k < n1; k++) E.line("  " + row(L.oDL + k) + " = " + A(sN, k) + " * " + num(M.invW[n1]) + ";");
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
  if (roles_lu_rows_ref()) {
  // ---- LU with one ROW per lane.  The columns the roles assembled are transposed through shared memory
  //      ([row][column][cell]); then NR adjacent lanes of a warp own one cell: lane group index g_ holds rows g_, g_ + NR,
  //      ... (n1 + 1 entries each, in registers, static indices: the column loop is unrolled).  Step c: the lanes that
  //      hold row c publish its entries c..n1 to a small per-cell buffer, everybody reads them back (broadcast), rows
  //      below take  a_rj -= (a_rc / a_cc) a_cj.  A warp owns its 32 / NR cells from here to the solution: no barrier,
  //      no named barrier, only __syncwarp.  Fast path = no row swap needed (the diagonal entry is the first row of
  //      maximal |a_rc|, r >= c: the oracle's rule); if any cell of the CTA needs one, the system -- still untouched in
  //      shared memory -- is solved by the generic pivoted loop below.
  const int RS = (n1 + NR - 1) / NR;                                   // row slots per lane
  const int NC1 = n1 + 1;
  auto R = [](int t, int j) { return "R" + I(t) + "_" + I(j); };
  // transposed store of the columns this role assembled
  E.line("{");
  for (int s = 0; s < NSL; s++) {
    E.line("  if (k" + I(s) + " <= " + I(n1) + ") { double *mt_ = sm_ + " + I(L.oR * 32) + " + k" + I(s) + " * 32 + lane;");
    for (int k = 0; k < n1; k++) E.line("    mt_[" + I(k * L.rstr) + "] = " + A(s, k) + ";");
    E.line("  }");
  }
  E.line("}");
  E.line("BAR();");
  // The column loop is ROLLED (the whole kernel has to stay close to the 32 KB instruction cache: straight-line code
  // streams from L2 at half an instruction per clock): after step c every row drops its column c, i.e. the update
  // writes column j into register j - 1, so the pivot column is always physical column 0 and the body is the same for
  // every c.  A row that has served as pivot row is frozen in shared memory (U store, triangular, per cell), where the
  // back-substitution reads it; its registers shift on as dead values.  The loop is cut into phases with fewer
  // physical columns and fewer live row slots.
  E.line("int bad = 0;");
  E.line("{");
  // lane = row group x CW + cell of the warp (CW = 32 / NR cells per warp): the CW lanes that own a row are adjacent,
  // so their 16-byte publishing stores go out as one shared-memory wavefront (one lane per quarter-warp costs four)
  const int CW = 32 / NR;
  E.line("  const int g_ = lane / " + I(CW) + ", cell_ = w * " + I(CW) + " + lane % " + I(CW) + ";");
  E.line("  const double *mr_ = sm_ + " + I(L.oR * 32) + " + g_ * " + I(L.rstr) + " + cell_;");
  E.line("  double *us_ = sm_ + " + I(L.oPB * 32) + " + cell_ * " + I(L.pbs) + ";     // U rows of this cell, row c at uoff(c)");
  for (int t = 0; t < RS; t++) {
    const bool part = NR * t + NR - 1 >= n1;                           // some lanes of this slot hold no row: zeros
    for (int j = 0; j < NC1; j++)
      E.line("  double " + R(t, j) + " = " + (part ? "g_ + " + I(NR * t) + " < " + I(n1) + " ? " : std::string("")) +
             "mr_[" + I(NR * t * L.rstr + j * 32) + "]" + (part ? " : 0.0" : "") + ";");
  }
  {
    std::string d = "  double ";
    for (int t = 0; t < RS; t++) d += "IP" + I(t) + " = 0.0, XS" + I(t) + " = 0.0" + (t + 1 < RS ? ", " : ";");
    E.line(d);
  }
  // The loop is software-pipelined: step c first updates the slot that holds row c + 1, publishes that row (with the
  // reciprocal of its diagonal entry, computed while the rest of the row is still being updated) and issues the loads of
  // step c + 1; the other slots are updated behind it, so the store -> load -> multiply chain of the next step is off
  // the critical path.  Two register sets (qa / qb) alternate; the loop body is two steps.
  // Phases [cs, ce): constant slot of the pivot row, constant slot of the next pivot row, constant set of live slots,
  // ncols = NC1 - cs physical columns.
  std::vector<int> cuts;
  {
    std::vector<char> cut(n1 + 1, 0);
    cut[0] = cut[n1] = 1;
    for (int t = 0; t < RS; t++) {
      if (NR * t < n1) cut[NR * t] = 1;                                // pivot slot changes
      if (NR * t + NR - 1 < n1) cut[NR * t + NR - 1] = 1;              // next-pivot slot changes, slot t goes dead
    }
    int last = 0;
    for (int c = 1; c <= n1; c++) {
      if (!cut[c]) continue;
      if (c - last >= 6) { int mid = last + (c - last) / 2; mid -= (mid - last) % 2; cut[mid] = 1; }   // fewer columns in the second half
      last = c;
    }
    for (int c = 0; c <= n1; c++) if (cut[c]) cuts.push_back(c);
  }
  {
    std::string d = "  double2 ";
    for (int j = 0; j < NC1; j += 2) d += "qa" + I(j) + ", qb" + I(j) + (j + 2 < NC1 ? ", " : ";");
    E.line(d);
    E.line("  double ipa, ipb;");
  }
  auto Q = [&](int b, int j) { return std::string(b ? "qb" : "qa") + I(j & ~1) + ((j & 1) ? ".y" : ".x"); };
  auto IPB = [&](int b) { return std::string(b ? "ipb" : "ipa"); };
  const int ipoff = L.pbs - 2;
  // publish row `cx` (held in slot t, nv valid entries) from the lanes g_ == cx % NR: predicated stores (inline PTX; as
  // an `if` the compiler branches around them and sinks the reciprocal's Newton steps into the branch, where nothing
  // overlaps them), then -- after whatever the caller puts in between -- the loads into register set b
  auto publish = [&](const std::string &cx, int t, int nv, const std::string &ind) {
    const int nv2 = (nv + 1) / 2 * 2;
    E.line(ind + "{ const unsigned ua_ = (unsigned)__cvta_generic_to_shared(us_ + uo_);");
    E.line(ind + "  const double ipn_ = rcp_nb(" + R(t, 0) + ");");
    E.line(ind + "  const int own_ = g_ == (" + cx + ") % " + I(NR) + ";");
    for (int j = 0; j < nv2; j += 2)
      E.line(ind + "  PST2(own_, ua_ + " + I(j * 8) + ", " + R(t, j) + ", " + (j + 1 < nv ? R(t, j + 1) : std::string("0.0")) + ");");
    E.line(ind + "  PST1(own_, (unsigned)__cvta_generic_to_shared(us_ + " + I(ipoff) + " + ((" + cx + ") & 1)), ipn_);");
    E.line(ind + "}");
  };
  auto load = [&](const std::string &cx, int b, int nv, const std::string &ind) {
    const int nv2 = (nv + 1) / 2 * 2;
    E.line(ind + "__syncwarp();");
    E.line(ind + "{ const double *ur_ = us_ + uo_;");
    for (int j = 0; j < nv2; j += 2) E.line(ind + "  " + std::string(b ? "qb" : "qa") + I(j) + " = *(const double2 *)(ur_ + " + I(j) + ");");
    E.line(ind + "  " + IPB(b) + " = us_[" + I(ipoff) + " + ((" + cx + ") & 1)];");
    E.line(ind + "}");
  };
  auto update_slot = [&](const std::string &cx, int t, int b, int ncols, const std::string &ind) {
    // rows <= c are dead values from here on (their U row is frozen in shared memory): they are updated like live rows,
    // unmasked -- only the pivot check has to leave them out
    E.line(ind + "{ const bool act = g_ + " + I(NR * t) + " > " + cx + "; const double l_ = " + R(t, 0) + " * " + IPB(b) + ";");
    E.line(ind + "  bad |= (int)(act & (fabs(" + R(t, 0) + ") > fabs(" + Q(b, 0) + ")));");
    for (int j = 1; j < ncols; j++) E.line(ind + "  " + R(t, j - 1) + " = fma(-l_, " + Q(b, j) + ", " + R(t, j) + ");");
    E.line(ind + "}");
  };
  // one elimination step with the pivot row in register set b; the next row goes to set 1 - b
  auto step = [&](const std::string &cx, int cs, int ce, int b, bool has_next, const std::string &ind) {
    const int ncols = NC1 - cs, t0 = cs / NR, t1 = (cs + 1) / NR < RS ? (cs + 1) / NR : RS - 1;
    (void)ce;
    E.line(ind + "uo_ += ((" + I(NC1) + " - (" + cx + ") + 1) >> 1) << 1;     // offset of row c + 1 (row lengths rounded up to even)");
    // slots other than the next pivot row's: the first one goes between the publishing stores' operands (the
    // reciprocal chain) and the stores' consumers, the rest behind the loads of the next row
    std::vector<int> others;
    for (int t = 0; t < RS; t++) {
      if (NR * t + NR - 1 <= cs) continue;                             // every row of the slot is <= c throughout the phase
      if (has_next && t == t1) continue;
      others.push_back(t);
    }
    size_t done = 0;
    if (has_next) {
      update_slot(cx, t1, b, ncols, ind);
      publish("(" + cx + ") + 1", t1, ncols - 1, ind);
      if (others.size() > 1) update_slot(cx, others[done++], b, ncols, ind);
      load("(" + cx + ") + 1", 1 - b, ncols - 1, ind);
    }
    E.line(ind + "bad |= !(fabs(" + Q(b, 0) + ") > 0.0);");
    E.line(ind + "if (g_ == (" + cx + ") % " + I(NR) + ") IP" + I(t0) + " = " + IPB(b) + ";");
    for (; done < others.size(); done++) update_slot(cx, others[done], b, ncols, ind);
  };
  E.line("  int uo_ = 0;");
  publish("0", 0, NC1, "  ");
  load("0", 0, NC1, "  ");
  int cur = 0;                                                         // register set that holds the pivot row at the phase start
  for (size_t ph = 0; ph + 1 < cuts.size(); ph++) {
    const int cs = cuts[ph], ce = cuts[ph + 1];
    if (cs >= ce) continue;
    const int npair = (ce - cs) / 2;
    const bool last_phase = ce == n1;
    // the very last step (c = n1 - 1) has no next row: keep it out of the paired loop
    int pairs = npair, rem = (ce - cs) % 2;
    if (last_phase && rem == 0) { pairs -= 1; rem = 2; }
    if (pairs > 0) {
      E.line("  #pragma unroll 1");
      E.line("  for (int c = " + I(cs) + "; c < " + I(cs + 2 * pairs) + "; c += 2) {");
      step("c", cs, ce, cur, true, "    ");
      step("c + 1", cs, ce, 1 - cur, true, "    ");
      E.line("  }");
    }
    int c = cs + 2 * pairs;
    for (; c < ce; c++) {
      step(I(c), cs, ce, cur, c + 1 < n1, "  ");
      cur = 1 - cur;
    }
  }
  // back-substitution from the U store: row r holds u_r,r .. u_r,n1-1, rhs_r at ur(r)[0 .. n1 - r]
  E.line("  bool okx = true;");
  {
    // offset of row r: sum_{i<r} roundup_even(NC1 - i)
    const std::string odd = (NC1 % 2 == 0) ? "(r >> 1)" : "((r + 1) >> 1)";
    E.line("  auto uoff = [](int r) { return r * " + I(NC1) + " - ((r * (r - 1)) >> 1) + " + odd + "; };");
  }
  for (int t = 0; t < RS; t++) {
    E.line("  const int r" + I(t) + " = g_ + " + I(NR * t) + ", o" + I(t) + " = uoff(r" + I(t) + " < " + I(n1) + " ? r" + I(t) + " : 0);");
    E.line("  double Y" + I(t) + " = r" + I(t) + " < " + I(n1) + " ? us_[o" + I(t) + " + " + I(n1) + " - r" + I(t) + "] : 0.0;");
  }
  // one loop per row slot of the pivot row (the slot index is then static: no selects)
  for (int t = 0; t < RS; t++) E.line("  const double *p" + I(t) + " = us_ + o" + I(t) + " - r" + I(t) + ";     // u_r,c of this lane's row at p[c]");
  for (int to = RS - 1; to >= 0; to--) {
    const int chi = std::min(n1 - 1, NR * to + NR - 1), clo = NR * to;
    E.line("  #pragma unroll 1");
    E.line("  for (int c = " + I(chi) + "; c >= " + I(clo) + "; c--) {");
    E.line("    const int go = c - " + I(clo) + ";");
    E.line("    double x_ = Y" + I(to) + " * IP" + I(to) + ";");
    E.line("    x_ = __shfl_sync(0xffffffffu, x_, go * " + I(CW) + " + lane % " + I(CW) + ");");
    E.line("    if (g_ == go) XS" + I(to) + " = x_;");
    for (int t = 0; t <= to; t++)                                        // rows of higher slots are all > c
      E.line("    if (r" + I(t) + " < c) Y" + I(t) + " = fma(-p" + I(t) + "[c], x_, Y" + I(t) + ");");
    E.line("  }");
  }
  for (int t = 0; t < RS; t++)
    E.line("  if (r" + I(t) + " < " + I(n1) + ") { if (!isfinite(XS" + I(t) + ")) okx = false; sm_[(" + I(L.oXS) + " + r" + I(t) + ") * 32 + cell_] = XS" + I(t) + "; }");
  E.line("  if (!okx) bad |= 2;     // non-finite solution: let the pivoted path decide (it raises the flag)");
  E.line("}");
  E.line("if (__syncthreads_or(bad)) {");
  // ---- slow path: generic partial pivoting on the untouched system in shared memory (lane = cell, roles split the columns)
  E.line("  #define SMA(r, c) sm_[" + I(L.oR * 32) + " + (r) * " + I(L.rstr) + " + (c) * 32 + lane]");
  E.line("  #pragma unroll 1");
  E.line("  for (int c = 0; c < " + I(n1) + "; c++) {");
  E.line("    int piv = c; double best = fabs(SMA(c, c));");
  E.line("    for (int r = c + 1; r < " + I(n1) + "; r++) { const double v = fabs(SMA(r, c)); if (v > best) { best = v; piv = r; } }");
  E.line("    if (!(best > 0.0)) ok = false;");
  E.line("    BAR();   // every role has chosen the pivot of column c before anyone swaps it");
  for (int s = 0; s < NSL; s++)
    E.line("    if (k" + I(s) + " >= c && k" + I(s) + " <= " + I(n1) + " && piv != c) { const double x_ = SMA(c, k" + I(s) + "); SMA(c, k" + I(s) + ") = SMA(piv, k" + I(s) + "); SMA(piv, k" + I(s) + ") = x_; }");
  E.line("    BAR();");
  E.line("    const double ip = 1.0 / SMA(c, c);     // column c is not written by the sweep below (only columns > c)");
  for (int s = 0; s < NSL; s++) {
    E.line("    if (k" + I(s) + " > c && k" + I(s) + " <= " + I(n1) + ") { const double pj = SMA(c, k" + I(s) + ");");
    E.line("      for (int r = 0; r < " + I(n1) + "; r++) if (r != c) SMA(r, k" + I(s) + ") = fma(-(SMA(r, c) * ip), pj, SMA(r, k" + I(s) + ")); }");
  }
  E.line("    if (w == 0) SM(" + I(L.oIP) + " + c) = ip;");
  E.line("    BAR();");
  E.line("  }");
  E.line("  if (w == " + I(wN) + ") {");
  E.line("    for (int k = 0; k < " + I(n1) + "; k++) { const double x_ = SMA(k, " + I(n1) + ") * SM(" + I(L.oIP) + " + k); if (!isfinite(x_)) ok = false; SM(" + I(L.oXS) + " + k) = x_; }");
  E.line("  }");
  E.line("  #undef SMA");
  E.line("}");
  } else {
  // ---- Gauss-Jordan elimination, column-distributed, one-column look-ahead (see the header); L is not kept: the
  //      right-hand side is column n1 of the system.  The column loop is a real loop (compact code, warm in the
  //      instruction cache): the update writes row p + 1 into row p, so the pivot row is always physical row 0
  //      (after n1 columns every surviving column is back in its original order) and only the slot is selected
  //      at run time, by warp-uniform branches.
  auto rot = [&](int s, const std::string &ind) {
    std::string l = ind + "{ const double P_ = " + A(s, 0) + ";";
    E.line(l);
    for (int p = 0; p + 1 < n1; p++) E.line(ind + "  " + A(s, p) + " = fma(-f" + I(p + 1) + ", P_, " + A(s, p + 1) + ");");
    E.line(ind + "  " + A(s, n1 - 1) + " = P_; }");
  };
  // owner of column cn (variables cn, pbn in scope), already rotated into cn's frame: physical rows 1..n1-1-cn are the
  // rows below the diagonal.  Publishes "needs a swap" and, if no cell does, the multipliers of all other rows.
  auto owner = [&](int s, const std::string &ind) {
    E.line(ind + "{ const double ac = fabs(" + A(s, 0) + "), ip = rcp_nb(" + A(s, 0) + ");");
    E.line(ind + "  const int nb_ = " + I(n1) + " - cn;");
    E.line(ind + "  int bad = !(ac > 0.0);                       // branch-free: 18 independent compares");
    for (int p = 1; p < n1; p++) E.line(ind + "  bad |= (int)(" + I(p) + " < nb_) & (int)(fabs(" + A(s, p) + ") > ac);");
    // multipliers are published unconditionally (garbage if a swap is needed: every role then leaves the loop
    // before using them), so nothing on the owner's critical path waits for a vote
    for (int p = 1; p < n1; p++) E.line(ind + "  SM(" + I(L.oF) + " + cn * " + I(n1) + " + " + I(p) + ") = " + A(s, p) + " * ip;");
    E.line(ind + "  SM(" + I(L.oIP) + " + cn) = ip;");
    E.line(ind + "  s_flag[cn * 64 + lane] = bad;");
    E.line(ind + "}");
  };
  E.line("int c0 = " + I(n1) + ";     // first column of the pivoted slow path (" + I(n1) + ": none)");
  E.line("if (w == 0) { const int cn = 0;");
  owner(0, "  ");
  E.line("  PUBLISH(1);");
  E.line("}");
  E.line("#pragma unroll 1");
  E.line("for (int c = 0; c < " + I(n1) + "; c++) {");
  E.line("  const int sc = c / " + I(NR) + ", oc = c % " + I(NR) + ";");
  E.line("  if (w != oc) AWAIT(1 + c % 15);     // column c published by its owner (producer / consumer barrier)");
  E.line("  const int fl_ = s_flag[c * 64 + lane];");
  for (int p = 1; p < n1; p++) E.line("  const double f" + I(p) + " = SM(" + I(L.oF) + " + c * " + I(n1) + " + " + I(p) + ");");
  E.line("  if (__any_sync(0xffffffffu, fl_ != 0)) { c0 = c; break; }");
  E.line("  const int cn = c + 1, ocn = cn % " + I(NR) + ", scn = cn / " + I(NR) + ";");
  E.line("  const bool la = cn < " + I(n1) + " && w == ocn;     // this role owns the next column: update it first, publish");
  E.line("  if (la) {");
  for (int s = 0; s < NSL; s++) {
    if (NR * s >= n1) break;
    E.line("    " + std::string(s ? "else " : "") + "if (scn == " + I(s) + ") {");
    rot(s, "      ");
    owner(s, "      ");
    E.line("    }");
    if (NR * (s + 1) >= n1 || s + 1 == NSL) E.line("    PUBLISH(1 + cn % 15);");
  }
  E.line("  }");
  for (int s = 0; s < NSL; s++) {
    std::string cond = "(sc < " + I(s) + " || (sc == " + I(s) + " && w > oc)) && !(la && scn == " + I(s) + ")";
    if (s == sN) cond += " && w <= " + I(wN);
    E.line("  if (" + cond + ") {");
    rot(s, "    ");
    E.line("  }");
  }
  E.line("}");
  // ---- fast path: the system is diagonal; the role holding the right-hand side scales it
  E.line("BAR();");
  E.line("if (c0 == " + I(n1) + ") {");
  E.line("  if (w == " + I(wN) + ") {");
  for (int k = 0; k < n1; k++) {
    E.line("    { const double x_ = " + A(sN, k) + " * " + row(L.oIP + k) + "; if (!isfinite(x_)) ok = false; " + row(L.oXS + k) + " = x_; }");
  }
  E.line("  }");
  E.line("} else {");
  // ---- slow path: spill the system, finish columns c0.. with partial pivoting in shared memory (generic loops)
  const int NC = n1 + 1;
  E.line("  #define SMA(r, c) sm_[((" + I(L.oR) + ") + (r) * " + I(NC) + " + (c)) * 32 + lane]");
  for (int s = 0; s < NSL; s++) {
    E.line("  if (k" + I(s) + " >= c0 && k" + I(s) + " <= " + I(n1) + ") {   // registers are rotated by c0 rows");
    for (int p = 0; p < n1; p++)
      E.line("    { int lr = " + I(p) + " + c0; if (lr >= " + I(n1) + ") lr -= " + I(n1) + "; SMA(lr, k" + I(s) + ") = " + A(s, p) + "; }");
    E.line("  }");
  }
  E.line("  BAR();");
  E.line("  #pragma unroll 1");
  E.line("  for (int c = c0; c < " + I(n1) + "; c++) {");
  E.line("    int piv = c; double best = fabs(SMA(c, c));");
  E.line("    for (int r = c + 1; r < " + I(n1) + "; r++) { const double v = fabs(SMA(r, c)); if (v > best) { best = v; piv = r; } }");
  E.line("    if (!(best > 0.0)) ok = false;");
  for (int s = 0; s < NSL; s++)
    E.line("    if (k" + I(s) + " >= c && k" + I(s) + " <= " + I(n1) + " && piv != c) { const double x_ = SMA(c, k" + I(s) + "); SMA(c, k" + I(s) + ") = SMA(piv, k" + I(s) + "); SMA(piv, k" + I(s) + ") = x_; }");
  E.line("    BAR();");
  E.line("    const double ip = 1.0 / SMA(c, c);");
  for (int s = 0; s < NSL; s++) {
    E.line("    if (k" + I(s) + " > c && k" + I(s) + " <= " + I(n1) + ") { const double pj = SMA(c, k" + I(s) + ");");
    E.line("      for (int r = 0; r < " + I(n1) + "; r++) if (r != c) SMA(r, k" + I(s) + ") = fma(-(SMA(r, c) * ip), pj, SMA(r, k" + I(s) + ")); }");
  }
  E.line("    if (w == 0) SM(" + I(L.oIP) + " + c) = ip;");
  E.line("    BAR();");
  E.line("  }");
  E.line("  if (w == " + I(wN) + ") {");
  E.line("    for (int k = 0; k < " + I(n1) + "; k++) { const double x_ = SMA(k, " + I(n1) + ") * SM(" + I(L.oIP) + " + k); if (!isfinite(x_)) ok = false; SM(" + I(L.oXS) + " + k) = x_; }");
  E.line("  }");
  E.line("  #undef SMA");
  E.line("}");
  }
  E.line("BAR();");
  for (int s = 0; s < NSL; s++)
    E.line("if (live && k" + I(s) + " < " + I(n1) + ") Up[(long long)(" + I(ndim + 2) + " + k" + I(s) + ") * a.pc] = ry" + I(s) +
           " + SM(" + I(L.oXS) + " + k" + I(s) + ");");
  E.line("if (!ok && live) *a.flag = 1;");
  E.line("asm volatile(\"cp.async.wait_all;\" ::: \"memory\");");
  E.line("BAR();   // shared rows are reused by the next turn; the prefetched inputs are visible to every role");
  E.line("lt = nlt; prel = nprel;");
  E.line("}");
  src += "}\n#undef PST2\n#undef PST1\n#undef SM\n#undef BAR\n#undef AWAIT\n#undef PUBLISH\n";
  return src;
}

}  // namespace chemgen
