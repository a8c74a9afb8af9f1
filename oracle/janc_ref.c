/* oracle/janc_ref.c -- CPU fp64 ORACLE for the JANC per-step update (arXiv 2504.13750).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It shares no
 * code, header, table or helper with the CUDA path (paper_2504_13750_b200/csrc) and
 * neither imports the other.
 *
 * It is the algorithm of PAPER.md section 4 written out step by step, in the paper's order
 * and notation, with the readings A1..A24 of SURVEY.md section 8(c) (listed in DESIGN.md):
 *   cons->prim + Newton T      PAPER.md:237-258 (eq 4.2-4.4), :306, :332
 *   cfl / alpha                PAPER.md:337, :292 (eq 4.11)
 *   ghost fill                 PAPER.md:295, :329, :97, :117, :213-216 (3 layers)
 *   LF split + WENO5 (JS)      PAPER.md:288-295 (eq 4.11)
 *   divergence                 PAPER.md:283-286 (eq 4.10)
 *   TVD-RK3
 *   rates, K_eq                PAPER.md:260-277 (eq 4.6-4.9)
 *   point-implicit             PAPER.md:297-304 (eq 4.12-4.13), :333, :340
 *   explicit source variant    PAPER.md:322 (source_terms advanced with the convection terms by the TVD RK3),
 *                              :338 (rhs = flux gradient + source_terms), :351-357 (advance_one_step without
 *                              advance_source_term); the source is the mechanism's own W_k omega_k of eq 4.6
 *   average-down
 *   crossover time advance     PAPER.md:186 (Fig 2a): level l at half the step of level l-1, deepest level first
 * No blocking, fusion or reordering beyond that.  OpenMP only splits independent cells/lines;
 * reductions are exact max, so results do not depend on the thread count.
 *
 * Pins: tests/test_oracle_*.py (closed forms, exact Riemann solution, conservation, finite differences, LAPACK,
 * brute force, ghost cells from global coordinates, mirrored periodic boxes; for the crossover advance and the
 * two-range thermo data see DESIGN.md section 3).  Parity unpinned: absolute accuracy of the
 * synthetic multi-step detonations (configs 1-4) -- only invariants apply there.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define RU 8.314472
#define NG 3
#define P_ATM 101325.0

enum { JREF_OK = 0, JREF_EINVAL = -1, JREF_ENOMEM = -2, JREF_ESTATE = -4, JREF_ENONFINITE = -5 };
enum { BC_PERIODIC = 0, BC_REFLECT = 1, BC_OUTFLOW = 2 };
enum { FK_NEIGHBOUR = 0, FK_PHYSICAL = 1, FK_COARSE = 2 };

typedef struct {
  int ndim;
  int n[3];
  double dx[3];
  int bc_lo[3], bc_hi[3];
  int n_patches;
  int n_levels, ratio;
} jref_grid;

typedef struct {
  int ns, nr;
  const double *W;
  const double *nasa;
  const int *nu_f, *nu_b;
  const double *A, *b, *Ta;
  const int *reversible;
  const int *third_body;
  const double *eff;
  const double *nasa_hi;   /* [ns][7] coefficients of the upper temperature range, NULL: single range (reading A7) */
  const double *T_mid;     /* [ns] switch temperature: T >= T_mid[k] uses nasa_hi[k] (Cantera-format data) */
} jref_mech;

typedef struct {
  int ns, nr;
  double *W, *nasa, *A, *b, *Ta, *eff;
  double *nasa_hi, *T_mid;     /* NULL: single range */
  int *nu_f, *nu_b, *reversible, *third_body;
} mech_t;

typedef struct jref_ctx {
  int explicit_src;            /* 1: chemical source added to the rhs of every RK stage */
  int only;                    /* -1: every level is advanced; 0 / 1: only the patches of that level (crossover advance) */
  jref_grid g;
  int np, nvar, have_mech, have_state;
  int P[3], G[3];
  long st[3], pc;
  mech_t m;
  int *level, *nbr, *parent, *fkind;
  double *U, *T, *p, *c;      /* [np][nvar][pc], [np][pc] ... */
  double *U0, *L;
  double dt_last;
  int flag;
} jref_ctx;

/* ------------------------------------------------------------------ thermo (eq 4.3-4.5) */
/* NASA-7 coefficients of species k at temperature T: the two-range form of the Cantera / Chemkin data the paper reads
 * (PAPER.md:258, :279): the upper set from T_mid upwards */
static const double *nasa_at(const mech_t *m, int k, double T) {
  return (m->nasa_hi && T >= m->T_mid[k]) ? m->nasa_hi + 7 * k : m->nasa + 7 * k;
}

static double cp_R(const mech_t *m, int k, double T) {
  const double *a = nasa_at(m, k, T);
  return a[0] + a[1] * T + a[2] * T * T + a[3] * T * T * T + a[4] * T * T * T * T;
}
static double h_R(const mech_t *m, int k, double T) { /* h_k/(Ru/W_k), eq 4.4 */
  const double *a = nasa_at(m, k, T);
  return a[0] * T + a[1] / 2 * T * T + a[2] / 3 * T * T * T + a[3] / 4 * T * T * T * T +
         a[4] / 5 * T * T * T * T * T + a[5];
}
static double s_R(const mech_t *m, int k, double T) { /* s_k/(Ru/W_k), eq 4.5 */
  const double *a = nasa_at(m, k, T);
  return a[0] * log(T) + a[1] * T + a[2] / 2 * T * T + a[3] / 3 * T * T * T +
         a[4] / 4 * T * T * T * T + a[6];
}

/* Newton-Raphson on e(T) = sum_k Y_k R_k (h_k/R_k - T) = e   (reading A6) */
static int newton_T(const mech_t *m, const double *Y, double e, double Tguess, double *Tout) {
  double T = Tguess;
  int it, conv = 0;
  for (it = 0; it < 50; it++) {
    double f = -e, cv = 0.0;
    for (int k = 0; k < m->ns; k++) {
      double Rk = RU / m->W[k];
      f += Y[k] * Rk * (h_R(m, k, T) - T);
      cv += Y[k] * Rk * (cp_R(m, k, T) - 1.0);
    }
    double dT = -f / cv;
    T += dT;
    if (fabs(dT) <= 1e-11 * fabs(T)) { conv = 1; break; }
  }
  *Tout = T;
  return conv && isfinite(T) && T > 0.0;
}

/* one cell: U -> (Y, u, T, p, gamma, c);  eq 4.2 */
static int cons2prim_cell(const mech_t *m, int ndim, const double *Uc, double Tguess, double *Y,
                          double *u, double *T, double *p, double *gam, double *c) {
  int ns = m->ns;
  double rho = Uc[0], ke = 0.0, ysum = 0.0, R = 0.0, cp = 0.0;
  for (int d = 0; d < ndim; d++) { u[d] = Uc[1 + d] / rho; ke += 0.5 * u[d] * u[d]; }
  for (int k = 0; k < ns - 1; k++) { Y[k] = Uc[ndim + 2 + k] / rho; ysum += Y[k]; }
  Y[ns - 1] = 1.0 - ysum;
  double e = (Uc[ndim + 1] - rho * ke) / rho;
  int ok = newton_T(m, Y, e, Tguess, T);
  for (int k = 0; k < ns; k++) {
    double Rk = RU / m->W[k];
    R += Y[k] * Rk;
    cp += Y[k] * Rk * cp_R(m, k, *T);
  }
  *p = rho * R * (*T);
  *gam = cp / (cp - R);
  *c = sqrt((*gam) * R * (*T));
  return ok && isfinite(*c);
}

/* ------------------------------------------------------------------ WENO5-JS (reading A1) */
static double weno5(const double *v) { /* v[0..4] = v_{-2..+2}; value at +1/2 */
  const double eps = 1e-6;
  double q0 = (2 * v[0] - 7 * v[1] + 11 * v[2]) / 6.0;
  double q1 = (-v[1] + 5 * v[2] + 2 * v[3]) / 6.0;
  double q2 = (2 * v[2] + 5 * v[3] - v[4]) / 6.0;
  double t;
  double b0, b1, b2;
  t = v[0] - 2 * v[1] + v[2]; b0 = 13.0 / 12.0 * t * t; t = v[0] - 4 * v[1] + 3 * v[2]; b0 += 0.25 * t * t;
  t = v[1] - 2 * v[2] + v[3]; b1 = 13.0 / 12.0 * t * t; t = v[1] - v[3];                b1 += 0.25 * t * t;
  t = v[2] - 2 * v[3] + v[4]; b2 = 13.0 / 12.0 * t * t; t = 3 * v[2] - 4 * v[3] + v[4]; b2 += 0.25 * t * t;
  double a0 = 0.1 / ((eps + b0) * (eps + b0));
  double a1 = 0.6 / ((eps + b1) * (eps + b1));
  double a2 = 0.3 / ((eps + b2) * (eps + b2));
  return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2);
}

/* ------------------------------------------------------------------ kinetics (eq 4.6-4.9) */
static double ipow(double x, int n) { double r = 1.0; for (int i = 0; i < n; i++) r *= x; return r; }

/* q_i and dq_i/dX_j at fixed T (readings A9, A10, A12) */
static void rates(const mech_t *m, double T, const double *X, double *q, double *dqdX) {
  int ns = m->ns, nr = m->nr;
  for (int i = 0; i < nr; i++) {
    const int *nf = m->nu_f + i * ns, *nb = m->nu_b + i * ns;
    double kf = m->A[i] * pow(T, m->b[i]) * exp(-m->Ta[i] / T);
    double kb = 0.0;
    if (m->reversible[i]) {
      double sum = 0.0; int dn = 0;
      for (int j = 0; j < ns; j++) {
        int d = nb[j] - nf[j];
        if (d) { sum += d * (s_R(m, j, T) - h_R(m, j, T) / T); dn += d; }
      }
      double Keq = exp(sum) * pow(P_ATM / (RU * T), (double)dn);
      kb = kf / Keq;
    }
    double pf = 1.0, pb = 1.0;
    for (int j = 0; j < ns; j++) { pf *= ipow(X[j], nf[j]); pb *= ipow(X[j], nb[j]); }
    double M = 1.0;
    if (m->third_body[i]) { M = 0.0; for (int j = 0; j < ns; j++) M += m->eff[i * ns + j] * X[j]; }
    double r = kf * pf - kb * pb;
    q[i] = M * r;
    for (int j = 0; j < ns; j++) {
      /* d/dX_j of prod_l X_l^nu_l = nu_j X_j^(nu_j-1) prod_{l!=j} X_l^nu_l */
      double dpf = 0.0, dpb = 0.0;
      if (nf[j] > 0) { dpf = nf[j] * ipow(X[j], nf[j] - 1); for (int l = 0; l < ns; l++) if (l != j) dpf *= ipow(X[l], nf[l]); }
      if (nb[j] > 0) { dpb = nb[j] * ipow(X[j], nb[j] - 1); for (int l = 0; l < ns; l++) if (l != j) dpb *= ipow(X[l], nb[l]); }
      double d = M * (kf * dpf - kb * dpb);
      if (m->third_body[i]) d += m->eff[i * ns + j] * r;
      dqdX[i * ns + j] = d;
    }
  }
}

/* omega_k (k < ns-1) and Jacobian d omega_k / d(rho Y_l) at fixed T, rho (reading A11) */
static void omega_jac(const mech_t *m, double T, double rho, const double *rhoY, double *omega,
                      double *J, double *work /* ns + nr + nr*ns */) {
  int ns = m->ns, nr = m->nr, n1 = ns - 1;
  double *X = work, *q = X + ns, *dq = q + nr;
  double s = 0.0;
  for (int k = 0; k < n1; k++) { X[k] = rhoY[k] / m->W[k]; s += rhoY[k]; }
  X[n1] = (rho - s) / m->W[n1];
  rates(m, T, X, q, dq);
  for (int k = 0; k < n1; k++) {
    double w = 0.0;
    for (int i = 0; i < nr; i++) w += (m->nu_b[i * ns + k] - m->nu_f[i * ns + k]) * q[i];
    omega[k] = m->W[k] * w;
    for (int l = 0; l < n1; l++) {
      double a = 0.0;
      for (int i = 0; i < nr; i++)
        a += (m->nu_b[i * ns + k] - m->nu_f[i * ns + k]) *
             (dq[i * ns + l] / m->W[l] - dq[i * ns + n1] / m->W[n1]);
      J[k * n1 + l] = m->W[k] * a;
    }
  }
}

/* Gaussian elimination with partial pivoting, A[n*n] row-major, b[n] -> x in b */
static int gauss_solve(int n, double *A, double *b) {
  for (int c = 0; c < n; c++) {
    int piv = c; double best = fabs(A[c * n + c]);
    for (int r = c + 1; r < n; r++) if (fabs(A[r * n + c]) > best) { best = fabs(A[r * n + c]); piv = r; }
    if (!(best > 0.0)) return 0;
    if (piv != c) {
      for (int j = 0; j < n; j++) { double t = A[c * n + j]; A[c * n + j] = A[piv * n + j]; A[piv * n + j] = t; }
      double t = b[c]; b[c] = b[piv]; b[piv] = t;
    }
    for (int r = c + 1; r < n; r++) {
      double f = A[r * n + c] / A[c * n + c];
      for (int j = c; j < n; j++) A[r * n + j] -= f * A[c * n + j];
      b[r] -= f * b[c];
    }
  }
  for (int r = n - 1; r >= 0; r--) {
    double s = b[r];
    for (int j = r + 1; j < n; j++) s -= A[r * n + j] * b[j];
    b[r] = s / A[r * n + r];
  }
  return 1;
}

/* (I - dt J) delta = dt omega   (eq 4.12) */
static int chem_cell(const mech_t *m, double T, double rho, const double *rhoY, double dt,
                     double *delta, double *work /* ns+nr+nr*ns + n1*n1 */) {
  int n1 = m->ns - 1;
  if (n1 == 0 || m->nr == 0) return 1;
  double *J = work + m->ns + m->nr + m->nr * m->ns;
  omega_jac(m, T, rho, rhoY, delta, J, work);
  for (int k = 0; k < n1; k++) {
    for (int l = 0; l < n1; l++) J[k * n1 + l] = (k == l ? 1.0 : 0.0) - dt * J[k * n1 + l];
    delta[k] *= dt;
  }
  return gauss_solve(n1, J, delta);
}

/* ------------------------------------------------------------------ context */
static void mech_free(mech_t *m) {
  free(m->W); free(m->nasa); free(m->A); free(m->b); free(m->Ta); free(m->eff); free(m->nasa_hi); free(m->T_mid);
  free(m->nu_f); free(m->nu_b); free(m->reversible); free(m->third_body);
  memset(m, 0, sizeof *m);
}
static void *dup_mem(const void *src, size_t bytes) {
  void *p = malloc(bytes ? bytes : 1);
  if (p && src && bytes) memcpy(p, src, bytes);
  return p;
}
static int mech_copy(mech_t *m, const jref_mech *in) {
  int ns = in->ns, nr = in->nr;
  if (ns < 1 || nr < 0) return JREF_EINVAL;
  mech_free(m);
  m->ns = ns; m->nr = nr;
  m->W = dup_mem(in->W, sizeof(double) * ns);
  m->nasa = dup_mem(in->nasa, sizeof(double) * 7 * ns);
  m->nu_f = dup_mem(in->nu_f, sizeof(int) * nr * ns);
  m->nu_b = dup_mem(in->nu_b, sizeof(int) * nr * ns);
  m->A = dup_mem(in->A, sizeof(double) * nr);
  m->b = dup_mem(in->b, sizeof(double) * nr);
  m->Ta = dup_mem(in->Ta, sizeof(double) * nr);
  m->reversible = dup_mem(in->reversible, sizeof(int) * nr);
  m->third_body = dup_mem(in->third_body, sizeof(int) * nr);
  m->nasa_hi = (in->nasa_hi && in->T_mid) ? dup_mem(in->nasa_hi, sizeof(double) * 7 * ns) : NULL;
  m->T_mid = (in->nasa_hi && in->T_mid) ? dup_mem(in->T_mid, sizeof(double) * ns) : NULL;
  m->eff = malloc(sizeof(double) * (nr * ns + 1));
  for (int i = 0; i < nr * ns; i++) m->eff[i] = in->eff ? in->eff[i] : 1.0;
  return JREF_OK;
}

int jref_create(const jref_grid *g, jref_ctx **out) {
  if (!g || !out || g->ndim < 1 || g->ndim > 3) return JREF_EINVAL;
  jref_ctx *c = calloc(1, sizeof *c);
  if (!c) return JREF_ENOMEM;
  c->g = *g;
  c->np = g->n_patches > 0 ? g->n_patches : 1;
  c->only = -1;
  if (g->n_patches <= 0) { c->g.n_levels = 1; }
  if (c->g.n_levels < 1 || c->g.n_levels > 2 || (c->g.n_levels == 2 && g->ratio != 2)) { free(c); return JREF_EINVAL; }
  c->pc = 1;
  for (int d = 0; d < 3; d++) {
    if (d < g->ndim) { if (g->n[d] < 1) { free(c); return JREF_EINVAL; } c->G[d] = NG; c->P[d] = g->n[d] + 2 * NG; }
    else { c->g.n[d] = 1; c->G[d] = 0; c->P[d] = 1; }
    c->st[d] = c->pc; c->pc *= c->P[d];
  }
  int nf = 2 * g->ndim;
  c->level = calloc(c->np, sizeof(int));
  c->nbr = malloc(sizeof(int) * c->np * nf);
  c->parent = malloc(sizeof(int) * c->np * (1 + g->ndim));
  c->fkind = malloc(sizeof(int) * c->np * nf);
  for (int i = 0; i < c->np * nf; i++) { c->nbr[i] = -1; c->fkind[i] = FK_PHYSICAL; }
  for (int i = 0; i < c->np * (1 + g->ndim); i++) c->parent[i] = -1;
  *out = c;
  return JREF_OK;
}

void jref_destroy(jref_ctx *c) {
  if (!c) return;
  mech_free(&c->m);
  free(c->level); free(c->nbr); free(c->parent); free(c->fkind);
  free(c->U); free(c->T); free(c->p); free(c->c); free(c->U0); free(c->L);
  free(c);
}

int jref_set_mechanism(jref_ctx *c, const jref_mech *in) {
  if (!c || !in) return JREF_EINVAL;
  int rc = mech_copy(&c->m, in);
  if (rc) return rc;
  c->nvar = c->g.ndim + 2 + in->ns - 1;
  size_t cells = (size_t)c->np * c->pc;
  free(c->U); free(c->T); free(c->p); free(c->c); free(c->U0); free(c->L);
  c->U = calloc(cells * c->nvar, sizeof(double));
  c->U0 = calloc(cells * c->nvar, sizeof(double));
  c->L = calloc(cells * c->nvar, sizeof(double));
  c->T = calloc(cells, sizeof(double));
  c->p = calloc(cells, sizeof(double));
  c->c = calloc(cells, sizeof(double));
  if (!c->U || !c->U0 || !c->L || !c->T || !c->p || !c->c) return JREF_ENOMEM;
  c->have_mech = 1; c->have_state = 0;
  return JREF_OK;
}

/* block lists: level[np]; nbr[np][2*ndim] (lo-x,hi-x,lo-y,...; -1 none);
 * parent[np][1+ndim] = (parent patch id, sub-region index per direction). */
int jref_set_blocks(jref_ctx *c, const int32_t *level, const int32_t *nbr, const int32_t *parent) {
  if (!c || c->g.n_patches <= 0 || !level || !nbr) return JREF_EINVAL;
  int nd = c->g.ndim, nf = 2 * nd;
  for (int p = 0; p < c->np; p++) {
    if (level[p] < 0 || level[p] >= c->g.n_levels) return JREF_EINVAL;
    c->level[p] = level[p];
    for (int f = 0; f < nf; f++) {
      int q = nbr[p * nf + f];
      if (q >= c->np || (q >= 0 && level[q] != level[p])) return JREF_EINVAL;
      c->nbr[p * nf + f] = q;
    }
    for (int e = 0; e <= nd; e++) c->parent[p * (1 + nd) + e] = parent ? parent[p * (1 + nd) + e] : -1;
    if (level[p] > 0) {
      int k = c->parent[p * (1 + nd)];
      if (k < 0 || k >= c->np || level[k] != level[p] - 1) return JREF_EINVAL;
      for (int e = 0; e < nd; e++) { int s = c->parent[p * (1 + nd) + 1 + e]; if (s < 0 || s >= c->g.ratio) return JREF_EINVAL; }
    }
  }
  /* what fills each face (readings A19, and SURVEY 8(c) step 8): same-level neighbour, else
   * (level>0) the coarse parent unless the face lies on the domain boundary, else physical BC */
  for (int p = 0; p < c->np; p++)
    for (int f = 0; f < nf; f++) {
      int kind;
      if (c->nbr[p * nf + f] >= 0) kind = FK_NEIGHBOUR;
      else if (c->level[p] == 0) kind = FK_PHYSICAL;
      else {
        int k = c->parent[p * (1 + nd)], d = f / 2, side = f % 2;
        int s = c->parent[p * (1 + nd) + 1 + d];
        int on_edge = side == 0 ? (s == 0) : (s == c->g.ratio - 1);
        kind = (on_edge && c->nbr[k * nf + f] < 0) ? FK_PHYSICAL : FK_COARSE;
      }
      c->fkind[p * nf + f] = kind;
    }
  return JREF_OK;
}

static inline long cidx(const jref_ctx *c, int i, int j, int k) {
  return (long)(i + c->G[0]) * c->st[0] + (long)(j + c->G[1]) * c->st[1] + (long)(k + c->G[2]) * c->st[2];
}

/* U: [np][nvar][nz][ny][nx] interior only, x fastest; T_guess nullable (1000 K, reading A6) */
int jref_set_state(jref_ctx *c, const double *U, const double *Tg) {
  if (!c || !U || !c->have_mech) return JREF_ESTATE;
  const int *n = c->g.n;
  long ic = (long)n[0] * n[1] * n[2];
  for (int p = 0; p < c->np; p++)
    for (int k = 0; k < n[2]; k++)
      for (int j = 0; j < n[1]; j++)
        for (int i = 0; i < n[0]; i++) {
          long s = ((long)k * n[1] + j) * n[0] + i, d = cidx(c, i, j, k);
          for (int v = 0; v < c->nvar; v++)
            c->U[((long)p * c->nvar + v) * c->pc + d] = U[((long)p * c->nvar + v) * ic + s];
          c->T[(long)p * c->pc + d] = Tg ? Tg[(long)p * ic + s] : 1000.0;
        }
  c->have_state = 1; c->flag = 0;
  return JREF_OK;
}

int jref_get_state(jref_ctx *c, double *U, double *T) {
  if (!c || !c->have_state) return JREF_ESTATE;
  const int *n = c->g.n;
  long ic = (long)n[0] * n[1] * n[2];
  for (int p = 0; p < c->np; p++)
    for (int k = 0; k < n[2]; k++)
      for (int j = 0; j < n[1]; j++)
        for (int i = 0; i < n[0]; i++) {
          long s = ((long)k * n[1] + j) * n[0] + i, d = cidx(c, i, j, k);
          if (U) for (int v = 0; v < c->nvar; v++)
            U[((long)p * c->nvar + v) * ic + s] = c->U[((long)p * c->nvar + v) * c->pc + d];
          if (T) T[(long)p * ic + s] = c->T[(long)p * c->pc + d];
        }
  return c->flag ? JREF_ENONFINITE : JREF_OK;
}

/* ------------------------------------------------------------------ step pieces */
/* cons->prim on the cells of every patch.  ghosts=0: interior only; 1: also face ghosts
 * (cells with exactly one index in the ghost range; corners are never read, reading A21).
 * Returns per-level, per-direction max(|u_d|+c) over INTERIOR cells (reading A3, A20). */
static void prim_all(jref_ctx *c, double *U, int ghosts, double smax[2][3]) {
  const int *n = c->g.n; int nd = c->g.ndim, ns = c->m.ns;
  for (int l = 0; l < 2; l++) for (int d = 0; d < 3; d++) smax[l][d] = 0.0;
  int bad = 0;
  for (int p = 0; p < c->np; p++) {
    int lev = c->level[p];
    if (c->only >= 0 && lev != c->only) continue;      /* crossover advance: one level at a time */
    double s0 = 0, s1 = 0, s2 = 0;
    int glo[3], ghi[3];
    for (int d = 0; d < 3; d++) { glo[d] = ghosts ? -c->G[d] : 0; ghi[d] = n[d] + (ghosts ? c->G[d] : 0); }
#pragma omp parallel for collapse(2) reduction(max : s0, s1, s2) reduction(| : bad) schedule(static)
    for (int k = glo[2]; k < ghi[2]; k++)
      for (int j = glo[1]; j < ghi[1]; j++) {
        double Y[64], u[3] = {0, 0, 0}, Uc[80];
        for (int i = glo[0]; i < ghi[0]; i++) {
          int og = (i < 0 || i >= n[0]) + (j < 0 || j >= n[1]) + (k < 0 || k >= n[2]);
          if (og > 1) continue;
          long id = cidx(c, i, j, k);
          for (int v = 0; v < c->nvar; v++) Uc[v] = U[((long)p * c->nvar + v) * c->pc + id];
          double T, pr, gam, cs;
          int ok = cons2prim_cell(&c->m, nd, Uc, c->T[(long)p * c->pc + id], Y, u, &T, &pr, &gam, &cs);
          c->T[(long)p * c->pc + id] = T; c->p[(long)p * c->pc + id] = pr; c->c[(long)p * c->pc + id] = cs;
          if (og == 0) {
            if (!ok) bad |= 1;
            double a;
            a = fabs(u[0]) + cs; if (a > s0) s0 = a;
            if (nd > 1) { a = fabs(u[1]) + cs; if (a > s1) s1 = a; }
            if (nd > 2) { a = fabs(u[2]) + cs; if (a > s2) s2 = a; }
          }
        }
      }
    (void)ns;
    if (s0 > smax[lev][0]) smax[lev][0] = s0;
    if (s1 > smax[lev][1]) smax[lev][1] = s1;
    if (s2 > smax[lev][2]) smax[lev][2] = s2;
  }
  if (bad) c->flag = 1;
}

static int floordiv(int a, int b) { int q = a / b; if ((a % b != 0) && ((a < 0) != (b < 0))) q--; return q; }

/* fill the 3 ghost layers of U and of the T guess on every face */
static void ghost_fill(jref_ctx *c, double *U) {
  const int *n = c->g.n; int nd = c->g.ndim, nf = 2 * nd, nv = c->nvar;
  for (int lev = 0; lev < c->g.n_levels; lev++)      /* level 0 first: level 1 injects from its padded parent */
    for (int p = 0; p < c->np; p++) {
      if (c->level[p] != lev) continue;
      if (c->only >= 0 && lev != c->only && !(lev == 0 && c->only == 1)) continue;   /* the fine level still needs its parents' ghosts */
      for (int d = 0; d < nd; d++)
        for (int side = 0; side < 2; side++) {
          int f = 2 * d + side, kind = c->fkind[p * nf + f];
          int bc = side == 0 ? c->g.bc_lo[d] : c->g.bc_hi[d];
          int lo[3] = {0, 0, 0}, hi[3] = {n[0], n[1], n[2]};
          for (int g = 1; g <= NG; g++) {
            lo[d] = side == 0 ? -g : n[d] - 1 + g; hi[d] = lo[d] + 1;
            for (int k = lo[2]; k < hi[2]; k++)
              for (int j = lo[1]; j < hi[1]; j++)
                for (int i = lo[0]; i < hi[0]; i++) {
                  int dst[3] = {i, j, k}, src[3] = {i, j, k};
                  int q = p; double sign = 1.0;
                  if (kind == FK_NEIGHBOUR || (kind == FK_PHYSICAL && bc == BC_PERIODIC)) {
                    if (kind == FK_NEIGHBOUR) q = c->nbr[p * nf + f];
                    src[d] = side == 0 ? n[d] - g : g - 1;
                  } else if (kind == FK_PHYSICAL && bc == BC_REFLECT) {   /* reading A15 */
                    src[d] = side == 0 ? g - 1 : n[d] - g; sign = -1.0;
                  } else if (kind == FK_PHYSICAL) {                        /* outflow, reading A14 */
                    src[d] = side == 0 ? 0 : n[d] - 1;
                  } else {                                                 /* coarse parent, one-to-four */
                    q = c->parent[p * (1 + nd)];
                    for (int e = 0; e < nd; e++)
                      src[e] = floordiv(c->parent[p * (1 + nd) + 1 + e] * n[e] + dst[e], c->g.ratio);
                  }
                  long di = cidx(c, dst[0], dst[1], dst[2]), si = cidx(c, src[0], src[1], src[2]);
                  for (int v = 0; v < nv; v++) {
                    double val = U[((long)q * nv + v) * c->pc + si];
                    if (v == 1 + d) val *= sign;
                    U[((long)p * nv + v) * c->pc + di] = val;
                  }
                  c->T[(long)p * c->pc + di] = c->T[(long)q * c->pc + si];
                }
          }
        }
    }
}

/* split fluxes f+ and f- of direction d at one cell (eq 4.11; F of PAPER.md:232) */
static void split_flux_cell(const jref_ctx *c, const double *U, int p, long id, int d, double alpha,
                            double *fp, double *fm) {
  int nd = c->g.ndim, nv = c->nvar;
  const double *Up = U + (long)p * nv * c->pc;
  double rho = Up[id], pr = c->p[(long)p * c->pc + id];
  double ud = Up[(long)(1 + d) * c->pc + id] / rho;
  for (int v = 0; v < nv; v++) {
    double Uv = Up[(long)v * c->pc + id], F;
    if (v == 0) F = Up[(long)(1 + d) * c->pc + id];
    else if (v <= nd) F = Uv * ud + (v == 1 + d ? pr : 0.0);
    else if (v == nd + 1) F = ud * (Uv + pr);
    else F = Uv * ud;
    fp[v] = 0.5 * (F + alpha * Uv);
    fm[v] = 0.5 * (F - alpha * Uv);
  }
}

/* L = - sum_d (Fhat_{+1/2} - Fhat_{-1/2}) / dx_d on interior cells (eq 4.10) */
static void flux_divergence(jref_ctx *c, const double *U, double alpha[2][3], double *L) {
  const int *n = c->g.n; int nd = c->g.ndim, nv = c->nvar;
  memset(L, 0, sizeof(double) * (size_t)c->np * nv * c->pc);
  for (int p = 0; p < c->np; p++) {
    int lev = c->level[p];
    if (c->only >= 0 && lev != c->only) continue;
    for (int d = 0; d < nd; d++) {
      double dx = c->g.dx[d]; for (int l = 0; l < lev; l++) dx /= c->g.ratio;
      double al = alpha[lev][d];
      int e1 = (d + 1) % 3, e2 = (d + 2) % 3;
#pragma omp parallel
      {
        double *Fh = malloc(sizeof(double) * (n[d] + 1) * nv);
        double *fp = malloc(sizeof(double) * 6 * nv), *fm = malloc(sizeof(double) * 6 * nv);
#pragma omp for collapse(2) schedule(static)
        for (int b = 0; b < n[e2]; b++)
          for (int a = 0; a < n[e1]; a++) {
            int ix[3]; ix[e1] = a; ix[e2] = b;
            for (int f = 0; f <= n[d]; f++) {         /* face between cells f-1 and f */
              for (int s = 0; s < 6; s++) {           /* cells f-3 .. f+2 */
                ix[d] = f - 3 + s;
                split_flux_cell(c, U, p, cidx(c, ix[0], ix[1], ix[2]), d, al, fp + s * nv, fm + s * nv);
              }
              for (int v = 0; v < nv; v++) {
                double vp[5], vm[5];
                for (int s = 0; s < 5; s++) { vp[s] = fp[s * nv + v]; vm[s] = fm[(5 - s) * nv + v]; }
                Fh[f * nv + v] = weno5(vp) + weno5(vm);
              }
            }
            for (int i = 0; i < n[d]; i++) {
              ix[d] = i;
              long id = cidx(c, ix[0], ix[1], ix[2]);
              for (int v = 0; v < nv; v++)
                L[((long)p * nv + v) * c->pc + id] -= (Fh[(i + 1) * nv + v] - Fh[i * nv + v]) / dx;
            }
          }
        free(Fh); free(fp); free(fm);
      }
    }
  }
}

/* rhs of PAPER.md:338: ghost fill -> update_aux -> flux gradient */
static void source_terms(jref_ctx *c, const double *U, double *L);

static void rhs(jref_ctx *c, double *U, double *L) {
  double s[2][3];
  ghost_fill(c, U);
  prim_all(c, U, 1, s);
  flux_divergence(c, U, s, L);
  if (c->explicit_src) source_terms(c, U, L);
}

static void chemistry(jref_ctx *c, double dt) {
  const int *n = c->g.n; int nd = c->g.ndim, nv = c->nvar, ns = c->m.ns, n1 = ns - 1;
  if (n1 == 0 || c->m.nr == 0) return;
  int bad = 0;
  for (int p = 0; p < c->np; p++) {
    if (c->only >= 0 && c->level[p] != c->only) continue;
#pragma omp parallel
    {
      double *work = malloc(sizeof(double) * (ns + c->m.nr + c->m.nr * ns + n1 * n1 + 2 * n1));
      double *ry = work + ns + c->m.nr + c->m.nr * ns + n1 * n1, *dl = ry + n1;
#pragma omp for collapse(2) reduction(| : bad) schedule(static)
      for (int k = 0; k < n[2]; k++)
        for (int j = 0; j < n[1]; j++)
          for (int i = 0; i < n[0]; i++) {
            long id = cidx(c, i, j, k);
            double *Up = c->U + (long)p * nv * c->pc;
            for (int s = 0; s < n1; s++) ry[s] = Up[(long)(nd + 2 + s) * c->pc + id];
            int ok = chem_cell(&c->m, c->T[(long)p * c->pc + id], Up[id], ry, dt, dl, work);
            for (int s = 0; s < n1; s++) {
              Up[(long)(nd + 2 + s) * c->pc + id] = ry[s] + dl[s];
              if (!isfinite(dl[s])) ok = 0;
            }
            if (!ok) bad |= 1;
          }
      free(work);
    }
  }
  if (bad) c->flag = 1;
}

/* four-to-one arithmetic mean onto covered coarse cells */
static void average_down(jref_ctx *c) {
  const int *n = c->g.n; int nd = c->g.ndim, nv = c->nvar, r = c->g.ratio;
  if (c->g.n_levels < 2) return;
  int rr[3] = {r, nd > 1 ? r : 1, nd > 2 ? r : 1};
  double w = 1.0 / (rr[0] * rr[1] * rr[2]);
  for (int p = 0; p < c->np; p++) {
    if (c->level[p] == 0) continue;
    int q = c->parent[p * (1 + nd)];
    int off[3] = {0, 0, 0};
    for (int e = 0; e < nd; e++) off[e] = c->parent[p * (1 + nd) + 1 + e] * (n[e] / r);
    for (int v = 0; v < nv; v++)
      for (int k = 0; k < n[2] / rr[2]; k++)
        for (int j = 0; j < n[1] / rr[1]; j++)
          for (int i = 0; i < n[0] / rr[0]; i++) {
            double s = 0.0;
            for (int kk = 0; kk < rr[2]; kk++)
              for (int jj = 0; jj < rr[1]; jj++)
                for (int ii = 0; ii < rr[0]; ii++)
                  s += c->U[((long)p * nv + v) * c->pc + cidx(c, i * rr[0] + ii, j * rr[1] + jj, k * rr[2] + kk)];
            c->U[((long)q * nv + v) * c->pc + cidx(c, off[0] + i, off[1] + j, off[2] + k)] = s * w;
          }
  }
}

/* aux_func.source_terms of the explicit variant: S_k = W_k omega_k(T, X) of eq 4.6-4.9 on the
 * species rows, evaluated on the stage state with the temperature update_aux has just recovered; added to L. */
static void source_terms(jref_ctx *c, const double *U, double *L) {
  const int *n = c->g.n; int nd = c->g.ndim, nv = c->nvar, ns = c->m.ns, n1 = ns - 1, nr = c->m.nr;
  if (n1 < 1 || nr < 1) return;
  for (int p = 0; p < c->np; p++) {
    if (c->only >= 0 && c->level[p] != c->only) continue;
    const double *Up = U + (long)p * nv * c->pc;
#pragma omp parallel
    {
      double *work = malloc(sizeof(double) * (size_t)(ns + nr + nr * ns));
      double *ry = malloc(sizeof(double) * ns), *om = malloc(sizeof(double) * ns), *J = malloc(sizeof(double) * (size_t)n1 * n1);
#pragma omp for collapse(2) schedule(static)
      for (int k = 0; k < n[2]; k++)
        for (int j = 0; j < n[1]; j++)
          for (int i = 0; i < n[0]; i++) {
            long id = cidx(c, i, j, k);
            for (int q = 0; q < n1; q++) ry[q] = Up[(long)(nd + 2 + q) * c->pc + id];
            omega_jac(&c->m, c->T[(long)p * c->pc + id], Up[id], ry, om, J, work);
            for (int q = 0; q < n1; q++) L[((long)p * nv + nd + 2 + q) * c->pc + id] += om[q];
          }
      free(work); free(ry); free(om); free(J);
    }
  }
}

/* advance_flux + advance_source_term of the patches selected by c->only over one step dt */
static void advance(jref_ctx *c, double dt, int do_chem) {
  size_t N = (size_t)c->np * c->nvar * c->pc;
  double s[2][3];
  memcpy(c->U0, c->U, N * sizeof(double));
  /* Shu-Osher SSP-RK3 in increment form (readings A4); L = 0 on patches that are not selected: they keep their state */
  rhs(c, c->U, c->L);
  for (size_t i = 0; i < N; i++) c->U[i] = c->U0[i] + dt * c->L[i];
  rhs(c, c->U, c->L);
  for (size_t i = 0; i < N; i++) c->U[i] = c->U0[i] + 0.25 * ((c->U[i] - c->U0[i]) + dt * c->L[i]);
  rhs(c, c->U, c->L);
  for (size_t i = 0; i < N; i++) c->U[i] = c->U0[i] + (2.0 / 3.0) * ((c->U[i] - c->U0[i]) + dt * c->L[i]);
  /* advance_source_term: update_aux -> solve_implicit_rate -> U + dU */
  prim_all(c, c->U, 0, s);
  if (do_chem == 1) chemistry(c, dt);
}

/* advance_one_step: CFL -> advance_flux (RK3) -> advance_source_term.
 * mode & 3: 0 no chemistry, 1 point-implicit after the RK3, 2 explicit: source inside every RK stage
 *           and no advance_source_term.
 * mode & 4: crossover time advance of a two-level block list (Fig 2a; reading B9): the step of
 *           a level is half that of the previous level and the deepest level is solved first -- two steps dt/2 of level
 *           1, its coarse-fine ghosts injected from the level-0 state at the START of the step (level 0 has not moved
 *           yet), then one step dt of level 0, then interpolate_fine_to_coarse.  dt = CFL * min dx(level 0) / max(|u|+c)
 *           (twice the synchronous step: both levels run at the same CFL number); cfl <= 0: dt_fixed is the level-0 step.
 *           Without the bit: synchronous advance, every level at the finest level's step (PAPER.md:186 Fig 2b, :460). */
int jref_step(jref_ctx *c, int nsteps, double cfl, double dt_fixed, int mode, double *t_adv) {
  if (!c || !c->have_state) return JREF_ESTATE;
  const int do_chem = mode & 3, crossover = (mode & 4) && c->g.n_levels == 2;
  c->explicit_src = do_chem == 2;
  double t = 0.0, s[2][3];
  for (int it = 0; it < nsteps; it++) {
    double dt = dt_fixed;
    if (cfl > 0.0) {                                   /* cfl(), reading A16/A17 */
      prim_all(c, c->U, 0, s);
      double smax = 0.0, dxmin = 1e300;
      for (int l = 0; l < 2; l++) for (int d = 0; d < c->g.ndim; d++) if (s[l][d] > smax) smax = s[l][d];
      for (int d = 0; d < c->g.ndim; d++) {
        double dx = c->g.dx[d];
        if (!crossover) for (int l = 1; l < c->g.n_levels; l++) dx /= c->g.ratio;
        if (dx < dxmin) dxmin = dx;
      }
      dt = cfl * dxmin / smax;
    }
    c->dt_last = dt;
    if (crossover) {
      c->only = 1; advance(c, 0.5 * dt, do_chem); advance(c, 0.5 * dt, do_chem);
      c->only = 0; advance(c, dt, do_chem);
      c->only = -1;
    } else {
      advance(c, dt, do_chem);
    }
    average_down(c);
    t += dt;
  }
  if (t_adv) *t_adv = t;
  return c->flag ? JREF_ENONFINITE : JREF_OK;
}

double jref_last_dt(const jref_ctx *c) { return c ? c->dt_last : 0.0; }

/* ------------------------------------------------------------------ fine-grained entry points (pins) */
double jref_weno5(const double *v) { return weno5(v); }

int jref_cons2prim(const jref_mech *in, int ndim, const double *Uc, double Tguess, double *out /* T,p,gamma,c */) {
  mech_t m; memset(&m, 0, sizeof m);
  if (mech_copy(&m, in)) return JREF_EINVAL;
  double Y[64], u[3];
  int ok = cons2prim_cell(&m, ndim, Uc, Tguess, Y, u, out, out + 1, out + 2, out + 3);
  mech_free(&m);
  return ok ? JREF_OK : JREF_ENONFINITE;
}

int jref_omega_jac(const jref_mech *in, double T, double rho, const double *rhoY, double *omega, double *J) {
  mech_t m; memset(&m, 0, sizeof m);
  if (mech_copy(&m, in)) return JREF_EINVAL;
  double *work = malloc(sizeof(double) * (m.ns + m.nr + m.nr * m.ns + 1));
  omega_jac(&m, T, rho, rhoY, omega, J, work);
  free(work); mech_free(&m);
  return JREF_OK;
}

/* rate of progress q_i of each reaction at (T, X[ns]) -- eq 4.7's bracket */
int jref_rates(const jref_mech *in, double T, const double *X, double *q) {
  mech_t m; memset(&m, 0, sizeof m);
  if (mech_copy(&m, in)) return JREF_EINVAL;
  double *dq = malloc(sizeof(double) * (m.nr * m.ns + 1));
  rates(&m, T, X, q, dq);
  free(dq); mech_free(&m);
  return JREF_OK;
}

int jref_chem_cell(const jref_mech *in, double T, double rho, const double *rhoY, double dt, double *delta) {
  mech_t m; memset(&m, 0, sizeof m);
  if (mech_copy(&m, in)) return JREF_EINVAL;
  int n1 = m.ns - 1;
  double *work = malloc(sizeof(double) * (m.ns + m.nr + m.nr * m.ns + n1 * n1 + 1));
  int ok = chem_cell(&m, T, rho, rhoY, dt, delta, work);
  free(work); mech_free(&m);
  return ok ? JREF_OK : JREF_ENONFINITE;
}

/* The same per-cell update (update_aux -> solve_implicit_rate) on a list of cells: Uc[ncell][nvar]
 * (cell-major), Tguess[ncell] -> delta[ncell][ns-1], Tout[ncell].  Cells are independent; OpenMP over cells. */
int jref_chem_cells(const jref_mech *in, int ndim, long ncell, const double *Uc, const double *Tguess, double dt,
                    double *delta, double *Tout) {
  mech_t m; memset(&m, 0, sizeof m);
  if (mech_copy(&m, in)) return JREF_EINVAL;
  int ns = m.ns, n1 = ns - 1, nvar = ndim + 2 + n1, bad = 0;
#pragma omp parallel
  {
    double *work = malloc(sizeof(double) * (size_t)(ns + m.nr + m.nr * ns + n1 * n1 + 1));
#pragma omp for reduction(| : bad) schedule(static)
    for (long i = 0; i < ncell; i++) {
      double Y[64], u[3], T, p, gam, cs;
      const double *U = Uc + i * nvar;
      int ok = cons2prim_cell(&m, ndim, U, Tguess[i], Y, u, &T, &p, &gam, &cs);
      ok &= chem_cell(&m, T, U[0], U + ndim + 2, dt, delta + i * n1, work);
      Tout[i] = T;
      if (!ok) bad |= 1;
    }
    free(work);
  }
  mech_free(&m);
  return bad ? JREF_ENONFINITE : JREF_OK;
}

int jref_gauss_solve(int n, double *A, double *b) { return gauss_solve(n, A, b) ? JREF_OK : JREF_ENONFINITE; }

/* Pin support: run ghost_fill on the current state and return the padded arrays (ghosts included),
 * Upad[np][nvar][pc] with pc = prod_d (n_d + 6), x fastest; Tpad[np][pc] nullable. */
int jref_debug_ghost_fill(jref_ctx *c, double *Upad, double *Tpad) {
  if (!c || !c->have_state || !Upad) return JREF_ESTATE;
  ghost_fill(c, c->U);
  memcpy(Upad, c->U, sizeof(double) * (size_t)c->np * c->nvar * c->pc);
  if (Tpad) memcpy(Tpad, c->T, sizeof(double) * (size_t)c->np * c->pc);
  return JREF_OK;
}

/* thread control for the timed baseline (results do not depend on it) */
int jref_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n; return 1;
#endif
}

/* ------------------------------------------------------------------ regridding (JAX-AMR "update refinement layer")
 * PAPER.md:73-75 (refinement criterion mask + buffer cells -> blocks to refine), :123 (update of the refinement layer
 * keeps the data of blocks with the same global index), :175-184 (get_refinement_grid_mask, get_refinement_block_mask,
 * get_refinement_block_info, get_refinement_block_data, find_and_update_unaltered_block), :115 (one-to-four).
 * Two levels, ratio 2; the level-0 patches are the first n0 entries of the list and tile the domain.  DESIGN.md reading
 * B12:
 *   1. mask (level-0 cells): max_d |rho(i + e_d) - rho(i - e_d)| / (2 rho(i)) > thr, on the level-0 state (covered cells
 *      hold the average of their fine cells) with its ghost layers filled;
 *   2. buffer: every cell within nbuf cells (in every direction: a box) of a masked cell is marked too, across patch
 *      boundaries and periodic sides, not across walls / outflow sides;
 *   3. a sub-region (level-0 patch k, sub-index s in {0,1}^ndim) is refined if it contains a marked cell;
 *   4. the new level-1 list follows the level-0 patches, ordered by parent, sub-index x fastest; same-level neighbours
 *      through the parents' neighbour lists;
 *   5. data: a block that existed before (same parent and sub-index) keeps its data, a new one is the one-to-four
 *      injection of its parent's sub-region (T likewise).
 * Outputs (caller-allocated for the worst case n0 (1 + 2^ndim) patches): level, nbr [2 ndim], parent [1 + ndim] per
 * patch; Unew [np_new][nvar][cells], Tnew [np_new][cells] in the interior layout of jref_set_state. */
int jref_regrid(jref_ctx *c, double thr, int nbuf, int *np_new, int32_t *level, int32_t *nbr, int32_t *parent,
                double *Unew, double *Tnew) {
  if (!c || !c->have_state || c->g.n_patches <= 0 || c->g.n_levels != 2 || nbuf < 0 || nbuf > 64) return JREF_EINVAL;
  const int nd = c->g.ndim, nf = 2 * nd, nv = c->nvar, nsub = 1 << nd;
  const int *n = c->g.n;
  int n0 = 0;
  while (n0 < c->np && c->level[n0] == 0) n0++;
  for (int p = n0; p < c->np; p++) if (c->level[p] != 1) return JREF_EINVAL;       /* level-0 patches first */
  const long ic = (long)n[0] * n[1] * n[2];
  /* 1. mask on the padded level-0 arrays (ghosts filled from neighbours / physical sides) */
  ghost_fill(c, c->U);
  unsigned char *mark = calloc((size_t)n0 * c->pc, 1), *tmp = calloc((size_t)n0 * c->pc, 1);
  if (!mark || !tmp) { free(mark); free(tmp); return JREF_ENOMEM; }
  for (int p = 0; p < n0; p++)
    for (int k = 0; k < n[2]; k++) for (int j = 0; j < n[1]; j++) for (int i = 0; i < n[0]; i++) {
      const double *rho = c->U + (long)p * nv * c->pc;
      long id = cidx(c, i, j, k);
      double g = 0.0;
      for (int d = 0; d < nd; d++) {
        double a = fabs(rho[id + c->st[d]] - rho[id - c->st[d]]) / (2.0 * rho[id]);
        if (a > g) g = a;
      }
      mark[(long)p * c->pc + id] = g > thr;
    }
  /* 2. buffer: nbuf passes of a one-cell box dilation; a pass reads the marks of neighbouring patches through a
   *    ghost layer of marks filled by the same neighbour rule (periodic sides wrap, other physical sides contribute 0) */
  for (int pass = 0; pass < nbuf; pass++) {
    /* ghost marks, one layer, direction by direction so that edge / corner cells arrive after nd sweeps */
    for (int d = 0; d < nd; d++)
      for (int p = 0; p < n0; p++)
        for (int side = 0; side < 2; side++) {
          int f = 2 * d + side, q = c->nbr[p * nf + f];
          int bc = side == 0 ? c->g.bc_lo[d] : c->g.bc_hi[d];
          if (q < 0 && bc == BC_PERIODIC) q = p;                     /* single patch across a periodic direction */
          int lo[3] = {0, 0, 0}, hi[3] = {n[0], n[1], n[2]};
          for (int e = 0; e < d; e++) { lo[e] = -1; hi[e] = n[e] + 1; }   /* include the ghost marks of earlier sweeps */
          lo[d] = side == 0 ? -1 : n[d]; hi[d] = lo[d] + 1;
          for (int k = lo[2]; k < hi[2]; k++) for (int j = lo[1]; j < hi[1]; j++) for (int i = lo[0]; i < hi[0]; i++) {
            int src[3] = {i, j, k};
            src[d] = side == 0 ? n[d] - 1 : 0;
            unsigned char v = 0;
            if (q >= 0 && (c->nbr[p * nf + f] >= 0 || bc == BC_PERIODIC)) v = mark[(long)q * c->pc + cidx(c, src[0], src[1], src[2])];
            mark[(long)p * c->pc + cidx(c, i, j, k)] = v;
          }
        }
    memcpy(tmp, mark, (size_t)n0 * c->pc);
    for (int p = 0; p < n0; p++)
      for (int k = 0; k < n[2]; k++) for (int j = 0; j < n[1]; j++) for (int i = 0; i < n[0]; i++) {
        unsigned char v = 0;
        for (int dk = (nd > 2 ? -1 : 0); dk <= (nd > 2 ? 1 : 0); dk++)
          for (int dj = (nd > 1 ? -1 : 0); dj <= (nd > 1 ? 1 : 0); dj++)
            for (int di = -1; di <= 1; di++) v |= tmp[(long)p * c->pc + cidx(c, i + di, j + dj, k + dk)];
        mark[(long)p * c->pc + cidx(c, i, j, k)] = v;
      }
  }
  free(tmp);
  /* 3. sub-regions that hold a marked cell */
  unsigned char *flag = calloc((size_t)n0 * nsub, 1);
  int *newid = malloc(sizeof(int) * (size_t)n0 * nsub), *oldid = malloc(sizeof(int) * (size_t)n0 * nsub);
  for (int p = 0; p < n0; p++)
    for (int k = 0; k < n[2]; k++) for (int j = 0; j < n[1]; j++) for (int i = 0; i < n[0]; i++)
      if (mark[(long)p * c->pc + cidx(c, i, j, k)]) {
        int s = (i >= n[0] / 2 ? 1 : 0) + (nd > 1 && j >= n[1] / 2 ? 2 : 0) + (nd > 2 && k >= n[2] / 2 ? 4 : 0);
        flag[p * nsub + s] = 1;
      }
  free(mark);
  /* 4. the new list */
  for (int q = 0; q < n0 * nsub; q++) { newid[q] = -1; oldid[q] = -1; }
  for (int p = n0; p < c->np; p++) {
    const int *par = c->parent + p * (1 + nd);
    int s = par[1] + (nd > 1 ? 2 * par[2] : 0) + (nd > 2 ? 4 * par[3] : 0);
    oldid[par[0] * nsub + s] = p;
  }
  int np2 = n0;
  for (int p = 0; p < n0; p++) for (int s = 0; s < nsub; s++) if (flag[p * nsub + s]) newid[p * nsub + s] = np2++;
  for (int p = 0; p < n0; p++) {
    level[p] = 0;
    for (int f = 0; f < nf; f++) nbr[p * nf + f] = c->nbr[p * nf + f];
    for (int e = 0; e <= nd; e++) parent[p * (1 + nd) + e] = -1;
  }
  for (int p = 0; p < n0; p++) for (int s = 0; s < nsub; s++) {
    int id = newid[p * nsub + s];
    if (id < 0) continue;
    level[id] = 1;
    parent[id * (1 + nd)] = p;
    for (int e = 0; e < nd; e++) parent[id * (1 + nd) + 1 + e] = (s >> e) & 1;
    for (int d = 0; d < nd; d++) for (int side = 0; side < 2; side++) {
      int sd = (s >> d) & 1, k2 = p, s2;
      if ((side == 0 && sd == 1) || (side == 1 && sd == 0)) s2 = s ^ (1 << d);            /* the sibling inside the parent */
      else { k2 = c->nbr[p * nf + 2 * d + side]; s2 = s ^ (1 << d); }                    /* across the parent's face */
      nbr[id * nf + 2 * d + side] = k2 >= 0 ? newid[k2 * nsub + s2] : -1;
    }
  }
  /* 5. data: level 0 as it is; level 1 carried over or injected */
  for (int p = 0; p < np2; p++) {
    int src = -1, par = -1, sub[3] = {0, 0, 0};
    if (p < n0) src = p;
    else {
      par = parent[p * (1 + nd)];
      for (int e = 0; e < nd; e++) sub[e] = parent[p * (1 + nd) + 1 + e];
      src = oldid[par * nsub + sub[0] + 2 * sub[1] + 4 * sub[2]];
    }
    for (int k = 0; k < n[2]; k++) for (int j = 0; j < n[1]; j++) for (int i = 0; i < n[0]; i++) {
      long o = ((long)k * n[1] + j) * n[0] + i, sid; int q;
      if (src >= 0) { q = src; sid = cidx(c, i, j, k); }
      else {                                            /* one-to-four: the coarse cell that contains this fine cell */
        q = par;
        sid = cidx(c, (sub[0] * n[0] + i) / 2, nd > 1 ? (sub[1] * n[1] + j) / 2 : 0, nd > 2 ? (sub[2] * n[2] + k) / 2 : 0);
      }
      for (int v = 0; v < nv; v++) Unew[((long)p * nv + v) * ic + o] = c->U[((long)q * nv + v) * c->pc + sid];
      Tnew[(long)p * ic + o] = c->T[(long)q * c->pc + sid];
    }
  }
  free(flag); free(newid); free(oldid);
  *np_new = np2;
  return JREF_OK;
}
