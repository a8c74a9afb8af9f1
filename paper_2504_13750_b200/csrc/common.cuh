// common.cuh -- shared definitions of the libjanc CUDA path (sm_100a, fp64).
// Independent of oracle/: nothing here is included by, or includes, the CPU oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define JANC_NG 3            // ghost layers
#define JANC_MAX_NS 32
#define JANC_MAX_NR 128
#define JANC_MAX_ORDER 6     // sum of stoichiometric coefficients on one side of a reaction
#define JANC_RU 8.314472
#define JANC_PATM 101325.0   // eq 4.9

#define JANC_MAX_TB 32       // third-body reactions
#define JANC_MAX_ENT 768     // sum over reactions of (reactant + product entries with multiplicity)

enum { FK_NEIGHBOUR = 0, FK_PHYSICAL = 1, FK_COARSE = 2 };

// One term of dq_i/dX_j (product rule on eq 4.7): +-(M k) * prod of the other species of that side.
struct DqEntry {
  unsigned char rx, side, nother, pad;
  unsigned char other[JANC_MAX_ORDER - 1];
  unsigned char pad2[3];
};

// Mechanism in constant memory (eq 4.3-4.9).  Reactant / product lists are expanded with
// multiplicity: prod_j X_j^nu_ij = prod_e X[sp[e]].
struct MechC {
  int ns, nr;
  double W[JANC_MAX_NS], invW[JANC_MAX_NS], Rk[JANC_MAX_NS];
  double nasa[JANC_MAX_NS][7];
  double nasa_hi[JANC_MAX_NS][7];            // two-range data: upper set, used from Tmid[k] upwards (two_range != 0)
  double Tmid[JANC_MAX_NS];
  int two_range;
  double lnA[JANC_MAX_NR], b[JANC_MAX_NR], Ta[JANC_MAX_NR];
  double Asign[JANC_MAX_NR];                 // sign(A) (A may not be <= 0; kept for safety: +1)
  signed char rev[JANC_MAX_NR], tb[JANC_MAX_NR], dn[JANC_MAX_NR];
  unsigned char nreac[JANC_MAX_NR], nprod[JANC_MAX_NR];
  unsigned char reac[JANC_MAX_NR][JANC_MAX_ORDER], prod[JANC_MAX_NR][JANC_MAX_ORDER];
  unsigned char tbi[JANC_MAX_NR];            // row of eff[] for a third-body reaction
  int ntb;
  double eff[JANC_MAX_TB][JANC_MAX_NS];      // a_ij of eq 4.7, third-body reactions only
  // tables of the register-resident chemistry kernel (chem.cuh, k_chem_reg)
  double dnu[JANC_MAX_NR][JANC_MAX_NS];      // nu^b - nu^f as doubles (dense rows, static row index)
  int col_start[JANC_MAX_NS + 1];            // derivative entries grouped by species column
  int nent;
  DqEntry ent[JANC_MAX_ENT];
};

// Geometry + device pointers handed to every kernel by value.
struct Params {
  int ndim, nvar, ns, np, nlev, ratio;
  int patch0;        // first patch the kernel acts on (block y + patch0); crossover advance: one level at a time
  double dt_scale;   // the step of this launch = scal[0] * dt_scale (crossover advance: 1/2 on level 1)
  int n[3];          // interior cells per patch
  int P[3];          // padded dims
  int G[3];          // ghost width per dim (3 or 0)
  long long st[3];   // strides in doubles
  long long pc;      // padded cells per patch
  double invdx[2][3];
  double dxmin;
  int bc_lo[3], bc_hi[3];
  // device arrays
  double *T, *p, *vel;        // [np][pc], [np][pc], [ndim][np][pc]
  const int *level, *nbr, *parent, *fkind;
  unsigned long long *slots;  // [2 parity][2 sub-step][3 stage][2 lev][3 dir] ordered-int max(|u_d|+c)
  double *scal;               // [0]=dt, [1]=t accumulated
  int *flag;                  // device error flag
};

#define JANC_NSLOT 72        // per parity: 36 = 2 sub-steps (crossover advance: level 1 takes two) x 3 stages x 2 levels x 3 directions
#define SLOTX(par, sub, stage, lev, d) (((((par) * 2 + (sub)) * 3 + (stage)) * 2 + (lev)) * 3 + (d))
#define SLOT(par, stage, lev, d) SLOTX(par, 0, stage, lev, d)

__device__ __forceinline__ long long cell_index(const Params &P, int i, int j, int k) {
  return (long long)(i + P.G[0]) * P.st[0] + (long long)(j + P.G[1]) * P.st[1] + (long long)(k + P.G[2]) * P.st[2];
}

// non-negative doubles order like their bit patterns: exact, order-independent max
__device__ __forceinline__ void atomic_max_nonneg(unsigned long long *addr, double v) {
  atomicMax(addr, (unsigned long long)__double_as_longlong(v));
}
__device__ __forceinline__ double slot_value(const unsigned long long *addr) {
  return __longlong_as_double((long long)*addr);
}

__device__ __forceinline__ int floordiv_i(int a, int b) {
  int q = a / b;
  if ((a % b != 0) && ((a < 0) != (b < 0))) q--;
  return q;
}
