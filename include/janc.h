/* janc.h -- C ABI of libjanc: the per-time-step update of the compressible multi-species
 * reacting Euler equations on uniform block-structured patches (arXiv 2504.13750, "JANC"),
 * implemented as hand-written sm_100a CUDA kernels in fp64.
 *
 * Citations are PAPER.md:<line> (section / equation).  Readings of silent or garbled passages
 * (A1..A24) are listed in DESIGN.md.
 *
 * Conventions
 *  - Every call returns an int status (JANC_OK = 0, negative = error); nothing throws or aborts
 *    across the ABI.  janc_last_error() gives a text for the last failure of a context.
 *  - The caller owns every buffer it passes; the library copies what it keeps.  Device memory
 *    for the state and all scratch comes from ONE caller-allocated workspace
 *    (janc_workspace_bytes / janc_bind_workspace); the library never allocates the big arrays.
 *  - All kernels are enqueued on the CUDA stream given to janc_create (a cudaStream_t passed as
 *    void*; NULL = legacy default stream).  janc_step is asynchronous unless t_advanced != NULL.
 *  - A device-side flag (non-finite value, T <= 0, Newton not converged, singular pivot) is
 *    reported as JANC_ENONFINITE by the next synchronising call (janc_step with t_advanced,
 *    janc_get_state, janc_status).
 *  - There is no CPU fallback: without a CUDA device janc_create returns JANC_ECUDA.
 *
 * State layout (PAPER.md:232 eq 4.1; :83, :179 block data [N, n_U, n_x, n_y]):
 *    U[np][nvar][nz][ny][nx], x fastest, interior cells only (no ghosts), fp64, with
 *    nvar = ndim + 2 + (ns-1) in the paper's order  rho, rho*u[, rho*v[, rho*w]], E,
 *    rho*Y_1 .. rho*Y_{ns-1};  np = max(1, n_patches).  T[np][nz][ny][nx] likewise.
 */
#ifndef JANC_H
#define JANC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct janc_ctx janc_ctx; /* opaque, owned by the library */

enum { JANC_OK = 0, JANC_EINVAL = -1, JANC_ENOMEM = -2, JANC_ECUDA = -3, JANC_ESTATE = -4, JANC_ENONFINITE = -5 };

/* Physical boundary kinds (readings A14, A15):
 * PERIODIC copies the opposite interior layers (uniform grid only; in block mode periodicity is
 * expressed through the neighbour lists), REFLECT mirrors about the face and negates the normal
 * momentum (slip wall), OUTFLOW copies the nearest interior cell (zero gradient,
 * the paper's "non-reflecting"). */
enum { JANC_BC_PERIODIC = 0, JANC_BC_REFLECT = 1, JANC_BC_OUTFLOW = 2,
       JANC_BC_EXCHANGE = 3 /* x sides of a uniform grid only: the ghost columns are filled by janc_halo (x-slab decomposition) */ };

typedef struct {
  int ndim;               /* 1, 2 or 3 (paper: 2; reading A18)                     */
  int n[3];               /* interior cells per direction (per patch in block mode)              */
  double dx[3];           /* level-0 spacing (m); level l uses dx / ratio^l                      */
  int bc_lo[3], bc_hi[3]; /* physical boundary kind per face                                     */
  int n_patches;          /* 0 = one uniform grid; > 0 = block-list mode        */
  int n_levels, ratio;    /* block mode: 1 or 2 levels, refine ratio 2          */
} janc_grid;

/* Reaction mechanism (eq 4.3-4.9).  Host arrays, copied by the call. */
typedef struct {
  int ns, nr;                /* species (>= 1), reactions (>= 0); ns <= 32, nr <= 128             */
  const double *W;           /* [ns] molar mass, kg/mol                                           */
  const double *nasa;        /* [ns][7] a0..a6 of eq 4.3-4.5, single range (reading A7)           */
  const int32_t *nu_f, *nu_b;/* [nr][ns] integer stoichiometry 0..3 (eq 4.6)                      */
  const double *A, *b, *Ta;  /* [nr] Arrhenius in SI (mol, m^3, s); Ta = Ea/Ru in K (eq 4.8)      */
  const int32_t *reversible; /* [nr] 0 => k_b = 0 (reading A10)                                   */
  const int32_t *third_body; /* [nr] 1 => rate multiplied by sum_j a_ij X_j (eq 4.7, reading A9)  */
  const double *eff;         /* [nr][ns] a_ij; NULL => all 1                                      */
  const double *nasa_hi;     /* [ns][7] two-range NASA-7 data (Cantera / Chemkin thermo):   */
  const double *T_mid;       /* [ns]    species k uses nasa_hi[k] for T >= T_mid[k], nasa[k] below; both NULL => */
                             /*         single range.  (The role-warp chemistry kernel is single-range only:    */
                             /*         two-range mechanisms of more than 13 species run the "jit-smem" kernel.) */
} janc_mech;

/* Chemkin-format mechanism reader (PAPER.md:279 "a chemkin-format reader", :400; two-range NASA-7 thermo, :258): host
 * only, needs no device.  mech_text: ELEMENTS / SPECIES / [THERMO] / REACTIONS sections; thermo_text (nullable): a
 * separate thermo file.  Supported subset = what eq 4.6-4.9 can express: Arrhenius reactions, reversible ("=", "<=>")
 * or not ("=>"), third bodies "+ M" with efficiency lines; units CAL/MOLE (default), KCAL/MOLE, JOULES/MOLE,
 * KJOULES/MOLE, KELVINS; element weights from a small built-in table or "X /w/".  Anything else (fall-off, PLOG, REV,
 * ...) is refused: JANC_EINVAL with a message in err (NUL-terminated, at most errcap bytes).  The result is in SI
 * (W kg/mol; A in mol, m^3, s; Ta = E / R_u in K), species in file order -- the LAST species is the one carried by
 * difference.  janc_mech_file_view fills a janc_mech whose pointers stay valid until janc_mech_file_free.
 * No mechanism data ships with the library. */
typedef struct janc_mech_file janc_mech_file;
int janc_mech_parse(const char *mech_text, const char *thermo_text, janc_mech_file **out, char *err, size_t errcap);
int janc_mech_file_view(const janc_mech_file *, janc_mech *view);
const char *janc_mech_file_species(const janc_mech_file *, int k);
void janc_mech_file_free(janc_mech_file *);

/* Create a context for one grid on CUDA device `device`; kernels go to `cuda_stream`.  JANC_EINVAL for a malformed
 * grid, including fewer than 3 cells along a direction whose sides are not both zero-gradient (the 3 ghost layers of
 * PAPER.md:295 are copies of 3 distinct interior cells under the periodic, mirror and neighbour-patch rules), or a
 * patch of 2^31 or more padded cells (more than one B200 holds). */
int janc_create(const janc_grid *grid, int device, void *cuda_stream, janc_ctx **out);

/* Options, as text (key, value); JANC_EINVAL for an unknown key or value.  The product runs the defaults; the other
 * values exist so that tests can reach every kernel and every host path without environment variables.
 *   "graph"            "1" (default) | "0"   replay one captured CUDA graph per step | eager launches
 *   "tma"              "1" (default) | "0"   2-D grids above 600 k cells and 3-D grids, with an even padded width: tiles
 *                      staged with cp.async.bulk.tensor (TMA) | with 8-byte cp.async (2-D) / staging loops (3-D)
 *   "halo"             "auto" (default) | "ghost"   auto: 2-D patches of <= 16 x 16 cells and 2-D grids below 600 k cells
 *                      gather their halo inside the flux kernel; ghost: k_ghost always materialises the ghost layers
 * and, only before janc_set_mechanism (JANC_ESTATE afterwards), the kernel selection of that call:
 *   "jit"              "1" (default) | "0"   mechanism-specialised kernels compiled with NVRTC | table-driven kernels
 *   "jit_max_unknowns" integer (default 12)  largest ns-1 of the one-thread-per-cell specialised chemistry kernel
 *   "jit_big"          "roles" (default) | "smem"   kernel for larger mechanisms
 *   "roles"            "8" (default) | "16"  role-warps per CTA of the role-warp chemistry kernel
 *   "roles_lu"         "rows" (default) | "columns"  its linear solve: LU with one row per lane inside a warp |
 *                      column-distributed Gauss-Jordan across the role warps
 *   "roles_newton"     "prim" (default) | "kernel"  where its T* = T(U*) comes from: a cons->prim launch in front of the
 *                      kernel | the Newton iteration inside the kernel */
int janc_set_option(janc_ctx *, const char *key, const char *value);

/* Mechanism must be set before the workspace is sized (nvar depends on ns).  A rejected mechanism (JANC_EINVAL) leaves
 * the context unchanged. */
int janc_set_mechanism(janc_ctx *, const janc_mech *);

/* Bytes of device memory the context needs (state with ghosts, RK registers, primitives,
 * reduction slots).  The caller allocates (e.g. torch.empty(..., device='cuda')) and binds a
 * 256-byte aligned device pointer; it must stay alive until janc_destroy. */
size_t janc_workspace_bytes(const janc_ctx *);
int janc_bind_workspace(janc_ctx *, void *dev_ptr, size_t bytes);

/* Block lists: level[np]; nbr[np][2*ndim] same-level neighbour patch ids in the
 * order lo-x, hi-x, lo-y, hi-y, lo-z, hi-z, -1 = none; parent[np][1+ndim] = (parent patch id,
 * sub-region index along x, y[, z] in 0..ratio-1), -1 on level 0.  Host arrays, copied.
 * A face without neighbour is filled from the physical BC on level 0; on level 1 by
 * piecewise-constant injection from the coarse parent unless the face lies on
 * the domain boundary (reading A19). */
int janc_set_blocks(janc_ctx *, const int32_t *level, const int32_t *nbr, const int32_t *parent);

/* Load the state.  U as laid out above; T_guess (nullable: 1000 K) seeds the Newton iteration
 * (reading A6).  on_device != 0: pointers are device pointers on the same device. */
int janc_set_state(janc_ctx *, const double *U, const double *T_guess, int on_device);

/* Advance nsteps of advance_one_step: cfl() -> advance_flux (TVD-RK3 over
 * rhs: ghost fill, update_aux, LF-split WENO5 fluxes, divergence) -> advance_source_term
 * (point-implicit chemistry, eq 4.12-4.13) [-> average-down in 2-level block mode, PAPER.md:188].
 * cfl > 0: dt = cfl * min_d dx_d(finest) / max(|u_d| + c) each step (reading A16);
 * cfl <= 0: dt = dt_fixed.  flags: bit 0 set => no chemistry at all (explicit variant of PAPER.md:351-357 with a zero
 * source_terms); bit 1 set => explicit variant with the mechanism's own source: S_k = W_k omega_k(T, X) (eq 4.6) is added to
 * the right-hand side of every RK stage and advance_source_term is not executed; returns JANC_ESTATE if
 * the run-time specialised source kernel is not available (no NVRTC).
 * bit 2 set => crossover time advance of a two-level block list (Fig 2a; reading B9) instead of
 * the synchronous one (Fig 2b): per step, two steps dt/2 of level 1 -- its coarse-fine ghosts injected from the level-0
 * state at the start of the step -- then one step dt of level 0, then the average-down; dt = cfl * min_d dx_d(level 0) /
 * max(|u_d| + c), or dt_fixed = the level-0 step.  Needs the patches ordered by level (JANC_EINVAL otherwise); ignored
 * on a single level.
 * t_advanced (host, nullable): receives the sum of dt; forces a stream synchronise. */
int janc_step(janc_ctx *, int nsteps, double cfl, double dt_fixed, int flags, double *t_advanced);

/* x-slab decomposition over several GPUs (split_grid, exchange_halo, parallel_rhs; one process per
 * GPU).  Every rank owns a slab of the grid along x with JANC_BC_EXCHANGE on its interior x sides and advances it with
 * janc_step_part instead of janc_step; between the parts the caller (paper_2504_13750_b200/slab.py: torch.distributed over
 * NCCL) max-reduces the reduction slots over the ranks and swaps the halo buffers.  Per step:
 *   PRIM(0) -> [all-reduce max of the slots] -> DT ->
 *   for stage s = 0, 1, 2:  (s > 0: PRIM(s) -> [all-reduce]) -> GHOST(s) -> janc_halo pack lo / hi ->
 *                           [send / receive] -> janc_halo unpack lo / hi -> FLUX(s)
 *   -> SOURCE.
 * The slots hold max(|u_d| + c) as the bit pattern of a non-negative double, which orders like an unsigned integer:
 * an integer MAX all-reduce is exact, so every rank computes the same dt and the same alpha as the undecomposed grid.
 * flags: 0, or 1 = no chemistry.  Uniform grids only; eager launches (no graph). */
enum { JANC_PART_PRIM = 0, JANC_PART_DT = 1, JANC_PART_GHOST = 2, JANC_PART_FLUX = 3, JANC_PART_SOURCE = 4 };
int janc_step_part(janc_ctx *, int part, int stage, double cfl, double dt_fixed, int flags);
/* Doubles in one halo buffer: (nvar + 2 + ndim) fields (U, T, p, u_d) x 3 columns x ny x nz. */
size_t janc_halo_doubles(const janc_ctx *);
/* unpack = 0: copy the 3 interior columns next to x side `side` (0 lo, 1 hi) of RK register `stage` (0 = U^n, 1 = U^(1),
 * 2 = U^(2)) and of T, p, u_d into the device buffer; unpack = 1: copy the buffer into the ghost columns of that side. */
int janc_halo(janc_ctx *, int stage, int side, double *buf_dev, int unpack);
/* Where the reduction slots sit inside the bound workspace (byte offset, number of 64-bit slots). */
int janc_reduction_slots(const janc_ctx *, size_t *byte_offset, size_t *count);

/* Regridding of a two-level block list (JAX-AMR "update refinement layer": PAPER.md:73-75 refinement criterion mask +
 * buffer cells, :123 / :184 unaltered blocks keep their data, :175-184 get_refinement_grid_mask / _block_mask / _block_info
 * / _block_data; reading B12).  The level-0 patches must be the first entries of the list and tile the domain.
 * janc_regrid_plan: marks the level-0 cells with max_d |rho(i+e_d) - rho(i-e_d)| / (2 rho(i)) > thr, adds nbuf buffer
 * cells in every direction (across patch boundaries and periodic sides), refines every fixed sub-region (parent, s in
 * {0,1}^ndim) that holds a marked cell, and returns the new list in host arrays sized for the worst case
 * n0 (1 + 2^ndim) patches: np_new, level[np], nbr[np][2 ndim], parent[np][1 + ndim] -- level 0 unchanged, then the
 * level-1 blocks ordered by parent and sub-index (x fastest).  janc_regrid_fill: the state of that list in the interior
 * layout of janc_set_state, U_new[np_new][nvar][cells], T_new[np_new][cells] (device or host): blocks that existed keep
 * their data, new ones are the one-to-four injection of their parent.  The caller then creates a context
 * for the new list (janc_create with n_patches = np_new, janc_set_blocks, janc_set_state).  Both calls synchronise and
 * use the RK scratch registers: call them between steps. */
int janc_regrid_plan(janc_ctx *, double thr, int nbuf, int32_t *np_new, int32_t *level, int32_t *nbr, int32_t *parent);
int janc_regrid_fill(janc_ctx *, double *U_new, double *T_new, int on_device);

/* dt of the most recent step (cfl()), read from the device; synchronises. */
int janc_last_dt(janc_ctx *, double *dt);

/* The stable time step of a state WITHOUT a workspace and without any allocation (cfl(): dt = cfl *
 * dx_min / max_d max_cells(|u_d| + c), with T, c from the cons->prim Newton iteration of PAPER.md:237-258, :306) -- for
 * callers that cannot call cudaMalloc (CUDA graph capture, serving loops).  A variant of the cons->prim + max-reduction
 * kernel whose per-CTA partial maxima and error flag live in a file-scope `static __device__` array of the library
 * (csrc/static_scratch.cuh; 256 B + JANC_STATIC_MAX_CELLS / 256 x 3 doubles = 1.5 MiB that every GPU which loads the
 * library holds until exit).  The context needs a mechanism only (janc_create + janc_set_mechanism; no workspace, blocks
 * or state): it supplies grid, dx_min, species data and the stream.
 *   U_dev   device, the interior layout of janc_set_state: [n_patches][nvar][nz][ny][nx]             (input, not modified)
 *   T_dev   device, [n_patches][nz][ny][nx] Newton starting temperatures, or NULL = 1000 K           (input, not modified)
 *   out_dev device, double[4]: dt, max(|u_x| + c), max(|u_y| + c), max(|u_z| + c) (0 for unused directions); dt is NaN
 *           if the Newton iteration failed in some cell (the maxima then exclude such cells)        (output)
 * Asynchronous on the context's stream; the caller owns all three buffers.  Returns JANC_EINVAL with a text in
 * janc_last_error if n_patches * cells per patch exceeds JANC_STATIC_MAX_CELLS, or cfl <= 0; JANC_ESTATE without a
 * mechanism.  Calls no cudaMalloc / cudaFree / allocating routine.  The first call of a context on a device resolves the
 * array's device address (cudaGetSymbolAddress, once per device) and, if another context's species tables sit in that
 * device's constant memory, drains the device and uploads its own: make that first call outside graph capture.
 * ALL calls of the process on one device share the array (it keeps the last call's contents; the flag word is cleared at
 * the start of every call): calls that overlap on the GPU -- different streams, or graphs replayed concurrently -- race;
 * calls on one stream are ordered and safe. */
#define JANC_STATIC_MAX_CELLS (1LL << 24)
int janc_cfl_dt_static(janc_ctx *, const double *U_dev, const double *T_dev, double cfl, double *out_dev);

/* Read the state back (U and/or T nullable).  Synchronises.  Returns JANC_ENONFINITE if the
 * device flag was raised since the last janc_set_state. */
int janc_get_state(janc_ctx *, double *U, double *T, int on_device);

/* Synchronise and return JANC_OK / JANC_ENONFINITE / JANC_ECUDA. */
int janc_status(janc_ctx *);

/* Number of kernel launches enqueued by this context since creation (diagnostic). */
long long janc_launch_count(const janc_ctx *);

/* Diagnostic: run the fused cons->prim + thermo kernel on the current
 * state and return T, p, c per interior cell ([np][nz][ny][nx] each, device or host). */
int janc_debug_cons2prim(janc_ctx *, double *T, double *p, double *c, int on_device);

/* Diagnostic: per-phase device time (ms, CUDA events on the context's stream) of ONE step at the
 * current state: out[0]=cons2prim+reduce, [1]=ghost fill, [2]=flux sweeps+divergence+RK,
 * [3]=chemistry, [4]=average-down, [5]=whole step; launches of each in n_out[0..5] (nullable).
 * Advances the state by one step with the given cfl/dt_fixed. */
int janc_profile_step(janc_ctx *, double cfl, double dt_fixed, float *ms_out, int *n_out);

/* Diagnostic: measured register-resident DFMA rate of the device, in DFMA/s (the FP64 ALU peak
 * used as roofline denominator for "bound":"alu"). */
int janc_measure_dfma_peak(int device, void *cuda_stream, double *dfma_per_s);

/* Which chemistry kernel the context runs: "jit" = the mechanism-specialised kernel generated and
 * compiled with NVRTC by janc_set_mechanism (csrc/chemgen.h; the counterpart of the paper's XLA JIT,
 * PAPER.md:24, :39), "reg" / "generic" = the table-driven kernels of csrc/chem.cuh (mechanisms with
 * NVRTC missing, or janc_set_option("jit", "0")), "jit-roles" / "jit-smem" = the specialised kernels for more than 12
 * unknowns, "none" before a mechanism is set.  janc_jit_log returns the NVRTC log / the reason the specialised kernel
 * is not used, and a note if the per-step CUDA graph could not be captured and the context fell back to eager launches. */
const char *janc_chem_kernel(const janc_ctx *);
const char *janc_jit_log(const janc_ctx *);

/* Diagnostic, needs no device: write the specialised CUDA source of a mechanism (NUL-terminated,
 * truncated to cap) to src_out (nullable), its length to src_len (nullable), and, if cubin_bytes is
 * non-NULL, compile it for sm_100a and return the cubin size.  JANC_ESTATE if NVRTC fails. */
int janc_jit_probe(const janc_mech *, int ndim, char *src_out, size_t cap, size_t *src_len, size_t *cubin_bytes);

const char *janc_last_error(const janc_ctx *);
void janc_destroy(janc_ctx *);

#ifdef __cplusplus
}
#endif
#endif /* JANC_H */
