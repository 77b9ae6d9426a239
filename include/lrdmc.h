/* include/lrdmc.h -- C-ABI of liblrdmc.so: the data-parallel hot path of load-balanced LRDMC
 * (arxiv 2508.12033, Nakano / Sorella / Casula) on one NVIDIA B200 (sm_100a), FP64.
 *
 * Citations "L<n>" are line numbers of the paper text with the equation / algorithm they
 * fall in; "Qn" are the readings of silent or garbled passages listed in DESIGN.md.
 *
 * Conventions
 *   - Every function returns int: 0 = LRDMC_OK, < 0 = hard error (nothing modified unless stated).
 *   - No process-global state: everything lives in the ctx (no environment variables are read; the text of a CUDA error is
 *     kept per ctx, see lrdmc_last_error).  Calls on DIFFERENT contexts may run concurrently from different threads and on
 *     different streams; calls on one ctx must be serialised by the caller.
 *   - "host"   pointer: ordinary CPU memory, read or written synchronously inside the call.
 *   - "device" pointer: CUDA device memory of the current device; used asynchronously on `stream`
 *     (a cudaStream_t passed as void*, NULL = legacy default stream).  The caller keeps such buffers alive
 *     until the stream has passed the call.
 *   - The library owns only the ctx (and small device tables inside it).  Walker storage is CALLER-owned
 *     device memory handed over with lrdmc_bind_walkers (e.g. a torch tensor).
 *   - No CPU fallback exists: without a CUDA device every call that needs one returns LRDMC_ECUDA.
 *   - Soft numerical events (W(x)-E_0 <= 0, node flags, non-finite weights) are counted in
 *     lrdmc_cycle_stats, never returned as errors.
 *   - Electron order: the n_up spin-up electrons first, then the n_dn spin-down ones.
 *   - Candidate (off-diagonal move) order: j = mesh*6N + 6*i + d, d = 0..5 <-> (+e1,-e1,+e2,-e2,+e3,-e3),
 *     e_k = k-th column of the step's random frame U (Eq.D3-D4).
 */
#ifndef LRDMC_H
#define LRDMC_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct lrdmc_ctx lrdmc_ctx; /* opaque; created by lrdmc_init, destroyed by lrdmc_free */

enum { LRDMC_OK = 0, LRDMC_EINVAL = -1, LRDMC_ESINGULAR = -2, LRDMC_ESTATE = -3, LRDMC_ECUDA = -4, LRDMC_ENOMEM = -5 };
enum { LRDMC_BALANCED = 0, LRDMC_CONVENTIONAL = 1 };
enum { LRDMC_SHELL_S = 0, LRDMC_SHELL_P = 1, LRDMC_SHELL_D = 2, LRDMC_SHELL_SLATER_S = 10 };
#define LRDMC_MAX_OCC 32 /* occupied MOs per spin supported by the kernels */

/* ---- problem statement (all arrays are HOST pointers and are COPIED by lrdmc_init) -------------------- */
typedef struct {
    int n_nuc;
    const double *Z;  /* [n_nuc] charge (Z, or Z_eff for a pseudo-atom) */
    const double *R;  /* [n_nuc][3] bohr */
    int n_up, n_dn;   /* n_up >= 1, n_dn >= 0, each <= LRDMC_MAX_OCC */
    const double *pp; /* NULL = all bare nuclei; else [n_nuc][4] = (alpha,beta,gamma,delta) of the local
                         pseudopotential v(r) = -(Z/r)(1-e^{-alpha r^2}) + Z alpha r e^{-beta r^2} + gamma e^{-delta r^2}
                         (reading Q14); alpha <= 0 marks a bare -Z/r nucleus */
    /* Non-local (semi-local) pseudopotential channels ("DLA", Eq.D1 "DTM", L625-L628):
     * nl == NULL or nl_K == 0: none.  Else nl [n_nuc][7] = (r_c, A_0, B_0, A_1, B_1, A_2, B_2): channel l of nucleus I is
     * v_l(r) = A_l exp(-B_l r^2) for r < r_c (r_c <= 0: no channels on that nucleus).  Each (electron i, centre I with
     * r_iI < r_c) adds the six candidates x_q = "electron i at R_I +- r_iI e_k" (octahedral rule in the step's frame) with
     * H_{x_q,x} = nu_q = (1/6) sum_l (2l+1) v_l(r_iI) P_l(cos theta_q) and rho_q = D(x_q)/D(x) (nl_dla != 0) or
     * Psi_G(x_q)/Psi_G(x) (nl_dla == 0); nu_q rho_q < 0: hop with Green's function -nu_q rho_q, > 0: into V_sf (Eq.D1).
     * nl_K = slots per electron = the largest number of cutoff spheres containing one point (1 <= nl_K <= 4; centres in range beyond the
     * nl_K-th are ignored -- a wrong nl_K is a caller error).  Candidate order: after the
     * 6 N n_mesh lattice hops, j = 6 N n_mesh + 6 (i nl_K + kk) + q, kk = rank of I among the centres in range (ascending),
     * q = 2k (+e_k), 2k+1 (-e_k); R[j] of lrdmc_step_debug holds -nu_q rho_q there (0: empty slot). */
    const double *nl;
    int nl_K, nl_dla;
} lrdmc_system;
typedef struct {
    int n_shell;
    const int *center;  /* [n_shell] nucleus index */
    const int *type;    /* [n_shell] LRDMC_SHELL_*: cartesian Gaussian primitives s (1 AO), p (x,y,z),
                           d (xx,xy,xz,yy,yz,zz), each normalised to unit self-overlap; or Slater s exp(-zeta r) */
    const double *zeta; /* [n_shell] > 0 */
    /* Contracted shells and real solid-harmonic d shells ("cc-pVTZ ... spherical (solid) harmonics"; L285).
     * n_cshell == 0 / cs_first == NULL: every shell above is a basis function set of its own.  Else the shells above are
     * PRIMITIVES and contracted shell cs is the run cs_first[cs] .. cs_first[cs+1]-1 (same centre, same type):
     * chi_cs,c = sum_k prim_coef[k] chi^prim_k,c; a d shell with cs_sph[cs] != 0 carries the five functions
     * z2 = zz - (xx+yy)/2, xz, yz, x2-y2 = (sqrt(3)/2)(xx - yy), xy of the normalised cartesian primitives (unit self-overlap
     * each for one primitive).  lrdmc_mo.n_ao and C_up / C_dn then refer to the CONTRACTED functions; lrdmc_init folds the
     * contraction into the primitive coefficient tables (host, once), the kernels are unchanged. */
    int n_cshell;
    const int *cs_first;      /* [n_cshell + 1] */
    const double *prim_coef;  /* [n_shell] */
    const int *cs_sph;        /* [n_cshell] */
} lrdmc_basis;
typedef struct {
    int n_ao;                 /* must equal the AO count implied by the shells */
    const double *C_up, *C_dn; /* [n_ao][n_up], [n_ao][n_dn] row-major: phi_m = sum_mu chi_mu C[mu][m] */
} lrdmc_mo;
typedef struct {
    double a_par, a_anti, b2; /* two-body Pade u2 = a r/(1+b2 r), a by spin pair; a = 0 disables */
    const double *c1, *b1;    /* [n_nuc] one-body Pade u1_I = -c1_I r/(1+b1_I r); c1 == NULL disables */
    /* Three-body (electron-electron-nucleus) Jastrow ("2+3-body Jastrow"; form = reading Q23):
     *   J3 = sum_{i<j} sum_{a,b} g_ab chi_a(r_i) chi_b(r_j),  chi_a(r) = dx^l dy^m dz^n exp(-zeta_a |d|^2),  d = r - R_{center_a},
     * g symmetric; s, p and cartesian d Gaussians (l + m + n <= 2, unnormalised: a norm is a factor of g).
     * n_j3 = 0 disables; at most 32 functions (LRDMC_EINVAL beyond). */
    int n_j3;
    const int *j3_center;     /* [n_j3] nucleus index */
    const double *j3_zeta;    /* [n_j3] > 0 */
    const double *j3_g;       /* [n_j3][n_j3] */
    const int *j3_lmn;        /* [n_j3][3] monomial exponents (l, m, n) of each function; NULL: all s functions */
} lrdmc_jastrow;
typedef struct {
    double a;      /* lattice spacing (Eq.D3) */
    double a2;     /* 0 = single mesh; > 0 = second spacing a' of the double mesh (reading Q13, g = 1/2) */
    uint64_t seed; /* Philox4x32-10 key; counter = (walker slot, cycle, step, purpose) (readings Q7, Q12) */
} lrdmc_lattice;

/* Psi_G = D_up D_dn exp(J) and the lattice-regularised fixed-node Hamiltonian of Appendix D (L554-L628).
 * Builds the device tables (sorted/padded shell list, MO coefficients pre-swizzled into FP64 tensor-core
 * B fragments with the AO norms folded in).  Errors: EINVAL (sizes, non-positive zeta/a, AO count), ECUDA, ENOMEM. */
int lrdmc_init(lrdmc_ctx **out, const lrdmc_system *, const lrdmc_basis *, const lrdmc_mo *, const lrdmc_jastrow *,
               const lrdmc_lattice *);
void lrdmc_free(lrdmc_ctx *);
const char *lrdmc_strerror(int code);      /* static text per error code */
/* Text of the last LRDMC_ECUDA of this ctx (cudaGetErrorString + source line; "" if none).  ctx == NULL: the text of the last
 * failed lrdmc_init of the CALLING THREAD (thread-local, like errno: a failed init leaves no ctx to ask). */
const char *lrdmc_last_error(const lrdmc_ctx *);
int lrdmc_n_candidates(const lrdmc_ctx *); /* P = 6 N n_mesh + 6 N nl_K */

/* Explicit tuning / test knobs (no environment variables).  Call BEFORE lrdmc_walker_bytes / lrdmc_bind_walkers (ESTATE once
 * walkers are bound: the buffer was carved for the old plan).
 *   LRDMC_OPT_TEAM_WARPS    value 0 = automatic (default), 1 = one warp per walker, 2/4/8/16 = a CTA of that
 *                           many warps per walker (north_star "one CTA or warp group per walker"); other values are rounded down to
 *                           a power of two.  The parity tests run every size.
 *   LRDMC_OPT_GLOBAL_TABLES value != 0: keep the MO-coefficient fragment tables and the MO cache in global memory even when
 *                           they fit shared memory (the code path of the 64-electron configuration, forced on small systems by tests).
 *   LRDMC_OPT_LISTED        candidate pass of lattice-only systems (no non-local slots, no three-body Jastrow) as a LISTED sweep: per-electron
 *                           lists of the shells within reach (every dropped exponent < -52) and Bc = C Dinv kept as rank-1-updated walker
 *                           state instead of recomputed.  value -1 = automatic (default), 0 = dense sweep, 1 = listed.
 *                           Ignored (dense) for systems with slots or a three-body Jastrow. */
enum { LRDMC_OPT_TEAM_WARPS = 1, LRDMC_OPT_GLOBAL_TABLES = 2, LRDMC_OPT_LISTED = 3 };
int lrdmc_set_option(lrdmc_ctx *, int option, int value);

/* ---- walker storage: structure of arrays in ONE caller-owned device buffer ---------------------------
 * positions (double-buffered for the branching gather), inverse Slater matrices per spin, cached MO
 * value/gradient/Laplacian rows, weights, per-walker observables, reconfiguration workspace.  256-byte aligned. */
size_t lrdmc_walker_bytes(const lrdmc_ctx *, int n_walkers);
int lrdmc_bind_walkers(lrdmc_ctx *, void *dev_buf /*device*/, size_t bytes, int n_walkers); /* EINVAL if too small */

/* Upload positions r [n_w][N][3] (device), build Dinv_sigma = D_sigma^{-1} by pivoted elimination and the MO
 * caches (row a13), weights <- 1.  Synchronises `stream`; returns ESINGULAR if any Slater matrix was singular (a pivot
 * <= 2^-44 max|D_ij|, reading Q24): the state IS set all the same, the singular walkers are dead (see n_singular below). */
int lrdmc_set_positions(lrdmc_ctx *, const double *r_dev, void *stream);

/* One branching interval for every walker (weights reset to 1 on entry, Alg.2 line 4 L401 / Alg.1 line 4 L350):
 *  BALANCED     (Alg.2, Eq.28-30): exactly n_moves times { evaluate; w *= bbar/(W-E0); heat-bath hop },
 *               then one measurement evaluation storing e_L, W and omega = w/(W-E0) (Eq.34, reading Q10).
 *  CONVENTIONAL (Alg.1, Eq.24-25): while tau_left > 0 { evaluate; tau_xi = min(-ln(1-xi)/bbar, tau_left);
 *               w *= exp(-tau_xi (e_L - E0)); tau_left -= tau_xi; hop unless the time ran out }, omega = w.
 *               Here E0 is the constant reference shift (Q8b); n_moves > 0 caps the evaluations, 0 = no cap.
 * `cycle` < 2^32 labels the random streams.  Asynchronous on `stream`. */
int lrdmc_propagate(lrdmc_ctx *, int mode, int n_moves, double tau, double E0, uint64_t cycle, void *stream);

/* Branching at fixed N_w (Eq.15-17) on the raw weights w: integer comb (prefix sum + search, indices
 * bit-exact by construction, reading Q21), gather of the surviving walkers, weights <- 1, wbar recorded (Eq.16),
 * inverses and caches rebuilt from the positions (reading Q15).  parents_dev (device, nullable) receives parent[k].
 * Asynchronous on `stream`. */
int lrdmc_reconfigure(lrdmc_ctx *, uint64_t cycle, int32_t *parents_dev, void *stream);

typedef struct {
    double wbar;     /* Eq.16: mean raw weight of the last reconfigure */
    double num, den; /* sum_k omega_k e_L,k and sum_k omega_k of the last propagate (Eq.20 L135 / Eq.34) */
    int64_t moves_min, moves_max, moves_sum; /* hops per walker in the last propagate */
    int64_t n_node_flag;    /* evaluations that saw at least one R_j < 0 */
    int64_t n_nonpos_diag;  /* evaluations with W(x)-E0 <= 0 (balanced; walker weight set to 0, reading Q16) */
    int64_t n_nonfinite;    /* walkers whose weight left the finite range (set to 0) */
    int64_t n_singular;     /* walkers whose Slater matrix was singular at the last (re)build -- after lrdmc_reconfigure: the
                               rebuild of that branching; before: set_positions / set_state.  Reading Q24: such a walker is DEAD
                               (zero inverses, never evaluated): the next propagate gives it w = omega = 0, the next branching
                               replaces it */
    double lockstep_idle_frac; /* 1 - sum n_k/(N_w max n_k): idle share of a lock-step batch (L168, App. C) */
    double barrier_idle_frac;  /* measured: 1 - sum_warps busy time / (resident warps x kernel span) */
    float propagate_ms, reconfigure_ms; /* CUDA-event durations of the last calls on their stream */
} lrdmc_cycle_stats;
/* Synchronises the stream of the last propagate/reconfigure and fills *out_host (host). */
int lrdmc_estimators(lrdmc_ctx *, lrdmc_cycle_stats *out_host);

/* Host-side estimators over generations (Eq.18-19): G_n^p = prod_{j=1..p} wbar_{n-j},
 * E = sum_n G_n^p e_n / sum_n G_n^p over n >= n_therm, e_n = num_n/den_n; sigma from a delete-one-block
 * jackknife over n_blocks blocks of generations (reading Q9).  All pointers host. */
int lrdmc_energy(const lrdmc_cycle_stats *recs, int n, int p, int n_therm, int n_blocks, double *E, double *sigma);

/* Parity hook: one evaluation + selection for every walker at (cycle, step) with NO state change.  Device outputs:
 * R [n_w][P]; scal [n_w][8] = { bbar, V_sf, W, e_L, b_x = bbar/(W-E0), tau_xi = -log1p(-u_tau)/bbar, node flag, u_sel };
 * jstar [n_w] (-1: no allowed move).  Runs the same device code as lrdmc_propagate. */
int lrdmc_step_debug(lrdmc_ctx *, double E0, uint64_t cycle, uint64_t step, double *R_dev, double *scal_dev,
                     int32_t *jstar_dev, void *stream);

/* State access (device arrays, any may be NULL): r [n_w][N][3], dinv_up [n_w][n_up][n_up], dinv_dn [n_w][n_dn][n_dn]
 * with Dinv[m][i] (sum_m D[i][m] Dinv[m][k] = delta_ik), w [n_w]. set_state with dinv == NULL rebuilds the inverses. */
int lrdmc_get_walkers(lrdmc_ctx *, double *r_dev, double *dinv_up_dev, double *dinv_dn_dev, double *w_dev, void *stream);
int lrdmc_set_state(lrdmc_ctx *, const double *r_dev, const double *dinv_up_dev, const double *dinv_dn_dev,
                    const double *w_dev, void *stream);
/* Per-walker observables of the last propagate (device, nullable): e_L, W, omega [n_w] doubles; n_moves [n_w] int64 */
int lrdmc_get_obs(lrdmc_ctx *, double *eL_dev, double *W_dev, double *omega_dev, int64_t *n_moves_dev, void *stream);

/* End-to-end convenience with HOST buffers (Alg.2 lines 2-13 L398-L420 / Alg.1): H2D of r_in [n_w][N][3], set_positions,
 * n_cycles x (propagate, reconfigure, estimators -> stats_out[c] (nullable, [n_cycles])), D2H of the final positions into r_out
 * (nullable).  Balanced mode feeds E0 back after each branching ("Update E_0", L232 / L418; reading Q8a): E0 <- running mean of
 * e_n = num_n/den_n over the generations so far, the mean restarting once at generation n_therm (0: never) so that the
 * equilibration transient does not stay in it; conventional mode keeps E0 (the constant shift of Q8b).  Walkers must be bound.
 * Synchronous.  Errors: EINVAL, ESTATE (no walkers bound), ESINGULAR (a Slater matrix of r_in had a zero pivot; nothing was
 * propagated, r_out untouched), ECUDA. */
int lrdmc_run_host(lrdmc_ctx *, const double *r_in_host, double *r_out_host, int mode, int n_moves, double tau, double E0,
                   uint64_t first_cycle, int n_cycles, int n_therm, lrdmc_cycle_stats *stats_out_host, void *stream);

/* Test hook for pin P11: fills out_dev [n][4] (uint32) with Philox4x32-10 blocks for counters ctr_dev [n][4], key[2]. */
int lrdmc_debug_philox(const uint32_t *ctr_dev, uint32_t key0, uint32_t key1, uint32_t *out_dev, int n, void *stream);
/* Test hook for row a0: out_dev [n][14] (device) = u1, u2, u3, u_sel, u_tau and the frame U[9] (row-major, versors = columns) that
 * walker slots 0..n-1 draw at (cycle, step) -- the same device functions the walker kernels call. */
int lrdmc_debug_draws(const lrdmc_ctx *, uint64_t cycle, uint64_t step, double *out_dev, int n, void *stream);
/* Diagnostics for bench.py: kernels launched by this ctx so far; and the launch shape lrdmc_propagate uses for the bound
 * walkers (grid, threads per CTA, dynamic shared memory, resident CTAs per SM; any pointer may be NULL), with
 * *team_warps = warps per walker: 1 = kernel k_propagate (warp per walker), > 1 = kernel k_propagate_team. */
int lrdmc_launch_count(const lrdmc_ctx *);
int lrdmc_launch_config(const lrdmc_ctx *, int *grid, int *block, int *smem_bytes, int *ctas_per_sm, int *team_warps);
/* 1 if the candidate pass of this ctx is the listed sweep (LRDMC_OPT_LISTED, or automatic for global-table systems), else 0 */
int lrdmc_listed_sweep(const lrdmc_ctx *);

/* ---- allocation-free entry point (csrc/comb_static.cu) -------------------------------------------------------------------------
 * The integer comb of the branching step alone (Eq.15-17, reading Q21: the arithmetic of lrdmc_reconfigure, bit for bit), for
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it): no ctx, no walker
 * buffer, and NO cudaMalloc / cudaFree / allocating library routine inside.  Its workspace (quantised weights and their prefix sums) is a
 * static device array of LRDMC_COMB_STATIC_MAX_WALKERS x 16 bytes = 1 MiB that every GPU loading the library holds until exit.
 *   w_dev       (device, in)  raw weights w [n_walkers]
 *   seed, cycle the run seed (lrdmc_lattice.seed) and the cycle label (< 2^32): the comb offset xi is the same Philox draw
 *               lrdmc_reconfigure(ctx, cycle) takes
 *   parents_dev (device, out) parent[k] [n_walkers] int32; identity if a weight is negative / non-finite or all are zero
 *   wbar_dev    (device, out, nullable) Eq.16 mean raw weight (0 in the degenerate case)
 * Asynchronous on `stream`.  ALL calls share the one scratch array: calls that overlap on the GPU (different streams or host threads)
 * race -- order them.  The array keeps the last call's contents; nothing in it has to be cleared (every call writes the entries it reads).
 * Errors: LRDMC_EINVAL for NULL pointers, n_walkers < 1, cycle >= 2^32 and for n_walkers > LRDMC_COMB_STATIC_MAX_WALKERS (nothing is
 * launched; use lrdmc_reconfigure for larger ensembles); LRDMC_ECUDA.  lrdmc_comb_static_error() returns the text of the calling thread's
 * last failure ("" if the last call succeeded).  lrdmc_comb_static_setup() resolves the array's device address for the current device
 * ahead of time (cudaGetSymbolAddress, once per device; lrdmc_comb_static does it on its first call otherwise). */
#define LRDMC_COMB_STATIC_MAX_WALKERS 65536
int lrdmc_comb_static(const double *w_dev, int n_walkers, uint64_t seed, uint64_t cycle, int32_t *parents_dev, double *wbar_dev,
                      void *stream);
int lrdmc_comb_static_setup(void);
const char *lrdmc_comb_static_error(void);

#ifdef __cplusplus
}
#endif
#endif
