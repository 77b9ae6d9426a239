/* oracle/lrdmc_ref.h -- interface of the CPU FP64 ORACLE for load-balanced LRDMC.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this.  It shares no code, header,
 * table or constant generator with the CUDA path (paper_2508_12033_b200/csrc, include/lrdmc.h).
 *
 * Everything is host memory, plain C, FP64.  Citations are PAPER.md line numbers (L...) plus the
 * equation / algorithm; "Qn" are the readings of silent or garbled passages listed in DESIGN.md.
 */
#ifndef LRDMC_REF_H
#define LRDMC_REF_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct lrdmc_ref_ctx lrdmc_ref_ctx;

enum { LRDMC_REF_OK = 0, LRDMC_REF_EINVAL = -1, LRDMC_REF_ESINGULAR = -2, LRDMC_REF_ESTATE = -3 };
enum { LRDMC_REF_BALANCED = 0, LRDMC_REF_CONVENTIONAL = 1 };

/* per-cycle record: Eq.34 (L227) / Eq.20 (L135) numerator and denominator, Eq.16 (L115) wbar */
typedef struct {
    double wbar, num, den;
    int64_t moves_min, moves_max, moves_sum;
    int64_t n_node_flag, n_nonpos_diag, n_nonfinite;
    double lockstep_idle_frac; /* 1 - sum_k n_k / (N_w max_k n_k): what a lock-step batch would idle */
    int64_t n_singular;        /* walkers whose Slater matrix was singular at the last (re)build (reading Q24) */
} lrdmc_ref_stats;

/* System description (all arrays copied).  pp == NULL: all-electron; else [n_nuc][4] local
 * pseudopotential parameters (alpha, beta, gamma, delta), alpha <= 0 meaning a bare Coulomb nucleus.
 * shell type: 0/1/2 = cartesian s/p/d Gaussian primitive, 10 = Slater-type s.  C_up [n_ao][n_up],
 * C_dn [n_ao][n_dn], row-major.  c1/b1 == NULL: no one-body Jastrow.  a2 == 0: single mesh. */
int lrdmc_ref_create(lrdmc_ref_ctx **out, int n_nuc, const double *Z, const double *Rnuc, const double *pp,
                     int n_up, int n_dn, int n_shell, const int *center, const int *type, const double *zeta,
                     int n_ao, const double *C_up, const double *C_dn, double a_par, double a_anti, double b2,
                     const double *c1, const double *b1, double a, double a2, uint64_t seed);
void lrdmc_ref_destroy(lrdmc_ref_ctx *);
int lrdmc_ref_n_candidates(const lrdmc_ref_ctx *); /* P = 6 N n_mesh (+ 6 N K non-local slots) */

/* Contracted shells and real solid-harmonic d shells (scope row f2; "cc-pVTZ basis sets ... The angular part of
 * the basis functions was expressed using spherical (solid) harmonics", L285 "cartesian").  The shells passed to create are then
 * PRIMITIVES; contracted shell cs is the run of consecutive primitive shells first[cs] .. first[cs+1]-1 (same centre, same type):
 *   chi_cs,c(r) = sum_k coef[k] chi^prim_k,c(r)      (each primitive normalised to unit self-overlap, reading Q14)
 * and for a d shell with sph[cs] != 0 the five real solid harmonics, each of unit self-overlap for a single primitive, in the order
 *   z2 = zz - (xx + yy)/2,  xz,  yz,  x2-y2 = (sqrt(3)/2)(xx - yy),  xy      (xx.. = the normalised cartesian d primitives).
 * n_ao and the MO matrices given to create refer to the CONTRACTED functions.  Call right after create. */
int lrdmc_ref_set_contraction(lrdmc_ref_ctx *, int n_cshell, const int *first /*[n_cshell+1]*/, const double *coef /*[n_shell]*/,
                              const int *sph /*[n_cshell]*/);

/* Three-body Jastrow (scope row f2; "the Jastrow factor used ... in the TurboRVB calculations", L285 "2+3-body Jastrow"):
 *   J3(x) = sum_{i<j} sum_{a,b} g_ab chi_a(r_i) chi_b(r_j),   chi_a(r) = dx^l dy^m dz^n exp(-zeta_a |d|^2),  d = r - R_{center_a},
 * s, p and cartesian d Gaussians on the nuclei: (l, m, n) = lmn[a], l + m + n <= 2, unnormalised (a norm is a factor of g); lmn NULL = all s.
 * g symmetric [n][n] (electron-electron-nucleus terms for a, b on one nucleus, e-e-n-n terms otherwise); added to J of Psi_G = D exp(J).
 * Any number of functions.  The functional form is named by the paper only: this is reading Q23 of DESIGN.md.  Call right after create. */
int lrdmc_ref_set_jastrow3(lrdmc_ref_ctx *, int n, const int *center, const double *zeta, const double *g, const int *lmn /*[n][3] or NULL*/);

/* Non-local (semi-local) pseudopotential, scope row f1 (L242 "DLA", L567 D1 "non-local pseudopotentials", L576 "DTM").
 * nl [n_nuc][7] = { r_c, A_0, B_0, A_1, B_1, A_2, B_2 }: channel l of nucleus I is v_l(r) = A_l exp(-B_l r^2) inside r < r_c
 * (synthetic Gaussian channels: the ccECP tables are not in the container); r_c <= 0: no non-local part on that nucleus.
 *   V_nl Psi(x)/Psi(x) = sum_i sum_I sum_l v_l(r_iI) (2l+1)/(4 pi) int P_l(cos th') Psi(.. R_I + r_iI Omega' ..)/Psi(x) dOmega'
 * with the integral on the 6-point octahedral rule (weights 1/6, exact to degree 3) along +-e_k of the step's random frame
 * ("and the discretized ECP mesh", L625-L628).  Each (electron i, centre I in range) gives 6 more candidates x_q with
 * H_{x_q,x} = nu_q = (1/6) sum_l (2l+1) v_l(r_iI) P_l(cos th_q) and ratio rho_q = D(x_q)/D(x) (dla = 1: determinant
 * locality, L576) or Psi_G(x_q)/Psi_G(x) (dla = 0: T-move form).  Fixed node (Eq.D1): nu_q rho_q < 0 -> allowed hop with
 * Green's function -nu_q rho_q; nu_q rho_q > 0 -> added to V_sf.  Slots: j = 6 N n_mesh + 6 (i K + kk) + q, kk = rank of
 * centre I among the centres in range of electron i (ascending I), q = 2k (+e_k) / 2k+1 (-e_k); R[j] holds the signed
 * Green's-function amplitude -nu_q rho_q (0 for an empty slot), i.e. the slot has "kappa = 1".  K = max centres in range of
 * one point (a property of the geometry; evaluation fails with EINVAL if exceeded).  Call before set_positions. */
int lrdmc_ref_set_nonlocal(lrdmc_ref_ctx *, int K, int dla, const double *nl);
/* nu_q and rho_q of every non-local slot at x in frame U (for the pins): nu, rho [6 N K], cand [6 N K][3] (nullable) */
int lrdmc_ref_nl_info(const lrdmc_ref_ctx *, const double *x, const double *dinv_up, const double *dinv_dn, const double U[9],
                      double *nu, double *rho, double *cand);

/* walkers.  Reading Q24 (the paper is silent; SURVEY row a13 "LRDMC_ESINGULAR if |D| = 0"): a walker whose Slater matrix has a
 * pivot <= 2^-44 max|D| at a (re)build is DEAD: its inverses are set to zero, it is never evaluated, the next propagate gives it
 * w = omega = 0 (e_L = W = 0, no moves), so the next branching replaces it.  set_positions returns ESINGULAR if there is any
 * (the state is set all the same); reconfigure reports them in the stats (n_singular). */
int lrdmc_ref_set_positions(lrdmc_ref_ctx *, int n_w, const double *r /*[n_w][N][3]*/);
int lrdmc_ref_get_state(const lrdmc_ref_ctx *, double *r, double *dinv_up, double *dinv_dn, double *w);
int lrdmc_ref_set_state(lrdmc_ref_ctx *, int n_w, const double *r, const double *dinv_up, const double *dinv_dn,
                        const double *w);
int lrdmc_ref_get_obs(const lrdmc_ref_ctx *, double *eL, double *W, double *omega, int64_t *n_moves);

/* the path: Alg.2 (L389-L423) / Alg.1 (L311-L387) inner loops, Eq.15-17 branching, Eq.20/34 sums */
int lrdmc_ref_propagate(lrdmc_ref_ctx *, int mode, int n_moves, double tau, double E0, uint64_t cycle);
int lrdmc_ref_reconfigure(lrdmc_ref_ctx *, uint64_t cycle, int32_t *parents_out /*nullable*/);
int lrdmc_ref_estimators(const lrdmc_ref_ctx *, lrdmc_ref_stats *out);
/* Walker k of this context draws from the random streams of slot `offset + k` (default 0): lets a test replay a few walkers
 * taken from the middle of a large ensemble. */
int lrdmc_ref_set_slot_offset(lrdmc_ref_ctx *, uint32_t offset);
int lrdmc_ref_set_threads(int n); /* OpenMP threads over walkers; returns the count in effect */

/* one evaluation + selection for every walker at (cycle, step), no state change.
 * scal[k][8] = { bbar, V_sf, W, e_L, b_x = bbar/(W-E0), tau_xi = -log1p(-u_tau)/bbar (unclipped),
 *                node flag (0/1), selection margin min_j |t - C_j| / C_{P-1} } */
int lrdmc_ref_step_debug(const lrdmc_ref_ctx *, double E0, uint64_t cycle, uint64_t step, double *R /*[n_w][P]*/,
                         double *scal /*[n_w][8]*/, int32_t *jstar /*[n_w]*/);

/* ---- primitives exported so the pins can reach every part on its own ---- */
void lrdmc_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double lrdmc_ref_uniform53(uint32_t lo, uint32_t hi);
void lrdmc_ref_draws(const lrdmc_ref_ctx *, uint32_t slot, uint64_t cycle, uint64_t step,
                     double u[5] /*u1,u2,u3,u_sel,u_tau*/);
void lrdmc_ref_frame(double u1, double u2, double u3, double U[9] /*row-major, columns = versors*/);
uint32_t lrdmc_ref_comb_r32(const lrdmc_ref_ctx *, uint64_t cycle);
int lrdmc_ref_comb(int n_w, const double *w, uint32_t r32, int32_t *parents, double *wbar, uint64_t *u_out /*nullable [n_w]*/,
                   uint64_t *T_out /*nullable*/, int *sh_out /*nullable*/);
int lrdmc_ref_ao(const lrdmc_ref_ctx *, const double r[3], double *val, double *grad /*[n_ao][3]*/, double *lap);
int lrdmc_ref_mo(const lrdmc_ref_ctx *, int spin, const double r[3], double *val, double *grad /*[O][3]*/, double *lap);
/* log|Psi_G| and sign from scratch (pivoted LU of the Slater matrices + full Jastrow double sum) */
int lrdmc_ref_logpsi(const lrdmc_ref_ctx *, const double *x /*[N][3]*/, double *logabs, int *sign);
/* Slater inverses from positions (a13); returns LRDMC_REF_ESINGULAR on a zero pivot */
int lrdmc_ref_build_inverse(const lrdmc_ref_ctx *, const double *x, double *dinv_up, double *dinv_dn);
/* one evaluation C2 at x with given inverses (NULL: built from x) and frame U.
 * scal[10] = { bbar, V_sf, W, e_L, node, V_ee, V_ii, K_diag = sum_j kappa_j, n_vmax_fired, e_L_continuum (D7 rhs) }
 * per-electron per[N][5] = { T_i, lap_i = nabla_i^2 Psi/Psi, v_ei(r_i), v_zv_i, v^a_ei_i } */
int lrdmc_ref_evaluate(const lrdmc_ref_ctx *, const double *x, const double *dinv_up, const double *dinv_dn,
                       const double U[9], double *R /*[P]*/, double *scal /*[10]*/, double *per /*[N][5]*/,
                       double *cand /*nullable [P][3] candidate positions*/);
/* heat-bath selection C4 on q_j = kappa_j max(R_j, 0) */
int lrdmc_ref_select(const lrdmc_ref_ctx *, const double *R, double u_sel, double *margin /*nullable*/);

#ifdef __cplusplus
}
#endif
#endif
