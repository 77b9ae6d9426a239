/* oracle/ref_internal.h -- private declarations of the CPU FP64 ORACLE (test infrastructure, not
 * product; see lrdmc_ref.h).  Nothing here is seen by the CUDA path. */
#ifndef LRDMC_REF_INTERNAL_H
#define LRDMC_REF_INTERNAL_H
#include "lrdmc_ref.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define REF_MAX_OCC 64   /* occupied MOs per spin the fixed-size scratch arrays allow */

struct lrdmc_ref_ctx {
    /* system */
    int n_nuc; double *Z, *Rn, *pp; /* pp NULL or [n_nuc][4] = alpha,beta,gamma,delta */
    int n_up, n_dn, N;
    /* basis */
    int n_shell, n_ao; int *center, *type, *ao0; double *zeta;
    /* contracted / spherical shells (scope row f2, L242 "cc-pVTZ ... spherical (solid) harmonics"): n_pao primitive AOs;
     * contracted shell cs = primitive shells [cs_first[cs], cs_first[cs+1]) with coefficients prim_coef; cs_sph: 5 real solid d */
    int n_pao, n_cshell, need_contraction; int *cs_first, *cs_sph; double *prim_coef;
    double *C_up, *C_dn;             /* [n_ao][n_up], [n_ao][n_dn] */
    /* Jastrow */
    double a_par, a_anti, b2; double *c1, *b1; /* c1 NULL: no one-body term */
    /* three-body (electron-electron-nucleus) Jastrow, scope row f2: J3 = sum_{i<j} sum_{ab} g_ab chi_a(r_i) chi_b(r_j),
     * chi_a(r) = dx^l dy^m dz^n exp(-zeta_a |d|^2), d = r - R_{c_a}, (l,m,n) = j3_lmn[a] (NULL: s functions), g symmetric [n_j3][n_j3] */
    int n_j3; int *j3_center, *j3_lmn; double *j3_zeta, *j3_g;
    /* lattice */
    double a, a2; int n_mesh; double amesh[2], gmesh[2], kappa[2]; /* kappa_m = g_m / (2 a_m^2) */
    int P;                           /* all candidates: P_lat lattice hops + 6 N nl_K non-local slots */
    int P_lat;                       /* 6 N n_mesh lattice hops (Eq.D4) */
    /* non-local (semi-local) pseudopotential channels, section 8(f) f1 (L242, L567, L576): per nucleus
     * nl[I][7] = { r_c, A_0, B_0, A_1, B_1, A_2, B_2 }: v_l(r) = A_l exp(-B_l r^2) for r < r_c; r_c <= 0: none */
    int nl_K, nl_dla; double *nl;
    uint64_t seed;
    double V_ii;
    /* walkers */
    int n_w; double *r, *dinv_up, *dinv_dn, *w, *eL, *W, *omega; int64_t *nmoves;
    int *flag_node, *flag_nonpos, *flag_nonfinite; /* per-walker event counts of the last cycle */
    int *dead;                       /* walker whose Slater matrix was singular at the last (re)build (reading Q24): weight 0, never evaluated */
    int64_t n_singular;              /* number of such walkers */
    double wbar; int have_obs;
    uint32_t slot0;                  /* random streams of walker k are keyed by slot slot0 + k (lrdmc_ref_set_slot_offset) */
};

static inline int ref_nocc(const lrdmc_ref_ctx *c, int spin) { return spin ? c->n_dn : c->n_up; }
static inline const double *ref_C(const lrdmc_ref_ctx *c, int spin) { return spin ? c->C_dn : c->C_up; }
/* electron i: spin 0 (up) for i < n_up, else spin 1; index inside its spin block */
static inline int ref_spin(const lrdmc_ref_ctx *c, int i) { return i < c->n_up ? 0 : 1; }
static inline int ref_local(const lrdmc_ref_ctx *c, int i) { return i < c->n_up ? i : i - c->n_up; }

/* candidate j -> (mesh block, electron, direction d in 0..5); displacement sign and versor index */
static inline double ref_kappa(const lrdmc_ref_ctx *c, int j) { return j < c->P_lat ? c->kappa[j / (6 * c->N)] : 1.0; }
static inline void ref_cand(const lrdmc_ref_ctx *c, int j, int *mesh, int *i, int *d)
{
    *mesh = j / (6 * c->N); j -= *mesh * 6 * c->N; *i = j / 6; *d = j % 6;
}

int ref_invert(int n, const double *A /*[n][n] row-major*/, double *Ainv, double *logabs, int *sign);
/* non-local slot j >= P_lat of configuration x in frame U: electron, target point, amplitude nu_q = V^nl_{x',x};
 * returns 0 if the slot is inactive (fewer than kk+1 centres in range) */
int ref_nl_slot(const lrdmc_ref_ctx *c, const double *x, const double U[9], int j, int *i_out, double rp[3], double *nu);
void ref_apply_move(const lrdmc_ref_ctx *c, double *x, double *dinv_up, double *dinv_dn, int i, const double rnew[3]);

#endif
