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
    double *C_up, *C_dn;             /* [n_ao][n_up], [n_ao][n_dn] */
    /* Jastrow */
    double a_par, a_anti, b2; double *c1, *b1; /* c1 NULL: no one-body term */
    /* lattice */
    double a, a2; int n_mesh; double amesh[2], gmesh[2], kappa[2]; /* kappa_m = g_m / (2 a_m^2) */
    int P;                           /* 6 N n_mesh candidates */
    uint64_t seed;
    double V_ii;
    /* walkers */
    int n_w; double *r, *dinv_up, *dinv_dn, *w, *eL, *W, *omega; int64_t *nmoves;
    int *flag_node, *flag_nonpos, *flag_nonfinite; /* per-walker event counts of the last cycle */
    double wbar; int have_obs;
};

static inline int ref_nocc(const lrdmc_ref_ctx *c, int spin) { return spin ? c->n_dn : c->n_up; }
static inline const double *ref_C(const lrdmc_ref_ctx *c, int spin) { return spin ? c->C_dn : c->C_up; }
/* electron i: spin 0 (up) for i < n_up, else spin 1; index inside its spin block */
static inline int ref_spin(const lrdmc_ref_ctx *c, int i) { return i < c->n_up ? 0 : 1; }
static inline int ref_local(const lrdmc_ref_ctx *c, int i) { return i < c->n_up ? i : i - c->n_up; }

/* candidate j -> (mesh block, electron, direction d in 0..5); displacement sign and versor index */
static inline void ref_cand(const lrdmc_ref_ctx *c, int j, int *mesh, int *i, int *d)
{
    *mesh = j / (6 * c->N); j -= *mesh * 6 * c->N; *i = j / 6; *d = j % 6;
}

int ref_invert(int n, const double *A /*[n][n] row-major*/, double *Ainv, double *logabs, int *sign);
void ref_apply_move(const lrdmc_ref_ctx *c, double *x, double *dinv_up, double *dinv_dn, int i, const double rnew[3]);

#endif
