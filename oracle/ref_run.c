/* oracle/ref_run.c -- ORACLE (test infrastructure): walker ensemble, the two projection loops
 * (Alg.2 L389-L423 load-balanced; Alg.1 L311-L387 conventional), branching (Eq.15-17) and the per-generation
 * sums of Eq.20 / Eq.34.  OpenMP over walkers only ("all walkers evolve independently", L25).
 */
#include "ref_internal.h"
#ifdef _OPENMP
#include <omp.h>
#endif

static double *dupd(const double *p, size_t n) { if (!p) return NULL; double *q = (double *)malloc(sizeof(double) * (n ? n : 1)); memcpy(q, p, sizeof(double) * n); return q; }
static int *dupi(const int *p, size_t n) { int *q = (int *)malloc(sizeof(int) * (n ? n : 1)); memcpy(q, p, sizeof(int) * n); return q; }

int lrdmc_ref_create(lrdmc_ref_ctx **out, int n_nuc, const double *Z, const double *Rnuc, const double *pp,
                     int n_up, int n_dn, int n_shell, const int *center, const int *type, const double *zeta,
                     int n_ao, const double *C_up, const double *C_dn, double a_par, double a_anti, double b2,
                     const double *c1, const double *b1, double a, double a2, uint64_t seed)
{
    if (!out || n_nuc < 1 || n_up < 1 || n_dn < 0 || n_up > REF_MAX_OCC || n_dn > REF_MAX_OCC || n_shell < 1 || !(a > 0.0) || a2 < 0.0)
        return LRDMC_REF_EINVAL;
    lrdmc_ref_ctx *c = (lrdmc_ref_ctx *)calloc(1, sizeof(*c));
    c->n_nuc = n_nuc; c->Z = dupd(Z, n_nuc); c->Rn = dupd(Rnuc, 3 * (size_t)n_nuc); c->pp = dupd(pp, 4 * (size_t)n_nuc);
    c->n_up = n_up; c->n_dn = n_dn; c->N = n_up + n_dn;
    c->n_shell = n_shell; c->center = dupi(center, n_shell); c->type = dupi(type, n_shell); c->zeta = dupd(zeta, n_shell);
    c->ao0 = (int *)malloc(sizeof(int) * (size_t)n_shell);
    int mu = 0;
    for (int s = 0; s < n_shell; ++s) {
        c->ao0[s] = mu;
        int t = type[s]; mu += (t == 0 || t == 10) ? 1 : (t == 1 ? 3 : (t == 2 ? 6 : -100000));
        if (center[s] < 0 || center[s] >= n_nuc || !(zeta[s] > 0.0)) mu = -100000;
    }
    if (mu < 0) { lrdmc_ref_destroy(c); return LRDMC_REF_EINVAL; }
    c->n_pao = mu; c->need_contraction = (mu != n_ao);      /* fewer functions than primitives: lrdmc_ref_set_contraction must follow */
    c->n_ao = n_ao; c->C_up = dupd(C_up, (size_t)n_ao * n_up); c->C_dn = dupd(C_dn, (size_t)n_ao * n_dn);
    c->a_par = a_par; c->a_anti = a_anti; c->b2 = b2; c->c1 = dupd(c1, n_nuc); c->b1 = c1 ? dupd(b1, n_nuc) : NULL;
    /* lattice: single mesh, or the double mesh of reading Q13: constant mixing g = 1/2 between a and a' */
    c->a = a; c->a2 = a2; c->n_mesh = a2 > 0.0 ? 2 : 1;
    c->amesh[0] = a; c->amesh[1] = a2; c->gmesh[0] = a2 > 0.0 ? 0.5 : 1.0; c->gmesh[1] = a2 > 0.0 ? 0.5 : 0.0;
    for (int m = 0; m < c->n_mesh; ++m) c->kappa[m] = c->gmesh[m] / (2.0 * c->amesh[m] * c->amesh[m]);
    c->P_lat = 6 * c->N * c->n_mesh; c->P = c->P_lat; c->seed = seed;
    c->V_ii = 0.0;
    for (int I = 0; I < n_nuc; ++I) for (int J = I + 1; J < n_nuc; ++J) {
        double dx = Rnuc[3 * I] - Rnuc[3 * J], dy = Rnuc[3 * I + 1] - Rnuc[3 * J + 1], dz = Rnuc[3 * I + 2] - Rnuc[3 * J + 2];
        c->V_ii += Z[I] * Z[J] / sqrt(dx * dx + dy * dy + dz * dz);
    }
    *out = c;
    return LRDMC_REF_OK;
}

static void free_walkers(lrdmc_ref_ctx *c)
{
    free(c->r); free(c->dinv_up); free(c->dinv_dn); free(c->w); free(c->eL); free(c->W); free(c->omega); free(c->nmoves);
    free(c->flag_node); free(c->flag_nonpos); free(c->flag_nonfinite); free(c->dead); c->dead = NULL; c->n_singular = 0;
    c->r = c->dinv_up = c->dinv_dn = c->w = c->eL = c->W = c->omega = NULL; c->nmoves = NULL;
    c->flag_node = c->flag_nonpos = c->flag_nonfinite = NULL; c->n_w = 0; c->have_obs = 0;
}

void lrdmc_ref_destroy(lrdmc_ref_ctx *c)
{
    if (!c) return;
    free_walkers(c);
    free(c->Z); free(c->Rn); free(c->pp); free(c->center); free(c->type); free(c->zeta); free(c->ao0);
    free(c->C_up); free(c->C_dn); free(c->c1); free(c->b1); free(c->nl); free(c->j3_center); free(c->j3_zeta); free(c->j3_g); free(c->j3_lmn); free(c->cs_first); free(c->cs_sph); free(c->prim_coef); free(c);
}

int lrdmc_ref_n_candidates(const lrdmc_ref_ctx *c) { return c->P; }

int lrdmc_ref_set_contraction(lrdmc_ref_ctx *c, int n_cshell, const int *first, const double *coef, const int *sph)
{
    if (!c || n_cshell < 1 || !first || !coef || !sph || first[0] != 0 || first[n_cshell] != c->n_shell || c->n_w) return LRDMC_REF_EINVAL;
    int nao = 0;
    for (int cs = 0; cs < n_cshell; ++cs) {
        if (first[cs + 1] <= first[cs]) return LRDMC_REF_EINVAL;
        int t = c->type[first[cs]], I = c->center[first[cs]];
        for (int k = first[cs]; k < first[cs + 1]; ++k) if (c->type[k] != t || c->center[k] != I) return LRDMC_REF_EINVAL;
        nao += (t == 1) ? 3 : (t == 2 ? (sph[cs] ? 5 : 6) : 1);
    }
    if (nao != c->n_ao) return LRDMC_REF_EINVAL;
    c->n_cshell = n_cshell; c->cs_first = dupi(first, (size_t)n_cshell + 1); c->cs_sph = dupi(sph, n_cshell); c->prim_coef = dupd(coef, c->n_shell);
    c->need_contraction = 0;
    return LRDMC_REF_OK;
}

int lrdmc_ref_set_jastrow3(lrdmc_ref_ctx *c, int n, const int *center, const double *zeta, const double *g, const int *lmn)
{
    if (!c || n < 0 || (n > 0 && (!center || !zeta || !g)) || c->n_w) return LRDMC_REF_EINVAL;
    for (int a = 0; a < n; ++a) {
        if (center[a] < 0 || center[a] >= c->n_nuc || !(zeta[a] > 0.0)) return LRDMC_REF_EINVAL;
        if (lmn && (lmn[3 * a] < 0 || lmn[3 * a + 1] < 0 || lmn[3 * a + 2] < 0 || lmn[3 * a] + lmn[3 * a + 1] + lmn[3 * a + 2] > 2)) return LRDMC_REF_EINVAL;
        for (int b = 0; b < n; ++b) if (g[a * n + b] != g[b * n + a]) return LRDMC_REF_EINVAL;
    }
    free(c->j3_center); free(c->j3_zeta); free(c->j3_g); free(c->j3_lmn);
    c->n_j3 = n; c->j3_center = n ? dupi(center, n) : NULL; c->j3_zeta = dupd(n ? zeta : NULL, n); c->j3_g = dupd(n ? g : NULL, (size_t)n * n);
    c->j3_lmn = (n && lmn) ? dupi(lmn, 3 * n) : NULL;
    return LRDMC_REF_OK;
}

int lrdmc_ref_set_nonlocal(lrdmc_ref_ctx *c, int K, int dla, const double *nl)
{
    if (!c || K < 0 || (K > 0 && !nl) || c->n_w) return LRDMC_REF_EINVAL;
    free(c->nl); c->nl = NULL; c->nl_K = 0; c->P = c->P_lat;
    if (K == 0) return LRDMC_REF_OK;
    c->nl = dupd(nl, 7 * (size_t)c->n_nuc); c->nl_K = K; c->nl_dla = dla ? 1 : 0;
    c->P = c->P_lat + 6 * c->N * K;
    return LRDMC_REF_OK;
}

int lrdmc_ref_set_slot_offset(lrdmc_ref_ctx *c, uint32_t offset) { if (!c) return LRDMC_REF_EINVAL; c->slot0 = offset; return LRDMC_REF_OK; }

int lrdmc_ref_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n; return 1;
#endif
}

static void alloc_walkers(lrdmc_ref_ctx *c, int n_w)
{
    free_walkers(c);
    size_t nw = (size_t)n_w, ou = (size_t)c->n_up * c->n_up, od = (size_t)c->n_dn * c->n_dn;
    c->n_w = n_w;
    c->r = (double *)calloc(nw * 3 * c->N, sizeof(double));
    c->dinv_up = (double *)calloc(nw * ou + 1, sizeof(double)); c->dinv_dn = (double *)calloc(nw * od + 1, sizeof(double));
    c->w = (double *)calloc(nw, sizeof(double)); c->eL = (double *)calloc(nw, sizeof(double));
    c->W = (double *)calloc(nw, sizeof(double)); c->omega = (double *)calloc(nw, sizeof(double));
    c->nmoves = (int64_t *)calloc(nw, sizeof(int64_t));
    c->flag_node = (int *)calloc(nw, sizeof(int)); c->flag_nonpos = (int *)calloc(nw, sizeof(int)); c->flag_nonfinite = (int *)calloc(nw, sizeof(int));
    c->dead = (int *)calloc(nw, sizeof(int));
    for (int k = 0; k < n_w; ++k) c->w[k] = 1.0;
}

/* inverses of every walker from its positions (row a13); singular walkers are marked dead, their inverses zeroed (reading Q24) */
static int rebuild_all(lrdmc_ref_ctx *c)
{
    size_t ou = (size_t)c->n_up * c->n_up, od = (size_t)c->n_dn * c->n_dn; int64_t bad = 0;
    #pragma omp parallel for schedule(dynamic) reduction(+:bad)
    for (int k = 0; k < c->n_w; ++k) {
        c->dead[k] = lrdmc_ref_build_inverse(c, c->r + (size_t)k * 3 * c->N, c->dinv_up + k * ou, c->dinv_dn + k * od) != 0;
        if (c->dead[k]) { memset(c->dinv_up + k * ou, 0, sizeof(double) * ou); memset(c->dinv_dn + k * od, 0, sizeof(double) * od); ++bad; }
    }
    c->n_singular = bad;
    return bad ? LRDMC_REF_ESINGULAR : LRDMC_REF_OK;
}

int lrdmc_ref_set_positions(lrdmc_ref_ctx *c, int n_w, const double *r)
{
    if (!c || n_w < 1 || !r) return LRDMC_REF_EINVAL;
    if (c->need_contraction) return LRDMC_REF_ESTATE;
    alloc_walkers(c, n_w);
    memcpy(c->r, r, sizeof(double) * (size_t)n_w * 3 * c->N);
    return rebuild_all(c);
}

int lrdmc_ref_get_state(const lrdmc_ref_ctx *c, double *r, double *dinv_up, double *dinv_dn, double *w)
{
    if (!c->n_w) return LRDMC_REF_ESTATE;
    size_t nw = (size_t)c->n_w;
    if (r) memcpy(r, c->r, sizeof(double) * nw * 3 * c->N);
    if (dinv_up) memcpy(dinv_up, c->dinv_up, sizeof(double) * nw * c->n_up * c->n_up);
    if (dinv_dn) memcpy(dinv_dn, c->dinv_dn, sizeof(double) * nw * c->n_dn * c->n_dn);
    if (w) memcpy(w, c->w, sizeof(double) * nw);
    return LRDMC_REF_OK;
}

int lrdmc_ref_set_state(lrdmc_ref_ctx *c, int n_w, const double *r, const double *dinv_up, const double *dinv_dn, const double *w)
{
    if (!c || n_w < 1 || !r) return LRDMC_REF_EINVAL;
    alloc_walkers(c, n_w);
    size_t nw = (size_t)n_w;
    memcpy(c->r, r, sizeof(double) * nw * 3 * c->N);
    if (dinv_up) {
        memcpy(c->dinv_up, dinv_up, sizeof(double) * nw * c->n_up * c->n_up);
        if (c->n_dn) memcpy(c->dinv_dn, dinv_dn, sizeof(double) * nw * c->n_dn * c->n_dn);
    } else rebuild_all(c);                     /* dead walkers are marked, not an error here (reading Q24) */
    if (w) memcpy(c->w, w, sizeof(double) * nw);
    return LRDMC_REF_OK;
}

int lrdmc_ref_get_obs(const lrdmc_ref_ctx *c, double *eL, double *W, double *omega, int64_t *n_moves)
{
    if (!c->have_obs) return LRDMC_REF_ESTATE;
    size_t nw = (size_t)c->n_w;
    if (eL) memcpy(eL, c->eL, sizeof(double) * nw); if (W) memcpy(W, c->W, sizeof(double) * nw);
    if (omega) memcpy(omega, c->omega, sizeof(double) * nw); if (n_moves) memcpy(n_moves, c->nmoves, sizeof(int64_t) * nw);
    return LRDMC_REF_OK;
}

/* candidate j of walker position x in frame U -> new position of its electron */
static void cand_pos(const lrdmc_ref_ctx *c, const double *x, const double U[9], int j, int *i_out, double rp[3])
{
    if (j >= c->P_lat) { double nu; ref_nl_slot(c, x, U, j, i_out, rp, &nu); return; }   /* non-local hop onto the quadrature point */
    int mesh, i, d; ref_cand(c, j, &mesh, &i, &d);
    int k = d / 2; double step = ((d % 2 == 0) ? 1.0 : -1.0) * c->amesh[mesh];
    rp[0] = x[3 * i] + step * U[k]; rp[1] = x[3 * i + 1] + step * U[3 + k]; rp[2] = x[3 * i + 2] + step * U[6 + k];
    *i_out = i;
}

/* one walker, one branching interval.  mode balanced: Alg.2 lines 4-8; conventional: Alg.1 lines 4-16. */
static void propagate_walker(lrdmc_ref_ctx *c, int k, int mode, int n_moves, double tau, double E0, uint64_t cycle)
{
    int N = c->N, P = c->P;
    if (c->dead[k]) {                                   /* singular at the last (re)build: dies at the next branching (reading Q24) */
        c->w[k] = 0.0; c->omega[k] = 0.0; c->eL[k] = 0.0; c->W[k] = 0.0; c->nmoves[k] = 0; c->flag_node[k] = 0; c->flag_nonpos[k] = 0;
        return;
    }
    double *x = c->r + (size_t)k * 3 * N;
    double *du = c->dinv_up + (size_t)k * c->n_up * c->n_up, *dd = c->dinv_dn + (size_t)k * c->n_dn * c->n_dn;
    double *R = (double *)malloc(sizeof(double) * (size_t)P), scal[10], u[5], U[9], rp[3];
    double w = 1.0, tau_left = tau;                     /* Alg.2 line 4 (L401) / Alg.1 line 4 (L350) */
    int64_t moves = 0; int nnode = 0, nnonpos = 0;
    int64_t cap = (mode == LRDMC_REF_BALANCED) ? n_moves : (n_moves > 0 ? n_moves : ((int64_t)1 << 30));
    for (uint64_t s = 0;; ++s) {
        lrdmc_ref_draws(c, c->slot0 + (uint32_t)k, cycle, s, u);
        lrdmc_ref_frame(u[0], u[1], u[2], U);
        lrdmc_ref_evaluate(c, x, du, dd, U, R, scal, NULL, NULL);
        double bbar = scal[0], W = scal[2], eL = scal[3];
        if (scal[4] != 0.0) ++nnode;
        int last = 0;
        if (mode == LRDMC_REF_BALANCED) {
            if ((int64_t)s == cap) {                    /* measurement evaluation at the final x (Q10; Eq.34) */
                double den = W - E0;
                if (!(den > 0.0)) { ++nnonpos; w = 0.0; c->omega[k] = 0.0; } else c->omega[k] = w / den;
                last = 1;
            } else {
                double den = W - E0;                    /* b_x = bbar/(W-E0) (Eq.29, Alg.2 line 6 L406) */
                if (!(den > 0.0)) { ++nnonpos; w = 0.0; } else w *= bbar / den;   /* Q16 */
            }
        } else {
            double tau_xi = -log1p(-u[4]) / bbar;       /* Eq.24 (L160), reading Q1 */
            if (!(tau_xi < tau_left) || (int64_t)s >= cap) { tau_xi = tau_left; last = 1; }   /* Alg.1 min[.,tau_left] (L362) */
            w *= exp(-tau_xi * (eL - E0));              /* Eq.25 (L164) with the constant shift of reading Q8b */
            tau_left -= tau_xi;
            if (last) c->omega[k] = w;                  /* Eq.20 (L135): plain weight */
        }
        if (last) { c->eL[k] = eL; c->W[k] = W; break; }
        int j = lrdmc_ref_select(c, R, u[3], NULL);     /* Alg.2 line 7 (L408) / Alg.1 */
        if (j >= 0) { int i; cand_pos(c, x, U, j, &i, rp); ref_apply_move(c, x, du, dd, i, rp); ++moves; }
    }
    if (!isfinite(w) || !isfinite(c->omega[k])) { c->flag_nonfinite[k] = 1; w = 0.0; c->omega[k] = 0.0; }
    c->w[k] = w; c->nmoves[k] = moves; c->flag_node[k] = nnode; c->flag_nonpos[k] = nnonpos;
    free(R);
}

int lrdmc_ref_propagate(lrdmc_ref_ctx *c, int mode, int n_moves, double tau, double E0, uint64_t cycle)
{
    if (!c || !c->n_w) return LRDMC_REF_ESTATE;
    if ((mode == LRDMC_REF_BALANCED && n_moves < 0) || (mode == LRDMC_REF_CONVENTIONAL && !(tau > 0.0)) || (mode != 0 && mode != 1)
        || cycle > 0xFFFFFFFFull) return LRDMC_REF_EINVAL;
    memset(c->flag_nonfinite, 0, sizeof(int) * (size_t)c->n_w);
    #pragma omp parallel for schedule(dynamic)
    for (int k = 0; k < c->n_w; ++k) propagate_walker(c, k, mode, n_moves, tau, E0, cycle);
    c->have_obs = 1;
    return LRDMC_REF_OK;
}

int lrdmc_ref_estimators(const lrdmc_ref_ctx *c, lrdmc_ref_stats *out)
{
    if (!c->have_obs) return LRDMC_REF_ESTATE;
    memset(out, 0, sizeof(*out));
    out->wbar = c->wbar; out->moves_min = INT64_MAX; out->n_singular = c->n_singular;
    for (int k = 0; k < c->n_w; ++k) {
        out->num += c->omega[k] * c->eL[k]; out->den += c->omega[k];   /* Eq.34 (L227) / Eq.20 (L135) */
        if (c->nmoves[k] < out->moves_min) out->moves_min = c->nmoves[k];
        if (c->nmoves[k] > out->moves_max) out->moves_max = c->nmoves[k];
        out->moves_sum += c->nmoves[k];
        out->n_node_flag += c->flag_node[k]; out->n_nonpos_diag += c->flag_nonpos[k]; out->n_nonfinite += c->flag_nonfinite[k];
    }
    out->lockstep_idle_frac = out->moves_max > 0 ? 1.0 - (double)out->moves_sum / ((double)c->n_w * (double)out->moves_max) : 0.0;
    return LRDMC_REF_OK;
}

/* Branching: comb on the raw weights w (Eq.15-17; L225 "Eqs.15-19 perfectly hold"), copy the survivors,
 * all weights <- 1 with wbar recorded (L129), inverses rebuilt from the positions (reading Q15). */
int lrdmc_ref_reconfigure(lrdmc_ref_ctx *c, uint64_t cycle, int32_t *parents_out)
{
    if (!c || !c->n_w) return LRDMC_REF_ESTATE;
    int n_w = c->n_w; size_t rec = 3 * (size_t)c->N;
    int32_t *par = (int32_t *)malloc(sizeof(int32_t) * (size_t)n_w);
    lrdmc_ref_comb(n_w, c->w, lrdmc_ref_comb_r32(c, cycle), par, &c->wbar, NULL, NULL, NULL);
    double *rn = (double *)malloc(sizeof(double) * (size_t)n_w * rec);
    for (int k = 0; k < n_w; ++k) memcpy(rn + k * rec, c->r + par[k] * rec, sizeof(double) * rec);
    memcpy(c->r, rn, sizeof(double) * (size_t)n_w * rec);
    for (int k = 0; k < n_w; ++k) c->w[k] = 1.0;
    if (parents_out) memcpy(parents_out, par, sizeof(int32_t) * (size_t)n_w);
    free(rn); free(par);
    rebuild_all(c);                             /* singular walkers: marked dead and counted in the stats (reading Q24), not an error */
    return LRDMC_REF_OK;
}

int lrdmc_ref_step_debug(const lrdmc_ref_ctx *c, double E0, uint64_t cycle, uint64_t step, double *R, double *scal, int32_t *jstar)
{
    if (!c || !c->n_w) return LRDMC_REF_ESTATE;
    int P = c->P;
    #pragma omp parallel for schedule(dynamic)
    for (int k = 0; k < c->n_w; ++k) {
        double u[5], U[9], s10[10], mg;
        lrdmc_ref_draws(c, c->slot0 + (uint32_t)k, cycle, step, u);
        lrdmc_ref_frame(u[0], u[1], u[2], U);
        lrdmc_ref_evaluate(c, c->r + (size_t)k * 3 * c->N, c->dinv_up + (size_t)k * c->n_up * c->n_up,
                           c->dinv_dn + (size_t)k * c->n_dn * c->n_dn, U, R + (size_t)k * P, s10, NULL, NULL);
        jstar[k] = lrdmc_ref_select(c, R + (size_t)k * P, u[3], &mg);
        double *o = scal + 8 * (size_t)k;
        o[0] = s10[0]; o[1] = s10[1]; o[2] = s10[2]; o[3] = s10[3]; o[4] = s10[0] / (s10[2] - E0);
        o[5] = -log1p(-u[4]) / s10[0]; o[6] = s10[4]; o[7] = mg;
    }
    return LRDMC_REF_OK;
}
