/* oracle/ref_wf.c -- ORACLE (test infrastructure): trial wavefunction Psi_G = D_up D_dn exp(J).
 *
 * The paper names the ansatz only ("Slater determinant x Jastrow", Gaussian basis: PAPER.md L242, L285,
 * "D_G determinant part" L576); the functional forms are DESIGN.md reading Q14:
 *   AO   cartesian Gaussian primitive  chi = N_lmn x^l y^m z^n exp(-zeta |r-R_c|^2),
 *        N_lmn = (2 zeta/pi)^(3/4) (4 zeta)^((l+m+n)/2) / sqrt((2l-1)!!(2m-1)!!(2n-1)!!)  (unit self-overlap),
 *        order s | x y z | xx xy xz yy yz zz;   type 10: Slater s, chi = exp(-zeta |r-R_c|).
 *   MO   phi_m(r) = sum_mu chi_mu(r) C[mu][m];  D_sigma[i][m] = phi_m(r_i).
 *   J    = sum_{i,I} u1_I(r_iI) + sum_{i<j} u2(r_ij),  u1_I = -c1_I r/(1+b1_I r),  u2 = a_ss' r/(1+b2 r).
 */
#include "ref_internal.h"

static const int CART_D[6][3] = { {2,0,0}, {1,1,0}, {1,0,1}, {0,2,0}, {0,1,1}, {0,0,2} };

static double dfact_odd(int k) /* (2k-1)!! */ { double f = 1.0; for (int j = 1; j <= k; ++j) f *= (2 * j - 1); return f; }

static double ipow(double v, int k) { double p = 1.0; for (int j = 0; j < k; ++j) p *= v; return p; }

/* one cartesian primitive and its gradient / Laplacian, written as polynomials (never divides by a coordinate):
 * d/dv [v^k e^{-z v^2}] = (k v^{k-1} - 2 z v^{k+1}) e,  d2/dv2 = (k(k-1) v^{k-2} - 2z(2k+1) v^k + 4 z^2 v^{k+2}) e */
static void cart_gto(double zeta, const int lmn[3], const double d[3], double *val, double g[3], double *lap)
{
    int L = lmn[0] + lmn[1] + lmn[2];
    double norm = pow(2.0 * zeta / M_PI, 0.75) * pow(4.0 * zeta, 0.5 * L)
                  / sqrt(dfact_odd(lmn[0]) * dfact_odd(lmn[1]) * dfact_odd(lmn[2]));
    double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
    double e = norm * exp(-zeta * r2);
    double f[3], f1[3], f2[3];
    for (int ax = 0; ax < 3; ++ax) {
        int k = lmn[ax]; double v = d[ax];
        f[ax] = ipow(v, k);
        f1[ax] = (k >= 1 ? k * ipow(v, k - 1) : 0.0) - 2.0 * zeta * ipow(v, k + 1);
        f2[ax] = (k >= 2 ? k * (k - 1) * ipow(v, k - 2) : 0.0) - 2.0 * zeta * (2 * k + 1) * ipow(v, k)
                 + 4.0 * zeta * zeta * ipow(v, k + 2);
    }
    *val = e * f[0] * f[1] * f[2];
    g[0] = e * f1[0] * f[1] * f[2]; g[1] = e * f[0] * f1[1] * f[2]; g[2] = e * f[0] * f[1] * f1[2];
    *lap = e * (f2[0] * f[1] * f[2] + f[0] * f2[1] * f[2] + f[0] * f[1] * f2[2]);
}

/* the primitive functions, one after the other in shell order */
static int ao_primitives(const lrdmc_ref_ctx *c, const double r[3], double *val, double *grad, double *lap)
{
    for (int s = 0; s < c->n_shell; ++s) {
        const double *Rc = c->Rn + 3 * c->center[s];
        double d[3] = { r[0] - Rc[0], r[1] - Rc[1], r[2] - Rc[2] };
        double z = c->zeta[s]; int mu = c->ao0[s];
        if (c->type[s] == 10) {         /* Slater s: grad = -z chi rhat, lap = chi (z^2 - 2 z / r) */
            double rr = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            double v = exp(-z * rr);
            val[mu] = v;
            for (int ax = 0; ax < 3; ++ax) grad[3 * mu + ax] = -z * v * d[ax] / rr;
            lap[mu] = v * (z * z - 2.0 * z / rr);
        } else if (c->type[s] == 0) {
            int lmn[3] = { 0, 0, 0 };
            cart_gto(z, lmn, d, &val[mu], &grad[3 * mu], &lap[mu]);
        } else if (c->type[s] == 1) {
            for (int k = 0; k < 3; ++k) {
                int lmn[3] = { k == 0, k == 1, k == 2 };
                cart_gto(z, lmn, d, &val[mu + k], &grad[3 * (mu + k)], &lap[mu + k]);
            }
        } else if (c->type[s] == 2) {
            for (int k = 0; k < 6; ++k) cart_gto(z, CART_D[k], d, &val[mu + k], &grad[3 * (mu + k)], &lap[mu + k]);
        } else return LRDMC_REF_EINVAL;
    }
    return LRDMC_REF_OK;
}

/* AO values: the primitives themselves, or the contracted / solid-harmonic functions of lrdmc_ref_set_contraction */
int lrdmc_ref_ao(const lrdmc_ref_ctx *c, const double r[3], double *val, double *grad, double *lap)
{
    if (c->need_contraction) return LRDMC_REF_ESTATE;
    if (!c->n_cshell) return ao_primitives(c, r, val, grad, lap);
    int np = c->n_pao;
    double *pv = (double *)malloc(sizeof(double) * 5 * (size_t)np), *pg = pv + np, *pl = pv + 4 * np;
    int rc = ao_primitives(c, r, pv, pg, pl);
    const double h3 = sqrt(3.0) / 2.0;
    int nu = 0;
    for (int cs = 0; cs < c->n_cshell; ++cs) {
        int t = c->type[c->cs_first[cs]], ncart = (t == 1) ? 3 : (t == 2 ? 6 : 1);
        double cv[6] = { 0 }, cg[18] = { 0 }, cl[6] = { 0 };                 /* contracted cartesian components */
        for (int k = c->cs_first[cs]; k < c->cs_first[cs + 1]; ++k)
            for (int q = 0; q < ncart; ++q) {
                int mu = c->ao0[k] + q; double d = c->prim_coef[k];
                cv[q] += d * pv[mu]; cl[q] += d * pl[mu];
                for (int ax = 0; ax < 3; ++ax) cg[3 * q + ax] += d * pg[3 * mu + ax];
            }
        if (t == 2 && c->cs_sph[cs]) {                                        /* xx xy xz yy yz zz -> z2, xz, yz, x2-y2, xy */
            double w[5][6] = { { -0.5, 0, 0, -0.5, 0, 1.0 }, { 0, 0, 1, 0, 0, 0 }, { 0, 0, 0, 0, 1, 0 }, { h3, 0, 0, -h3, 0, 0 }, { 0, 1, 0, 0, 0, 0 } };
            for (int m = 0; m < 5; ++m, ++nu) {
                double v = 0, l = 0, g[3] = { 0, 0, 0 };
                for (int q = 0; q < 6; ++q) { v += w[m][q] * cv[q]; l += w[m][q] * cl[q]; for (int ax = 0; ax < 3; ++ax) g[ax] += w[m][q] * cg[3 * q + ax]; }
                val[nu] = v; lap[nu] = l; for (int ax = 0; ax < 3; ++ax) grad[3 * nu + ax] = g[ax];
            }
        } else for (int q = 0; q < ncart; ++q, ++nu) { val[nu] = cv[q]; lap[nu] = cl[q]; for (int ax = 0; ax < 3; ++ax) grad[3 * nu + ax] = cg[3 * q + ax]; }
    }
    free(pv);
    return rc;
}

int lrdmc_ref_mo(const lrdmc_ref_ctx *c, int spin, const double r[3], double *val, double *grad, double *lap)
{
    int O = ref_nocc(c, spin), A = c->n_ao; const double *C = ref_C(c, spin);
    double *av = (double *)malloc(sizeof(double) * 5 * (size_t)A), *ag = av + A, *al = av + 4 * A;
    int rc = lrdmc_ref_ao(c, r, av, ag, al);
    for (int m = 0; m < O; ++m) {
        double v = 0, gx = 0, gy = 0, gz = 0, l = 0;
        for (int mu = 0; mu < A; ++mu) {
            double cm = C[(size_t)mu * O + m];
            v += av[mu] * cm; gx += ag[3 * mu] * cm; gy += ag[3 * mu + 1] * cm; gz += ag[3 * mu + 2] * cm; l += al[mu] * cm;
        }
        if (val) val[m] = v;
        if (grad) { grad[3 * m] = gx; grad[3 * m + 1] = gy; grad[3 * m + 2] = gz; }
        if (lap) lap[m] = l;
    }
    free(av);
    return rc;
}

/* Gauss-Jordan inverse with partial (row) pivoting; also log|det| and its sign.
 * ESINGULAR when a pivot is not above 2^-44 max|A_ij| (reading Q24 of DESIGN.md: "|D| = 0" in FP64.  Two identical rows -- two
 * same-spin electrons at one point -- leave a pivot of rounding size ~2^-52 max|A|, not an exact zero; a matrix whose pivots fall
 * below 2^-44 has lost all but 8 bits of its inverse anyway). */
int ref_invert(int n, const double *A, double *Ainv, double *logabs, int *sign)
{
    double la = 0.0; int sg = 1;
    if (n == 0) { if (logabs) *logabs = 0.0; if (sign) *sign = 1; return LRDMC_REF_OK; }
    double amax = 0.0;
    for (int i = 0; i < n * n; ++i) if (fabs(A[i]) > amax) amax = fabs(A[i]);
    const double tiny = ldexp(amax, -44);
    double *M = (double *)malloc(sizeof(double) * 2 * (size_t)n * n);
    for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) { M[i * 2 * n + j] = A[i * n + j]; M[i * 2 * n + n + j] = (i == j); }
    for (int col = 0; col < n; ++col) {
        int piv = col; double best = fabs(M[col * 2 * n + col]);
        for (int i = col + 1; i < n; ++i) if (fabs(M[i * 2 * n + col]) > best) { best = fabs(M[i * 2 * n + col]); piv = i; }
        if (!(best > tiny) || !isfinite(best)) { free(M); return LRDMC_REF_ESINGULAR; }
        if (piv != col) { for (int j = 0; j < 2 * n; ++j) { double t = M[col * 2 * n + j]; M[col * 2 * n + j] = M[piv * 2 * n + j]; M[piv * 2 * n + j] = t; } sg = -sg; }
        double p = M[col * 2 * n + col];
        la += log(fabs(p)); if (p < 0) sg = -sg;
        for (int j = 0; j < 2 * n; ++j) M[col * 2 * n + j] /= p;
        for (int i = 0; i < n; ++i) if (i != col) {
            double f = M[i * 2 * n + col];
            if (f != 0.0) for (int j = 0; j < 2 * n; ++j) M[i * 2 * n + j] -= f * M[col * 2 * n + j];
        }
    }
    if (Ainv) for (int i = 0; i < n; ++i) for (int j = 0; j < n; ++j) Ainv[i * n + j] = M[i * 2 * n + n + j];
    if (logabs) *logabs = la; if (sign) *sign = sg;
    free(M);
    return LRDMC_REF_OK;
}

static void slater_matrix(const lrdmc_ref_ctx *c, int spin, const double *x, double *D /*[O][O]: D[i][m]*/)
{
    int O = ref_nocc(c, spin), off = spin ? c->n_up : 0;
    for (int i = 0; i < O; ++i) lrdmc_ref_mo(c, spin, x + 3 * (off + i), D + (size_t)i * O, NULL, NULL);
}

/* Dinv_sigma[m][i] with sum_m D[i][m] Dinv[m][k] = delta_ik  (row-major [O][O]) */
int lrdmc_ref_build_inverse(const lrdmc_ref_ctx *c, const double *x, double *dinv_up, double *dinv_dn)
{
    for (int spin = 0; spin < 2; ++spin) {
        int O = ref_nocc(c, spin); if (!O) continue;
        double *D = (double *)malloc(sizeof(double) * (size_t)O * O);
        slater_matrix(c, spin, x, D);
        int rc = ref_invert(O, D, spin ? dinv_dn : dinv_up, NULL, NULL);
        free(D);
        if (rc) return rc;
    }
    return LRDMC_REF_OK;
}

static double pade(double cc, double b, double r) { return cc * r / (1.0 + b * r); }

/* log|Psi_G| and sign from scratch: pivoted elimination of both Slater matrices + the full Jastrow double sum */
int lrdmc_ref_logpsi(const lrdmc_ref_ctx *c, const double *x, double *logabs, int *sign)
{
    double la = 0.0; int sg = 1;
    for (int spin = 0; spin < 2; ++spin) {
        int O = ref_nocc(c, spin); if (!O) continue;
        double *D = (double *)malloc(sizeof(double) * (size_t)O * O), l; int s;
        slater_matrix(c, spin, x, D);
        int rc = ref_invert(O, D, NULL, &l, &s);
        free(D);
        if (rc) return rc;
        la += l; sg *= s;
    }
    double J = 0.0;
    for (int i = 0; i < c->N; ++i) {
        if (c->c1) for (int I = 0; I < c->n_nuc; ++I) {
            double dx = x[3 * i] - c->Rn[3 * I], dy = x[3 * i + 1] - c->Rn[3 * I + 1], dz = x[3 * i + 2] - c->Rn[3 * I + 2];
            J -= pade(c->c1[I], c->b1[I], sqrt(dx * dx + dy * dy + dz * dz));
        }
        for (int j = i + 1; j < c->N; ++j) {
            double dx = x[3 * i] - x[3 * j], dy = x[3 * i + 1] - x[3 * j + 1], dz = x[3 * i + 2] - x[3 * j + 2];
            double aij = ref_spin(c, i) == ref_spin(c, j) ? c->a_par : c->a_anti;
            J += pade(aij, c->b2, sqrt(dx * dx + dy * dy + dz * dz));
        }
    }
    /* three-body term, written as defined: sum_{i<j} sum_{ab} g_ab chi_a(r_i) chi_b(r_j), chi = monomial (j3_lmn, 1 without) x Gaussian */
    for (int i = 0; i < c->N; ++i) for (int j = i + 1; j < c->N; ++j)
        for (int a = 0; a < c->n_j3; ++a) for (int b = 0; b < c->n_j3; ++b) {
            const double *Ra = c->Rn + 3 * c->j3_center[a], *Rb = c->Rn + 3 * c->j3_center[b];
            double da2 = 0.0, db2 = 0.0, pa = 1.0, pb = 1.0;
            for (int ax = 0; ax < 3; ++ax) {
                double u = x[3 * i + ax] - Ra[ax], v = x[3 * j + ax] - Rb[ax]; da2 += u * u; db2 += v * v;
                if (c->j3_lmn) { pa *= pow(u, c->j3_lmn[3 * a + ax]); pb *= pow(v, c->j3_lmn[3 * b + ax]); }
            }
            J += c->j3_g[a * c->n_j3 + b] * pa * exp(-c->j3_zeta[a] * da2) * pb * exp(-c->j3_zeta[b] * db2);
        }
    *logabs = la + J; *sign = sg;
    return LRDMC_REF_OK;
}

/* Apply the move "electron i -> rnew" (row a10 of the scope table; not in the paper, standard QMC):
 * Sherman-Morrison for the replacement of row i of D_sigma by phi(rnew).  With rho = sum_m phi_m Dinv[m][i]
 * (the determinant ratio) and s_k = sum_m phi_m Dinv[m][k]:
 *   Dinv'[m][i] = Dinv[m][i] / rho,   Dinv'[m][k] = Dinv[m][k] - Dinv[m][i] s_k / rho  (k != i). */
void ref_apply_move(const lrdmc_ref_ctx *c, double *x, double *dinv_up, double *dinv_dn, int i, const double rnew[3])
{
    int spin = ref_spin(c, i), il = ref_local(c, i), O = ref_nocc(c, spin);
    double *Dinv = spin ? dinv_dn : dinv_up;
    double phi[REF_MAX_OCC], s[REF_MAX_OCC], col[REF_MAX_OCC];
    lrdmc_ref_mo(c, spin, rnew, phi, NULL, NULL);
    for (int k = 0; k < O; ++k) { double t = 0.0; for (int m = 0; m < O; ++m) t += phi[m] * Dinv[m * O + k]; s[k] = t; }
    double rho = s[il];
    for (int m = 0; m < O; ++m) col[m] = Dinv[m * O + il];
    for (int m = 0; m < O; ++m)
        for (int k = 0; k < O; ++k)
            Dinv[m * O + k] = (k == il) ? col[m] / rho : Dinv[m * O + k] - col[m] * s[k] / rho;
    x[3 * i] = rnew[0]; x[3 * i + 1] = rnew[1]; x[3 * i + 2] = rnew[2];
}
