/* oracle/ref_ham.c -- ORACLE (test infrastructure): one evaluation of the lattice-regularised fixed-node
 * Hamiltonian at a configuration x (Appendix D) and the heat-bath selection
 * (Eq.29, Alg.2 line 7 L408).  Written in the paper's order; no blocking, no fusion.
 */
#include "ref_internal.h"

/* Pade pair term u = c r/(1+b r): value, u' = c/(1+br)^2, lap u = u'' + 2u'/r = 2c/(r (1+br)^3) */
static void pade3(double cc, double b, double r, double *u, double *du, double *lapu)
{
    double q = 1.0 + b * r;
    *u = cc * r / q; *du = cc / (q * q); *lapu = 2.0 * cc / (r * q * q * q);
}

/* bare or local-pseudopotential electron-ion potential of nucleus I at distance r (reading Q14):
 *   all-electron: -Z/r;   local PP: -(Z/r)(1-e^{-alpha r^2}) + Z alpha r e^{-beta r^2} + gamma e^{-delta r^2} */
static double v_nuc(const lrdmc_ref_ctx *c, int I, double r)
{
    double Z = c->Z[I];
    if (!c->pp || !(c->pp[4 * I] > 0.0)) return -Z / r;
    double al = c->pp[4 * I], be = c->pp[4 * I + 1], ga = c->pp[4 * I + 2], de = c->pp[4 * I + 3];
    return Z * expm1(-al * r * r) / r + Z * al * r * exp(-be * r * r) + ga * exp(-de * r * r);
}

/* lower bound v^a_ei of Eq.D10 (L620): -Z/max(r,a) for a bare nucleus; -Z_eff/r for an ECP nucleus (L623) */
static double v_nuc_bound(const lrdmc_ref_ctx *c, int I, double r)
{
    if (!c->pp || !(c->pp[4 * I] > 0.0)) return -c->Z[I] / (r > c->a ? r : c->a);
    return -c->Z[I] / r;
}

static double dist(const double *p, const double *q)
{
    double dx = p[0] - q[0], dy = p[1] - q[1], dz = p[2] - q[2];
    return sqrt(dx * dx + dy * dy + dz * dz);
}

/* chi_a(r) = dx^l dy^m dz^n exp(-zeta_a |d|^2), d = r - R_a, of the three-body Jastrow (l = m = n = 0 without j3_lmn), optionally
 * with gradient and Laplacian.  Per axis, u(v) = v^k exp(-zeta v^2):  u' = (k v^(k-1) - 2 zeta v^(k+1)) e,
 * u'' = (k (k-1) v^(k-2) - 2 zeta (2k+1) v^k + 4 zeta^2 v^(k+2)) e; chi is the product of the three axis functions. */
static double ipow(double v, int k) { double p = 1.0; for (int q = 0; q < k; ++q) p *= v; return k < 0 ? 0.0 : p; }
static double j3_chi(const lrdmc_ref_ctx *c, int a, const double r[3], double g[3], double *lap)
{
    const double *Ra = c->Rn + 3 * c->j3_center[a]; double z = c->j3_zeta[a];
    double u[3], u1[3], u2[3];
    for (int ax = 0; ax < 3; ++ax) {
        int k = c->j3_lmn ? c->j3_lmn[3 * a + ax] : 0; double v = r[ax] - Ra[ax], e = exp(-z * v * v);
        u[ax] = ipow(v, k) * e;
        u1[ax] = (k * ipow(v, k - 1) - 2.0 * z * ipow(v, k + 1)) * e;
        u2[ax] = (k * (k - 1) * ipow(v, k - 2) - 2.0 * z * (2 * k + 1) * ipow(v, k) + 4.0 * z * z * ipow(v, k + 2)) * e;
    }
    if (g) { g[0] = u1[0] * u[1] * u[2]; g[1] = u[0] * u1[1] * u[2]; g[2] = u[0] * u[1] * u1[2]; }
    if (lap) *lap = u2[0] * u[1] * u[2] + u[0] * u2[1] * u[2] + u[0] * u[1] * u2[2];
    return u[0] * u[1] * u[2];
}
/* V_a(i) = sum_{j != i} sum_b g_ab chi_b(r_j): the three-body field electron i feels through basis function a */
static double j3_field(const lrdmc_ref_ctx *c, const double *x, int i, int a)
{
    double V = 0.0;
    for (int j = 0; j < c->N; ++j) if (j != i) for (int b = 0; b < c->n_j3; ++b) V += c->j3_g[a * c->n_j3 + b] * j3_chi(c, b, x + 3 * j, NULL, NULL);
    return V;
}

/* the part of J that involves electron i when it sits at ri (other electrons at x) */
static double jastrow_of_electron(const lrdmc_ref_ctx *c, const double *x, int i, const double ri[3])
{
    double J = 0.0;
    for (int a = 0; a < c->n_j3; ++a) J += j3_chi(c, a, ri, NULL, NULL) * j3_field(c, x, i, a);   /* g symmetric: i<j and j<i pairs alike */
    if (c->c1) for (int I = 0; I < c->n_nuc; ++I) { double r = dist(ri, c->Rn + 3 * I); J -= c->c1[I] * r / (1.0 + c->b1[I] * r); }
    for (int j = 0; j < c->N; ++j) if (j != i) {
        double r = dist(ri, x + 3 * j), aij = ref_spin(c, i) == ref_spin(c, j) ? c->a_par : c->a_anti;
        J += aij * r / (1.0 + c->b2 * r);
    }
    return J;
}

/* ---- non-local pseudopotential candidates (scope row f1; definition in lrdmc_ref.h) ------------------------------- */
/* centres in range of a point: nuclei with r_c > 0 and |ri - R_I| < r_c, ascending I; returns their number */
static int nl_in_range(const lrdmc_ref_ctx *c, const double ri[3], int *list)
{
    int n = 0;
    if (c->nl) for (int I = 0; I < c->n_nuc; ++I) if (c->nl[7 * I] > 0.0 && dist(ri, c->Rn + 3 * I) < c->nl[7 * I]) list[n++] = I;
    return n;
}

int ref_nl_slot(const lrdmc_ref_ctx *c, const double *x, const double U[9], int j, int *i_out, double rp[3], double *nu)
{
    int s = (j - c->P_lat) / 6, q = (j - c->P_lat) % 6, i = s / c->nl_K, kk = s % c->nl_K;
    int *list = (int *)malloc(sizeof(int) * (size_t)c->n_nuc);
    int n = nl_in_range(c, x + 3 * i, list), I = kk < n ? list[kk] : -1;
    free(list);
    *i_out = i;
    if (I < 0) return 0;
    const double *ri = x + 3 * i, *RI = c->Rn + 3 * I, *par = c->nl + 7 * I;
    double r = dist(ri, RI);
    int k = q / 2; double sgn = (q % 2 == 0) ? 1.0 : -1.0;
    double e[3] = { U[k], U[3 + k], U[6 + k] };                       /* versor k = column k of the frame */
    for (int ax = 0; ax < 3; ++ax) rp[ax] = RI[ax] + sgn * r * e[ax];  /* quadrature point on the sphere |r' - R_I| = r_iI */
    double ct = sgn * (e[0] * (ri[0] - RI[0]) + e[1] * (ri[1] - RI[1]) + e[2] * (ri[2] - RI[2])) / r;   /* cos(theta_q) */
    double P[3] = { 1.0, ct, 0.5 * (3.0 * ct * ct - 1.0) }, v = 0.0;   /* Legendre P_0, P_1, P_2 */
    for (int l = 0; l < 3; ++l) v += (2 * l + 1) * par[1 + 2 * l] * exp(-par[2 + 2 * l] * r * r) * P[l];
    *nu = v / 6.0;                                                     /* octahedral rule: six points, weight 1/6 each */
    return 1;
}

/* rho_q: determinant ratio (dla) or full wavefunction ratio of moving electron i to rp */
static double nl_ratio(const lrdmc_ref_ctx *c, const double *x, const double *const dinv[2], int i, const double rp[3])
{
    int spin = ref_spin(c, i), il = ref_local(c, i), O = ref_nocc(c, spin);
    double phi[REF_MAX_OCC];
    lrdmc_ref_mo(c, spin, rp, phi, NULL, NULL);
    double dr = 0.0; for (int m = 0; m < O; ++m) dr += phi[m] * dinv[spin][m * O + il];
    if (c->nl_dla) return dr;                                          /* D_G(x')/D_G(x), L576 */
    return dr * exp(jastrow_of_electron(c, x, i, rp) - jastrow_of_electron(c, x, i, x + 3 * i));
}

int lrdmc_ref_nl_info(const lrdmc_ref_ctx *c, const double *x, const double *dinv_up, const double *dinv_dn, const double U[9],
                      double *nu, double *rho, double *cand)
{
    const double *dinv[2] = { dinv_up, dinv_dn };
    for (int j = c->P_lat; j < c->P; ++j) {
        int i, o = j - c->P_lat; double rp[3] = { 0, 0, 0 }, v = 0.0;
        int act = ref_nl_slot(c, x, U, j, &i, rp, &v);
        nu[o] = act ? v : 0.0; rho[o] = act ? nl_ratio(c, x, dinv, i, rp) : 0.0;
        if (cand) { cand[3 * o] = rp[0]; cand[3 * o + 1] = rp[1]; cand[3 * o + 2] = rp[2]; }
    }
    return LRDMC_REF_OK;
}

int lrdmc_ref_evaluate(const lrdmc_ref_ctx *c, const double *x, const double *dinv_up_in, const double *dinv_dn_in,
                       const double U[9], double *R, double *scal, double *per, double *cand)
{
    int N = c->N, P = c->P_lat;
    double *own = NULL; const double *dinv[2] = { dinv_up_in, dinv_dn_in };
    if (!dinv_up_in) {
        own = (double *)calloc((size_t)(c->n_up * c->n_up + c->n_dn * c->n_dn + 1), sizeof(double));
        int rc = lrdmc_ref_build_inverse(c, x, own, own + c->n_up * c->n_up);
        if (rc) { free(own); return rc; }
        dinv[0] = own; dinv[1] = own + c->n_up * c->n_up;
    }
    /* --- step 1+2 (C2): candidates x_j (Eq.D4: electron i displaced by +-a along the versors) and
     *     ratios R_j = Psi_G(x_j)/Psi_G(x) = [sum_m phi_m(r') Dinv[m][i]] exp(J(x_j)-J(x)) */
    for (int j = 0; j < P; ++j) {
        int mesh, i, d; ref_cand(c, j, &mesh, &i, &d);
        int k = d / 2; double sgn = (d % 2 == 0) ? 1.0 : -1.0, step = sgn * c->amesh[mesh];
        double rp[3] = { x[3 * i] + step * U[k], x[3 * i + 1] + step * U[3 + k], x[3 * i + 2] + step * U[6 + k] };
        if (cand) { cand[3 * j] = rp[0]; cand[3 * j + 1] = rp[1]; cand[3 * j + 2] = rp[2]; }
        int spin = ref_spin(c, i), il = ref_local(c, i), O = ref_nocc(c, spin);
        double phi[REF_MAX_OCC];
        lrdmc_ref_mo(c, spin, rp, phi, NULL, NULL);
        double dr = 0.0; for (int m = 0; m < O; ++m) dr += phi[m] * dinv[spin][m * O + il];
        double dJ = jastrow_of_electron(c, x, i, rp) - jastrow_of_electron(c, x, i, x + 3 * i);
        R[j] = dr * exp(dJ);
    }
    /* --- step 3: fixed node (Eq.D1).  Kinetic hops have H_{x',x} = -kappa_j < 0, so
     *     s_{x',x} > 0  <=>  R_j < 0 (node crossing): those are removed and summed into V_sf >= 0 */
    double bbar = 0.0, Vsf = 0.0, Kdiag = 0.0; int node = 0;
    for (int j = 0; j < P; ++j) {
        double kap = c->kappa[j / (6 * N)];
        Kdiag += kap;                                   /* K^a_{x,x} = sum_j kappa_j = 3N/a^2 (Eq.D5) */
        if (R[j] > 0.0) bbar += kap * R[j];             /* bbar_x of Eq.29 (L199), summed in index order */
        else if (R[j] < 0.0) { Vsf -= kap * R[j]; node = 1; }
    }
    /* --- non-local pseudopotential candidates (f1): amplitude -nu_q rho_q; fixed node by the sign of H_{x',x} Psi'/Psi
     *     (Eq.D1 "for the non-local pseudopotentials ... chosen simply to guarantee the non-negativity");
     *     the D11 trigger looks at the wavefunction sign, rho_q < 0 ("(and ECP)", L625-L628) */
    double enl = 0.0;
    if (c->P > c->P_lat) {
        int *list = (int *)malloc(sizeof(int) * (size_t)c->n_nuc);
        for (int i = 0; i < N; ++i) if (nl_in_range(c, x + 3 * i, list) > c->nl_K) { free(list); free(own); return LRDMC_REF_EINVAL; }
        free(list);
        for (int j = c->P_lat; j < c->P; ++j) {
            int i; double rp[3] = { 0, 0, 0 }, nu = 0.0;
            R[j] = 0.0;
            if (cand) { cand[3 * j] = cand[3 * j + 1] = cand[3 * j + 2] = 0.0; }
            if (!ref_nl_slot(c, x, U, j, &i, rp, &nu)) continue;
            if (cand) { cand[3 * j] = rp[0]; cand[3 * j + 1] = rp[1]; cand[3 * j + 2] = rp[2]; }
            double rho = nl_ratio(c, x, dinv, i, rp);
            R[j] = -nu * rho;
            enl += nu * rho;                            /* V_nl Psi / Psi on the quadrature (its share of e_L, Eq.D7) */
            if (R[j] > 0.0) bbar += R[j];               /* allowed non-local hop: G = -H_{x',x} rho */
            else if (R[j] < 0.0) Vsf -= R[j];           /* s_{x',x} > 0: localised into V_sf (Eq.D1) */
            if (rho < 0.0) node = 1;
        }
    }
    /* --- step 4: per electron, continuum pieces and the regularised electron-ion potential (D6-D11) */
    double Vee = 0.0, sum_vopt = 0.0, eL_cont = 0.0; int n_vmax = 0;
    for (int i = 0; i < N; ++i) {
        int spin = ref_spin(c, i), il = ref_local(c, i), O = ref_nocc(c, spin);
        const double *ri = x + 3 * i;
        double val[REF_MAX_OCC], grad[3 * REF_MAX_OCC], lap[REF_MAX_OCC];
        lrdmc_ref_mo(c, spin, ri, val, grad, lap);
        double G[3] = { 0, 0, 0 }, Ld = 0.0;             /* grad_i D / D and lap_i D / D through the inverse */
        for (int m = 0; m < O; ++m) {
            double di = dinv[spin][m * O + il];
            G[0] += grad[3 * m] * di; G[1] += grad[3 * m + 1] * di; G[2] += grad[3 * m + 2] * di; Ld += lap[m] * di;
        }
        double gJ[3] = { 0, 0, 0 }, lJ = 0.0, vei = 0.0, vbound = 0.0;
        for (int I = 0; I < c->n_nuc; ++I) {
            const double *RI = c->Rn + 3 * I; double r = dist(ri, RI);
            if (c->c1) {
                double u, du, lu; pade3(-c->c1[I], c->b1[I], r, &u, &du, &lu);
                for (int ax = 0; ax < 3; ++ax) gJ[ax] += du * (ri[ax] - RI[ax]) / r;
                lJ += lu;
            }
            vei += v_nuc(c, I, r); vbound += v_nuc_bound(c, I, r);
        }
        for (int j = 0; j < N; ++j) if (j != i) {
            const double *rj = x + 3 * j; double r = dist(ri, rj), u, du, lu;
            pade3(ref_spin(c, j) == spin ? c->a_par : c->a_anti, c->b2, r, &u, &du, &lu);
            for (int ax = 0; ax < 3; ++ax) gJ[ax] += du * (ri[ax] - rj[ax]) / r;
            lJ += lu;
            if (j > i) Vee += 1.0 / r;
        }
        for (int a = 0; a < c->n_j3; ++a) {              /* three-body Jastrow: grad_i J3 = sum_a grad chi_a(r_i) V_a(i), same for the Laplacian */
            double ga[3], la, V = j3_field(c, x, i, a);
            j3_chi(c, a, ri, ga, &la);
            for (int ax = 0; ax < 3; ++ax) gJ[ax] += ga[ax] * V;
            lJ += la * V;
        }
        /* lap_i Psi / Psi for Psi = D exp(J) */
        double lap_i = Ld + 2.0 * (G[0] * gJ[0] + G[1] * gJ[1] + G[2] * gJ[2]) + lJ + (gJ[0] * gJ[0] + gJ[1] * gJ[1] + gJ[2] * gJ[2]);
        /* discretised Laplacian of Eq.D3 (L582) on Psi_G, over Psi_G: all six ratios, both signs */
        double T_i = 0.0;
        for (int mesh = 0; mesh < c->n_mesh; ++mesh) {
            double s = 0.0; for (int d = 0; d < 6; ++d) s += R[mesh * 6 * N + 6 * i + d];
            T_i += c->gmesh[mesh] * (s - 6.0) / (c->amesh[mesh] * c->amesh[mesh]);
        }
        double vzv = vei + 0.5 * (T_i - lap_i);          /* Eq.D8 (L610) */
        double vmax = vzv > vbound ? vzv : vbound;       /* Eq.D9 (L615) */
        double vopt = node ? vmax : vzv;                 /* Eq.D11 (L625), "at least one x_j" read globally (Q5) */
        if (node && vbound > vzv) ++n_vmax;
        sum_vopt += vopt;
        eL_cont += -0.5 * lap_i + vei;
        if (per) { per[5 * i] = T_i; per[5 * i + 1] = lap_i; per[5 * i + 2] = vei; per[5 * i + 3] = vzv; per[5 * i + 4] = vbound; }
    }
    /* --- step 5: diagonal element W(x) = H^FN_{x,x} (L628 plus the kinetic diagonal of Eq.D5, reading Q3)
     *     and local energy e_L = -bbar + W (L223) */
    double W = Kdiag + sum_vopt + Vee + c->V_ii + Vsf;
    scal[0] = bbar; scal[1] = Vsf; scal[2] = W; scal[3] = -bbar + W; scal[4] = node; scal[5] = Vee; scal[6] = c->V_ii;
    scal[7] = Kdiag; scal[8] = n_vmax; scal[9] = eL_cont + Vee + c->V_ii + enl;   /* right-hand side of Eq.D7 (L604) */
    free(own);
    return LRDMC_REF_OK;
}

/* Heat-bath selection (Eq.29: p_{x',x} = kappa_j R_j / bbar_x on the allowed moves).  q_j = kappa_j max(R_j,0);
 * C_j = q_0 + ... + q_j summed sequentially in index order; t = u C_{P-1}; j* = min{ j : C_j > t };
 * if rounding leaves none, the last j with q_j > 0.  Returns -1 when no move is allowed (bbar = 0).
 * margin = min_j |t - C_j| / C_{P-1}: how close the draw came to a bin edge (near-tie report, Q12). */
int lrdmc_ref_select(const lrdmc_ref_ctx *c, const double *R, double u_sel, double *margin)
{
    int P = c->P, jstar = -1, last = -1;
    double tot = 0.0;
    for (int j = 0; j < P; ++j) if (R[j] > 0.0) { tot += ref_kappa(c, j) * R[j]; last = j; }
    if (margin) *margin = 1.0;
    if (last < 0) return -1;
    double t = u_sel * tot, C = 0.0, mg = 1.0;
    for (int j = 0; j < P; ++j) {
        if (R[j] > 0.0) C += ref_kappa(c, j) * R[j];
        if (jstar < 0 && C > t) jstar = j;
        double dm = fabs(t - C) / tot; if (dm < mg) mg = dm;
    }
    if (margin) *margin = mg;
    return jstar >= 0 ? jstar : last;
}
