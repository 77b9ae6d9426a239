/* oracle/ref_rng.c -- ORACLE (test infrastructure): random numbers, lattice frame, reconfiguration comb.
 *
 * The paper only says "xi is a uniform variate in [0,1)" (Eq.17, L146 Eq.21, L358 Alg.1)
 * and that the versors "rotate with random angles along the simulation" (L596).  The generator and
 * the frame distribution are readings Q7/Q12 of DESIGN.md: Philox4x32-10 (Salmon et al., SC'11),
 * counter = (walker slot, cycle, step, purpose), key = 64-bit run seed; a Haar-uniform rotation from
 * three uniforms through a unit quaternion (Shoemake 1992).  The CUDA path re-implements the same
 * counter-based generator independently; no code is shared.
 */
#include "ref_internal.h"

/* Philox4x32-10: ten rounds of  (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * the key bumped by the Weyl constants between rounds. */
void lrdmc_ref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* 53-bit uniform in [0,1): the top 53 bits of the 64-bit word hi:lo times 2^-53 */
double lrdmc_ref_uniform53(uint32_t lo, uint32_t hi)
{
    uint64_t v = ((uint64_t)hi << 32) | lo;
    return (double)(v >> 11) * (1.0 / 9007199254740992.0);
}

static void block(const lrdmc_ref_ctx *c, uint32_t slot, uint64_t cycle, uint64_t step, uint32_t purpose, uint32_t out[4])
{
    uint32_t ctr[4] = { slot, (uint32_t)cycle, (uint32_t)step, purpose };
    uint32_t key[2] = { (uint32_t)c->seed, (uint32_t)(c->seed >> 32) };
    lrdmc_ref_philox4x32_10(ctr, key, out);
}

/* purpose 0 -> (u1,u2); purpose 1 -> (u3,u_sel); purpose 2 -> (u_tau, unused) */
void lrdmc_ref_draws(const lrdmc_ref_ctx *c, uint32_t slot, uint64_t cycle, uint64_t step, double u[5])
{
    uint32_t o[4];
    block(c, slot, cycle, step, 0, o); u[0] = lrdmc_ref_uniform53(o[0], o[1]); u[1] = lrdmc_ref_uniform53(o[2], o[3]);
    block(c, slot, cycle, step, 1, o); u[2] = lrdmc_ref_uniform53(o[0], o[1]); u[3] = lrdmc_ref_uniform53(o[2], o[3]);
    block(c, slot, cycle, step, 2, o); u[4] = lrdmc_ref_uniform53(o[0], o[1]);
}

uint32_t lrdmc_ref_comb_r32(const lrdmc_ref_ctx *c, uint64_t cycle)
{
    uint32_t o[4];
    block(c, 0xFFFFFFFFu, cycle, 0, 3, o);
    return o[0];
}

/* Random lattice frame (L596).  Unit quaternion q = (x,y,z,w) =
 * (sqrt(1-u1) sin 2 pi u2, sqrt(1-u1) cos 2 pi u2, sqrt(u1) sin 2 pi u3, sqrt(u1) cos 2 pi u3)
 * is uniform on S^3; its rotation matrix U is Haar-uniform on SO(3).  U row-major; the three
 * versors e_1,e_2,e_3 of Eq.D3 are the COLUMNS of U. */
void lrdmc_ref_frame(double u1, double u2, double u3, double U[9])
{
    const double two_pi = 6.283185307179586476925286766559;
    double s1 = sqrt(1.0 - u1), s2 = sqrt(u1);
    double x = s1 * sin(two_pi * u2), y = s1 * cos(two_pi * u2);
    double z = s2 * sin(two_pi * u3), w = s2 * cos(two_pi * u3);
    U[0] = 1.0 - 2.0 * (y * y + z * z); U[1] = 2.0 * (x * y - z * w);       U[2] = 2.0 * (x * z + y * w);
    U[3] = 2.0 * (x * y + z * w);       U[4] = 1.0 - 2.0 * (x * x + z * z); U[5] = 2.0 * (y * z - x * w);
    U[6] = 2.0 * (x * z - y * w);       U[7] = 2.0 * (y * z + x * w);       U[8] = 1.0 - 2.0 * (x * x + y * y);
}

/* Reconfiguration at fixed N_w (Eq.15-17), integer form (reading Q21).
 *   p_alpha = w_alpha / sum w (Eq.15);  comb Z_k = (xi + k)/N_w, k = 0..N_w-1 (Eq.17, xi = r32/2^32);
 *   new walker k copies the first old walker beta whose cumulative normalised weight exceeds Z_k (L121).
 * Weights are first quantised to integers u_alpha = floor(w_alpha 2^sh) with sh chosen so that the
 * total T < 2^62; the comparison  P_beta / T > (r32 + k 2^32) / (N_w 2^32)  is then done exactly in
 * 128-bit integers, so the indices do not depend on floating-point summation order.
 * wbar = T 2^-sh / N_w (Eq.16).  Degenerate input (no positive finite weight): parents = identity, wbar = 0. */
int lrdmc_ref_comb(int n_w, const double *w, uint32_t r32, int32_t *parents, double *wbar, uint64_t *u_out,
                   uint64_t *T_out, int *sh_out)
{
    if (n_w <= 0) return LRDMC_REF_EINVAL;
    double m = 0.0; int bad = 0;
    for (int k = 0; k < n_w; ++k) { if (!(w[k] >= 0.0) || isinf(w[k])) bad = 1; else if (w[k] > m) m = w[k]; }
    if (bad || !(m > 0.0)) {
        for (int k = 0; k < n_w; ++k) parents[k] = k;
        if (wbar) *wbar = 0.0; if (T_out) *T_out = 0; if (sh_out) *sh_out = 0;
        if (u_out) memset(u_out, 0, sizeof(uint64_t) * (size_t)n_w);
        return bad ? LRDMC_REF_EINVAL : LRDMC_REF_OK;
    }
    int e; (void)frexp(m, &e);                       /* m = f 2^e, f in [0.5,1) */
    int L = 1; while ((1 << L) < n_w) ++L;           /* max(1, ceil(log2 N_w)) */
    int sh = 62 - L - e;
    uint64_t *u = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)n_w), T = 0;
    for (int k = 0; k < n_w; ++k) { u[k] = (uint64_t)floor(ldexp(w[k], sh)); T += u[k]; }
    unsigned __int128 scale = (unsigned __int128)(uint64_t)n_w << 32;
    uint64_t Pb = u[0]; int beta = 0;
    for (int k = 0; k < n_w; ++k) {
        unsigned __int128 rhs = ((unsigned __int128)r32 + ((unsigned __int128)(uint64_t)k << 32)) * T;
        while (beta < n_w - 1 && !((unsigned __int128)Pb * scale > rhs)) { ++beta; Pb += u[beta]; }
        parents[k] = beta;
    }
    if (wbar) *wbar = ldexp((double)T, -sh) / (double)n_w;
    if (u_out) memcpy(u_out, u, sizeof(uint64_t) * (size_t)n_w);
    if (T_out) *T_out = T; if (sh_out) *sh_out = sh;
    free(u);
    return LRDMC_REF_OK;
}
