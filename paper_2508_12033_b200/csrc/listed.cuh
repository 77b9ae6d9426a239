// listed.cuh -- the candidate pass as a LISTED sweep (template bit EXT = 4 of the walker kernels): chosen automatically for the systems whose tables
// live in global memory (64 electrons, 600 AOs), available on any lattice-only system through LRDMC_OPT_LISTED.
//
// Rows a1-a4 of the scope table in column form (wavefunction.cuh: sum_m phi_m(r') Dinv[m][i] = sum_mu chi_mu(r') Bc[mu][i], Bc = C Dinv),
// with two changes against the dense sweep of ao_columns:
//   (1) Gaussian sparsity.  Most (electron, shell) pairs of an extended system contribute nothing: a shell is LISTED for the six displaced
//       points x0 +- step e_k of an electron only when |x0 - R_shell| < step + srad(zeta) (common.cuh LRDMC_LIST_THR: every exponent of an
//       unlisted shell is below -52 in any frame, its terms below 1e-22 of the norm).  Counted on thermalised configurations: 58 % of the
//       pairs of the 64-electron configuration and 41 % of the water-methane-shaped one are unlisted.  The test
//       depends on the positions only, so the lists (bytes, per electron and list group) are kept with the walker state in shared memory
//       and rebuilt for the electron that hopped.
//   (2) Bc is STATE, not recomputed: Bc [electron][n_aop] of the walker lives in a global scratch of the resident CTA / warp, is built when
//       the walker is loaded and follows the inverse by the same rank-1 formula after every hop
//       (Bc'[:,k] = Bc[:,k] - Bc[:,i] s_k / rho, Bc'[:,i] = Bc[:,i] / rho: 2 A n_s flop instead of 2 A O n_s on the tensor pipe).
// The sweep keeps the lane map of the dense pass -- a quad per row (mesh, electron), lane t takes every fourth entry of ITS electron's
// list -- so the four shares meet in a quad shuffle and the Jastrow ratios of the same 8 rows reuse the geometry (evaluate.cuh,
// listed_phase_b); 8-row batches are independent, a team deals them to its warps.  The oracle never screens.
#pragma once
#include "common.cuh"
#include "fastmath.cuh"

// Per-walker lists (shared memory, bytes): cnt [n_lg][N] listed-shell counts, then lst [N][lt] slot numbers (relative to the list group's first
// slot), the groups of an electron at lg_off[lg].  A shell is listed for electron i when |r_i - R_shell| < step_max + srad: the test depends on the
// position only, so the lists are kept with the walker state and rebuilt for the electron that hopped.
__device__ __forceinline__ void list_build(const DevSys &S, const double *shells, const double *srad, unsigned char *lw, int i, double x, double y, double z,
                                           double step_max, int lane)
{
    unsigned char *cnt = lw, *lrow = lw + S.n_lg * S.N + i * S.lt;
    for (int lg = 0; lg < S.n_lg; ++lg) {
        unsigned w[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int ql = lane + 32 * h; const bool in = ql < S.lg_n[lg];
            const int q = S.lg_slot0[lg] + (in ? ql : 0);
            const double4 sh = reinterpret_cast<const double4 *>(shells)[q];
            const double dx = x - sh.x, dy = y - sh.y, dz = z - sh.z, rad = step_max + srad[q];
            w[h] = __ballot_sync(0xffffffffu, in && rad > 0.0 && dx * dx + dy * dy + dz * dz < rad * rad);
        }
        unsigned char *l = lrow + S.lg_off[lg];
        const unsigned below = (1u << lane) - 1u; const int n0 = __popc(w[0]);
        if ((w[0] >> lane) & 1u) l[__popc(w[0] & below)] = (unsigned char)lane;
        if ((w[1] >> lane) & 1u) l[n0 + __popc(w[1] & below)] = (unsigned char)(lane + 32);
        if (lane == 0) cnt[lg * S.N + i] = (unsigned char)(n0 + __popc(w[1]));
    }
}

// Bc = C Dinv of one walker, [electron][n_aop], by the threads tid = 0 .. nthr-1 (a warp or a CTA): thread = one AO row of C (slot-major, norms
// folded in), eight inverse columns at a time.  Built when the walker is loaded (reading Q15: the state is rebuilt wherever the inverse is).
__device__ __forceinline__ void build_bc(const DevSys &S, const double *dinv0, const double *dinv1, double *__restrict__ bc, int tid, int nthr)
{
    const int A = S.n_aop, OS = S.OS;
    for (int sp = 0; sp < 2; ++sp) {
        const int ns = sp ? S.n_dn : S.n_up, off = sp ? S.n_up : 0;
        if (!ns) continue;
        const double *__restrict__ cn = S.cn[sp], *dinv = sp ? dinv1 : dinv0;
        for (int ao = tid; ao < A; ao += nthr) {
            const double *crow = cn + (size_t)ao * OS;
            for (int il0 = 0; il0 < ns; il0 += 8) {
                double acc[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) acc[j] = 0.0;
                for (int m = 0; m < ns; ++m) {
                    const double cv = __ldg(crow + m); const double *dr = dinv + m * ns + il0;   // columns beyond n_s read padding, never stored
#pragma unroll
                    for (int j = 0; j < 8; ++j) acc[j] = fma(cv, dr[j], acc[j]);
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) if (il0 + j < ns) bc[(size_t)(off + il0 + j) * A + ao] = acc[j];
            }
        }
    }
}

// Bc follows the inverse by the same rank-1 formula after electron i (spin sp, column il) hopped: Bc'[:,k] = Bc[:,k] - Bc[:,il] s_k / rho,
// Bc'[:,il] = Bc[:,il] / rho.  Thread = one AO (consecutive threads on consecutive AOs: coalesced), eight columns in flight at a time; a thread
// touches the entries of its own AOs only, so no barrier is needed inside.
__device__ __forceinline__ void bc_rank1_update(const DevSys &S, double *bc, int sp, int il, int ns, const double *sk, double irho, int tid, int nthr)
{
    const size_t A = (size_t)S.n_aop;
    double *b0 = bc + (size_t)(sp ? S.n_up : 0) * A;
    for (int ao = tid; ao < (int)A; ao += nthr) {
        double *p = b0 + ao;
        const double f = __ldcg(p + (size_t)il * A) * irho;
        for (int k0 = 0; k0 < ns; k0 += 8, p += 8 * A) {
            double v[8];
#pragma unroll
            for (int q = 0; q < 8; ++q) v[q] = (k0 + q < ns) ? __ldcg(p + q * A) : 0.0;
#pragma unroll
            for (int q = 0; q < 8; ++q) if (k0 + q < ns) __stcg(p + q * A, (k0 + q == il) ? f : fma(-f, sk[k0 + q], v[q]));
        }
    }
}

// geometry of one shell against a row: distances and the six exponent arguments of x0 +- av[k] (as LRDMC_GEOM / LRDMC_EXPS of ao_columns)
struct SixGeom { double dx0, dy0, dz0, z; double e[6]; };
__device__ __forceinline__ SixGeom six_gaussians(const double4 s, double x0, double y0, double z0, const double (&av)[3][3], double a2, const double *etab)
{
    SixGeom G; G.z = s.w;
    G.dx0 = x0 - s.x; G.dy0 = y0 - s.y; G.dz0 = z0 - s.z;
    const double q0 = fma(G.dx0, G.dx0, fma(G.dy0, G.dy0, fma(G.dz0, G.dz0, a2)));
    double sk[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) sk[k] = fma(av[k][0], G.dx0, fma(av[k][1], G.dy0, av[k][2] * G.dz0));
    const double zq0 = -G.z * q0; const bool far_ = zq0 < 0.5 * LRDMC_EXP_XMIN;
    const double zq = far_ ? 0.5 * LRDMC_EXP_XMIN : zq0, tz = far_ ? 0.0 : -2.0 * G.z;
    double ex_[6];
#pragma unroll
    for (int k = 0; k < 3; ++k) { ex_[2 * k] = fma(tz, sk[k], zq); ex_[2 * k + 1] = fma(-tz, sk[k], zq); }
    exp_tab_n<6>(ex_, G.e, etab);
    return G;
}

// The listed sweep of ONE row per quad (lane = 4 g + t: row g of the batch, t = which of four listed shells taken together): the share of lane t in
//     sum over the listed shells of chi(x0 +- av[k]) . Bc[i][.]        (the determinant ratios of the six candidates of electron i on this mesh);
// the caller adds the four lanes of a quad.  Every quad walks ITS electron's lists; a list group takes ceil(max over the 8 rows of n / 4) iterations.
//   lw this walker's lists, bc its Bc [N][n_aop], valid = the quad holds a row (idle quads run with coefficient 0).
__device__ __forceinline__ void ao_listed_quad(const DevSys &S, const double *__restrict__ shells, const double *__restrict__ etab, const unsigned char *lw,
                                               const double *__restrict__ bc, int i, bool valid, double x0, double y0, double z0, const double (&av)[3][3], double a2,
                                               int lane, double (&acc)[6])
{
    const int t = lane & 3, N = S.N;
    const unsigned char *cnt = lw + i, *lrow = lw + S.n_lg * N + i * S.lt;
    const double *bci = bc + (size_t)i * S.n_aop;
#pragma unroll
    for (int d = 0; d < 6; ++d) acc[d] = 0.0;
    for (int lg = 0; lg < S.n_lg; ++lg) {
        const int n = valid ? cnt[lg * N] : 0;
        const int nmax = __reduce_max_sync(0xffffffffu, n);
        const unsigned char *l = lrow + S.lg_off[lg];
        const double *bcr = bci + S.lg_ao0[lg];
        const double4 *sh4 = reinterpret_cast<const double4 *>(shells) + S.lg_slot0[lg];
        const int type = S.lg_type[lg];
        if (type == 0) {                                                  // Slater s: exp(-z r)
            for (int k0 = 0; k0 < nmax; k0 += 4) {
                const bool ok = k0 + t < n; const int q = ok ? l[k0 + t] : 0;
                const double b = ok ? bcr[q] : 0.0;
                const double4 s = sh4[q]; const double dx0 = x0 - s.x, dy0 = y0 - s.y, dz0 = z0 - s.z;
                const double q0 = fma(dx0, dx0, fma(dy0, dy0, fma(dz0, dz0, a2)));
#pragma unroll
                for (int kk = 0; kk < 3; ++kk) {
                    const double sk = fma(av[kk][0], dx0, fma(av[kk][1], dy0, av[kk][2] * dz0));
                    const double qp = fma(2.0, sk, q0), qm = fma(-2.0, sk, q0);
                    acc[2 * kk] = fma(exp_tab(exp_arg_floor(-s.w * (qp * fast_rsqrt(qp))), etab), b, acc[2 * kk]);
                    acc[2 * kk + 1] = fma(exp_tab(exp_arg_floor(-s.w * (qm * fast_rsqrt(qm))), etab), b, acc[2 * kk + 1]);
                }
            }
        } else if (type == 1) {                                           // s Gaussians
            for (int k0 = 0; k0 < nmax; k0 += 4) {
                const bool ok = k0 + t < n; const int q = ok ? l[k0 + t] : 0;
                const double b = ok ? bcr[q] : 0.0;
                const SixGeom G = six_gaussians(sh4[q], x0, y0, z0, av, a2, etab);
#pragma unroll
                for (int d = 0; d < 6; ++d) acc[d] = fma(G.e[d], b, acc[d]);
            }
        } else if (type == 2) {                                           // p Gaussians: e (bc . (d0 +- a e_k))
            for (int k0 = 0; k0 < nmax; k0 += 4) {
                const bool ok = k0 + t < n; const int q = ok ? l[k0 + t] : 0;
                const double *bp = bcr + 3 * q;
                const double bx = ok ? bp[0] : 0.0, by = ok ? bp[1] : 0.0, bz = ok ? bp[2] : 0.0;
                const SixGeom G = six_gaussians(sh4[q], x0, y0, z0, av, a2, etab);
                const double l0 = fma(bx, G.dx0, fma(by, G.dy0, bz * G.dz0));
#pragma unroll
                for (int kk = 0; kk < 3; ++kk) {
                    const double lk = fma(bx, av[kk][0], fma(by, av[kk][1], bz * av[kk][2]));
                    acc[2 * kk] = fma(G.e[2 * kk], l0 + lk, acc[2 * kk]);
                    acc[2 * kk + 1] = fma(G.e[2 * kk + 1], l0 - lk, acc[2 * kk + 1]);
                }
            }
        } else {                                                          // d Gaussians: e Q(d), Q(d0 +- v) = Q(d0) +- v.grad Q(d0) + Q(v)
            for (int k0 = 0; k0 < nmax; k0 += 4) {
                const bool ok = k0 + t < n; const int q = ok ? l[k0 + t] : 0;
                const double *bp = bcr + 6 * q;
                double b[6];
#pragma unroll
                for (int j = 0; j < 6; ++j) b[j] = ok ? bp[j] : 0.0;
                const SixGeom G = six_gaussians(sh4[q], x0, y0, z0, av, a2, etab);
                const double gx = fma(2.0 * b[0], G.dx0, fma(b[1], G.dy0, b[2] * G.dz0));
                const double gy = fma(b[1], G.dx0, fma(2.0 * b[3], G.dy0, b[4] * G.dz0));
                const double gz = fma(b[2], G.dx0, fma(b[4], G.dy0, 2.0 * b[5] * G.dz0));
                const double Q0 = 0.5 * fma(gx, G.dx0, fma(gy, G.dy0, gz * G.dz0));
#pragma unroll
                for (int kk = 0; kk < 3; ++kk) {
                    const double vx = av[kk][0], vy = av[kk][1], vz = av[kk][2];
                    const double lin = fma(gx, vx, fma(gy, vy, gz * vz));
                    const double Qv = fma(vx, fma(b[0], vx, fma(b[1], vy, b[2] * vz)), fma(vy, fma(b[3], vy, b[4] * vz), b[5] * vz * vz));
                    const double Qs = Q0 + Qv;
                    acc[2 * kk] = fma(G.e[2 * kk], Qs + lin, acc[2 * kk]);
                    acc[2 * kk + 1] = fma(G.e[2 * kk + 1], Qs - lin, acc[2 * kk + 1]);
                }
            }
        }
    }
}
