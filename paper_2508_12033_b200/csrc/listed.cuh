// listed.cuh -- the candidate pass of the LARGE systems (tables in global memory: 64 electrons, 600 AOs) as a LISTED sweep.
//
// Rows a1-a4 of the scope table in column form (wavefunction.cuh: sum_m phi_m(r') Dinv[m][i] = sum_mu chi_mu(r') Bc[mu][i], Bc = C Dinv),
// with two changes against the dense sweep of ao_columns:
//   (1) Gaussian sparsity.  In a 12-bohr cluster most (electron, shell) pairs contribute nothing: a shell is LISTED for a row of six
//       displaced points x0 +- step e_k only when |x0 - R_shell| < step + srad(zeta) (common.cuh LRDMC_LIST_THR: every exponent of an
//       unlisted shell is below -52 in any frame, its terms below 1e-22 of the norm).  Counted on thermalised configurations: 58 % of
//       the pairs of the 64-electron configuration are unlisted.  The test depends on positions only, so the
//       lists are 64-bit masks per (electron, list group) kept with the walker state and refreshed for the electron that hopped.
//   (2) Bc is STATE, not recomputed: the CTA keeps Bc [electron][n_aop] of its walker in global scratch, builds it when the walker
//       is loaded and updates it with the same rank-1 formula as the inverse after every hop
//       (Bc'[:,k] = Bc[:,k] - Bc[:,i] s_k / rho, Bc'[:,i] = Bc[:,i] / rho: 2 A n_s flop instead of 2 A O n_s on the tensor pipe).
// Work is dealt by ROWS (mesh, electron), a batch of at most 16 rows per warp: the lanes of the warp split every row's list of a
// type group into pieces of c consecutive listed shells (c minimal with sum_rows ceil(n_row / c) <= 32), sweep c pairs each, and add
// their shares by a segmented shuffle reduction.  The Jastrow ratios of the same rows follow in the same warp, so a warp finishes
// R_j of its rows without meeting the others.
#pragma once
#include "common.cuh"
#include "fastmath.cuh"

__device__ __forceinline__ int warp_sum_int(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// position of the n-th (0-based) set bit of a 64-bit mask (n < popcount)
__device__ __forceinline__ int nth_set_bit64(unsigned long long m, int n)
{
    const unsigned lo = (unsigned)m, hi = (unsigned)(m >> 32);
    const int pl = __popc(lo);
    return n < pl ? (int)__fns(lo, 0, n + 1) : 32 + (int)__fns(hi, 0, n - pl + 1);
}

// Listed-shell masks of one point for the list groups lg = first, first + stride, ...: bit q of group lg = slot lg_slot0 + q is within
// step_max + srad of (x, y, z).  One warp; lane 0 writes am_i[lg].
__device__ __forceinline__ void list_masks(const DevSys &S, const double *shells, const double *srad, unsigned long long *am_i, double x, double y,
                                           double z, double step_max, int lane, int first, int stride)
{
    for (int lg = first; lg < S.n_lg; lg += stride) {
        unsigned w[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int ql = lane + 32 * h; const bool in = ql < S.lg_n[lg];
            const int q = S.lg_slot0[lg] + (in ? ql : 0);
            const double4 sh = reinterpret_cast<const double4 *>(shells)[q];
            const double dx = x - sh.x, dy = y - sh.y, dz = z - sh.z, rad = step_max + srad[q];
            w[h] = __ballot_sync(0xffffffffu, in && rad > 0.0 && dx * dx + dy * dy + dz * dz < rad * rad);
        }
        if (lane == 0) am_i[lg] = ((unsigned long long)w[1] << 32) | w[0];
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

// The listed sweep of the rows rho0 .. rho0 + nrows - 1 (row = mesh N + electron; nrows <= 32, best <= 16) by ONE warp:
// R[mesh 6N + 6 i + d] <- sum over the listed shells of chi(x_i +- a_mesh e_k) . Bc[i][.]   (the determinant ratio of candidate (i, d)).
//   r_el [N][3] positions, U the step's frame, am [N][n_lg] listed-shell masks, bc [N][n_aop] this walker's Bc.
__device__ __forceinline__ void ao_listed_warp(const DevSys &S, const double *__restrict__ shells, const double *__restrict__ etab,
                                               const double *__restrict__ r_el, const double *__restrict__ U, const unsigned long long *__restrict__ am,
                                               const double *__restrict__ bc, int rho0, int nrows, double *__restrict__ R, int lane)
{
    const int N = S.N, A = S.n_aop;
    const bool inr = lane < nrows;
    const int my_rho = rho0 + (inr ? lane : 0), my_mesh = my_rho / N, my_i = my_rho - my_mesh * N;
    if (inr) { double *Ro = R + my_mesh * 6 * N + 6 * my_i;
#pragma unroll
        for (int d = 0; d < 6; ++d) Ro[d] = 0.0; }
    __syncwarp();
    for (int lg = 0; lg < S.n_lg; ++lg) {
        const unsigned long long mk = inr ? am[my_i * S.n_lg + lg] : 0ull;
        const int n_r = __popcll(mk);
        const int total = warp_sum_int(n_r);
        if (total == 0) continue;                                        // (uniform)
        int c = (total + 31) >> 5;
        for (;;) { if (warp_sum_int((n_r + c - 1) / c) <= 32) break; ++c; }
        const int m_r = (n_r + c - 1) / c;                                // lanes of this row
        int incl = m_r;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
        const int start = incl - m_r, used = __shfl_sync(0xffffffffu, incl, 31);
        int mmax = m_r;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mmax = max(mmax, __shfl_xor_sync(0xffffffffu, mmax, o));
        int row = 0;
        for (int r = 1; r < nrows; ++r) { const int s = __shfl_sync(0xffffffffu, start, r); if (lane >= s) row = r; }
        const bool has = lane < used;
        const int rstart = __shfl_sync(0xffffffffu, start, row), rend = rstart + __shfl_sync(0xffffffffu, m_r, row);   // lanes [rstart, rend) share the row
        unsigned long long m = __shfl_sync(0xffffffffu, mk, row);
        const int piece = lane - rstart;
        if (has && piece > 0) m &= ~0ull << nth_set_bit64(m, piece * c);  // this lane's piece starts at listed shell number piece * c
        if (!has) m = 0ull;
        const int rho = rho0 + row, mesh = rho / N, i = rho - mesh * N;
        const double x0 = r_el[3 * i], y0 = r_el[3 * i + 1], z0 = r_el[3 * i + 2], am_ = S.amesh[mesh], a2 = am_ * am_;
        double av[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) { av[k][0] = am_ * U[k]; av[k][1] = am_ * U[3 + k]; av[k][2] = am_ * U[6 + k]; }
        const double *bcr = bc + (size_t)i * A + S.lg_ao0[lg];
        const double4 *sh4 = reinterpret_cast<const double4 *>(shells) + S.lg_slot0[lg];
        const int type = S.lg_type[lg];
        double acc[6];
#pragma unroll
        for (int d = 0; d < 6; ++d) acc[d] = 0.0;
        if (type == 0) {                                                  // Slater s: exp(-z r)
            for (int k = 0; k < c; ++k) {
                const bool valid = m != 0ull; const int q = valid ? __ffsll((long long)m) - 1 : 0; m &= m - 1ull;
                const double b = valid ? bcr[q] : 0.0;
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
            for (int k = 0; k < c; ++k) {
                const bool valid = m != 0ull; const int q = valid ? __ffsll((long long)m) - 1 : 0; m &= m - 1ull;
                const double b = valid ? bcr[q] : 0.0;
                const SixGeom G = six_gaussians(sh4[q], x0, y0, z0, av, a2, etab);
#pragma unroll
                for (int d = 0; d < 6; ++d) acc[d] = fma(G.e[d], b, acc[d]);
            }
        } else if (type == 2) {                                           // p Gaussians: e (bc . (d0 +- a e_k))
            for (int k = 0; k < c; ++k) {
                const bool valid = m != 0ull; const int q = valid ? __ffsll((long long)m) - 1 : 0; m &= m - 1ull;
                const double *bp = bcr + 3 * q;
                const double bx = valid ? bp[0] : 0.0, by = valid ? bp[1] : 0.0, bz = valid ? bp[2] : 0.0;
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
            for (int k = 0; k < c; ++k) {
                const bool valid = m != 0ull; const int q = valid ? __ffsll((long long)m) - 1 : 0; m &= m - 1ull;
                const double *bp = bcr + 6 * q;
                double b[6];
#pragma unroll
                for (int j = 0; j < 6; ++j) b[j] = valid ? bp[j] : 0.0;
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
        // the lanes of a row add up (suffix sums inside [rstart, rend)); the row's first lane adds the group's share to R
        for (int o = 1; o < mmax; o <<= 1) {
#pragma unroll
            for (int d = 0; d < 6; ++d) { const double v = __shfl_down_sync(0xffffffffu, acc[d], o); if (lane + o < rend) acc[d] += v; }
        }
        if (has && piece == 0) { double *Ro = R + mesh * 6 * N + 6 * i;
#pragma unroll
            for (int d = 0; d < 6; ++d) Ro[d] += acc[d]; }
        __syncwarp();
    }
}
