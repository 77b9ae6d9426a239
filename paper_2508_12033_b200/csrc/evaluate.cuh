// evaluate.cuh -- one evaluation of the lattice-regularised fixed-node Hamiltonian at a walker's configuration
// (Appendix D; rows a1, a4-a10 of the scope table), by ONE WARP on shared-memory state.
#pragma once
#include "common.cuh"
#include "fastmath.cuh"
#include "philox.cuh"
#include "wavefunction.cuh"
#include "listed.cuh"

struct WarpState {            // per-warp views (shared memory; moc may live in global memory for large systems)
    double *r, *dinv[2], *moc, *R, *el, *ob, *U;
    double *j3;               // three-body Jastrow (systems that have one): chi3 [N][j3s] = chi_a(r_j), then V3 [N][j3s], then S3 [j3s]
    unsigned char *lw;        // listed sweep: this walker's listed-shell lists (listed.cuh: counts [n_lg][N], slots [N][lt])
    double *bc;               // listed sweep: this walker's Bc = C Dinv [N][n_aop] (global scratch of the resident warp / CTA, rank-1 updated)
};
struct EvalOut { double bbar, Vsf, W, eL; int node;
                 double c_loc, c_excl; };   // per LANE: sum of the allowed amplitudes of the lane's candidate chunk, and of the chunks before it (select_move)

__device__ __forceinline__ int spin_of(const DevSys &S, int i) { return i < S.n_up ? 0 : 1; }

// electron-ion potential of one nucleus and its lower bound (Eq.D10; ECP rule L623)
__device__ __forceinline__ void nuc_potential(double a_cut, const double *nu, double r, double ir, double &v, double &vb)
{
    const double Z = nu[3];
    if (nu[10] != 0.0) {
        const double r2 = r * r;
        v = Z * expm1(-nu[6] * r2) * ir + Z * nu[6] * r * exp_nonpos(-nu[7] * r2) + nu[8] * exp_nonpos(-nu[9] * r2);
        vb = -Z * ir;
    } else { v = -Z * ir; vb = (r > a_cut) ? -Z * ir : -Z / a_cut; }
}

// One-body cache of electron i (depends on its own position only): ob[i][0..6] = J1_i, grad J1 (3), lap J1, v_ei, v^a_ei.
// Nuclei are spread over the lanes; called for every electron when a walker is loaded and for the mover after a hop.
__device__ __forceinline__ void refresh_onebody(int n_nuc, int has_j1, double a_cut, const double *nuc, double *ob_i, double xi, double yi, double zi, int lane)
{
    LRDMC_ASSUME_SHARED(nuc); LRDMC_ASSUME_SHARED(ob_i);
    double J = 0.0, gx = 0.0, gy = 0.0, gz = 0.0, lJ = 0.0, vei = 0.0, vb = 0.0;
    for (int I = lane; I < n_nuc; I += 32) {
        const double *nu = nuc + I * LRDMC_NUC_STRIDE;
        const double dx = xi - nu[0], dy = yi - nu[1], dz = zi - nu[2], r2 = dx * dx + dy * dy + dz * dz;
        const double ir = fast_rsqrt(r2), r = r2 * ir;
        if (has_j1) {                                              // u1 = -c1 r/(1+b1 r): u' = c/(1+br)^2, lap u = 2c/(r (1+br)^3)
            const double c = -nu[4], iq = fast_rcp(1.0 + nu[5] * r), du = c * iq * iq * ir;
            J += c * r * iq; gx += du * dx; gy += du * dy; gz += du * dz; lJ += 2.0 * du * iq;
        }
        double v, b; nuc_potential(a_cut, nu, r, ir, v, b); vei += v; vb += b;
    }
    J = warp_sum(J); gx = warp_sum(gx); gy = warp_sum(gy); gz = warp_sum(gz); lJ = warp_sum(lJ); vei = warp_sum(vei); vb = warp_sum(vb);
    if (lane == 0) { ob_i[0] = J; ob_i[1] = gx; ob_i[2] = gy; ob_i[3] = gz; ob_i[4] = lJ; ob_i[5] = vei; ob_i[6] = vb; }
}

// Three-body Jastrow (reading Q23): chi_a(r) = dx^l dy^m dz^n exp(-zeta_a |r - R_a|^2) of electron j, lane per function (zero beyond n_j3).
__device__ __forceinline__ double mono_pow(double v, int k) { return k == 0 ? 1.0 : (k == 1 ? v : v * v); }     // v^k, k = 0, 1, 2
__device__ __forceinline__ void refresh_j3_row(const DevSys &S, const double *nuc, double *chi3_j, double x, double y, double z, int lane)
{
    if (lane < S.j3s) {
        double v = 0.0;
        if (lane < S.n_j3) {
            const double *nu = nuc + S.j3_center[lane] * LRDMC_NUC_STRIDE;
            const double dx = x - nu[0], dy = y - nu[1], dz = z - nu[2];
            v = exp_nonpos(-S.j3_zeta[lane] * (dx * dx + dy * dy + dz * dz));
            if (S.j3_poly) { const int q = S.j3_lmn[lane]; v *= mono_pow(dx, q & 3) * mono_pow(dy, (q >> 2) & 3) * mono_pow(dz, (q >> 4) & 3); }
        }
        chi3_j[lane] = v;
    }
}

// The fields V_a(i) = sum_b g_ab (S_b - chi_b(r_i)), S_b = sum_j chi_b(r_j), of all electrons (start of every evaluation) by the threads
// tid = 0 .. nthr-1 of a warp (SYNC = __syncwarp) or of a CTA (__syncthreads): j3 = chi3 [N][j3s], V3 [N][j3s], S3 [j3s]; g staged in the tables.
template <typename SYNC>
__device__ __forceinline__ void j3_fields(const DevSys &S, const double *__restrict__ g3, double *j3, int tid, int nthr, SYNC sync)
{
    const int N = S.N, J = S.j3s;
    double *chi3 = j3, *V3 = j3 + N * J, *S3 = V3 + N * J;
    for (int b = tid; b < J; b += nthr) { double sb = 0.0; for (int j = 0; j < N; ++j) sb += chi3[j * J + b]; S3[b] = sb; }
    sync();
    for (int idx = tid; idx < N * J; idx += nthr) {
        const int i = idx / J, a = idx - i * J;
        double v = 0.0;
        for (int b = 0; b < J; b += 4) {
#pragma unroll
            for (int q = 0; q < 4; ++q) v += g3[a * J + b + q] * (S3[b + q] - chi3[i * J + b + q]);
        }
        V3[idx] = v;
    }
    sync();
}

// J3 terms of electron i in the continuum pieces (phase A): J += sum_a chi_a V_a, grad and Laplacian alike.  s functions:
// grad chi = -2 zeta d chi, lap chi = (4 zeta^2 r^2 - 6 zeta) chi.  With monomials, per axis u(v) = v^k e^{-zeta v^2}:
// u' = (k v^(k-1) - 2 zeta v^(k+1)) e, u'' = (k (k-1) v^(k-2) - 2 zeta (2k+1) v^k + 4 zeta^2 v^(k+2)) e, chi = product of the three axes.
__device__ __forceinline__ void j3_axis(double v, int k, double z, double &f, double &f1, double &f2)
{
    const double v2 = v * v, tz = 2.0 * z, fz2 = 4.0 * z * z;
    f = mono_pow(v, k);
    f1 = k == 0 ? -tz * v : (k == 1 ? 1.0 - tz * v2 : (2.0 - tz * v2) * v);
    f2 = k == 0 ? fz2 * v2 - tz : (k == 1 ? (fz2 * v2 - 3.0 * tz) * v : 2.0 + (fz2 * v2 - 5.0 * tz) * v2);
}
__device__ __forceinline__ void j3_electron_terms(const DevSys &S, const double *nuc, const double *chi3_i, const double *V3_i, double xi, double yi, double zi,
                                                  double &J, double &gx, double &gy, double &gz, double &lJ)
{
    for (int a = 0; a < S.n_j3; ++a) {
        const double *nu = nuc + S.j3_center[a] * LRDMC_NUC_STRIDE, z = S.j3_zeta[a];
        const double dx = xi - nu[0], dy = yi - nu[1], dz = zi - nu[2], V = V3_i[a];
        const int q = S.j3_poly ? S.j3_lmn[a] : 0;
        if (q == 0) {
            const double cv = chi3_i[a] * V, tz = -2.0 * z * cv;
            J += cv; gx += tz * dx; gy += tz * dy; gz += tz * dz;
            lJ += (4.0 * z * z * (dx * dx + dy * dy + dz * dz) - 6.0 * z) * cv;
        } else {
            const double eV = exp_nonpos(-z * (dx * dx + dy * dy + dz * dz)) * V;
            double fx, fx1, fx2, fy, fy1, fy2, fz, fz1, fz2;
            j3_axis(dx, q & 3, z, fx, fx1, fx2); j3_axis(dy, (q >> 2) & 3, z, fy, fy1, fy2); j3_axis(dz, (q >> 4) & 3, z, fz, fz1, fz2);
            J += chi3_i[a] * V; gx += fx1 * fy * fz * eV; gy += fx * fy1 * fz * eV; gz += fx * fy * fz1 * eV;
            lJ += (fx2 * fy * fz + fx * fy2 * fz + fx * fy * fz2) * eV;
        }
    }
}

// Pade term c r/(1 + b r) = c/(b + 1/r) of one partner at the six displaced points of an electron:
// |d0 +- a e_k|^2 = |d0|^2 + a^2 +- 2 a e_k.d0 (d0 = electron - partner), one reciprocal square root and one reciprocal each.
__device__ __forceinline__ void pade_six(double dx, double dy, double dz, const double (&av)[3][3], double a2, double c, double b, double (&J)[6])
{
    const double q0 = fma(dx, dx, fma(dy, dy, fma(dz, dz, a2)));
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double sk = fma(av[k][0], dx, fma(av[k][1], dy, av[k][2] * dz));
        J[2 * k] = fma(c, fast_rcp(b + fast_rsqrt(fma(2.0, sk, q0))), J[2 * k]);
        J[2 * k + 1] = fma(c, fast_rcp(b + fast_rsqrt(fma(-2.0, sk, q0))), J[2 * k + 1]);
    }
}

// R_j = (determinant ratio) * exp(J' - J) of the six candidates of a quad's row, from the lanes' shares: after the quad sums every lane holds the six
// sums; lane t finishes candidates d = t and (t < 2) d = 4 + t and stores them itself -- two exponentials per lane instead of six inlined copies
// (the extended kernels' hot loop has to fit the instruction cache), same arithmetic per candidate.
__device__ __forceinline__ void finish_ratios(const double (&acc)[6], const double (&Jn)[6], double Jo, const double *etab, int t, bool valid, double *Ro)
{
    double A[6], J[6];
#pragma unroll
    for (int d = 0; d < 6; ++d) { A[d] = quad_sum(acc[d]); J[d] = quad_sum(Jn[d]); }
    const double a0 = t == 0 ? A[0] : (t == 1 ? A[1] : (t == 2 ? A[2] : A[3])), j0 = t == 0 ? J[0] : (t == 1 ? J[1] : (t == 2 ? J[2] : J[3]));
    const double a1 = t == 0 ? A[4] : A[5], j1 = t == 0 ? J[4] : J[5];
    const double r0 = a0 * exp_tab(j0 - Jo, etab), r1 = a1 * exp_tab(j1 - Jo, etab);
    if (valid) { Ro[t] = r0; if (t < 2) Ro[4 + t] = r1; }
}

// Three-body Jastrow at the six displaced points x0 +- av[k] of one electron (reading Q23): Jn[d] += sum_a chi_a(point d) V_a,
// the functions dealt over the `stride` lanes that share the electron (t = this lane's index among them, a = a0 + t): six table
// exponentials per function in the same +- form as the AOs.  The trip count is uniform in the warp (exp_tab_n synchronises it).
template <bool POLY>
__device__ __forceinline__ void j3_six_loop(const DevSys &S, const Tables &T, const double *V3, double x0, double y0, double z0, const double (&av)[3][3],
                                            double a2, int t, double (&Jn)[6], int a_first, int a_stride)
{
    for (int a0 = a_first; a0 < S.n_j3; a0 += a_stride) {
        const bool on = a0 + t < S.n_j3; const int a = on ? a0 + t : 0;
        const double *np_ = T.nuc + S.j3_center[a] * LRDMC_NUC_STRIDE, z = S.j3_zeta[a];
        const double dx = x0 - np_[0], dy = y0 - np_[1], dz = z0 - np_[2], q0 = fma(dx, dx, fma(dy, dy, fma(dz, dz, a2)));
        double ex_[6], e_[6];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double sk = fma(av[k][0], dx, fma(av[k][1], dy, av[k][2] * dz));
            ex_[2 * k] = exp_arg_floor(-z * fma(2.0, sk, q0)); ex_[2 * k + 1] = exp_arg_floor(-z * fma(-2.0, sk, q0));
        }
        exp_tab_n<6>(ex_, e_, T.etab);
        const double Va = on ? V3[a] : 0.0;
        if (POLY) {                    // monomial factor at the displaced points d0 +- av[k]
            const int q = S.j3_lmn[a], kx = q & 3, ky = (q >> 2) & 3, kz = (q >> 4) & 3;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double pp = mono_pow(dx + av[k][0], kx) * mono_pow(dy + av[k][1], ky) * mono_pow(dz + av[k][2], kz);
                const double pm = mono_pow(dx - av[k][0], kx) * mono_pow(dy - av[k][1], ky) * mono_pow(dz - av[k][2], kz);
                Jn[2 * k] = fma(e_[2 * k] * pp, Va, Jn[2 * k]); Jn[2 * k + 1] = fma(e_[2 * k + 1] * pm, Va, Jn[2 * k + 1]);
            }
        } else {
#pragma unroll
            for (int d = 0; d < 6; ++d) Jn[d] = fma(e_[d], Va, Jn[d]);
        }
    }
}
__device__ __forceinline__ void j3_six(const DevSys &S, const Tables &T, const double *V3, double x0, double y0, double z0, const double (&av)[3][3],
                                       double a2, int t, double (&Jn)[6], int a_first = 0, int a_stride = 4)
{
    if (S.j3_poly) j3_six_loop<true>(S, T, V3, x0, y0, z0, av, a2, t, Jn, a_first, a_stride);      // uniform: a property of the system
    else j3_six_loop<false>(S, T, V3, x0, y0, z0, av, a2, t, Jn, a_first, a_stride);
}

// ---- non-local pseudopotential candidates (scope row f1; include/lrdmc.h lrdmc_system.nl) ------------------------------
// The kk-th centre in range of the point (x,y,z): nuclei with r_c > 0 and |r - R_I| < r_c in ascending order.  Returns its index
// (-1: fewer than kk+1 in range) and the distance.  Every lane runs the same loop on the same data (uniform result).
__device__ __forceinline__ int nl_centre(const DevSys &S, const double *nuc, double x, double y, double z, int kk, double &r_out)
{
    int seen = 0;
    for (int I = 0; I < S.n_nuc; ++I) {
        const double *nu = nuc + I * LRDMC_NUC_STRIDE, rc = nu[LRDMC_NL_OFF];
        if (!(rc > 0.0)) continue;
        const double dx = x - nu[0], dy = y - nu[1], dz = z - nu[2], r = sqrt(dx * dx + dy * dy + dz * dz);
        if (r < rc) { if (seen == kk) { r_out = r; return I; } ++seen; }
    }
    r_out = 0.0;
    return -1;
}

// Phase B of a system WITH non-local slots, by one warp: lattice blocks and slot blocks go through ONE loop with ONE ao_columns /
// pade_six call site.  The six quadrature points R_I +- r_iI e_k of a slot have exactly the +-(a e_k) structure of the lattice hops,
// about the CENTRE R_I with step r_iI, so a slot pass is a lattice pass with per-lane arguments (x0 = R_I, av = r_iI e_k, the
// Dinv column of the slot's electron); nu_q = (1/6) sum_l (2l+1) v_l(r) P_l(+-e_k . rhat).  Two inlined copies of the shell sweep
// doubled the hot instruction footprint: ncu showed 2.3 "no instruction" stall cycles per issue and the kernel at 35 % issue
// utilisation.  Returns the node flag raised by the slots (rho_q < 0).
template <int NT, bool TS, bool J3>
__device__ __forceinline__ int phase_b_with_nonlocal(const DevSys &S, const WarpState &ws, const Tables &T, const double *Jold, int lane)
{
    const int t = lane & 3, g = lane >> 2, N = S.N, K = S.nl_K, n_nuc = S.n_nuc;
    const int nb0 = (S.n_up + 7) / 8, nbm = nb0 + (S.n_dn + 7) / 8, n_lat = S.n_mesh * nbm;
    // Slots in range of a centre are few (about 2.5 of 16 at C3): list them first (lane per slot, ballot), then sweep 8 LISTED
    // slots per pass.  With one coefficient table for both spins (same_C) a pass may mix spins (per-lane inverse, per-lane n_s);
    // otherwise the list is cut at the first spin-down slot.  The list (N K <= 4 N ints) lives in the s_k / old-column scratch of the hop (free during an evaluation).
    int *list = reinterpret_cast<int *>(ws.el + 2 * N);
    int n_act = 0, n_act_up = 0;
    for (int s0 = 0; s0 < N * K; s0 += 32) {
        const int sl = s0 + lane; const bool in = sl < N * K;
        const int i = in ? sl / K : 0, kk = in ? sl - i * K : 0;
        double r;
        const bool act = in && nl_centre(S, T.nuc, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], kk, r) >= 0;
        const unsigned m = __ballot_sync(0xffffffffu, act);
        if (act) list[n_act + __popc(m & ((1u << lane) - 1u))] = sl;
        if (in) { double *Ro = ws.R + S.P_lat + 6 * sl;
#pragma unroll
            for (int d = 0; d < 6; ++d) Ro[d] = 0.0; }
        n_act_up += __popc(__ballot_sync(0xffffffffu, act && i < S.n_up));
        n_act += __popc(m);
    }
    __syncwarp();
    const int cut = S.same_C ? n_act : n_act_up;                    // passes never straddle `cut`
    const int n_p0 = (cut + 7) / 8, n_nlp = n_p0 + (n_act - cut + 7) / 8;
    int node_nl = 0;
    for (int pass = 0; pass < n_lat + n_nlp; ++pass) {
        const bool is_nl = pass >= n_lat;
        int sp, il, kk = 0, mesh = 0, i; bool valid;
        if (!is_nl) {
            mesh = pass / nbm; const int rem = pass - mesh * nbm; sp = rem >= nb0 ? 1 : 0;
            const int il0 = 8 * (sp ? rem - nb0 : rem), ns_ = sp ? S.n_dn : S.n_up;
            valid = il0 + g < ns_; il = valid ? il0 + g : 0; i = (sp ? S.n_up : 0) + il;
        } else {
            const int b = pass - n_lat, lo = b < n_p0 ? 8 * b : cut + 8 * (b - n_p0), hi = b < n_p0 ? cut : n_act;
            valid = lo + g < hi;
            const int sl = list[valid ? lo + g : lo];               // an idle row repeats the pass's first slot (its result is dropped)
            i = sl / K; kk = sl - i * K; sp = i < S.n_up ? 0 : 1; il = sp ? i - S.n_up : i;
        }
        const int ns = sp ? S.n_dn : S.n_up;
        const double xi = ws.r[3 * i], yi = ws.r[3 * i + 1], zi = ws.r[3 * i + 2];
        double x0 = xi, y0 = yi, z0 = zi, step = S.amesh[mesh], r = 0.0;
        const double *nu = T.nuc;
        if (is_nl) {
            const int I = nl_centre(S, T.nuc, xi, yi, zi, kk, r);   // listed slots are in range: I >= 0
            nu = T.nuc + I * LRDMC_NUC_STRIDE; x0 = nu[0]; y0 = nu[1]; z0 = nu[2]; step = r;
        }
        const double a2 = step * step;
        double av[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) { av[k][0] = step * ws.U[k]; av[k][1] = step * ws.U[3 + k]; av[k][2] = step * ws.U[6 + k]; }
        double acc[6], Jn[6];
        ao_columns<NT, TS>(S, T.shells, sp ? T.cf[1] : T.cf[0], T.etab, sp ? ws.dinv[1] : ws.dinv[0], ns, il, x0, y0, z0, av, a2, lane, acc);
#pragma unroll
        for (int d = 0; d < 6; ++d) Jn[d] = 0.0;
        if (!is_nl || !S.nl_dla) {
            if (S.has_j1) for (int I = t; I < n_nuc; I += 4) {
                const double *np_ = T.nuc + I * LRDMC_NUC_STRIDE;
                pade_six(x0 - np_[0], y0 - np_[1], z0 - np_[2], av, a2, -np_[4], np_[5], Jn);
            }
            for (int j = t; j < N; j += 4) {
                const double c = (j == i) ? 0.0 : ((spin_of(S, j) == sp) ? S.a_par : S.a_anti);
                pade_six(x0 - ws.r[3 * j], y0 - ws.r[3 * j + 1], z0 - ws.r[3 * j + 2], av, a2, c, S.b2, Jn);
            }
        }
        if (J3 && (!is_nl || !S.nl_dla)) j3_six(S, T, ws.j3 + (N + i) * S.j3s, x0, y0, z0, av, a2, t, Jn);
        const double Jo = Jold[i];
        if (!is_nl) {
            finish_ratios(acc, Jn, Jo, T.etab, t, valid, ws.R + mesh * 6 * N + 6 * i);
        } else {
            double nuq[6];
            {
                const double ir = 1.0 / r, hx = (xi - nu[0]) * ir, hy = (yi - nu[1]) * ir, hz = (zi - nu[2]) * ir;   // rhat of the electron about the centre
                const double r2 = r * r, *ch = nu + LRDMC_NL_OFF;
                const double v0 = ch[1] * exp_nonpos(-ch[2] * r2), v1 = 3.0 * ch[3] * exp_nonpos(-ch[4] * r2), v2 = 5.0 * ch[5] * exp_nonpos(-ch[6] * r2);
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double ct = ws.U[k] * hx + ws.U[3 + k] * hy + ws.U[6 + k] * hz, p2 = 0.5 * (3.0 * ct * ct - 1.0);
                    nuq[2 * k] = (v0 + v1 * ct + v2 * p2) * (1.0 / 6.0);
                    nuq[2 * k + 1] = (v0 - v1 * ct + v2 * p2) * (1.0 / 6.0);
                }
            }
            double *Ro = ws.R + S.P_lat + 6 * (i * K + kk);
#pragma unroll
            for (int d = 0; d < 6; ++d) {
                double rho = quad_sum(acc[d]);
                if (!S.nl_dla) rho *= exp_tab(quad_sum(Jn[d]) - Jo, T.etab);
                if (valid && t == 0) { Ro[d] = -nuq[d] * rho; if (rho < 0.0) node_nl = 1; }
            }
        }
    }
    return node_nl;
}

// Position an accepted move j puts its electron at: lattice hop r_i +- a e_k, or the quadrature point of a non-local slot.
template <bool SLOTS>
__device__ __forceinline__ void move_target(const DevSys &S, const WarpState &ws, const double *nuc, int j, int &i, double &px, double &py, double &pz)
{
    const int N = S.N;
    if (!SLOTS || j < S.P_lat) {
        const int mesh = j / (6 * N), jj = j - mesh * 6 * N, d = jj - 6 * (jj / 6), k = d >> 1;
        i = jj / 6;
        const double step = (d & 1) ? -S.amesh[mesh] : S.amesh[mesh];
        px = ws.r[3 * i] + step * ws.U[k]; py = ws.r[3 * i + 1] + step * ws.U[3 + k]; pz = ws.r[3 * i + 2] + step * ws.U[6 + k];
    } else {
        const int o = j - S.P_lat, slot = o / 6, q = o - 6 * slot, k = q >> 1, kk = slot % S.nl_K;
        i = slot / S.nl_K;
        double r;
        const int I = nl_centre(S, nuc, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], kk, r);
        const double *nu = nuc + (I < 0 ? 0 : I) * LRDMC_NUC_STRIDE, step = (q & 1) ? -r : r;
        px = nu[0] + step * ws.U[k]; py = nu[1] + step * ws.U[3 + k]; pz = nu[2] + step * ws.U[6 + k];
    }
}

// One term of the cumulative sums: the product kappa_j R_j is rounded before the add (reading Q12), in phase_c and in select_move alike.
__device__ __forceinline__ double amp_add(double run, double kap, double Rj) { return __dadd_rn(run, __dmul_rn(kap, Rj)); }
template <bool SLOTS>
__device__ __forceinline__ double kappa_of(const DevSys &S, int j)
{
    return SLOTS ? (j < 6 * S.N ? S.kappa[0] : (j < S.P_lat ? S.kappa[1] : 1.0))   // non-local slots hold -nu_q rho_q itself
                 : S.kappa[j >= 6 * S.N ? 1 : 0];
}

// Phase C (row a7) of one evaluation, by one warp on the candidate ratios R[P] left in shared memory.
// node0: node flag already raised by the non-local candidates (rho_q < 0), any lane.
template <bool SLOTS = false>
__device__ __forceinline__ EvalOut phase_c(const DevSys &S, const WarpState &ws, const double *lap_s, double Vee, int lane, int node0 = 0)
{
    const int N = S.N;
    // ---- phase C (row a7): fixed-node split (Eq.D1) and the cumulative sums C_j of the allowed amplitudes in candidate
    //      order (row a9 searches them).  Each lane owns a contiguous chunk; chunk totals are scanned across the warp
    //      (reading Q12: the summation order is free, a draw closer than 1e-9 to a bin edge is a reported near-tie).
    //      C_j = (sum over the lane's chunk up to j) + (sum of the chunks before): only the two per-lane numbers are kept
    //      (EvalOut.c_loc / c_excl); select_move re-walks the one chunk that holds the selected move -- no C_j array.
    const int P = S.P, chunk = (P + 31) >> 5, j0 = lane * chunk;
    double vsf_part = 0.0, loc = 0.0; int node = node0;
    for (int e = 0; e < chunk; ++e) {
        const int j = j0 + e;
        if (j < P) {
            const double Rj = ws.R[j];
            const double kap = kappa_of<SLOTS>(S, j);
            if (Rj > 0.0) loc = amp_add(loc, kap, Rj);
            else if (Rj < 0.0) { vsf_part -= kap * Rj; if (!SLOTS || j < S.P_lat) node = 1; }
        }
    }
    double inc = loc;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const double v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
    double excl = __shfl_up_sync(0xffffffffu, inc, 1); if (lane == 0) excl = 0.0;
    const double bbar = __shfl_sync(0xffffffffu, inc, 31);
    const double Vsf = warp_sum(vsf_part);
    node = __any_sync(0xffffffffu, node);
    double vsum = 0.0;
    for (int i = lane; i < N; i += 32) {
        double T = 0.0;
        for (int mesh = 0; mesh < S.n_mesh; ++mesh) {
            const double *Rm = ws.R + mesh * 6 * N + 6 * i;
            double s = Rm[0]; s += Rm[1]; s += Rm[2]; s += Rm[3]; s += Rm[4]; s += Rm[5];
            T += S.g_over_a2[mesh] * (s - 6.0);                      // discretised Laplacian of Eq.D3 over Psi_G
        }
        const double *ob = ws.ob + 8 * i;
        const double vzv = ob[5] + 0.5 * (T - lap_s[i]);              // Eq.D8
        vsum += node ? fmax(vzv, ob[6]) : vzv;                        // Eq.D9 / D11 (reading Q5: global node flag)
    }
    vsum = warp_sum(vsum);
    EvalOut o;
    o.bbar = bbar; o.Vsf = Vsf; o.node = node;
    o.W = S.Kdiag + vsum + Vee + S.V_ii + Vsf;                        // L628 + kinetic diagonal of Eq.D5 (reading Q3)
    o.eL = o.W - bbar;                                                // L223
    o.c_loc = loc; o.c_excl = excl;
    return o;
}

// Phase B as a LISTED sweep (listed.cuh; EXT bit 2) of the 8-row batches first, first + stride, ... of the rows (mesh, electron) by one warp:
// quad per row, the determinant ratios from the walker's stored Bc over the electron's own shell lists, the Jastrow ratios of the same
// rows from the same geometry, R_j = ratio * exp(J' - J).  Rows are independent, so a warp finishes its batches without meeting the others.
__device__ __forceinline__ void listed_phase_b(const DevSys &S, const WarpState &ws, const Tables &T, const double *Jold, int first, int stride, int lane)
{
    const int N = S.N, n_nuc = S.n_nuc, t = lane & 3, g = lane >> 2, n_rows = S.n_mesh * N;
    for (int r0 = 8 * first; r0 < n_rows; r0 += 8 * stride) {
        const bool valid = r0 + g < n_rows;
        const int rho = valid ? r0 + g : r0, mesh = rho / N, i = rho - mesh * N, sp = spin_of(S, i);
        const double x0 = ws.r[3 * i], y0 = ws.r[3 * i + 1], z0 = ws.r[3 * i + 2], am_ = S.amesh[mesh], a2 = am_ * am_;
        double av[3][3], acc[6], Jn[6];
#pragma unroll
        for (int k = 0; k < 3; ++k) { av[k][0] = am_ * ws.U[k]; av[k][1] = am_ * ws.U[3 + k]; av[k][2] = am_ * ws.U[6 + k]; }
        ao_listed_quad(S, T.shells, T.etab, ws.lw, ws.bc, i, valid, x0, y0, z0, av, a2, lane, acc);
#pragma unroll
        for (int d = 0; d < 6; ++d) Jn[d] = 0.0;
        if (S.has_j1) for (int I = t; I < n_nuc; I += 4) {
            const double *np_ = T.nuc + I * LRDMC_NUC_STRIDE;
            pade_six(x0 - np_[0], y0 - np_[1], z0 - np_[2], av, a2, -np_[4], np_[5], Jn);
        }
        for (int j = t; j < N; j += 4) {
            const double c = (j == i) ? 0.0 : ((spin_of(S, j) == sp) ? S.a_par : S.a_anti);
            pade_six(x0 - ws.r[3 * j], y0 - ws.r[3 * j + 1], z0 - ws.r[3 * j + 2], av, a2, c, S.b2, Jn);
        }
        const double Jo = Jold[i];
        finish_ratios(acc, Jn, Jo, T.etab, t, valid, ws.R + mesh * 6 * N + 6 * i);
    }
}

// EXT (extended kernels, separate instantiations so that each system pays only for what it has): bit 0 = non-local
// pseudopotential slots (row f1), bit 1 = three-body Jastrow (row f2), bit 2 = listed candidate sweep on stored Bc (listed.cuh; lattice-only systems).
template <int NT, bool TS, int EXT = 0>
__device__ __forceinline__ EvalOut evaluate_walker(const DevSys &S, const WarpState &ws, const Tables &T, int lane)
{
    constexpr bool SLOTS = (EXT & 1) != 0, J3 = (EXT & 2) != 0, LISTED = (EXT & 4) != 0;
    const int N = S.N, n_nuc = S.n_nuc;
    const int t = lane & 3, g = lane >> 2;
    double *Jold = ws.el, *lap_s = ws.el + N;

    // ---- phase A (row a6): per-electron continuum pieces.  Two lanes per electron split the e-e partners; the
    //      one-body parts come from the cache.
    if (J3) j3_fields(S, T.j3g, ws.j3, lane, 32, [] { __syncwarp(); });     // three-body fields V_a(i) of this evaluation
    double vee_part = 0.0;
    for (int i0 = 0; i0 < N; i0 += 16) {
        const int i = i0 + (lane >> 1), sub = lane & 1;
        const bool act = i < N;
        const int ii = act ? i : 0;
        const int sp = spin_of(S, ii), il = sp ? ii - S.n_up : ii, ns = sp ? S.n_dn : S.n_up;
        const double xi = ws.r[3 * ii], yi = ws.r[3 * ii + 1], zi = ws.r[3 * ii + 2];
        double J = 0.0, gx = 0.0, gy = 0.0, gz = 0.0, lJ = 0.0, ve = 0.0;
        for (int j = sub; j < N; j += 2) if (j != ii) {
            const double dx = xi - ws.r[3 * j], dy = yi - ws.r[3 * j + 1], dz = zi - ws.r[3 * j + 2], r2 = dx * dx + dy * dy + dz * dz;
            const double ir = fast_rsqrt(r2), r = r2 * ir;
            const double c = (spin_of(S, j) == sp) ? S.a_par : S.a_anti, iq = fast_rcp(1.0 + S.b2 * r), du = c * iq * iq * ir;
            J += c * r * iq; gx += du * dx; gy += du * dy; gz += du * dz; lJ += 2.0 * du * iq;
            if (j > ii) ve += ir;
        }
        // grad D / D and lap D / D through the stored inverse and the cached MO rows: the two lanes split the MOs
        const double *mc = ws.moc + (size_t)ii * 5 * S.OS, *di = (sp ? ws.dinv[1] : ws.dinv[0]) + il;
        double Gx = 0.0, Gy = 0.0, Gz = 0.0, Ld = 0.0;
        for (int m = sub; m < ns; m += 2) {
            const double d = di[m * ns];
            Gx += mc[S.OS + m] * d; Gy += mc[2 * S.OS + m] * d; Gz += mc[3 * S.OS + m] * d; Ld += mc[4 * S.OS + m] * d;
        }
#define PAIR_SUM(v) v += __shfl_xor_sync(0xffffffffu, v, 1)
        PAIR_SUM(J); PAIR_SUM(gx); PAIR_SUM(gy); PAIR_SUM(gz); PAIR_SUM(lJ); PAIR_SUM(Gx); PAIR_SUM(Gy); PAIR_SUM(Gz); PAIR_SUM(Ld);
#undef PAIR_SUM
        if (act) vee_part += ve;
        if (act && sub == 0) {
            const double *ob = ws.ob + 8 * ii;
            gx += ob[1]; gy += ob[2]; gz += ob[3];
            if (J3) j3_electron_terms(S, T.nuc, ws.j3 + ii * S.j3s, ws.j3 + (N + ii) * S.j3s, xi, yi, zi, J, gx, gy, gz, lJ);
            Jold[ii] = J + ob[0];
            lap_s[ii] = Ld + 2.0 * (Gx * gx + Gy * gy + Gz * gz) + (lJ + ob[4]) + (gx * gx + gy * gy + gz * gz);
        }
    }
    const double Vee = warp_sum(vee_part);
    __syncwarp();

    // ---- phase B (rows a1-a5): the 6 n_s candidates of each spin, 8 electrons (48 points) per warp pass in column form
    if (LISTED) listed_phase_b(S, ws, T, Jold, 0, 1, lane);
    if (!SLOTS && !LISTED) for (int mesh = 0; mesh < S.n_mesh; ++mesh) {
        const double am = S.amesh[mesh], a2 = am * am;
        double av[3][3];                                             // av[k] = a e_k, e_k = k-th column of U (Eq.D3-D4)
#pragma unroll
        for (int k = 0; k < 3; ++k) { av[k][0] = am * ws.U[k]; av[k][1] = am * ws.U[3 + k]; av[k][2] = am * ws.U[6 + k]; }
        for (int sp = 0; sp < 2; ++sp) {
            const int ns = sp ? S.n_dn : S.n_up, off = sp ? S.n_up : 0;
            for (int il0 = 0; il0 < ns; il0 += 8) {
                const bool valid = il0 + g < ns;
                const int il = valid ? il0 + g : 0, i = off + il;
                const double x0 = ws.r[3 * i], y0 = ws.r[3 * i + 1], z0 = ws.r[3 * i + 2];
                double acc[6], Jn[6];
                ao_columns<NT, TS>(S, T.shells, sp ? T.cf[1] : T.cf[0], T.etab, sp ? ws.dinv[1] : ws.dinv[0], ns, il, x0, y0, z0, av, a2, lane, acc);
                // Jastrow ratio (row a5): the 4 lanes of the quad split the partners; u = c r/(1 + b r) = c/(b + 1/r)
#pragma unroll
                for (int d = 0; d < 6; ++d) Jn[d] = 0.0;
                if (S.has_j1) for (int I = t; I < n_nuc; I += 4) {
                    const double *nu = T.nuc + I * LRDMC_NUC_STRIDE;
                    pade_six(x0 - nu[0], y0 - nu[1], z0 - nu[2], av, a2, -nu[4], nu[5], Jn);
                }
                for (int j = t; j < N; j += 4) {
                    const double c = (j == i) ? 0.0 : ((spin_of(S, j) == sp) ? S.a_par : S.a_anti);
                    pade_six(x0 - ws.r[3 * j], y0 - ws.r[3 * j + 1], z0 - ws.r[3 * j + 2], av, a2, c, S.b2, Jn);
                }
                if (J3) j3_six(S, T, ws.j3 + (N + i) * S.j3s, x0, y0, z0, av, a2, t, Jn);
                const double Jo = Jold[i];
                finish_ratios(acc, Jn, Jo, T.etab, t, valid, ws.R + mesh * 6 * N + 6 * i);
            }
        }
    }
    // ---- systems with non-local pseudopotential slots (row f1): lattice blocks and slot blocks in one loop
    int node_nl = 0;
    if (SLOTS) node_nl = phase_b_with_nonlocal<NT, TS, J3>(S, ws, T, Jold, lane);
    __syncwarp();

    const EvalOut o = phase_c<SLOTS>(S, ws, lap_s, Vee, lane, node_nl);
    __syncwarp();
    return o;
}

// Heat-bath selection (Eq.29): j* = min{ j : C_j > u C_{P-1} } with C_j as phase_c defines them (e = the EvalOut of THIS warp's phase_c);
// fallback = last allowed move; -1 if none is allowed.  All lanes return the same j*.
template <bool SLOTS = false>
__device__ __forceinline__ int select_move(const DevSys &S, const WarpState &ws, const EvalOut &e, double u_sel, int lane)
{
    LRDMC_ASSUME_SHARED(ws.R);
    const int P = S.P, chunk = (P + 31) >> 5, j0 = lane * chunk;
    const double mine = e.c_loc + e.c_excl;                            // C_j of the last candidate of this lane's chunk
    const double tot = __shfl_sync(0xffffffffu, mine, (P - 1) / chunk);  // C_{P-1}
    if (!(tot > 0.0)) return -1;
    const double thr = __dmul_rn(u_sel, tot);
    const unsigned hit = __ballot_sync(0xffffffffu, j0 < P && e.c_loc > 0.0 && mine > thr);   // (a chunk without an allowed move cannot hold j*)
    if (hit) {                                                         // the first chunk whose last C_j passes holds j*: its lane walks it again
        const int L = __ffs(hit) - 1; int js = -1;
        if (lane == L) {
            double run = 0.0;
            for (int q = 0; q < chunk && js < 0; ++q) {
                const int j = j0 + q;
                if (j < P) { const double Rj = ws.R[j]; if (Rj > 0.0) { run = amp_add(run, kappa_of<SLOTS>(S, j), Rj); if (run + e.c_excl > thr) js = j; } }
            }
        }
        return __shfl_sync(0xffffffffu, js, L);
    }
    int last = -1;                                                     // rounding left no C_j > thr: last j with q_j > 0
    for (int j = lane; j < P; j += 32) if (ws.R[j] > 0.0) last = j;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
    return last;
}

// Apply move j (row a10): r_i <- r'_j, refresh the cached MO rows and the one-body cache of electron i, Sherman-Morrison on Dinv_sigma.
template <int NT, bool TS, int EXT = 0>
__device__ __forceinline__ void apply_move(const DevSys &S, const WarpState &ws, const Tables &T, int j, int lane)
{
    const int N = S.N; int i; double px, py, pz;
    move_target<(EXT & 1) != 0>(S, ws, T.nuc, j, i, px, py, pz);
    const int sp = spin_of(S, i), il = sp ? i - S.n_up : i, ns = sp ? S.n_dn : S.n_up;
    double *mc = ws.moc + (size_t)i * 5 * S.OS;
    __syncwarp();
    refresh_mo_cache<NT, LRDMC_BF_SMEM(TS, EXT)>(S, T.shells, sp ? T.bf[1] : T.bf[0], T.etab, mc, px, py, pz, lane);
    refresh_onebody(S.n_nuc, S.has_j1, S.a, T.nuc, ws.ob + 8 * i, px, py, pz, lane);
    if (EXT & 2) refresh_j3_row(S, T.nuc, ws.j3 + i * S.j3s, px, py, pz, lane);
    if (EXT & 4) list_build(S, T.shells, T.srad, ws.lw, i, px, py, pz, fmax(S.amesh[0], S.amesh[1]), lane);   // the mover's listed shells at its new position
    if (lane == 0) { ws.r[3 * i] = px; ws.r[3 * i + 1] = py; ws.r[3 * i + 2] = pz; }
    __syncwarp();
    // s_k = sum_m phi_m Dinv[m][k];  rho = s_il;  Dinv'[m][il] = Dinv[m][il]/rho;  Dinv'[m][k] = Dinv[m][k] - Dinv[m][il] s_k / rho
    double *dinv = sp ? ws.dinv[1] : ws.dinv[0], *sk = ws.el + 2 * N, *col = ws.el + 3 * N;   // scratch: s_k and the old column il (n_s <= N each)
    for (int kk = lane; kk < ns; kk += 32) {
        double s = 0.0;
        for (int m = 0; m < ns; ++m) s += mc[m] * dinv[m * ns + kk];
        sk[kk] = s; col[kk] = dinv[kk * ns + il];
    }
    __syncwarp();
    const double irho = 1.0 / sk[il];
    for (int idx = lane; idx < ns * ns; idx += 32) {
        const int m = idx / ns, kk = idx - m * ns;
        const double ci = col[m] * irho;
        dinv[idx] = (kk == il) ? ci : dinv[idx] - ci * sk[kk];
    }
    if (EXT & 4) bc_rank1_update(S, ws.bc, sp, il, ns, sk, irho, lane, 32);
    __syncwarp();
}
