// evaluate.cuh -- one evaluation of the lattice-regularised fixed-node Hamiltonian at a walker's configuration
// (Appendix D; rows a1, a4-a10 of the scope table), by ONE WARP on shared-memory state.
#pragma once
#include "common.cuh"
#include "philox.cuh"
#include "wavefunction.cuh"

struct WarpState {            // per-warp views (shared memory; moc may live in global memory for large systems)
    double *r, *dinv[2], *moc, *R, *cum, *el;
};
struct EvalOut { double bbar, Vsf, W, eL; int node; };

__device__ __forceinline__ int spin_of(const DevSys &S, int i) { return i < S.n_up ? 0 : 1; }

// Pade pair terms (reading Q14): u = c r/(1+b r), u' = c/(1+br)^2, lap u = 2c/(r (1+br)^3)
__device__ __forceinline__ double pade_u(double c, double b, double r) { return c * r / (1.0 + b * r); }

// electron-ion potential of one nucleus and its lower bound (Eq.D10; ECP rule L623)
__device__ __forceinline__ void nuc_potential(const DevSys &S, const double *nu, double r, double &v, double &vb)
{
    double Z = nu[3];
    if (nu[10] != 0.0) {
        double r2 = r * r;
        v = Z * expm1(-nu[6] * r2) / r + Z * nu[6] * r * exp(-nu[7] * r2) + nu[8] * exp(-nu[9] * r2);
        vb = -Z / r;
    } else { v = -Z / r; vb = -Z / fmax(r, S.a); }
}

template <int NT>
__device__ __forceinline__ EvalOut evaluate_walker(const DevSys &S, const WarpState &ws, const double *shells, const double *const bf[2],
                                                   const double *nuc, const double U[9], int lane)
{
    const int N = S.N, n_nuc = S.n_nuc;
    const int t = lane & 3, g = lane >> 2;
    double *Jold = ws.el, *vei_s = ws.el + N, *vb_s = ws.el + 2 * N, *lap_s = ws.el + 3 * N;

    // ---- phase A (row a6): per-electron continuum pieces.  lane <-> electron.
    double vee_part = 0.0;
    for (int i = lane; i < N; i += 32) {
        const int sp = spin_of(S, i), il = sp ? i - S.n_up : i, ns = sp ? S.n_dn : S.n_up;
        const double xi = ws.r[3 * i], yi = ws.r[3 * i + 1], zi = ws.r[3 * i + 2];
        double J = 0.0, gx = 0.0, gy = 0.0, gz = 0.0, lJ = 0.0, vei = 0.0, vb = 0.0;
        for (int I = 0; I < n_nuc; ++I) {
            const double *nu = nuc + I * LRDMC_NUC_STRIDE;
            double dx = xi - nu[0], dy = yi - nu[1], dz = zi - nu[2], r = sqrt(dx * dx + dy * dy + dz * dz);
            if (S.has_j1) {
                double c = -nu[4], q = 1.0 + nu[5] * r, iq = 1.0 / q, du = c * iq * iq / r;
                J += c * r * iq; gx += du * dx; gy += du * dy; gz += du * dz; lJ += 2.0 * du * iq;
            }
            double v, b; nuc_potential(S, nu, r, v, b); vei += v; vb += b;
        }
        for (int j = 0; j < N; ++j) if (j != i) {
            double dx = xi - ws.r[3 * j], dy = yi - ws.r[3 * j + 1], dz = zi - ws.r[3 * j + 2], r = sqrt(dx * dx + dy * dy + dz * dz);
            double c = (spin_of(S, j) == sp) ? S.a_par : S.a_anti, q = 1.0 + S.b2 * r, iq = 1.0 / q, du = c * iq * iq / r;
            J += c * r * iq; gx += du * dx; gy += du * dy; gz += du * dz; lJ += 2.0 * du * iq;
            if (j > i) vee_part += 1.0 / r;
        }
        // grad D / D and lap D / D through the stored inverse and the cached MO rows
        const double *mc = ws.moc + (size_t)i * 5 * S.OS, *di = ws.dinv[sp] + il;
        double Gx = 0.0, Gy = 0.0, Gz = 0.0, Ld = 0.0;
        for (int m = 0; m < ns; ++m) {
            double d = di[m * ns];
            Gx += mc[S.OS + m] * d; Gy += mc[2 * S.OS + m] * d; Gz += mc[3 * S.OS + m] * d; Ld += mc[4 * S.OS + m] * d;
        }
        Jold[i] = J; vei_s[i] = vei; vb_s[i] = vb;
        lap_s[i] = Ld + 2.0 * (Gx * gx + Gy * gy + Gz * gz) + lJ + (gx * gx + gy * gy + gz * gz);
    }
    const double Vee = warp_sum(vee_part);
    __syncwarp();

    // ---- phase B (rows a1-a5): candidates in batches of 8 points through the tensor-core MO pass
    for (int mesh = 0; mesh < S.n_mesh; ++mesh) {
        const double am = S.amesh[mesh];
        for (int sp = 0; sp < 2; ++sp) {
            const int ns = sp ? S.n_dn : S.n_up, off = sp ? S.n_up : 0, npts = 6 * ns;
            if (ns == 0) continue;
            const double *dinv = ws.dinv[sp];
            for (int q0 = 0; q0 < npts; q0 += 8) {
                const bool valid = q0 + g < npts;
                const int q = valid ? q0 + g : 0, il = q / 6, d = q - 6 * il, i = off + il, k = d >> 1;
                const double step = (d & 1) ? -am : am;
                const double px = ws.r[3 * i] + step * U[k], py = ws.r[3 * i + 1] + step * U[3 + k], pz = ws.r[3 * i + 2] + step * U[6 + k];
                double acc[NT][2];
                mo_pass<NT, false>(S, shells, bf[sp], px, py, pz, lane, acc);
                // determinant ratio (row a4): sum_m phi_m(r') Dinv[m][il]; this lane holds m = 8 nt + 2t, +1 (rows beyond n_s are zero-padded)
                double part = 0.0;
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                    int m = 8 * nt + 2 * t;
                    part += acc[nt][0] * dinv[m * ns + il] + acc[nt][1] * dinv[(m + 1) * ns + il];
                }
                const double dr = quad_sum(part);
                // Jastrow ratio (row a5): partners split over the 4 lanes of the quad
                double Jn = 0.0;
                if (S.has_j1) for (int I = t; I < n_nuc; I += 4) {
                    const double *nu = nuc + I * LRDMC_NUC_STRIDE;
                    double dx = px - nu[0], dy = py - nu[1], dz = pz - nu[2];
                    Jn -= pade_u(nu[4], nu[5], sqrt(dx * dx + dy * dy + dz * dz));
                }
                for (int j = t; j < N; j += 4) if (j != i) {
                    double dx = px - ws.r[3 * j], dy = py - ws.r[3 * j + 1], dz = pz - ws.r[3 * j + 2];
                    Jn += pade_u((spin_of(S, j) == sp) ? S.a_par : S.a_anti, S.b2, sqrt(dx * dx + dy * dy + dz * dz));
                }
                Jn = quad_sum(Jn);
                if (valid && t == 0) ws.R[mesh * 6 * N + 6 * i + d] = dr * exp(Jn - Jold[i]);
            }
        }
    }
    __syncwarp();

    // ---- phase C (row a7): fixed-node split (Eq.D1), sequential cumulative sums in candidate order (row a9 needs them)
    double bbar = 0.0, Vsf = 0.0; int node = 0;
    if (lane == 0) {
        const int P = S.P, sixN = 6 * N;
        for (int mesh = 0, j = 0; mesh < S.n_mesh; ++mesh) {
            const double kap = S.kappa[mesh];
            for (int jj = 0; jj < sixN; ++jj, ++j) {
                double Rj = ws.R[j];
                if (Rj > 0.0) bbar = __dadd_rn(bbar, __dmul_rn(kap, Rj));
                else if (Rj < 0.0) { Vsf -= kap * Rj; node = 1; }
                ws.cum[j] = bbar;
            }
        }
        (void)P;
    }
    bbar = __shfl_sync(0xffffffffu, bbar, 0); Vsf = __shfl_sync(0xffffffffu, Vsf, 0); node = __shfl_sync(0xffffffffu, node, 0);
    double vsum = 0.0;
    for (int i = lane; i < N; i += 32) {
        double T = 0.0;
        for (int mesh = 0; mesh < S.n_mesh; ++mesh) {
            const double *Rm = ws.R + mesh * 6 * N + 6 * i;
            double s = Rm[0]; s += Rm[1]; s += Rm[2]; s += Rm[3]; s += Rm[4]; s += Rm[5];
            T += S.g_over_a2[mesh] * (s - 6.0);                      // discretised Laplacian of Eq.D3 over Psi_G
        }
        double vzv = vei_s[i] + 0.5 * (T - lap_s[i]);                 // Eq.D8
        double vopt = node ? fmax(vzv, vb_s[i]) : vzv;                // Eq.D9 / D11 (reading Q5: global node flag)
        vsum += vopt;
    }
    vsum = warp_sum(vsum);
    EvalOut o;
    o.bbar = bbar; o.Vsf = Vsf; o.node = node;
    o.W = S.Kdiag + vsum + Vee + S.V_ii + Vsf;                        // L628 + kinetic diagonal of Eq.D5 (reading Q3)
    o.eL = o.W - bbar;                                                // L223
    __syncwarp();
    return o;
}

// Heat-bath selection (Eq.29): j* = min{ j : C_j > u C_{P-1} } on the sequential cumulative sums left in ws.cum;
// fallback = last allowed move; -1 if none is allowed.  All lanes return the same j*.
__device__ __forceinline__ int select_move(const DevSys &S, const WarpState &ws, double u_sel, int lane)
{
    const int P = S.P;
    const double tot = ws.cum[P - 1];
    if (!(tot > 0.0)) return -1;
    const double thr = __dmul_rn(u_sel, tot);
    for (int j0 = 0; j0 < P; j0 += 32) {
        int j = j0 + lane;
        unsigned hit = __ballot_sync(0xffffffffu, j < P && ws.cum[j] > thr);
        if (hit) return j0 + __ffs(hit) - 1;
    }
    int last = -1;                                                     // rounding left no C_j > thr: last j with q_j > 0
    for (int j = lane; j < P; j += 32) if (ws.R[j] > 0.0) last = j;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
    return last;
}

// Apply move j (row a10): r_i <- r'_j, refresh the cached MO rows of electron i, Sherman-Morrison on Dinv_sigma.
template <int NT>
__device__ __forceinline__ void apply_move(const DevSys &S, const WarpState &ws, const double *shells, const double *const bf[2],
                                           const double U[9], int j, int lane)
{
    const int N = S.N, mesh = j / (6 * N), jj = j - mesh * 6 * N, i = jj / 6, d = jj - 6 * i, k = d >> 1;
    const int sp = spin_of(S, i), il = sp ? i - S.n_up : i, ns = sp ? S.n_dn : S.n_up;
    const double step = (d & 1) ? -S.amesh[mesh] : S.amesh[mesh];
    const double px = ws.r[3 * i] + step * U[k], py = ws.r[3 * i + 1] + step * U[3 + k], pz = ws.r[3 * i + 2] + step * U[6 + k];
    double *mc = ws.moc + (size_t)i * 5 * S.OS;
    __syncwarp();
    refresh_mo_cache<NT>(S, shells, bf[sp], mc, px, py, pz, lane);
    if (lane == 0) { ws.r[3 * i] = px; ws.r[3 * i + 1] = py; ws.r[3 * i + 2] = pz; }
    __syncwarp();
    // s_k = sum_m phi_m Dinv[m][k];  rho = s_il;  Dinv'[m][il] = Dinv[m][il]/rho;  Dinv'[m][k] = Dinv[m][k] - Dinv[m][il] s_k / rho
    double *dinv = ws.dinv[sp], *sk = ws.el + 4 * N, *col = ws.el + 5 * N;   // scratch: s_k and the old column il (n_s <= N each)
    for (int kk = lane; kk < ns; kk += 32) {
        double s = 0.0;
        for (int m = 0; m < ns; ++m) s += mc[m] * dinv[m * ns + kk];
        sk[kk] = s; col[kk] = dinv[kk * ns + il];
    }
    __syncwarp();
    const double rho = sk[il];
    for (int idx = lane; idx < ns * ns; idx += 32) {
        int m = idx / ns, kk = idx - m * ns;
        dinv[idx] = (kk == il) ? col[m] / rho : dinv[idx] - col[m] * sk[kk] / rho;
    }
    __syncwarp();
}
