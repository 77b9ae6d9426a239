// team.cuh -- the projection kernel in TEAM form: one CTA of TW warps works on ONE walker (north_star: "one CTA or warp
// group per walker").  Same arithmetic per candidate as the warp-per-walker kernel of propagate.cuh; what changes is who
// does it:
//   * few walkers (the paper runs 100 walkers per GPU, L289): with one warp per walker 100 warps would sit on 148 SMs.
//     The candidate pass of an evaluation is cut into work units (8-electron block) x (shell part) that the TW warps take
//     in turn; partial determinant ratios and partial Jastrow sums meet in shared memory.
//   * large systems (64 electrons, 600 AOs): one walker's state is 36 KB of shared memory, so warp-per-walker leaves one warp
//     per scheduler (ncu: 6 % warps active, FP64 pipe 21 %).  Here TW warps share that one state.
// The walker queue, the weight rules (Alg.2 lines 4-8 L401-L410 / Alg.1) and the HBM layout are those of k_propagate.
#pragma once
#include "propagate.cuh"
#include "listed.cuh"

__device__ __forceinline__ void load_walker_team(const DevSys &S, const DevWalk &W, WarpState &ws, const double *nuc, int k, int TW)
{
    const int N = S.N, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, wt = tid >> 5;
    for (int i = tid; i < 3 * N; i += nthr) ws.r[i] = W.r[(size_t)k * 3 * N + i];
    for (int sp = 0; sp < 2; ++sp) {
        const int ns = sp ? S.n_dn : S.n_up, tot = S.dinv_rows[sp] * ns;
        const double *src = W.dinv[sp] + (size_t)k * ns * ns;
        for (int i = tid; i < tot; i += nthr) ws.dinv[sp][i] = (i < ns * ns) ? src[i] : 0.0;
    }
    const size_t mocn = (size_t)N * 5 * S.OS;
    if (S.moc_in_smem) { for (int i = tid; i < (int)mocn; i += nthr) ws.moc[i] = W.moc[(size_t)k * mocn + i]; }
    else ws.moc = W.moc + (size_t)k * mocn;
    __syncthreads();
    for (int i = wt; i < N; i += TW) {
        refresh_onebody(S.n_nuc, S.has_j1, S.a, nuc, ws.ob + 8 * i, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], lane);
        if (S.n_j3) refresh_j3_row(S, nuc, ws.j3 + i * S.j3s, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], lane);
    }
    __syncthreads();
}

__device__ __forceinline__ void store_walker_team(const DevSys &S, const DevWalk &W, const WarpState &ws, int k)
{
    const int N = S.N, tid = threadIdx.x, nthr = blockDim.x;
    for (int i = tid; i < 3 * N; i += nthr) W.r[(size_t)k * 3 * N + i] = ws.r[i];
    for (int sp = 0; sp < 2; ++sp) {
        const int ns = sp ? S.n_dn : S.n_up;
        double *dst = W.dinv[sp] + (size_t)k * ns * ns;
        for (int i = tid; i < ns * ns; i += nthr) dst[i] = ws.dinv[sp][i];
    }
    const size_t mocn = (size_t)N * 5 * S.OS;
    if (S.moc_in_smem) for (int i = tid; i < (int)mocn; i += nthr) W.moc[(size_t)k * mocn + i] = ws.moc[i];
}

// The draws of step `step` of walker `slot` (row a0) by one warp: frame U in out[0..8], u_sel in out[10], u_tau in out[11].
__device__ __forceinline__ void team_step_frame(const DevSys &S, double *out, uint32_t slot, uint32_t cycle, uint32_t step, bool need_tau, int lane)
{
    const StepDraws d = step_draws(S, slot, cycle, step, need_tau);
    if (lane == 0) {
        double U[9]; lattice_frame(d.u1, d.u2, d.u3, U);
#pragma unroll
        for (int i = 0; i < 9; ++i) out[i] = U[i];
        out[10] = d.u_sel; out[11] = d.u_tau;
    }
}

// One evaluation by the team.  The result is valid in warp 0 only (it runs phase C); ws.R is complete for everyone
// after the caller's next barrier.  s_vee: TW doubles of static shared memory.
// BCS: parked Bc entries (wavefunction.cuh, ao_columns): bcs_cta = this CTA's scratch [block of a mesh][k-step pair][lane];
// reuse_spin = the spin that did not hop since the last evaluation (-1: none).  A unit's entries are parked and taken back by the
// same warp: unit -> warp is a fixed map, and P.mesh_share says that both meshes of a block land on the same warp.
template <int NT, bool TS, int EXT, bool BCS>
__device__ __forceinline__ EvalOut evaluate_team(const DevSys &S, const TeamPlan &P, const WarpState &ws, const Tables &T, double *scr, double *s_vee, int *s_node,
                                                 double2 *bcs_cta, int reuse_spin)
{
    constexpr bool LISTED = (EXT & 4) != 0;        // listed sweep on the CTA's rank-1-updated Bc (listed.cuh); BCS: parked Bc entries of the dense sweep
    const int N = S.N, n_nuc = S.n_nuc, TW = P.TW, NP = P.NP, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, wt = tid >> 5;
    const int t = lane & 3, g = lane >> 2;
    constexpr bool NL = (EXT & 1) != 0, J3 = (EXT & 2) != 0;      // non-local slots / three-body Jastrow (separate instantiations)
    double *Jold = ws.el, *lap_s = ws.el + N;

    if (J3) j3_fields(S, T.j3g, ws.j3, tid, nthr, [] { __syncthreads(); });     // three-body fields V_a(i) of this evaluation (evaluate.cuh)
    // ---- phase A (row a6): per-electron continuum pieces; P.lpe lanes of one warp per electron split the partners and the MOs
    {
        const int LPE = P.lpe, epp = nthr / LPE;
        double vee_part = 0.0;
        for (int i0 = 0; i0 < N; i0 += epp) {
            const int i = i0 + tid / LPE, sub = tid & (LPE - 1);
            const bool act = i < N;
            const int ii = act ? i : 0;
            const int sp = spin_of(S, ii), il = sp ? ii - S.n_up : ii, ns = sp ? S.n_dn : S.n_up;
            const double xi = ws.r[3 * ii], yi = ws.r[3 * ii + 1], zi = ws.r[3 * ii + 2];
            double J = 0.0, gx = 0.0, gy = 0.0, gz = 0.0, lJ = 0.0, ve = 0.0;
            for (int j = sub; j < N; j += LPE) if (j != ii) {
                const double dx = xi - ws.r[3 * j], dy = yi - ws.r[3 * j + 1], dz = zi - ws.r[3 * j + 2], r2 = dx * dx + dy * dy + dz * dz;
                const double ir = fast_rsqrt(r2), r = r2 * ir;
                const double c = (spin_of(S, j) == sp) ? S.a_par : S.a_anti, iq = fast_rcp(1.0 + S.b2 * r), du = c * iq * iq * ir;
                J += c * r * iq; gx += du * dx; gy += du * dy; gz += du * dz; lJ += 2.0 * du * iq;
                if (j > ii) ve += ir;
            }
            const double *mc = ws.moc + (size_t)ii * 5 * S.OS, *di = (sp ? ws.dinv[1] : ws.dinv[0]) + il;
            double Gx = 0.0, Gy = 0.0, Gz = 0.0, Ld = 0.0;
            for (int m = sub; m < ns; m += LPE) {
                const double d = di[m * ns];
                Gx += mc[S.OS + m] * d; Gy += mc[2 * S.OS + m] * d; Gz += mc[3 * S.OS + m] * d; Ld += mc[4 * S.OS + m] * d;
            }
            for (int o = 1; o < LPE; o <<= 1) {
#define GRP_SUM(v) v += __shfl_xor_sync(0xffffffffu, v, o)
                GRP_SUM(J); GRP_SUM(gx); GRP_SUM(gy); GRP_SUM(gz); GRP_SUM(lJ); GRP_SUM(Gx); GRP_SUM(Gy); GRP_SUM(Gz); GRP_SUM(Ld);
#undef GRP_SUM
            }
            if (act) vee_part += ve;
            if (act && sub == 0) {
                const double *ob = ws.ob + 8 * ii;
                gx += ob[1]; gy += ob[2]; gz += ob[3];
                if (J3) j3_electron_terms(S, T.nuc, ws.j3 + ii * S.j3s, ws.j3 + (N + ii) * S.j3s, xi, yi, zi, J, gx, gy, gz, lJ);
                Jold[ii] = J + ob[0];
                lap_s[ii] = Ld + 2.0 * (Gx * gx + Gy * gy + Gz * gz) + (lJ + ob[4]) + (gx * gx + gy * gy + gz * gz);
            }
        }
        vee_part = warp_sum(vee_part);
        if (lane == 0) s_vee[wt] = vee_part;
    }
    if (NL && wt == TW - 1) {        // list the slots in range of a centre (ballot), clear the others; list in the hop's s_k / old-column scratch (free during an evaluation)
        int *lst = reinterpret_cast<int *>(ws.el + 2 * N);
        const int Kk = S.nl_K; int na = 0, nup = 0;
        for (int s0 = 0; s0 < N * Kk; s0 += 32) {
            const int sl = s0 + lane; const bool in = sl < N * Kk;
            const int i = in ? sl / Kk : 0, kk = in ? sl - i * Kk : 0;
            double r;
            const bool act = in && nl_centre(S, T.nuc, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], kk, r) >= 0;
            const unsigned m = __ballot_sync(0xffffffffu, act);
            if (act) lst[na + __popc(m & ((1u << lane) - 1u))] = sl;
            if (in) {
                if (NP == 1) { double *Ro = ws.R + S.P_lat + 6 * sl;
#pragma unroll
                    for (int d = 0; d < 6; ++d) Ro[d] = 0.0; }
                else scr[P.o_nu + (size_t)sl * 7 + 6] = 0.0;
            }
            nup += __popc(__ballot_sync(0xffffffffu, act && i < S.n_up));
            na += __popc(m);
        }
        if (lane == 0) { s_node[1] = na; s_node[2] = S.same_C ? na : nup; }
    }
    __syncthreads();

    if (LISTED) {
        // ---- phase B as a listed sweep (rows a1-a5): 8-row batches (mesh, electron) per warp; the listed sweep leaves the
        //      determinant ratios in R, the Jastrow ratios of the same rows follow in the same warp (quad per row)
        listed_phase_b(S, ws, T, Jold, wt, TW, lane);        // 8-row batches wt, wt + TW, ...; ws.bc = this CTA's Bc (set by the kernel)
        __syncthreads();
        EvalOut o; o.bbar = 0.0; o.Vsf = 0.0; o.W = 0.0; o.eL = 0.0; o.node = 0;
        if (wt == 0) {
            double Vee = 0.0;
            for (int w = 0; w < TW; ++w) Vee += s_vee[w];
            o = phase_c<false>(S, ws, lap_s, Vee, lane, 0);
        }
        return o;
    }

    // ---- phase B (rows a1-a5, f1): work units (mesh, spin, 8-electron block, shell part) and, with non-local slots, (pass of 8
    //      LISTED slots, shell part); unit v -> warp v mod TW.  One loop, one ao_columns call site for both kinds.
    const int nb_mesh = P.nblk[0] + P.nblk[1], K = S.nl_K;
    const int *list = reinterpret_cast<const int *>(ws.el + 2 * N);
    const int n_act = NL ? s_node[1] : 0, cut = NL ? s_node[2] : 0, n_p0 = (cut + 7) / 8, n_nlp = n_p0 + (n_act - cut + 7) / 8;
    for (int v = wt; v < P.n_units + n_nlp * NP; v += TW) {
        const bool is_nl = NL && v >= P.n_units;
        const int u = is_nl ? v - P.n_units : v, part = u % NP, blk = u / NP;
        int sp, il, i, kk = 0, mesh = 0, rem = 0; bool valid;
        if (!is_nl) {
            mesh = blk / nb_mesh; rem = blk - mesh * nb_mesh; sp = rem >= P.nblk[0] ? 1 : 0;
            const int il0 = 8 * (sp ? rem - P.nblk[0] : rem), ns_ = sp ? S.n_dn : S.n_up;
            valid = il0 + g < ns_; il = valid ? il0 + g : 0; i = (sp ? S.n_up : 0) + il;
        } else {
            const int lo = blk < n_p0 ? 8 * blk : cut + 8 * (blk - n_p0), hi = blk < n_p0 ? cut : n_act;
            valid = lo + g < hi;
            const int sl = list[valid ? lo + g : lo];
            i = sl / K; kk = sl - i * K; sp = i < S.n_up ? 0 : 1; il = sp ? i - S.n_up : i;
        }
        const int ns = sp ? S.n_dn : S.n_up;
        const double xi = ws.r[3 * i], yi = ws.r[3 * i + 1], zi = ws.r[3 * i + 2];
        double x0 = xi, y0 = yi, z0 = zi, step = S.amesh[mesh], r = 0.0;
        const double *nu = T.nuc;
        if (is_nl) {
            const int I = nl_centre(S, T.nuc, xi, yi, zi, kk, r);   // listed slots are in range
            nu = T.nuc + I * LRDMC_NUC_STRIDE; x0 = nu[0]; y0 = nu[1]; z0 = nu[2]; step = r;
        }
        const double a2 = step * step;
        double av[3][3];
#pragma unroll
        for (int k = 0; k < 3; ++k) { av[k][0] = step * ws.U[k]; av[k][1] = step * ws.U[3 + k]; av[k][2] = step * ws.U[6 + k]; }
        double acc[6], Jn[6];
        if (BCS && !is_nl) {
            double2 *bq = bcs_cta + (size_t)rem * S.n_kpairs * 32 + lane;
            if ((mesh > 0 && P.mesh_share) || sp == reuse_spin)
                ao_columns<NT, TS, true, 2>(S, T.shells, sp ? T.cf[1] : T.cf[0], T.etab, sp ? ws.dinv[1] : ws.dinv[0], ns, il, x0, y0, z0, av, a2, lane, acc, &P, &P.col[part], bq);
            else
                ao_columns<NT, TS, true, 1>(S, T.shells, sp ? T.cf[1] : T.cf[0], T.etab, sp ? ws.dinv[1] : ws.dinv[0], ns, il, x0, y0, z0, av, a2, lane, acc, &P, &P.col[part], bq);
        } else
        ao_columns<NT, TS, true>(S, T.shells, sp ? T.cf[1] : T.cf[0], T.etab, sp ? ws.dinv[1] : ws.dinv[0], ns, il, x0, y0, z0, av, a2, lane, acc, &P, &P.col[part]);
#pragma unroll
        for (int d = 0; d < 6; ++d) Jn[d] = 0.0;
        if (!is_nl || !S.nl_dla) {
            if (S.has_j1) for (int I = t + 4 * part; I < n_nuc; I += 4 * NP) {
                const double *np_ = T.nuc + I * LRDMC_NUC_STRIDE;
                pade_six(x0 - np_[0], y0 - np_[1], z0 - np_[2], av, a2, -np_[4], np_[5], Jn);
            }
            for (int j = t + 4 * part; j < N; j += 4 * NP) {
                const double c = (j == i) ? 0.0 : ((spin_of(S, j) == sp) ? S.a_par : S.a_anti);
                pade_six(x0 - ws.r[3 * j], y0 - ws.r[3 * j + 1], z0 - ws.r[3 * j + 2], av, a2, c, S.b2, Jn);
            }
        }
        if (J3 && (!is_nl || !S.nl_dla))                             // three-body Jastrow: the functions are dealt over (part, quad lane)
            j3_six(S, T, ws.j3 + (N + i) * S.j3s, x0, y0, z0, av, a2, t, Jn, 4 * part, 4 * NP);
        double nuq[6];
#pragma unroll
        for (int d = 0; d < 6; ++d) nuq[d] = 0.0;
        if (is_nl && part == 0) {                                    // nu_q = (1/6) sum_l (2l+1) v_l(r) P_l(+-e_k . rhat)
            const double ir = 1.0 / r, hx = (xi - nu[0]) * ir, hy = (yi - nu[1]) * ir, hz = (zi - nu[2]) * ir;
            const double r2 = r * r, *ch = nu + LRDMC_NL_OFF;
            const double v0 = ch[1] * exp_nonpos(-ch[2] * r2), v1 = 3.0 * ch[3] * exp_nonpos(-ch[4] * r2), v2 = 5.0 * ch[5] * exp_nonpos(-ch[6] * r2);
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double ct = ws.U[k] * hx + ws.U[3 + k] * hy + ws.U[6 + k] * hz, p2 = 0.5 * (3.0 * ct * ct - 1.0);
                nuq[2 * k] = (v0 + v1 * ct + v2 * p2) * (1.0 / 6.0);
                nuq[2 * k + 1] = (v0 - v1 * ct + v2 * p2) * (1.0 / 6.0);
            }
        }
        if (NP == 1) {
            const double Jo = Jold[i];
            double *Ro = is_nl ? ws.R + S.P_lat + 6 * (i * K + kk) : ws.R + mesh * 6 * N + 6 * i;
#pragma unroll
            for (int d = 0; d < 6; ++d) {
                double rho = quad_sum(acc[d]);
                if (!is_nl || !S.nl_dla) rho *= exp_tab(quad_sum(Jn[d]) - Jo, T.etab);
                if (valid && t == 0) { Ro[d] = is_nl ? -nuq[d] * rho : rho; if (is_nl && rho < 0.0) atomicOr(s_node, 1); }
            }
        } else {
            double *q = is_nl ? scr + P.o_nl + ((size_t)(i * K + kk) * NP + part) * 12 : scr + ((size_t)(mesh * N + i) * NP + part) * 12;
#pragma unroll
            for (int d = 0; d < 6; ++d) {
                const double A = quad_sum(acc[d]), J = quad_sum(Jn[d]);
                if (valid && t == 0) { q[d] = A; q[6 + d] = J; }
            }
            if (is_nl && part == 0 && valid && t == 0) {
                double *qn = scr + P.o_nu + (size_t)(i * K + kk) * 7;
#pragma unroll
                for (int d = 0; d < 6; ++d) qn[d] = nuq[d];
                qn[6] = 1.0;
            }
        }
    }
    __syncthreads();
    if (NP > 1) {                      // the parts of a candidate meet: R = (sum of determinant shares) exp(sum of Jastrow shares - J_old)
        for (int p = tid; p < S.P_lat; p += nthr) {
            const int mesh = p / (6 * N), rem = p - mesh * 6 * N, i = rem / 6, d = rem - 6 * i;
            const double *q = scr + (size_t)(mesh * N + i) * NP * 12;
            double A = 0.0, J = 0.0;
            for (int part = 0; part < NP; ++part) { A += q[part * 12 + d]; J += q[part * 12 + 6 + d]; }
            ws.R[p] = A * exp_tab(J - Jold[i], T.etab);
        }
        if (NL) for (int p = S.P_lat + tid; p < S.P; p += nthr) {  // non-local slots: R = -nu_q rho_q
            const int o = p - S.P_lat, slot = o / 6, d = o - 6 * slot, i = slot / S.nl_K;
            const double *q = scr + P.o_nl + (size_t)slot * NP * 12, *qn = scr + P.o_nu + (size_t)slot * 7;
            if (qn[6] == 0.0) { ws.R[p] = 0.0; continue; }          // slot not listed: no centre in range
            double A = 0.0, J = 0.0;
            for (int part = 0; part < NP; ++part) { A += q[part * 12 + d]; J += q[part * 12 + 6 + d]; }
            const double rho = S.nl_dla ? A : A * exp_tab(J - Jold[i], T.etab);
            ws.R[p] = -qn[d] * rho;
            if (rho < 0.0) atomicOr(s_node, 1);
        }
        __syncthreads();
    }
    EvalOut o; o.bbar = 0.0; o.Vsf = 0.0; o.W = 0.0; o.eL = 0.0; o.node = 0;
    if (wt == 0) {
        double Vee = 0.0;
        for (int w = 0; w < TW; ++w) Vee += s_vee[w];
        o = phase_c<NL>(S, ws, lap_s, Vee, lane, NL ? *s_node : 0);
    }
    return o;
}

// Apply move j (row a10) by the team: warp w takes part P.mo[w] of the derivative pass of the mover (value, gradient, Laplacian
// rows by DMMA), the partial rows meet in scr; Sherman-Morrison on Dinv_sigma over all threads.
template <int NT, bool TS, int EXT>
__device__ __forceinline__ void apply_move_team(const DevSys &S, const TeamPlan &P, const WarpState &ws, const Tables &T, double *scr, int j, double *bc = nullptr)
{
    constexpr bool LISTED = (EXT & 4) != 0;
    const int N = S.N, TW = P.TW, tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, wt = tid >> 5;   // warp 0 holds the lightest shell part (s shells): it also refreshes the one-body cache
    int i; double px, py, pz;
    move_target<(EXT & 1) != 0>(S, ws, T.nuc, j, i, px, py, pz);
    const int sp = spin_of(S, i), il = sp ? i - S.n_up : i, ns = sp ? S.n_dn : S.n_up;
    double *mc = ws.moc + (size_t)i * 5 * S.OS;
    const int rows = 5 * S.OS;
    {
        double acc[NT][2];
        mo_pass<NT, true, LRDMC_BF_SMEM(TS, EXT), true>(S, T.shells, sp ? T.bf[1] : T.bf[0], T.etab, px, py, pz, lane, acc, &P, &P.mo[wt]);
        const int t = lane & 3, g = lane >> 2;
        if (g < 5) {
            double *q = scr + (size_t)wt * rows + g * S.OS;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) { q[8 * nt + 2 * t] = acc[nt][0]; q[8 * nt + 2 * t + 1] = acc[nt][1]; }
        }
    }
    if (wt == 0) { refresh_onebody(S.n_nuc, S.has_j1, S.a, T.nuc, ws.ob + 8 * i, px, py, pz, lane); if (EXT & 2) refresh_j3_row(S, T.nuc, ws.j3 + i * S.j3s, px, py, pz, lane); }
    if (LISTED && wt == TW - 1)            // the mover's shell lists at its new position
        list_build(S, T.shells, T.srad, ws.lw, i, px, py, pz, fmax(S.amesh[0], S.amesh[1]), lane);
    __syncthreads();                                   // every thread has read the old position
    for (int idx = tid; idx < rows; idx += nthr) {
        double s = 0.0;
        for (int w = 0; w < TW; ++w) s += scr[(size_t)w * rows + idx];
        mc[idx] = s;
    }
    if (tid == 0) { ws.r[3 * i] = px; ws.r[3 * i + 1] = py; ws.r[3 * i + 2] = pz; }
    __syncthreads();
    // s_k = sum_m phi_m Dinv[m][k];  rho = s_il;  Dinv'[m][il] = Dinv[m][il]/rho;  Dinv'[m][k] = Dinv[m][k] - Dinv[m][il] s_k / rho
    double *dinv = sp ? ws.dinv[1] : ws.dinv[0], *sk = ws.el + 2 * N, *col = ws.el + 3 * N;
    for (int kk = tid; kk < ns; kk += nthr) {
        double s = 0.0;
        for (int m = 0; m < ns; ++m) s += mc[m] * dinv[m * ns + kk];
        sk[kk] = s; col[kk] = dinv[kk * ns + il];
    }
    __syncthreads();
    const double irho = 1.0 / sk[il];
    for (int idx = tid; idx < ns * ns; idx += nthr) {
        const int m = idx / ns, kk = idx - m * ns;
        const double ci = col[m] * irho;
        dinv[idx] = (kk == il) ? ci : dinv[idx] - ci * sk[kk];
    }
    if (LISTED) bc_rank1_update(S, bc, sp, il, ns, sk, irho, tid, nthr);   // Bc = C Dinv follows the inverse (listed.cuh)
    __syncthreads();
}

template <int NT, bool TS, int EXT>
__global__ void __launch_bounds__(LRDMC_TEAM_MAX_WARPS * 32, 1) k_propagate_team(DevSys S, DevWalk W, TeamPlan P, int mode, int n_moves, double tau, double E0, uint32_t cycle)
{
    extern __shared__ __align__(16) double smem[];
    __shared__ double s_vee[LRDMC_TEAM_MAX_WARPS];
    __shared__ double s_frame[2][12];   // per step parity: lattice frame U [9], pad, u_sel, u_tau (team_step_frame)
    __shared__ int s_ctrl[8];      // [0] walker, [1] last, [2] selected move, [3] node flag of the slots, [4] listed slots, [5] spin cut of the list
    stage_tables(S, smem);
    const int tid = threadIdx.x, lane = tid & 31, wt = tid >> 5;
    const Tables T = table_pointers<TS, LRDMC_BF_SMEM(TS, EXT)>(S, smem);
    WarpState ws = warp_views(S, smem, 0);
    double *scr = smem + S.tables_doubles + P.o_scr;
    constexpr bool LISTED = (EXT & 4) != 0;                     // listed sweep on stored, rank-1-updated Bc
    constexpr bool BCS = !TS && LRDMC_BC_STORE && !LISTED;      // large systems, dense sweep: parked Bc entries
    double2 *bcs_cta = (BCS || LISTED) ? reinterpret_cast<double2 *>(W.bcs + (size_t)blockIdx.x * W.bcs_stride) : nullptr;
    if (LISTED) ws.bc = W.bcs + (size_t)blockIdx.x * W.bcs_stride;
    const unsigned long long t_start = globaltimer_ns();
    for (;;) {
        if (tid == 0) s_ctrl[0] = atomicAdd(W.counter, 1);
        __syncthreads();
        const int k = s_ctrl[0];
        if (k >= W.n_w) break;
        if (W.dead[k]) {                                        // singular at the last (re)build (reading Q24): weight 0, not evaluated
            if (tid == 0) {
                W.w[k] = 0.0; W.eL[k] = 0.0; W.W[k] = 0.0; W.omega[k] = 0.0; W.nmoves[k] = 0;
                W.flags[3 * k] = 0; W.flags[3 * k + 1] = 0; W.flags[3 * k + 2] = 0;
            }
            __syncthreads();                                    // everyone has read s_ctrl[0]
            continue;
        }
        load_walker_team(S, W, ws, T.nuc, k, P.TW);
        if (LISTED) {                                           // listed sweep: shell lists of every electron, Bc of this walker
            for (int i = wt; i < S.N; i += P.TW)
                list_build(S, T.shells, T.srad, ws.lw, i, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], fmax(S.amesh[0], S.amesh[1]), lane);
            build_bc(S, ws.dinv[0], ws.dinv[1], reinterpret_cast<double *>(bcs_cta), tid, blockDim.x);
            __syncthreads();
        }
        uint32_t s = 0; int reuse_spin = -1;
        double w = 1.0, tau_left = tau, omega = 0.0, eL_last = 0.0, W_last = 0.0; long long moves = 0; int n_node = 0, n_nonpos = 0;
        // The draws and the frame of step s depend on (walker, cycle, s) alone: the last warp prepares those of step s + 1 in the
        // other half of s_frame while the leader warp runs phase C and the selection of step s -- off the critical path of the step.
        if (wt == P.TW - 1) team_step_frame(S, s_frame[0], (uint32_t)k, cycle, 0u, mode == LRDMC_CONVENTIONAL, lane);
        if (tid == 0) s_ctrl[3] = 0;
        __syncthreads();
        for (;;) {
            double *fr = s_frame[s & 1];
            ws.U = fr;
            const EvalOut e = evaluate_team<NT, TS, EXT, BCS>(S, P, ws, T, scr, s_vee, &s_ctrl[3], bcs_cta, reuse_spin);
            if (wt == P.TW - 1) team_step_frame(S, s_frame[(s + 1) & 1], (uint32_t)k, cycle, s + 1, mode == LRDMC_CONVENTIONAL, lane);
            if (wt == 0) {                                       // the leader warp keeps the weight (same rules as k_propagate)
                StepDraws d; d.u_sel = fr[10]; d.u_tau = fr[11];
                if (lane == 0) s_ctrl[3] = 0;                    // node flag of the slots: consumed by phase C, clear for the next evaluation
                n_node += e.node;
                bool last = false;
                if (mode == LRDMC_BALANCED) {
                    const double den = e.W - E0;                       // b_x = bbar/(W - E0)   (Eq.29)
                    if ((int)s == n_moves) {                           // measurement evaluation (reading Q10; Eq.34)
                        if (!(den > 0.0)) { ++n_nonpos; w = 0.0; omega = 0.0; } else omega = w / den;
                        last = true;
                    } else if (!(den > 0.0)) { ++n_nonpos; w = 0.0; }  // reading Q16
                    else w *= e.bbar / den;                            // Alg.2 line 6 (L406)
                } else {
                    double tx = -log1p(-d.u_tau) / e.bbar;             // Eq.24 (L160)
                    if (!(tx < tau_left) || (n_moves > 0 && (int)s >= n_moves)) { tx = tau_left; last = true; }   // min[., tau_left] (L362)
                    w *= exp(-tx * (e.eL - E0));                       // Eq.25 (L164), constant shift of reading Q8b
                    tau_left -= tx;
                    if (last) omega = w;
                }
                int j = -1;
                if (!last) j = select_move<(EXT & 1) != 0>(S, ws, e, d.u_sel, lane);      // Alg.2 line 7 (L408)
                else { eL_last = e.eL; W_last = e.W; }
                if (lane == 0) { s_ctrl[1] = last ? 1 : 0; s_ctrl[2] = j; }
            }
            __syncthreads();
            const bool last = s_ctrl[1] != 0; const int j = s_ctrl[2];
            if (last) break;
            if (j >= 0) {
                apply_move_team<NT, TS, EXT>(S, P, ws, T, scr, j, reinterpret_cast<double *>(bcs_cta)); ++moves;
                const int im = j < S.P_lat ? (j % (6 * S.N)) / 6 : (j - S.P_lat) / (6 * S.nl_K);   // the electron that hopped
                reuse_spin = 1 - spin_of(S, im);
            } else reuse_spin = -1;
            ++s;
        }
        store_walker_team(S, W, ws, k);
        if (tid == 0) {
            int nonfinite = 0;
            if (!isfinite(w) || !isfinite(omega)) { nonfinite = 1; w = 0.0; omega = 0.0; }
            W.w[k] = w; W.eL[k] = eL_last; W.W[k] = W_last; W.omega[k] = omega; W.nmoves[k] = moves;
            W.flags[3 * k] = n_node; W.flags[3 * k + 1] = n_nonpos; W.flags[3 * k + 2] = nonfinite;
        }
        if (!S.moc_in_smem) { ws = warp_views(S, smem, 0); if (LISTED) ws.bc = W.bcs + (size_t)blockIdx.x * W.bcs_stride; }
        __syncthreads();                                        // the state and s_ctrl are free for the next walker
    }
    if (tid == 0) { W.timing[2 * blockIdx.x] = t_start; W.timing[2 * blockIdx.x + 1] = globaltimer_ns(); }
}

