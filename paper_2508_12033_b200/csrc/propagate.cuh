// propagate.cuh -- the persistent walker kernels: one warp = one walker, state resident in shared memory for the
// whole branching interval (HBM is touched once per walker per cycle); walkers are pulled from a device-side queue
// so that the stochastic trip counts of the conventional mode (L168) do not leave SMs idle.
#pragma once
#include "evaluate.cuh"

// ---- shared-memory staging -------------------------------------------------------------------------------------
__device__ __forceinline__ void stage_tables(const DevSys &S, double *smem)
{
    for (int i = threadIdx.x; i < S.n_slots * 4; i += blockDim.x) smem[S.off_shells + i] = S.shells[i];
    for (int i = threadIdx.x; i < S.n_nuc * LRDMC_NUC_STRIDE; i += blockDim.x) smem[S.off_nuc + i] = S.nuc[i];
    for (int i = threadIdx.x; i < S.n_slots; i += blockDim.x) smem[S.off_srad + i] = S.srad[i];
    for (int i = threadIdx.x; i < S.j3s * S.j3s; i += blockDim.x) smem[S.off_j3g + i] = S.j3g[i];
    if (S.bf_in_smem) {
        const int nb = S.bfm_in_smem ? S.n_ksteps * S.NT[0] * 32 : 0;
        for (int i = threadIdx.x; i < nb; i += blockDim.x) smem[S.off_bf[0] + i] = S.bfrag[0][i];
        if (!S.same_C && S.n_dn > 0) for (int i = threadIdx.x; i < nb; i += blockDim.x) smem[S.off_bf[1] + i] = S.bfrag[1][i];
        const int nc = S.cf_in_smem ? S.n_kpairs * 2 * S.NT[0] * 32 : 0;
        for (int i = threadIdx.x; i < nc; i += blockDim.x) smem[S.off_cf[0] + i] = S.cfrag[0][i];
        if (!S.same_C && S.n_dn > 0) for (int i = threadIdx.x; i < nc; i += blockDim.x) smem[S.off_cf[1] + i] = S.cfrag[1][i];
    }
    for (int i = threadIdx.x; i < 256; i += blockDim.x) smem[i] = S.etab[i];        // off_etab == 0 by construction
    __syncthreads();
}

// TS (tables + MO cache in shared memory): every pointer below is "shared base + offset" with no global alternative, so the
// compiler's address-space inference emits LDS/STS.  !TS (64-electron config): fragments / cache stay in global memory.
// BFS: the derivative-pass fragments `bf` are in shared memory (LRDMC_BF_SMEM), else global.
template <bool TS, bool BFS = TS>
__device__ __forceinline__ Tables table_pointers(const DevSys &S, const double *smem)
{
    Tables T;
    T.shells = smem + S.off_shells; T.nuc = smem + S.off_nuc; T.etab = smem; T.srad = smem + S.off_srad; T.j3g = smem + S.off_j3g;
    if (BFS) { T.bf[0] = smem + S.off_bf[0]; T.bf[1] = smem + (S.same_C ? S.off_bf[0] : S.off_bf[1]); }
    else { T.bf[0] = S.bfrag[0]; T.bf[1] = S.bfrag[1]; }        // global memory only: a single provenance per pointer (see lrdmc_init)
    if (TS) { T.cf[0] = smem + S.off_cf[0]; T.cf[1] = smem + (S.same_C ? S.off_cf[0] : S.off_cf[1]); }
    else { T.cf[0] = S.cfrag[0]; T.cf[1] = S.cfrag[1]; }
    return T;
}

__device__ __forceinline__ WarpState warp_views(const DevSys &S, double *smem, int warp)
{
    double *base = smem + S.tables_doubles + (size_t)warp * S.per_warp_doubles;
    WarpState ws;
    ws.r = base + S.o_r; ws.dinv[0] = base + S.o_dinv[0]; ws.dinv[1] = base + S.o_dinv[1];
    ws.moc = base + S.o_moc; ws.R = base + S.o_R; ws.el = base + S.o_el; ws.ob = base + S.o_ob; ws.U = base + S.o_U; ws.j3 = base + S.o_j3;
    ws.lw = reinterpret_cast<unsigned char *>(base + S.o_am); ws.bc = nullptr;
    return ws;
}

// the step's lattice frame, computed by lane 0 and published in shared memory (the versors are indexed by direction)
__device__ __forceinline__ void publish_frame(const WarpState &ws, const StepDraws &d, int lane)
{
    __syncwarp();
    if (lane == 0) { double U[9]; lattice_frame(d.u1, d.u2, d.u3, U);
#pragma unroll
        for (int i = 0; i < 9; ++i) ws.U[i] = U[i]; }
    __syncwarp();
}

// The draws and frames of the steps s0 .. s0 + LRDMC_FRAME_BATCH - 1 of walker `slot`, one LANE per step (they depend on (slot, cycle, step) alone): the
// Philox rounds and the frame's sincos / sqrt sequences are warp instructions whichever lanes need them, so preparing four steps costs what one did.
// fr = the warp's frame buffer [S.frame_batch][LRDMC_FRAME_STRIDE].
__device__ __forceinline__ void prepare_frames(const DevSys &S, double *fr, uint32_t slot, uint32_t cycle, uint32_t s0, bool need_tau, int lane)
{
    __syncwarp();
    const StepDraws d = step_draws(S, slot, cycle, s0 + (lane < S.frame_batch ? lane : 0), need_tau);
    if (lane < S.frame_batch) {
        double U[9]; lattice_frame(d.u1, d.u2, d.u3, U);
        double *o = fr + lane * LRDMC_FRAME_STRIDE;
#pragma unroll
        for (int i = 0; i < 9; ++i) o[i] = U[i];
        o[10] = d.u_sel; o[11] = d.u_tau;
    }
    __syncwarp();
}

// LISTED (EXT bit 2): also the shell lists of every electron and Bc = C Dinv of this walker in the warp's global scratch ws.bc.
template <bool TS, bool LISTED = false>
__device__ __forceinline__ void load_walker(const DevSys &S, const DevWalk &W, WarpState &ws, const Tables &T, int k, int lane, bool with_dinv, bool with_onebody = true)
{
    const int N = S.N;
    for (int i = lane; i < 3 * N; i += 32) ws.r[i] = W.r[(size_t)k * 3 * N + i];
    for (int sp = 0; sp < 2; ++sp) {
        const int ns = sp ? S.n_dn : S.n_up, tot = S.dinv_rows[sp] * ns;
        const double *src = W.dinv[sp] + (size_t)k * ns * ns;
        for (int i = lane; i < tot; i += 32) ws.dinv[sp][i] = (with_dinv && i < ns * ns) ? src[i] : 0.0;
    }
    const size_t mocn = (size_t)N * 5 * S.OS;
    if (TS) { for (int i = lane; i < (int)mocn; i += 32) ws.moc[i] = W.moc[(size_t)k * mocn + i]; }
    else ws.moc = W.moc + (size_t)k * mocn;
    __syncwarp();
    const double *nuc = T.nuc;
    if (with_onebody && S.n_j3) for (int i = 0; i < N; ++i) refresh_j3_row(S, nuc, ws.j3 + i * S.j3s, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], lane);
    if (with_onebody) for (int i = 0; i < N; ++i) refresh_onebody(S.n_nuc, S.has_j1, S.a, nuc, ws.ob + 8 * i, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], lane);
    if (LISTED) {
        for (int i = 0; i < N; ++i) list_build(S, T.shells, T.srad, ws.lw, i, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], fmax(S.amesh[0], S.amesh[1]), lane);
        build_bc(S, ws.dinv[0], ws.dinv[1], ws.bc, lane, 32);
    }
    __syncwarp();
}

__device__ __forceinline__ void store_walker(const DevSys &S, const DevWalk &W, const WarpState &ws, int k, int lane)
{
    const int N = S.N;
    __syncwarp();
    for (int i = lane; i < 3 * N; i += 32) W.r[(size_t)k * 3 * N + i] = ws.r[i];
    for (int sp = 0; sp < 2; ++sp) {
        const int ns = sp ? S.n_dn : S.n_up;
        double *dst = W.dinv[sp] + (size_t)k * ns * ns;
        for (int i = lane; i < ns * ns; i += 32) dst[i] = ws.dinv[sp][i];
    }
    const size_t mocn = (size_t)N * 5 * S.OS;
    if (S.moc_in_smem) for (int i = lane; i < (int)mocn; i += 32) W.moc[(size_t)k * mocn + i] = ws.moc[i];
    __syncwarp();
}

// ---- the projection kernel (Alg.2 lines 4-8 L401-L410 / Alg.1 lines 4-16 L350-L374) ----------------------------
// WPBK: the warps per CTA the kernel is compiled for (launch bound; registers per thread = 65536 / (LRDMC_MINB 32 WPBK)).
template <int NT, bool TS, int EXT, int WPBK = LRDMC_WPB>
__global__ void __launch_bounds__(WPBK * 32, LRDMC_MINB) k_propagate(DevSys S, DevWalk W, int mode, int n_moves, double tau, double E0, uint32_t cycle)
{
    extern __shared__ __align__(16) double smem[];
    stage_tables(S, smem);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, gwarp = blockIdx.x * (blockDim.x >> 5) + warp;
    const Tables T = table_pointers<TS, LRDMC_BF_SMEM(TS, EXT)>(S, smem);
    WarpState ws = warp_views(S, smem, warp);
    if (EXT & 4) ws.bc = W.bcs + (size_t)gwarp * W.bcs_stride;
    double *const frames = ws.U;             // [LRDMC_FRAME_BATCH][LRDMC_FRAME_STRIDE]; ws.U points at the current step's frame
    const unsigned long long t_start = globaltimer_ns();
    // The warps of a CTA meet at a barrier once per step, whatever walker and step index each of them is at: they then run
    // the same code region at the same time and share the small instruction caches (L0 6 KB, L1.5 32 KB against 140 KB of
    // kernel).  A warp whose walker is finished takes the next one from the device-side queue at once, so the stochastic
    // trip counts of the conventional mode (L168) cost no idle lanes; in balanced mode all warps of a CTA reload together.
    bool have = false; int k = 0; uint32_t s = 0;
    double w = 1.0, tau_left = tau; long long moves = 0; int n_node = 0, n_nonpos = 0;
    for (;;) {
        while (!have) {
            if (lane == 0) k = atomicAdd(W.counter, 1);
            k = __shfl_sync(0xffffffffu, k, 0);
            if (k >= W.n_w) break;
            if (W.dead[k]) {                                   // singular at the last (re)build (reading Q24): weight 0, not evaluated
                if (lane == 0) {
                    W.w[k] = 0.0; W.eL[k] = 0.0; W.W[k] = 0.0; W.omega[k] = 0.0; W.nmoves[k] = 0;
                    W.flags[3 * k] = 0; W.flags[3 * k + 1] = 0; W.flags[3 * k + 2] = 0;
                }
                continue;
            }
            load_walker<TS, (EXT & 4) != 0>(S, W, ws, T, k, lane, true);
            have = true; s = 0; w = 1.0; tau_left = tau; moves = 0; n_node = 0; n_nonpos = 0;
        }
        if (LRDMC_LOCKSTEP) { if (!__syncthreads_or(have)) break; if (!have) continue; }
        else if (!have) break;
        if ((s & (S.frame_batch - 1)) == 0) prepare_frames(S, frames, (uint32_t)k, cycle, s, mode == LRDMC_CONVENTIONAL, lane);
        ws.U = frames + (s & (S.frame_batch - 1)) * LRDMC_FRAME_STRIDE;
        StepDraws d; d.u_sel = ws.U[10]; d.u_tau = ws.U[11];
        const EvalOut e = evaluate_walker<NT, TS, EXT>(S, ws, T, lane);
        n_node += e.node;
        bool last = false; double omega = 0.0;
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
        if (!last) {
            const int j = select_move<(EXT & 1) != 0>(S, ws, e, d.u_sel, lane);   // Alg.2 line 7 (L408)
            if (j >= 0) { apply_move<NT, TS, EXT>(S, ws, T, j, lane); ++moves; }
            ++s;
            continue;
        }
        int nonfinite = 0;
        if (!isfinite(w) || !isfinite(omega)) { nonfinite = 1; w = 0.0; omega = 0.0; }
        store_walker(S, W, ws, k, lane);
        if (lane == 0) {
            W.w[k] = w; W.eL[k] = e.eL; W.W[k] = e.W; W.omega[k] = omega; W.nmoves[k] = moves;
            W.flags[3 * k] = n_node; W.flags[3 * k + 1] = n_nonpos; W.flags[3 * k + 2] = nonfinite;
        }
        if (!TS) { ws = warp_views(S, smem, warp); if (EXT & 4) ws.bc = W.bcs + (size_t)gwarp * W.bcs_stride; }   // load_walker pointed ws.moc at the walker's global rows
        have = false;
    }
    if (lane == 0) { W.timing[2 * gwarp] = t_start; W.timing[2 * gwarp + 1] = globaltimer_ns(); }
}

// ---- parity hook: one evaluation + selection, no state change ---------------------------------------------------
template <int NT, bool TS, int EXT, int WPBK = LRDMC_WPB>
__global__ void __launch_bounds__(WPBK * 32, LRDMC_MINB) k_step_debug(DevSys S, DevWalk W, double E0, uint32_t cycle, uint32_t step, double *R_out,
                                                    double *scal_out, int *jstar_out)
{
    extern __shared__ __align__(16) double smem[];
    stage_tables(S, smem);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    const Tables T = table_pointers<TS, LRDMC_BF_SMEM(TS, EXT)>(S, smem);
    WarpState ws = warp_views(S, smem, warp);
    for (int k = blockIdx.x * wpb + warp; k < W.n_w; k += gridDim.x * wpb) {
        if (EXT & 4) ws.bc = W.bcs + (size_t)(blockIdx.x * wpb + warp) * W.bcs_stride;
        load_walker<TS, (EXT & 4) != 0>(S, W, ws, T, k, lane, true);
        const StepDraws d = step_draws(S, (uint32_t)k, cycle, step, true);
        publish_frame(ws, d, lane);
        const EvalOut e = evaluate_walker<NT, TS, EXT>(S, ws, T, lane);
        const int j = select_move<(EXT & 1) != 0>(S, ws, e, d.u_sel, lane);
        for (int p = lane; p < S.P; p += 32) R_out[(size_t)k * S.P + p] = ws.R[p];
        if (lane == 0) {
            double *o = scal_out + 8 * (size_t)k;
            o[0] = e.bbar; o[1] = e.Vsf; o[2] = e.W; o[3] = e.eL; o[4] = e.bbar / (e.W - E0);
            o[5] = -log1p(-d.u_tau) / e.bbar; o[6] = (double)e.node; o[7] = d.u_sel;
            jstar_out[k] = j;
        }
        if (!S.moc_in_smem) ws = warp_views(S, smem, warp);
        __syncwarp();
    }
}

// ---- (re)build of the inverses and MO caches from the positions (row a13) ---------------------------------------
template <int NT, bool TS, bool BFS>
__global__ void __launch_bounds__(LRDMC_WPB * 32) k_rebuild(DevSys S, DevWalk W, int do_invert)
{
    extern __shared__ __align__(16) double smem[];
    stage_tables(S, smem);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, wpb = blockDim.x >> 5;
    const Tables T = table_pointers<TS, BFS>(S, smem);
    WarpState ws = warp_views(S, smem, warp);
    const int N = S.N;
    for (int k = blockIdx.x * wpb + warp; k < W.n_w; k += gridDim.x * wpb) {
        load_walker<TS>(S, W, ws, T, k, lane, !(do_invert & 1), false);
        if (!(do_invert & 2)) for (int i = 0; i < N; ++i) {
            const int sp = spin_of(S, i);
            refresh_mo_cache<NT, BFS>(S, T.shells, T.bf[sp], T.etab, ws.moc + (size_t)i * 5 * S.OS, ws.r[3 * i], ws.r[3 * i + 1], ws.r[3 * i + 2], lane);
        }
        __syncwarp();
        if (do_invert & 1) {
            bool ok = true;
            for (int sp = 0; sp < 2; ++sp) {
                const int ns = sp ? S.n_dn : S.n_up, off = sp ? S.n_up : 0;
                if (!ns) continue;
                double *A = ws.dinv[sp];
                for (int idx = lane; idx < ns * ns; idx += 32) { int i = idx / ns, m = idx - i * ns; A[idx] = ws.moc[(size_t)(off + i) * 5 * S.OS + m]; }
                __syncwarp();
                if (!warp_invert(A, ns, ns, reinterpret_cast<int *>(ws.el), lane)) ok = false;      // row permutation: n_s ints in the per-electron scratch (4 N doubles)
                __syncwarp();
            }
            if (!ok) {       // reading Q24: a singular walker is dead (zero inverses, weight 0 in the next propagate) and counted
                for (int sp = 0; sp < 2; ++sp) { const int ns = sp ? S.n_dn : S.n_up; for (int idx = lane; idx < ns * ns; idx += 32) ws.dinv[sp][idx] = 0.0; }
                if (lane == 0) { atomicOr(W.counter + 1, 1); atomicAdd(reinterpret_cast<unsigned long long *>(W.n_sing), 1ull); }
            }
            if (lane == 0) W.dead[k] = ok ? 0 : 1;
        }
        store_walker(S, W, ws, k, lane);
        if (!S.moc_in_smem) ws = warp_views(S, smem, warp);
    }
}
