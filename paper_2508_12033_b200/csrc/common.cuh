// common.cuh -- shared device/host declarations of liblrdmc (CUDA path; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/lrdmc.h"

// __builtin_assume(__isShared(p)) made nvcc 12.9 delete the hop (apply_move) from k_propagate: measured, reverted.
// Address spaces are inferred instead: with TS every per-warp pointer is "shared base + offset" with no global alternative.
#define LRDMC_ASSUME_SHARED(p) ((void)0)
#ifndef LRDMC_WPB
#define LRDMC_WPB 8            // warps (= walkers in flight) per CTA
#endif
#ifndef LRDMC_WPB_EXT
#define LRDMC_WPB_EXT 6        // second instantiation of the extended kernels (non-local slots / three-body Jastrow) for systems whose state leaves room
#endif                         // for 6 or 7 warps only: 7 cannot be spread evenly over the 4 schedulers (lrdmc.cu plan_smem), and 192 threads lift the register cap to 168
#ifndef LRDMC_MINB
#define LRDMC_MINB 2           // CTAs per SM the register allocation must allow
#endif
#ifndef LRDMC_LOCKSTEP
#define LRDMC_LOCKSTEP 1        // balanced mode: the warps of a CTA step together (one barrier per step)
#endif
#ifndef LRDMC_BC_STORE
#define LRDMC_BC_STORE 1         // Bc kept between evaluations: listed sweep (listed.cuh), or parked entries of the dense sweep of the large systems (ao_columns BCS)
#endif
// Systems with a three-body Jastrow keep the fragment table `bf` of the mover's derivative pass (12.8 KB at 200 AOs, read once per move, the same for every
// walker: L1-resident) in global memory, so that their larger per-walker state still leaves room for 8 warps per CTA.  EXT is the kernels' feature mask.
#define LRDMC_BF_SMEM(TS, EXT) ((TS) && !((EXT) & 2))
#define LRDMC_FRAME_BATCH 4    // warp-per-walker kernel: the draws and lattice frames of up to this many consecutive steps are prepared at once, one lane per step
                               // (DevSys.frame_batch = 4, 2 or 1: the largest that costs no warp of occupancy, lrdmc.cu plan_smem)
#define LRDMC_FRAME_STRIDE 12  // doubles per prepared step: U [9], pad, u_sel, u_tau
#define LRDMC_NUC_STRIDE 20  // doubles per nucleus row: Rx Ry Rz Z c1 b1 alpha beta gamma delta is_pp pad | r_c A0 B0 A1 B1 A2 B2 pad (non-local channels)
#define LRDMC_NL_OFF 12      // first non-local entry of a nucleus row
#define LRDMC_NL_MAX_K 4
#define LRDMC_J3_MAX 32       // three-body Jastrow functions, at most (lane per function in the row refresh)
#define LRDMC_EL_ARRAYS 4     // per-electron scratch arrays in shared memory: Jold, lap, s_k, old column
#define LRDMC_MAX_LG 8        // list groups of the listed candidate sweep: (shell type, chunk of at most 64 sorted shell slots)
// Screening of the listed candidate sweep: a shell is listed for a row of six displaced points
// x0 +- step e_k when |x0 - R_shell| < step + srad, srad = sqrt(LRDMC_LIST_THR / zeta) (Gaussians) or LRDMC_LIST_THR / zeta (Slater):
// every exponent of an unlisted shell is below -LRDMC_LIST_THR in ANY frame (|x0 +- step e - R| >= |x0 - R| - step).
#define LRDMC_LIST_THR 52.0

// Everything a kernel needs to know about the system; passed by value (fits the 4 KB parameter space).
struct DevSys {
    int N, n_up, n_dn, n_nuc, P, n_mesh;   // P = all candidates = P_lat + 6 N nl_K
    int P_lat, nl_K, nl_dla;               // 6 N n_mesh lattice hops; non-local pseudopotential slots per electron (0: none); determinant-locality flag
    int n_it[4];          // DMMA k-iterations (4 shells each) per shell group: 0 Slater-s, 1 s, 2 p, 3 d
    int n_slots;          // 4 * sum n_it  (sorted + padded shell list)
    int n_ksteps;         // n_it[0] + n_it[1] + 3 n_it[2] + 6 n_it[3]  = (padded AO count)/4
    int NT[2];            // 8-wide MO tiles per spin
    int OS;               // MO stride of the cache rows, 8*max(NT)
    int same_C;           // C_dn == C_up: one fragment table
    int has_j1, has_pp;
    double amesh[2], gmesh[2], kappa[2], g_over_a2[2];
    double a_par, a_anti, b2, V_ii, Kdiag, a;
    // three-body Jastrow J3 = sum_{i<j} sum_ab g_ab chi_a(r_i) chi_b(r_j), chi_a = dx^l dy^m dz^n exp(-zeta_a |r - R_a|^2) (extended kernels only)
    int n_j3, j3s;             // functions; j3s = row stride of the per-walker arrays and of g = n_j3 rounded up to a multiple of 4
    int j3_poly;               // some function has a monomial factor (p / d functions): l | m << 2 | n << 4 in j3_lmn
    int j3_center[LRDMC_J3_MAX], j3_lmn[LRDMC_J3_MAX]; double j3_zeta[LRDMC_J3_MAX];
    const double *j3g; int off_j3g;   // g [j3s][j3s] (zero padded): global copy, staged into the shared tables at off_j3g
    uint32_t key0, key1;
    // device tables (global memory copies; staged into shared memory when they fit)
    const double *shells;      // [n_slots][4] = cx cy cz zeta
    const double *bfrag[2];    // [n_ksteps][NT][32] FP64 mma B fragments, AO norms folded in
    const double *nuc;         // [n_nuc][LRDMC_NUC_STRIDE]
    const double *etab;        // [256] 2^(j/256) for exp_tab
    const double *cfrag[2];    // [n_kpairs][2 NT][32] FP64 mma B fragments of the Bc = C Dinv product (ao_columns), norms folded in
    int n_kpairs, off_cf[2];   // pairs of k-steps (each shell group padded to an even number of k-steps)
    // listed candidate sweep (team kernel of the large systems): sorted slots in list groups of one type and at most 64 slots
    int n_lg, lg_type[LRDMC_MAX_LG], lg_slot0[LRDMC_MAX_LG], lg_n[LRDMC_MAX_LG], lg_ao0[LRDMC_MAX_LG];
    int lg_off[LRDMC_MAX_LG], lt;   // byte offset of a list group inside an electron's list row; lt = bytes per electron (sum of lg_n, multiple of 4)
    int n_aop;                 // AO count of the sorted, padded shell list (slot-major: components of a shell are consecutive)
    int off_srad, o_am;        // shared memory: srad [n_slots] in the tables; per walker: the listed-shell lists (listed.cuh), (N (lt + n_lg) + 7) / 8 doubles
    const double *srad;        // [n_slots] screening radii (LRDMC_LIST_THR); padded slots: -1e300 (never listed)
    const double *cn[2];       // [n_aop][OS] MO coefficients with the AO norms folded in, slot-major (Bc = C Dinv by rows)
    // shared-memory plan (units: doubles)
    int frame_batch;                           // steps per prepared batch of draws / frames (power of two <= LRDMC_FRAME_BATCH)
    int bf_in_smem, moc_in_smem, cf_in_smem;   // cf_in_smem: the pair table of ao_columns is staged too (not with the listed sweep)
    int bfm_in_smem;                           // the fragment table `bf` of the mover's derivative pass is staged too (LRDMC_BF_SMEM: not with a three-body Jastrow)
    int off_shells, off_nuc, off_bf[2], off_etab, tables_doubles;
    int o_r, o_dinv[2], o_moc, o_R, o_el, o_ob, o_U, o_j3, per_warp_doubles;   // o_j3: chi3 [N][j3s], V3 [N][j3s], S3 [j3s] (systems with a J3)
    int dinv_rows[2];     // padded row count 8*NT
};

// ---- team mode (team.cuh): one CTA of TW warps works on ONE walker --------------------------------------------------
// A shell part = per shell group [lo, hi) ranges of 4-shell iterations of the sorted, padded shell list.
struct ShellPart { int lo[4], hi[4]; };
#define LRDMC_TEAM_MAX_WARPS 16
#define LRDMC_TEAM_MAX_PARTS 8
struct TeamPlan {
    int TW;               // warps per walker (= blockDim.x / 32)
    int NP;               // shell parts of the candidate pass (work units = electron blocks x NP)
    int lpe;              // lanes per electron in phase A (power of two, 2..32)
    int nblk[2];          // 8-electron blocks per spin
    int n_units;          // n_mesh (nblk[0] + nblk[1]) NP
    int nblk_nl[2], n_units_nl, o_nl, o_nu;   // non-local slot blocks (8 slots) per spin, their units, scratch offsets (partials, nu_q)
    int it_base[4];       // first 4-shell iteration of each shell group
    int kstep_base[4];    // first mma k-step of each group in the `bf` fragment table
    int pair_base[4];     // first k-step pair of each group in the `cf` fragment table
    int mesh_share;       // both meshes of a block are handled by the same warp: the second takes the first's parked Bc entries
    int o_scr, scr_doubles; // scratch (partial sums) behind the walker state, in doubles from the state base
    int listed;           // the candidate pass is the listed sweep (listed.cuh): 8-row batches (mesh, electron) dealt to the warps
    ShellPart col[LRDMC_TEAM_MAX_PARTS];     // parts of ao_columns (groups 0-2 start on even iterations: k-step pairs)
    ShellPart mo[LRDMC_TEAM_MAX_WARPS];      // parts of the derivative pass of the mover (one per warp)
};

// Table pointers as a kernel sees them (shared memory, or global memory for the fragments of the largest systems)
struct Tables { const double *shells, *nuc, *bf[2], *cf[2], *etab, *srad, *j3g; };

// Walker storage (views into the caller's buffer)
struct DevWalk {
    int n_w;
    double *r;            // current positions [n_w][3N]
    double *r_alt;        // gather target
    double *dinv[2];      // [n_w][n_s*n_s]
    double *moc;          // [n_w][N][5][OS] cached MO value/grad/lap rows at each electron
    double *moc_alt;      // gather target of the cache rows (they depend on the positions only: copies of the parent's are exact)
    double *w, *eL, *W, *omega;
    long long *nmoves;
    int *flags;           // [n_w][3] node / nonpos / nonfinite counts of the last propagate
    int *dead;            // [n_w] 1: Slater matrix singular at the last (re)build (reading Q24): weight 0, never evaluated
    long long *n_sing;    // device counter of such walkers (lives in the ctx's DevStats)
    unsigned long long *wq, *prefix; // comb workspace
    int *parents;
    unsigned long long *timing;      // [max_warps][2] globaltimer start/end per resident warp
    double *stats;        // device copy of the reduced numbers (see k_reduce_obs)
    int *counter;         // dynamic walker queue head; [1] = singular flag
    double *bcs;          // per resident team CTA / warp of the warp-per-walker kernel: Bc = C Dinv of its walker, [electron][n_aop] (listed sweep, updated rank-1 with the inverse),
                          // or the parked Bc entries [block of a mesh][k-step pair][lane][2] of ao_columns BCS; NULL if unused
    size_t bcs_stride;    // doubles per CTA
    int bcs_ctas;         // CTAs the scratch was sized for
};

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double quad_sum(double v)
{
    v += __shfl_xor_sync(0xffffffffu, v, 1);
    v += __shfl_xor_sync(0xffffffffu, v, 2);
    return v;
}
__device__ __forceinline__ unsigned long long globaltimer_ns()
{
    unsigned long long t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t;
}
