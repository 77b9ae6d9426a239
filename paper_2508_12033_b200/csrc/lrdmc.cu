// lrdmc.cu -- C-ABI of liblrdmc.so (see include/lrdmc.h).  Host logic only: table construction, the shared-memory
// plan, kernel launches, CUDA-event timing.  Every step of the path runs in the kernels of the *.cuh files.
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "philox.cuh"
#include "wavefunction.cuh"
#include "evaluate.cuh"
#include "propagate.cuh"
#include "kernels.h"
#include "reconfigure.cuh"
#include "api_internal.h"

// CUDA errors: the text goes into the context (lrdmc_last_error); every function that uses CK has a ctx pointer named `c`.
#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { snprintf(c->msg, sizeof c->msg, "%s at %s:%d", cudaGetErrorString(e_), __FILE__, __LINE__); return LRDMC_ECUDA; } } while (0)
// lrdmc_init has no context to hand back when it fails: its text is kept per calling thread (like errno), read with lrdmc_last_error(NULL).
static thread_local char t_init_msg[256] = "";

struct lrdmc_ctx {
    DevSys S; DevWalk W;
    void *d_tables; DevStats *d_stats, *h_stats;   // h_stats: pinned staging of the per-generation sums (read back on the ctx's own stream)
    int ext;        // 0 lattice only, bit 0: non-local slots, bit 1: three-body Jastrow
    int NT, ts, wpb, ctas_per_sm, sm_count, smem_bytes, grid_max; size_t smem_per_sm;
    int bound, have_prop, have_reconf, state_ok;
    cudaEvent_t ev[4]; cudaStream_t last_stream;
    int launches;   // kernels launched so far (bench.py reports it)
    char msg[256];  // text of the last CUDA error of this context (lrdmc_last_error)
    int opt_team, opt_global_tables, opt_listed; // lrdmc_set_option (opt_listed: -1 automatic, 0 dense, 1 listed)
    int listed;                                 // the candidate pass of this system is the listed sweep (EXT = 4)
    size_t n_sh, n_nuc_d, bf_n, cf_n;           // table sizes in doubles (shared-memory plan)
    // team mode (team.cuh): chosen at lrdmc_bind_walkers from N_w and the footprint; team_tw == 1 -> warp-per-walker kernel
    TeamPlan team; int team_tw, team_smem, team_ctas_per_sm, team_grid_max, pair_base[5];
};

extern "C" const char *lrdmc_strerror(int code)
{
    switch (code) {
    case LRDMC_OK: return "ok";
    case LRDMC_EINVAL: return "invalid argument";
    case LRDMC_ESINGULAR: return "singular Slater matrix";
    case LRDMC_ESTATE: return "call order: walkers not bound / positions not set / nothing propagated";
    case LRDMC_ECUDA: return "CUDA error (text: lrdmc_last_error)";
    case LRDMC_ENOMEM: return "system does not fit the shared-memory plan";
    default: return "unknown error";
    }
}

static double odd_dfact(int k) { double f = 1.0; for (int j = 1; j <= k; ++j) f *= (2 * j - 1); return f; }
static double gto_norm(double z, int l, int m, int n)
{
    return pow(2.0 * z / M_PI, 0.75) * pow(4.0 * z, 0.5 * (l + m + n)) / sqrt(odd_dfact(l) * odd_dfact(m) * odd_dfact(n));
}
static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ---- shared-memory plan: either every table and the MO cache sit in shared memory (TS kernels), or the fragment tables and
// the cache are read from global memory (large systems; LRDMC_OPT_GLOBAL_TABLES forces this path for tests).  No mixed case: a
// fragment pointer that may be shared OR global makes nvcc 12.9 infer "shared" for it (cvta.to.shared + ld.shared on a global
// address).  Re-run by lrdmc_set_option; the device tables themselves do not depend on it.
static int plan_smem(lrdmc_ctx *c)
{
    DevSys &S = c->S;
    cudaDeviceProp prop; int dev = 0; CK(cudaGetDevice(&dev)); CK(cudaGetDeviceProperties(&prop, dev));
    c->sm_count = prop.multiProcessorCount; c->smem_per_sm = prop.sharedMemPerMultiprocessor;
    const size_t bf_n = c->bf_n, cf_n = c->cf_n;
    const size_t bf_doubles = (bf_n + cf_n) * (S.same_C ? 1 : 2);
    const size_t moc_doubles = (size_t)S.N * 5 * S.OS;
    const bool fits = bf_doubles * 8 <= 64 * 1024 && moc_doubles * 8 <= 12 * 1024 && !c->opt_global_tables;
    S.bf_in_smem = fits; S.moc_in_smem = fits; S.bfm_in_smem = fits && !S.n_j3;     // LRDMC_BF_SMEM (common.cuh)
    size_t o = 0;
    S.off_etab = (int)o; o += 256;              // always first: exp_tab addresses it as (dynamic smem base) + 8 j
    S.off_shells = (int)o; o += align_up(c->n_sh, 2);
    S.off_nuc = (int)o; o += align_up(c->n_nuc_d, 2);
    S.off_srad = (int)o; o += align_up((size_t)S.n_slots, 2);
    S.off_j3g = (int)o; o += (size_t)S.j3s * S.j3s;
    // listed sweep (EXT = 4): lattice-only systems; automatic = the systems whose tables live in global memory (64 electrons, 600 AOs)
    c->listed = !S.nl_K && !S.n_j3 && LRDMC_BC_STORE && (c->opt_listed < 0 ? !fits : c->opt_listed != 0);
    S.off_bf[0] = (int)o; if (S.bfm_in_smem) o += bf_n;
    S.off_bf[1] = (int)o; if (S.bfm_in_smem && !S.same_C) o += bf_n;
    S.cf_in_smem = S.bf_in_smem && !c->listed;
    S.off_cf[0] = (int)o; if (S.bf_in_smem && !c->listed) o += cf_n;            // the pair table of ao_columns is not used by the listed sweep
    S.off_cf[1] = (int)o; if (S.bf_in_smem && !S.same_C && !c->listed) o += cf_n;
    S.tables_doubles = (int)align_up(o, 2);
    size_t w = 0;
    S.o_r = (int)w; w += align_up(3 * (size_t)S.N, 2);
    S.o_dinv[0] = (int)w; w += align_up((size_t)S.dinv_rows[0] * S.n_up, 2);
    S.o_dinv[1] = (int)w; w += align_up((size_t)S.dinv_rows[1] * S.n_dn, 2);
    S.o_moc = (int)w; if (S.moc_in_smem) w += align_up(moc_doubles, 2);
    S.o_R = (int)w; w += align_up((size_t)S.P, 2);
    S.o_el = (int)w; w += align_up((size_t)LRDMC_EL_ARRAYS * S.N, 2);
    S.o_ob = (int)w; w += 8 * (size_t)S.N;      // one-body cache: J1, grad J1, lap J1, v_ei, v^a_ei per electron
    S.o_j3 = (int)w; if (S.n_j3) w += (size_t)S.N * 2 * S.j3s + S.j3s;   // three-body Jastrow: chi3, V3, S3
    S.o_am = (int)w; if (c->listed) w += ((size_t)S.N * (S.lt + S.n_lg) + 7) / 8;       // listed-shell lists (listed.cuh)
    S.o_U = (int)w;                             // last: prepared draws + lattice frames of S.frame_batch steps (propagate.cuh prepare_frames)
    const size_t per_sm = prop.sharedMemPerMultiprocessor, per_blk_max = prop.sharedMemPerBlockOptin, reserve = 1024;
    // warps per CTA that LRDMC_MINB CTAs of `pw` doubles per warp leave room for.  The hardware deals the warps of the resident CTAs round-robin over the
    // 4 schedulers and the warps of a CTA meet at a barrier every step: with 7 (5) warps per CTA the fullest scheduler sets the pace of all -- 2 x 7 warps
    // run at the pace of 16 -- so 7 and 5 are never chosen.  Measured (C3nl / C3j3, 7 -> 6 warps): 75.6 -> 71.7 ms, 61.4 -> 58.2 ms.
    auto warps_for = [&](size_t pw) {
        int n = LRDMC_WPB;
        while (n > 1 && (((size_t)S.tables_doubles + (size_t)n * pw) * 8 + reserve) * LRDMC_MINB > per_sm) --n;
        return (n == 7 || n == 5) ? n - 1 : n;
    };
    S.frame_batch = 1;                          // the largest batch of prepared frames that costs no warp of occupancy
    c->wpb = warps_for(w + LRDMC_FRAME_STRIDE);
    for (int fb = LRDMC_FRAME_BATCH; fb > 1; fb >>= 1) if (warps_for(w + (size_t)fb * LRDMC_FRAME_STRIDE) == c->wpb) { S.frame_batch = fb; break; }
    w += (size_t)S.frame_batch * LRDMC_FRAME_STRIDE;
    S.per_warp_doubles = (int)w;
    c->smem_bytes = (int)(((size_t)S.tables_doubles + (size_t)c->wpb * S.per_warp_doubles) * 8);
    if ((size_t)c->smem_bytes > per_blk_max) return LRDMC_ENOMEM;
#define SET_SMEM(K) CK(cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem_bytes))
#define SET_ALL(NTV, TSV, BFV) SET_SMEM((k_rebuild<NTV, TSV, BFV>))
    SET_ALL(1, true, true); SET_ALL(2, true, true); SET_ALL(4, true, true); SET_ALL(1, true, false); SET_ALL(2, true, false); SET_ALL(4, true, false);
    SET_ALL(1, false, false); SET_ALL(2, false, false); SET_ALL(4, false, false);
#undef SET_ALL
#undef SET_SMEM
    c->ts = S.bf_in_smem && S.moc_in_smem;
    c->ext = c->listed ? 4 : (S.nl_K ? 1 : 0) | (S.n_j3 ? 2 : 0);     // which instantiation of the walker kernels this system runs (kernels.cu)
    LRDMC_K_CALL(c->ext, lrdmc_k_set_smem, c->smem_bytes);
    const int occ = LRDMC_K_CALL(c->ext, lrdmc_k_occupancy, c->NT, c->ts, c->wpb * 32, c->smem_bytes);
    CK(cudaGetLastError());
    c->ctas_per_sm = occ > 0 ? occ : 1;
    c->grid_max = c->sm_count * c->ctas_per_sm;
    return LRDMC_OK;
}

static int init_device(lrdmc_ctx *c, const std::vector<double> &h_sh, const std::vector<double> &h_nuc, const std::vector<double> &h_et,
                       const std::vector<double> (&h_bf)[2], const std::vector<double> (&h_cf)[2], const std::vector<double> &h_srad, const std::vector<double> &h_j3g,
                       const std::vector<double> (&h_cn)[2])
{
    DevSys &S = c->S;
    int ndev = 0; CK(cudaGetDeviceCount(&ndev));
    const size_t bf_n = c->bf_n, cf_n = c->cf_n;
    const size_t cn_n = h_cn[0].size();
    const size_t bytes = (h_sh.size() + h_nuc.size() + h_et.size() + h_srad.size() + h_j3g.size() + (bf_n + cf_n + cn_n) * (S.same_C ? 1 : 2)) * sizeof(double);
    CK(cudaMalloc(&c->d_tables, bytes));
    double *d = (double *)c->d_tables;
    CK(cudaMemcpy(d, h_sh.data(), h_sh.size() * 8, cudaMemcpyHostToDevice)); S.shells = d; d += h_sh.size();
    CK(cudaMemcpy(d, h_nuc.data(), h_nuc.size() * 8, cudaMemcpyHostToDevice)); S.nuc = d; d += h_nuc.size();
    CK(cudaMemcpy(d, h_et.data(), h_et.size() * 8, cudaMemcpyHostToDevice)); S.etab = d; d += h_et.size();
    CK(cudaMemcpy(d, h_bf[0].data(), bf_n * 8, cudaMemcpyHostToDevice)); S.bfrag[0] = d; d += bf_n;
    if (!S.same_C) { CK(cudaMemcpy(d, h_bf[1].data(), bf_n * 8, cudaMemcpyHostToDevice)); S.bfrag[1] = d; d += bf_n; } else S.bfrag[1] = S.bfrag[0];
    S.cfrag[0] = S.cfrag[1] = d;
    if (cf_n) {
        CK(cudaMemcpy(d, h_cf[0].data(), cf_n * 8, cudaMemcpyHostToDevice)); d += cf_n;
        if (!S.same_C) { CK(cudaMemcpy(d, h_cf[1].data(), cf_n * 8, cudaMemcpyHostToDevice)); S.cfrag[1] = d; d += cf_n; }
    }
    CK(cudaMemcpy(d, h_srad.data(), h_srad.size() * 8, cudaMemcpyHostToDevice)); S.srad = d; d += h_srad.size();
    S.j3g = d; if (h_j3g.size()) { CK(cudaMemcpy(d, h_j3g.data(), h_j3g.size() * 8, cudaMemcpyHostToDevice)); d += h_j3g.size(); }
    CK(cudaMemcpy(d, h_cn[0].data(), cn_n * 8, cudaMemcpyHostToDevice)); S.cn[0] = S.cn[1] = d; d += cn_n;
    if (!S.same_C) { CK(cudaMemcpy(d, h_cn[1].data(), cn_n * 8, cudaMemcpyHostToDevice)); S.cn[1] = d; d += cn_n; }
    CK(cudaMalloc((void **)&c->d_stats, sizeof(DevStats)));
    CK(cudaMemset(c->d_stats, 0, sizeof(DevStats)));
    CK(cudaMallocHost((void **)&c->h_stats, sizeof(DevStats)));
    for (int i = 0; i < 4; ++i) CK(cudaEventCreate(&c->ev[i]));
    return plan_smem(c);
}

extern "C" int lrdmc_init(lrdmc_ctx **out, const lrdmc_system *sys, const lrdmc_basis *bas, const lrdmc_mo *mo, const lrdmc_jastrow *jas,
                          const lrdmc_lattice *lat)
{
    if (!out || !sys || !bas || !mo || !jas || !lat) return LRDMC_EINVAL;
    if (sys->n_nuc < 1 || sys->n_up < 1 || sys->n_dn < 0 || sys->n_up > LRDMC_MAX_OCC || sys->n_dn > LRDMC_MAX_OCC) return LRDMC_EINVAL;
    if (bas->n_shell < 1 || !(lat->a > 0.0) || lat->a2 < 0.0 || !sys->Z || !sys->R || !mo->C_up || (sys->n_dn && !mo->C_dn)) return LRDMC_EINVAL;
    // ---- shells: sort by group (Slater s, s, p, d), pad each group to a multiple of 4
    static const int ncomp[4] = { 1, 1, 3, 6 };
    static const int lmn[4][6][3] = { { {0,0,0} }, { {0,0,0} }, { {1,0,0}, {0,1,0}, {0,0,1} }, { {2,0,0}, {1,1,0}, {1,0,1}, {0,2,0}, {0,1,1}, {0,0,2} } };
    std::vector<int> ao0(bas->n_shell), group(bas->n_shell);
    int n_ao = 0;
    for (int s = 0; s < bas->n_shell; ++s) {
        int t = bas->type[s], g = t == LRDMC_SHELL_SLATER_S ? 0 : (t == LRDMC_SHELL_S ? 1 : (t == LRDMC_SHELL_P ? 2 : (t == LRDMC_SHELL_D ? 3 : -1)));
        if (g < 0 || bas->center[s] < 0 || bas->center[s] >= sys->n_nuc || !(bas->zeta[s] > 0.0)) return LRDMC_EINVAL;
        group[s] = g; ao0[s] = n_ao; n_ao += ncomp[g];
    }
    // ---- contracted / solid-harmonic shells: fold the contraction into primitive coefficient matrices (include/lrdmc.h, lrdmc_basis)
    std::vector<double> Cfold[2];
    const double *Cup = mo->C_up, *Cdn = mo->C_dn;
    if (bas->n_cshell > 0 && bas->cs_first) {
        if (!bas->prim_coef || !bas->cs_sph || bas->cs_first[0] != 0 || bas->cs_first[bas->n_cshell] != bas->n_shell) return LRDMC_EINVAL;
        static const double h3 = 0.86602540378443864676;           // sqrt(3)/2;  rows: z2, xz, yz, x2-y2, xy over xx xy xz yy yz zz
        static const double SPH[5][6] = { { -0.5, 0, 0, -0.5, 0, 1.0 }, { 0, 0, 1, 0, 0, 0 }, { 0, 0, 0, 0, 1, 0 }, { h3, 0, 0, -h3, 0, 0 }, { 0, 1, 0, 0, 0, 0 } };
        int nc = 0;
        for (int cs = 0; cs < bas->n_cshell; ++cs) {
            const int k0 = bas->cs_first[cs], k1 = bas->cs_first[cs + 1];
            if (k1 <= k0) return LRDMC_EINVAL;
            for (int k = k0; k < k1; ++k) if (bas->type[k] != bas->type[k0] || bas->center[k] != bas->center[k0]) return LRDMC_EINVAL;
            nc += (group[k0] == 3 && bas->cs_sph[cs]) ? 5 : ncomp[group[k0]];
        }
        if (nc != mo->n_ao) return LRDMC_EINVAL;
        for (int sp = 0; sp < 2; ++sp) {
            const int ns = sp ? sys->n_dn : sys->n_up; const double *C = sp ? mo->C_dn : mo->C_up;
            Cfold[sp].assign((size_t)n_ao * (ns > 0 ? ns : 1), 0.0);
            int nu0 = 0;
            for (int cs = 0; cs < bas->n_cshell; ++cs) {
                const int k0 = bas->cs_first[cs], k1 = bas->cs_first[cs + 1], g = group[k0];
                const bool sph = g == 3 && bas->cs_sph[cs];
                const int nfun = sph ? 5 : ncomp[g];
                for (int k = k0; k < k1; ++k) for (int q = 0; q < ncomp[g]; ++q) for (int f = 0; f < nfun; ++f) {
                    const double w = bas->prim_coef[k] * (sph ? SPH[f][q] : (f == q ? 1.0 : 0.0));
                    if (w != 0.0) for (int m = 0; m < ns; ++m) Cfold[sp][(size_t)(ao0[k] + q) * ns + m] += w * C[(size_t)(nu0 + f) * ns + m];
                }
                nu0 += nfun;
            }
        }
        Cup = Cfold[0].data(); Cdn = Cfold[1].data();
    } else if (n_ao != mo->n_ao) return LRDMC_EINVAL;
    lrdmc_ctx *c = (lrdmc_ctx *)calloc(1, sizeof(lrdmc_ctx));
    if (!c) return LRDMC_ENOMEM;
    c->opt_listed = -1;
    DevSys &S = c->S;
    S.N = sys->n_up + sys->n_dn; S.n_up = sys->n_up; S.n_dn = sys->n_dn; S.n_nuc = sys->n_nuc;
    S.n_mesh = lat->a2 > 0.0 ? 2 : 1; S.P_lat = 6 * S.N * S.n_mesh; S.a = lat->a;
    S.nl_K = (sys->nl && sys->nl_K > 0) ? sys->nl_K : 0; S.nl_dla = sys->nl_dla ? 1 : 0;
    if (S.nl_K > LRDMC_NL_MAX_K) { free(c); return LRDMC_EINVAL; }
    S.P = S.P_lat + 6 * S.N * S.nl_K;
    S.amesh[0] = lat->a; S.amesh[1] = lat->a2; S.gmesh[0] = S.n_mesh == 2 ? 0.5 : 1.0; S.gmesh[1] = S.n_mesh == 2 ? 0.5 : 0.0;
    S.Kdiag = 0.0;
    for (int m = 0; m < S.n_mesh; ++m) {
        S.kappa[m] = S.gmesh[m] / (2.0 * S.amesh[m] * S.amesh[m]); S.g_over_a2[m] = S.gmesh[m] / (S.amesh[m] * S.amesh[m]);
    }
    for (int j = 0; j < S.P_lat; ++j) S.Kdiag += S.kappa[j / (6 * S.N)];      // K^a_{x,x} = sum_j kappa_j = 3N/a^2 (Eq.D5)
    S.a_par = jas->a_par; S.a_anti = jas->a_anti; S.b2 = jas->b2; S.has_j1 = jas->c1 != NULL; S.has_pp = sys->pp != NULL;
    S.n_j3 = jas->n_j3 > 0 ? jas->n_j3 : 0; S.j3s = (S.n_j3 + 3) & ~3; S.j3_poly = 0;
    if (S.n_j3 > LRDMC_J3_MAX || (S.n_j3 && (!jas->j3_center || !jas->j3_zeta || !jas->j3_g))) { free(c); return LRDMC_EINVAL; }
    for (int a = 0; a < S.n_j3; ++a) {
        if (jas->j3_center[a] < 0 || jas->j3_center[a] >= sys->n_nuc || !(jas->j3_zeta[a] > 0.0)) { free(c); return LRDMC_EINVAL; }
        S.j3_center[a] = jas->j3_center[a]; S.j3_zeta[a] = jas->j3_zeta[a]; S.j3_lmn[a] = 0;
        if (jas->j3_lmn) {
            const int *q = jas->j3_lmn + 3 * a;
            if (q[0] < 0 || q[1] < 0 || q[2] < 0 || q[0] + q[1] + q[2] > 2) { free(c); return LRDMC_EINVAL; }
            S.j3_lmn[a] = q[0] | (q[1] << 2) | (q[2] << 4); if (S.j3_lmn[a]) S.j3_poly = 1;
        }
    }
    S.key0 = (uint32_t)lat->seed; S.key1 = (uint32_t)(lat->seed >> 32);
    S.V_ii = 0.0;
    for (int I = 0; I < sys->n_nuc; ++I) for (int J = I + 1; J < sys->n_nuc; ++J) {
        double dx = sys->R[3 * I] - sys->R[3 * J], dy = sys->R[3 * I + 1] - sys->R[3 * J + 1], dz = sys->R[3 * I + 2] - sys->R[3 * J + 2];
        S.V_ii += sys->Z[I] * sys->Z[J] / sqrt(dx * dx + dy * dy + dz * dz);
    }
    std::vector<int> slot_shell; int base[4];
    for (int g = 0; g < 4; ++g) {
        base[g] = (int)slot_shell.size();
        for (int s = 0; s < bas->n_shell; ++s) if (group[s] == g) slot_shell.push_back(s);
        while ((slot_shell.size() - base[g]) % 4) slot_shell.push_back(-1);
        S.n_it[g] = ((int)slot_shell.size() - base[g]) / 4;
    }
    S.n_slots = (int)slot_shell.size();
    S.n_ksteps = S.n_it[0] + S.n_it[1] + 3 * S.n_it[2] + 6 * S.n_it[3];
    int omax = sys->n_up > sys->n_dn ? sys->n_up : sys->n_dn, nt = (omax + 7) / 8;
    c->NT = nt <= 1 ? 1 : (nt == 2 ? 2 : 4);
    S.NT[0] = S.NT[1] = c->NT; S.OS = 8 * c->NT; S.dinv_rows[0] = S.dinv_rows[1] = 8 * c->NT;
    S.same_C = (sys->n_dn == 0) || (sys->n_dn == sys->n_up && (Cdn == Cup || !memcmp(Cup, Cdn, sizeof(double) * (size_t)n_ao * sys->n_up)));
    // ---- host images of the tables
    std::vector<double> h_sh((size_t)S.n_slots * 4), h_nuc((size_t)S.n_nuc * LRDMC_NUC_STRIDE, 0.0);
    for (int q = 0; q < S.n_slots; ++q) {
        int s = slot_shell[q];
        if (s < 0) { h_sh[4 * q] = h_sh[4 * q + 1] = h_sh[4 * q + 2] = 0.0; h_sh[4 * q + 3] = 1.0; continue; }
        const double *Rc = sys->R + 3 * bas->center[s];
        h_sh[4 * q] = Rc[0]; h_sh[4 * q + 1] = Rc[1]; h_sh[4 * q + 2] = Rc[2]; h_sh[4 * q + 3] = bas->zeta[s];
    }
    for (int I = 0; I < S.n_nuc; ++I) {
        double *nu = &h_nuc[(size_t)I * LRDMC_NUC_STRIDE];
        nu[0] = sys->R[3 * I]; nu[1] = sys->R[3 * I + 1]; nu[2] = sys->R[3 * I + 2]; nu[3] = sys->Z[I];
        nu[4] = jas->c1 ? jas->c1[I] : 0.0; nu[5] = jas->c1 ? (jas->b1 ? jas->b1[I] : 1.0) : 1.0;
        if (S.nl_K) for (int q = 0; q < 7; ++q) nu[LRDMC_NL_OFF + q] = sys->nl[7 * I + q];
        if (sys->pp && sys->pp[4 * I] > 0.0) { nu[6] = sys->pp[4 * I]; nu[7] = sys->pp[4 * I + 1]; nu[8] = sys->pp[4 * I + 2]; nu[9] = sys->pp[4 * I + 3]; nu[10] = 1.0; }
    }
    const size_t bf_n = (size_t)S.n_ksteps * c->NT * 32;
    std::vector<double> h_bf[2], h_et(256);
    for (int j = 0; j < 256; ++j) h_et[j] = exp2((double)j / 256.0);       // table of exp_tab
    for (int sp = 0; sp < (S.same_C ? 1 : 2); ++sp) {
        const int ns = sp ? sys->n_dn : sys->n_up; const double *C = sp ? Cdn : Cup;
        h_bf[sp].assign(bf_n, 0.0);
        int kstep = 0;
        for (int g = 0; g < 4; ++g) for (int it = 0; it < S.n_it[g]; ++it) for (int comp = 0; comp < ncomp[g]; ++comp, ++kstep)
            for (int t = 0; t < c->NT; ++t) for (int lane = 0; lane < 32; ++lane) {
                int gp = lane >> 2, tp = lane & 3, s = slot_shell[base[g] + 4 * it + tp], m = 8 * t + gp;
                if (s < 0 || m >= ns) continue;
                double nrm = g == 0 ? 1.0 : gto_norm(bas->zeta[s], lmn[g][comp][0], lmn[g][comp][1], lmn[g][comp][2]);
                h_bf[sp][((size_t)kstep * c->NT + t) * 32 + lane] = nrm * C[(size_t)(ao0[s] + comp) * ns + m];
            }
    }
    // ---- pair table of ao_columns: B fragments of Bc[ao][el] = sum_m C[ao][m] Dinv[m][el], two k-steps per mma column set.
    //      mma column n = 2 slot + parity (k-step 2 pair + parity of the group's own sequence), mma k = MO 4 j + k.
    int pair_base[5]; pair_base[0] = 0;
    for (int g = 0; g < 4; ++g) pair_base[g + 1] = pair_base[g] + (ncomp[g] * S.n_it[g] + 1) / 2;
    S.n_kpairs = pair_base[4];
    for (int g = 0; g < 5; ++g) c->pair_base[g] = pair_base[g];
    const int NA = 2 * c->NT;
    const size_t cf_n = (size_t)S.n_kpairs * NA * 32;
    std::vector<double> h_cf[2];
    for (int sp = 0; sp < (S.same_C ? 1 : 2) && cf_n; ++sp) {
        const int ns = sp ? sys->n_dn : sys->n_up; const double *C = sp ? Cdn : Cup;
        h_cf[sp].assign(cf_n, 0.0);
        for (int g = 0; g < 4; ++g) for (int it = 0; it < S.n_it[g]; ++it) for (int comp = 0; comp < ncomp[g]; ++comp) {
            const int q = it * ncomp[g] + comp, pair = pair_base[g] + q / 2, par = q & 1;
            for (int slot = 0; slot < 4; ++slot) {
                const int s = slot_shell[base[g] + 4 * it + slot];
                if (s < 0) continue;
                const double nrm = g == 0 ? 1.0 : gto_norm(bas->zeta[s], lmn[g][comp][0], lmn[g][comp][1], lmn[g][comp][2]);
                for (int j = 0; j < NA; ++j) for (int k = 0; k < 4; ++k) {
                    const int m = 4 * j + k; if (m >= ns) continue;
                    h_cf[sp][((size_t)pair * NA + j) * 32 + 4 * (2 * slot + par) + k] = nrm * C[(size_t)(ao0[s] + comp) * ns + m];
                }
            }
        }
    }
    // ---- listed candidate sweep: list groups (one shell type, at most 64 slots each), slot-major coefficient rows, screening radii
    {
        S.n_lg = 0; S.n_aop = 0; S.lt = 0;
        int ao_run = 0;
        for (int g = 0; g < 4; ++g) {
            const int nsl = 4 * S.n_it[g];
            for (int s0 = 0; s0 < nsl; s0 += 64) {
                if (S.n_lg == LRDMC_MAX_LG) { free(c); return LRDMC_ENOMEM; }
                S.lg_type[S.n_lg] = g; S.lg_slot0[S.n_lg] = base[g] + s0; S.lg_n[S.n_lg] = nsl - s0 < 64 ? nsl - s0 : 64;
                S.lg_ao0[S.n_lg] = ao_run + s0 * ncomp[g]; S.lg_off[S.n_lg] = S.lt; S.lt += S.lg_n[S.n_lg]; ++S.n_lg;
            }
            ao_run += nsl * ncomp[g];
        }
        S.n_aop = ao_run;
    }
    std::vector<double> h_srad(S.n_slots), h_cn[2];
    {
        double amax = lat->a > lat->a2 ? lat->a : lat->a2; (void)amax;
        for (int q = 0; q < S.n_slots; ++q) {
            const int s = slot_shell[q];
            h_srad[q] = s < 0 ? -1e300 : (group[s] == 0 ? LRDMC_LIST_THR / bas->zeta[s] : sqrt(LRDMC_LIST_THR / bas->zeta[s]));
        }
        for (int sp = 0; sp < (S.same_C ? 1 : 2); ++sp) {
            const int ns = sp ? sys->n_dn : sys->n_up; const double *C = sp ? Cdn : Cup;
            h_cn[sp].assign((size_t)S.n_aop * S.OS, 0.0);
            int row = 0;
            for (int g = 0; g < 4; ++g) for (int q = base[g]; q < base[g] + 4 * S.n_it[g]; ++q) for (int comp = 0; comp < ncomp[g]; ++comp, ++row) {
                const int s = slot_shell[q]; if (s < 0) continue;
                const double nrm = g == 0 ? 1.0 : gto_norm(bas->zeta[s], lmn[g][comp][0], lmn[g][comp][1], lmn[g][comp][2]);
                for (int m = 0; m < ns; ++m) h_cn[sp][(size_t)row * S.OS + m] = nrm * C[(size_t)(ao0[s] + comp) * ns + m];
            }
        }
    }
    // ---- device copies (every CUDA call checked; on failure the text moves to the calling thread's slot and the ctx is freed)
    c->n_sh = h_sh.size(); c->n_nuc_d = h_nuc.size(); c->bf_n = bf_n; c->cf_n = cf_n;
    std::vector<double> h_j3g((size_t)S.j3s * S.j3s, 0.0);          // three-body couplings g [j3s][j3s], zero padded
    for (int a = 0; a < S.n_j3; ++a) for (int b = 0; b < S.n_j3; ++b) h_j3g[(size_t)a * S.j3s + b] = jas->j3_g[a * S.n_j3 + b];
    const int rc = init_device(c, h_sh, h_nuc, h_et, h_bf, h_cf, h_srad, h_j3g, h_cn);
    if (rc != LRDMC_OK) { snprintf(t_init_msg, sizeof t_init_msg, "%s", c->msg); lrdmc_free(c); return rc; }
    *out = c;
    return LRDMC_OK;
}

extern "C" void lrdmc_free(lrdmc_ctx *c)
{
    if (!c) return;
    if (c->d_tables) cudaFree(c->d_tables);
    if (c->d_stats) cudaFree(c->d_stats);
    if (c->h_stats) cudaFreeHost(c->h_stats);
    for (int i = 0; i < 4; ++i) if (c->ev[i]) cudaEventDestroy(c->ev[i]);
    free(c);
}

extern "C" int lrdmc_n_candidates(const lrdmc_ctx *c) { return c ? c->S.P : LRDMC_EINVAL; }

extern "C" const char *lrdmc_last_error(const lrdmc_ctx *c) { return c ? c->msg : t_init_msg; }

extern "C" int lrdmc_set_option(lrdmc_ctx *c, int option, int value)
{
    if (!c) return LRDMC_EINVAL;
    if (c->bound) return LRDMC_ESTATE;            // the walker buffer was carved with the old plan
    switch (option) {
    case LRDMC_OPT_TEAM_WARPS:
        if (value < 0 || value > LRDMC_TEAM_MAX_WARPS) return LRDMC_EINVAL;
        c->opt_team = value; return LRDMC_OK;
    case LRDMC_OPT_GLOBAL_TABLES:
        c->opt_global_tables = value != 0; return plan_smem(c);
    case LRDMC_OPT_LISTED:
        if (value < -1 || value > 1) return LRDMC_EINVAL;
        c->opt_listed = value; return plan_smem(c);
    default: return LRDMC_EINVAL;
    }
}

// ---- walker buffer carving -------------------------------------------------------------------------------------
static size_t carve(const lrdmc_ctx *c, int n_w, char *base, DevWalk *W)
{
    const DevSys &S = c->S; size_t o = 0; const size_t nw = (size_t)n_w;
#define TAKE(field, type, count) do { if (W) W->field = (type *)(base + o); o = align_up(o + sizeof(type) * (count), 256); } while (0)
    TAKE(r, double, nw * 3 * S.N); TAKE(r_alt, double, nw * 3 * S.N);
    TAKE(dinv[0], double, nw * S.n_up * S.n_up); TAKE(dinv[1], double, nw * S.n_dn * S.n_dn + 1);
    TAKE(moc, double, nw * S.N * 5 * S.OS); TAKE(moc_alt, double, nw * S.N * 5 * S.OS);
    TAKE(w, double, nw); TAKE(eL, double, nw); TAKE(W, double, nw); TAKE(omega, double, nw);
    TAKE(nmoves, long long, nw); TAKE(flags, int, nw * 3); TAKE(dead, int, nw);
    TAKE(wq, unsigned long long, nw); TAKE(prefix, unsigned long long, nw); TAKE(parents, int, nw);
    {   // parked Bc entries of the team kernel of the large systems (ao_columns BCS): [resident CTA][block of a mesh][k-step pair][lane][2]
        const bool use = LRDMC_BC_STORE && (!c->ts || c->listed);
        size_t stride = (size_t)((S.n_up + 7) / 8 + (S.n_dn + 7) / 8) * S.n_kpairs * 64;
        if (c->listed) stride = (size_t)S.N * S.n_aop;       // listed sweep: Bc [electron][n_aop] per resident walker
        const size_t cta_bytes = ((size_t)S.tables_doubles + S.per_warp_doubles) * 8 + 1024;
        size_t per_sm = c->smem_per_sm / cta_bytes; if (per_sm > 32) per_sm = 32; if (per_sm < 1) per_sm = 1;   // resident team CTAs per SM, at most
        size_t n_res = per_sm * c->sm_count;                  // team CTAs (plan_team clamps the grid to this) ...
        if (c->listed) {                                      // ... or the resident warps of the warp-per-walker kernel; never more than the walkers
            if ((size_t)c->grid_max * c->wpb > n_res) n_res = (size_t)c->grid_max * c->wpb;
            if (n_res > nw + LRDMC_WPB) n_res = nw + LRDMC_WPB;
        }
        if (W) { W->bcs_stride = use ? stride : 0; W->bcs_ctas = use ? (int)n_res : 0; }
        TAKE(bcs, double, use ? stride * n_res : 0);
        if (W && !use) W->bcs = NULL;
    }
    TAKE(timing, unsigned long long, 2 * (size_t)(c->grid_max * c->wpb > c->sm_count * 32 ? c->grid_max * c->wpb : c->sm_count * 32)); TAKE(counter, int, 64);
#undef TAKE
    return o;
}

extern "C" size_t lrdmc_walker_bytes(const lrdmc_ctx *c, int n_walkers)
{
    if (!c || n_walkers < 1) return 0;
    return carve(c, n_walkers, NULL, NULL) + 256;
}

// ---- team mode planning (team.cuh) ----------------------------------------------------------------------------------
// Cut the sorted shell list into K parts of about equal cost.  Unit = two 4-shell iterations in groups 0-2 when `pairs`
// (a part of ao_columns must start on a k-step pair), else one iteration; units go to parts by their cumulative cost.
// `lead` is work part 0 has besides its shells, in the same cost units (the team's warp 0 also refreshes the one-body cache).
static void partition_shells(const int n_it[4], const double cost[4], bool pairs, int K, ShellPart *out, double lead = 0.0)
{
    struct Unit { int g, lo, hi; double c; };
    std::vector<Unit> units; double total = 0.0;
    for (int g = 0; g < 4; ++g) {
        const int stepu = (pairs && g < 3) ? 2 : 1;
        for (int it = 0; it < n_it[g]; it += stepu) {
            const int hi = it + stepu < n_it[g] ? it + stepu : n_it[g];
            units.push_back({ g, it, hi, cost[g] * (hi - it) }); total += cost[g] * (hi - it);
        }
    }
    for (int k = 0; k < K; ++k) for (int g = 0; g < 4; ++g) out[k].lo[g] = out[k].hi[g] = 0;
    double cum = lead; total += lead;
    for (const Unit &u : units) {
        int k = total > 0.0 ? (int)((cum + 0.5 * u.c) / total * K) : 0;
        if (k > K - 1) k = K - 1;
        if (out[k].hi[u.g] == out[k].lo[u.g]) out[k].lo[u.g] = u.lo;
        out[k].hi[u.g] = u.hi; cum += u.c;
    }
}

// Choose the team size for n_w walkers.  Warp-per-walker (team_tw = 1) when the walkers alone fill the resident warp slots;
// otherwise 4 warps per walker: for few walkers (n_w up to 3/8 of the warp slots), and for the large systems whose 36 KB state
// leaves one warp per scheduler.  lrdmc_set_option(LRDMC_OPT_TEAM_WARPS, tw) forces a size (1: warp-per-walker).
static void plan_team(lrdmc_ctx *c, int n_w)
{
    const DevSys &S = c->S; TeamPlan &P = c->team;
    c->team_tw = 1;
    int tw = 1;
    const long slots = (long)c->grid_max * c->wpb;
    if (!c->ts) tw = c->listed ? 8 : 4;   // listed sweep (listed.cuh): measured at C5 N_w = 4096, TW = 4 / 8 / 16: 2.27 / 2.82 / 2.64 M walker-moves/s
    else if ((long)n_w * 8 <= 3 * slots) tw = 4;   // measured on C3/C4 (profiles/r1_team_kernel.md): 4 warps per walker beat 2, 8 and 16 at every N_w,
                                                   // and beat warp-per-walker up to N_w of about 3/8 of the resident warp slots
    if (c->opt_team > 0) tw = c->opt_team;        // LRDMC_OPT_TEAM_WARPS (tests force 1, 2, 4, 8, 16)
    int p2 = 1; while (p2 * 2 <= tw && p2 * 2 <= LRDMC_TEAM_MAX_WARPS) p2 *= 2;
    tw = p2;
    if (tw <= 1) return;
    memset(&P, 0, sizeof P);
    static const int ncomp[4] = { 1, 1, 3, 6 };
    P.TW = tw;
    P.nblk[0] = (S.n_up + 7) / 8; P.nblk[1] = (S.n_dn + 7) / 8;
    const int nblk = S.n_mesh * (P.nblk[0] + P.nblk[1]);
    int it_total = 0;
    for (int g = 0; g < 4; ++g) {
        P.it_base[g] = it_total; it_total += S.n_it[g];
        P.kstep_base[g] = g ? P.kstep_base[g - 1] + ncomp[g - 1] * S.n_it[g - 1] : 0;
        P.pair_base[g] = c->pair_base[g];
    }
    int np = 1; while (nblk * np < tw && np < LRDMC_TEAM_MAX_PARTS && 2 * np <= (it_total + 1) / 2) np *= 2;
    P.NP = np; P.n_units = nblk * np;
    P.mesh_share = S.n_mesh == 2 && ((P.nblk[0] + P.nblk[1]) * np) % tw == 0;
    int lpe = 32; while (lpe > 1 && (tw * 32) / lpe < S.N) lpe >>= 1;     // largest power of two with one pass over the electrons
    P.lpe = lpe;
    // relative cost of a 4-shell iteration by group (s with one exponent per row, contracted s, p, d): measured on C3, N_w = 100 / 400, against
    // the derivative pass of wavefunction.cuh (one product per row): 9.61 -> 10.33 and 27.65 -> 28.96 M walker-moves/s over the former { 1.5, 1, 3, 6 }
    const double cost_col[4] = { 2.0, 1.0, 1.45, 2.1 }, cost_mo[4] = { 1.3, 1.0, 1.5, 2.2 };
    partition_shells(S.n_it, cost_col, true, np, P.col);
    partition_shells(S.n_it, cost_mo, false, tw, P.mo, 3.0);
    P.nblk_nl[0] = (S.n_up * S.nl_K + 7) / 8; P.nblk_nl[1] = (S.n_dn * S.nl_K + 7) / 8; P.n_units_nl = (P.nblk_nl[0] + P.nblk_nl[1]) * np;
    const size_t scr_lat = np > 1 ? (size_t)S.n_mesh * S.N * np * 12 : 0, scr_nl = np > 1 ? (size_t)S.N * S.nl_K * np * 12 : 0,
                 scr_nu = np > 1 ? (size_t)S.N * S.nl_K * 7 : 0, scr_col = scr_lat + scr_nl + scr_nu, scr_mo = (size_t)tw * 5 * S.OS;
    P.o_nl = (int)scr_lat; P.o_nu = (int)(scr_lat + scr_nl);
    P.o_scr = S.per_warp_doubles; P.scr_doubles = (int)align_up(scr_col > scr_mo ? scr_col : scr_mo, 2);
    const int smem = (int)(((size_t)S.tables_doubles + S.per_warp_doubles + P.scr_doubles) * 8);
    const int occ = LRDMC_K_CALL(c->ext, lrdmc_k_team_occupancy, c->NT, c->ts, tw * 32, smem);
    if (cudaGetLastError() != cudaSuccess || occ < 1) return;             // does not fit: stay with warp-per-walker
    P.listed = c->listed;
    c->team_tw = tw; c->team_smem = smem; c->team_ctas_per_sm = occ; c->team_grid_max = c->sm_count * occ;
    if (c->W.bcs && c->team_grid_max > c->W.bcs_ctas) c->team_grid_max = c->W.bcs_ctas;   // the parked-entry scratch is indexed by blockIdx.x
}

extern "C" int lrdmc_bind_walkers(lrdmc_ctx *c, void *dev_buf, size_t bytes, int n_walkers)
{
    if (!c || !dev_buf || n_walkers < 1 || n_walkers > (1 << 20)) return LRDMC_EINVAL;
    char *base = (char *)align_up((size_t)dev_buf, 256);
    if (carve(c, n_walkers, NULL, NULL) + (size_t)(base - (char *)dev_buf) > bytes) return LRDMC_EINVAL;
    carve(c, n_walkers, base, &c->W);
    c->W.n_sing = &c->d_stats->n_singular;
    plan_team(c, n_walkers);
    c->W.n_w = n_walkers; c->bound = 1; c->state_ok = 0; c->have_prop = c->have_reconf = 0;
    return LRDMC_OK;
}

// ---- launch helpers -----------------------------------------------------------------------------------------------
static int grid_for(const lrdmc_ctx *c) { int g = (c->W.n_w + c->wpb - 1) / c->wpb; return g < c->grid_max ? g : c->grid_max; }
// Warp-per-walker launch of lrdmc_propagate: an SM's time grows with its resident warps (the kernel is dispatch-bound), so an
// ensemble that does not fill the warp slots is spread over ALL resident CTAs with fewer warps each, instead of filling some SMs
// with full CTAs (N_w = 1200 on C4: 150 CTAs x 8 warps put 16 walkers on two SMs -> 4.44 ms; 240 x 5 warps -> 10 per SM).
static void propagate_shape(const lrdmc_ctx *c, int *grid, int *warps)
{
    int w = (c->W.n_w + c->grid_max - 1) / c->grid_max; if (w > c->wpb) w = c->wpb; if (w < 1) w = 1;
    int g = (c->W.n_w + w - 1) / w; if (g > c->grid_max) g = c->grid_max;
    *grid = g; *warps = w;
}
#define LAUNCH_(KERNEL, NTV, TSV, NLV, grid, stream, ...) KERNEL<NTV, TSV, NLV><<<grid, c->wpb * 32, c->smem_bytes, stream>>>(__VA_ARGS__)
#define DISPATCH_NL_(KERNEL, NLV, grid, stream, ...)                                                             \
    do {                                                                                                         \
        if (c->ts) {                                                                                             \
            if (c->NT == 1) LAUNCH_(KERNEL, 1, true, NLV, grid, stream, __VA_ARGS__);                            \
            else if (c->NT == 2) LAUNCH_(KERNEL, 2, true, NLV, grid, stream, __VA_ARGS__);                       \
            else LAUNCH_(KERNEL, 4, true, NLV, grid, stream, __VA_ARGS__);                                       \
        } else {                                                                                                 \
            if (c->NT == 1) LAUNCH_(KERNEL, 1, false, NLV, grid, stream, __VA_ARGS__);                           \
            else if (c->NT == 2) LAUNCH_(KERNEL, 2, false, NLV, grid, stream, __VA_ARGS__);                      \
            else LAUNCH_(KERNEL, 4, false, NLV, grid, stream, __VA_ARGS__);                                      \
        }                                                                                                        \
        ++c->launches;                                                                                           \
    } while (0)

static int rebuild(lrdmc_ctx *c, int do_invert /* bit 0: invert, bit 1: the MO cache is valid */, cudaStream_t st)
{
    CK(cudaMemsetAsync(c->W.counter, 0, 64 * sizeof(int), st));
    if (do_invert & 1) CK(cudaMemsetAsync(c->W.n_sing, 0, sizeof(long long), st));
    else CK(cudaMemsetAsync(c->W.dead, 0, sizeof(int) * (size_t)c->W.n_w, st));     // inverses supplied by the caller: nobody is dead
    if (c->S.bfm_in_smem) DISPATCH_NL_(k_rebuild, true, grid_for(c), st, c->S, c->W, do_invert);      // third argument: LRDMC_BF_SMEM
    else DISPATCH_NL_(k_rebuild, false, grid_for(c), st, c->S, c->W, do_invert);
    CK(cudaGetLastError());
    return LRDMC_OK;
}

static void fill_ones(lrdmc_ctx *c, cudaStream_t st);
__global__ void k_fill(double *p, double v, int n) { for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) p[i] = v; }
static void fill_ones(lrdmc_ctx *c, cudaStream_t st) { k_fill<<<(c->W.n_w + 255) / 256, 256, 0, st>>>(c->W.w, 1.0, c->W.n_w); ++c->launches; }

extern "C" int lrdmc_set_positions(lrdmc_ctx *c, const double *r_dev, void *stream)
{
    if (!c || !r_dev) return LRDMC_EINVAL;
    if (!c->bound) return LRDMC_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemcpyAsync(c->W.r, r_dev, sizeof(double) * (size_t)c->W.n_w * 3 * c->S.N, cudaMemcpyDeviceToDevice, st));
    fill_ones(c, st);
    int rc = rebuild(c, 1, st); if (rc) return rc;
    int flag[2] = { 0, 0 };
    CK(cudaMemcpyAsync(flag, c->W.counter, sizeof flag, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    c->state_ok = 1; c->have_prop = c->have_reconf = 0; c->last_stream = st;
    return flag[1] ? LRDMC_ESINGULAR : LRDMC_OK;
}

extern "C" int lrdmc_set_state(lrdmc_ctx *c, const double *r_dev, const double *du, const double *dd, const double *w_dev, void *stream)
{
    if (!c || !r_dev) return LRDMC_EINVAL;
    if (!c->bound) return LRDMC_ESTATE;
    cudaStream_t st = (cudaStream_t)stream; const DevSys &S = c->S; const size_t nw = (size_t)c->W.n_w;
    CK(cudaMemcpyAsync(c->W.r, r_dev, sizeof(double) * nw * 3 * S.N, cudaMemcpyDeviceToDevice, st));
    if (du) {
        CK(cudaMemcpyAsync(c->W.dinv[0], du, sizeof(double) * nw * S.n_up * S.n_up, cudaMemcpyDeviceToDevice, st));
        if (S.n_dn) { if (!dd) return LRDMC_EINVAL; CK(cudaMemcpyAsync(c->W.dinv[1], dd, sizeof(double) * nw * S.n_dn * S.n_dn, cudaMemcpyDeviceToDevice, st)); }
    }
    if (w_dev) CK(cudaMemcpyAsync(c->W.w, w_dev, sizeof(double) * nw, cudaMemcpyDeviceToDevice, st)); else fill_ones(c, st);
    int rc = rebuild(c, du ? 0 : 1, st); if (rc) return rc;
    c->state_ok = 1; c->have_prop = c->have_reconf = 0; c->last_stream = st;
    return LRDMC_OK;
}

extern "C" int lrdmc_get_walkers(lrdmc_ctx *c, double *r_dev, double *du, double *dd, double *w_dev, void *stream)
{
    if (!c) return LRDMC_EINVAL;
    if (!c->bound || !c->state_ok) return LRDMC_ESTATE;
    cudaStream_t st = (cudaStream_t)stream; const DevSys &S = c->S; const size_t nw = (size_t)c->W.n_w;
    if (r_dev) CK(cudaMemcpyAsync(r_dev, c->W.r, sizeof(double) * nw * 3 * S.N, cudaMemcpyDeviceToDevice, st));
    if (du) CK(cudaMemcpyAsync(du, c->W.dinv[0], sizeof(double) * nw * S.n_up * S.n_up, cudaMemcpyDeviceToDevice, st));
    if (dd && S.n_dn) CK(cudaMemcpyAsync(dd, c->W.dinv[1], sizeof(double) * nw * S.n_dn * S.n_dn, cudaMemcpyDeviceToDevice, st));
    if (w_dev) CK(cudaMemcpyAsync(w_dev, c->W.w, sizeof(double) * nw, cudaMemcpyDeviceToDevice, st));
    return LRDMC_OK;
}

extern "C" int lrdmc_get_obs(lrdmc_ctx *c, double *eL, double *Wd, double *om, int64_t *nm, void *stream)
{
    if (!c) return LRDMC_EINVAL;
    if (!c->have_prop) return LRDMC_ESTATE;
    cudaStream_t st = (cudaStream_t)stream; const size_t nw = (size_t)c->W.n_w;
    if (eL) CK(cudaMemcpyAsync(eL, c->W.eL, 8 * nw, cudaMemcpyDeviceToDevice, st));
    if (Wd) CK(cudaMemcpyAsync(Wd, c->W.W, 8 * nw, cudaMemcpyDeviceToDevice, st));
    if (om) CK(cudaMemcpyAsync(om, c->W.omega, 8 * nw, cudaMemcpyDeviceToDevice, st));
    if (nm) CK(cudaMemcpyAsync(nm, c->W.nmoves, 8 * nw, cudaMemcpyDeviceToDevice, st));
    return LRDMC_OK;
}

extern "C" int lrdmc_propagate(lrdmc_ctx *c, int mode, int n_moves, double tau, double E0, uint64_t cycle, void *stream)
{
    if (!c) return LRDMC_EINVAL;
    if (!c->bound || !c->state_ok) return LRDMC_ESTATE;
    if ((mode != LRDMC_BALANCED && mode != LRDMC_CONVENTIONAL) || n_moves < 0 || (mode == LRDMC_CONVENTIONAL && !(tau > 0.0)) || cycle > 0xFFFFFFFFull
        || !std::isfinite(E0)) return LRDMC_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    CK(cudaMemsetAsync(c->W.counter, 0, 64 * sizeof(int), st));
    const bool team = c->team_tw > 1;
    int grid = team ? (c->W.n_w < c->team_grid_max ? c->W.n_w : c->team_grid_max) : 0, warps = c->wpb;
    if (!team) propagate_shape(c, &grid, &warps);
    CK(cudaEventRecord(c->ev[0], st));
    if (team) LRDMC_K_CALL(c->ext, lrdmc_k_team, c->NT, c->ts, grid, c->team_tw * 32, c->team_smem, st, c->S, c->W, c->team, mode, n_moves, tau, E0, (uint32_t)cycle);
    else LRDMC_K_CALL(c->ext, lrdmc_k_propagate, c->NT, c->ts, grid, warps * 32, c->smem_bytes, st, c->S, c->W, mode, n_moves, tau, E0, (uint32_t)cycle);
    ++c->launches;
    CK(cudaEventRecord(c->ev[1], st));
    CK(cudaGetLastError());
    k_reduce_obs<<<1, 1024, 0, st>>>(c->W, c->d_stats, team ? grid : grid * warps); ++c->launches;
    CK(cudaGetLastError());
    c->have_prop = 1; c->last_stream = st;
    return LRDMC_OK;
}

extern "C" int lrdmc_reconfigure(lrdmc_ctx *c, uint64_t cycle, int32_t *parents_dev, void *stream)
{
    if (!c) return LRDMC_EINVAL;
    if (!c->bound || !c->state_ok) return LRDMC_ESTATE;
    if (cycle > 0xFFFFFFFFull) return LRDMC_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    // comb random number: counter (0xFFFFFFFF, cycle, 0, 3), word 0 -- same block function as the device generator, run on the host
    uint32_t ctr[4] = { 0xFFFFFFFFu, (uint32_t)cycle, 0u, 3u }, k0 = c->S.key0, k1 = c->S.key1;
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * ctr[0], p1 = (uint64_t)0xCD9E8D57u * ctr[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ ctr[1] ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ ctr[3] ^ k1, n3 = (uint32_t)p0;
        ctr[0] = n0; ctr[1] = n1; ctr[2] = n2; ctr[3] = n3; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    CK(cudaEventRecord(c->ev[2], st));
    const int split = c->W.n_w > 8192;        // large ensembles: the search (one 128-bit binary search per slot) runs on the whole device
    k_comb<<<1, COMB_THREADS, 0, st>>>(c->W, ctr[0], c->d_stats, parents_dev, !split); ++c->launches;
    CK(cudaGetLastError());
    if (split) { k_comb_search<<<(c->W.n_w + 255) / 256, 256, 0, st>>>(c->W, ctr[0], c->d_stats, parents_dev); ++c->launches; CK(cudaGetLastError()); }
    const int rec = 3 * c->S.N;
    size_t total = (size_t)c->W.n_w * (rec + c->S.N * 5 * c->S.OS / 2); int gb = (int)((total + 255) / 256); if (gb > c->sm_count * 16) gb = c->sm_count * 16;
    k_gather<<<gb, 256, 0, st>>>(c->W, rec, c->S.N * 5 * c->S.OS); ++c->launches;
    CK(cudaGetLastError());
    double *tmp = c->W.r; c->W.r = c->W.r_alt; c->W.r_alt = tmp;
    tmp = c->W.moc; c->W.moc = c->W.moc_alt; c->W.moc_alt = tmp;
    int rc = rebuild(c, 1 | 2, st); if (rc) return rc;          // invert from the gathered cache rows (reading Q15)
    CK(cudaEventRecord(c->ev[3], st));
    c->have_reconf = 1; c->last_stream = st;
    return LRDMC_OK;
}

extern "C" int lrdmc_estimators(lrdmc_ctx *c, lrdmc_cycle_stats *out)
{
    if (!c || !out) return LRDMC_EINVAL;
    if (!c->have_prop) return LRDMC_ESTATE;
    // read back on the stream of the last call and wait for that stream only: other contexts' streams keep running
    CK(cudaMemcpyAsync(c->h_stats, c->d_stats, sizeof(DevStats), cudaMemcpyDeviceToHost, c->last_stream));
    CK(cudaStreamSynchronize(c->last_stream));
    const DevStats h = *c->h_stats;
    memset(out, 0, sizeof *out);
    out->wbar = c->have_reconf ? h.wbar : 0.0; out->num = h.num; out->den = h.den;
    out->moves_min = h.moves_min; out->moves_max = h.moves_max; out->moves_sum = h.moves_sum;
    out->n_node_flag = h.n_node; out->n_nonpos_diag = h.n_nonpos; out->n_nonfinite = h.n_nonfinite; out->n_singular = h.n_singular;
    out->lockstep_idle_frac = h.moves_max > 0 ? 1.0 - (double)h.moves_sum / ((double)c->W.n_w * (double)h.moves_max) : 0.0;
    out->barrier_idle_frac = (h.span_ns > 0.0 && h.n_warps > 0) ? 1.0 - h.busy_ns / (h.span_ns * h.n_warps) : 0.0;
    cudaEventElapsedTime(&out->propagate_ms, c->ev[0], c->ev[1]);
    if (c->have_reconf) cudaEventElapsedTime(&out->reconfigure_ms, c->ev[2], c->ev[3]);
    cudaGetLastError();
    return LRDMC_OK;
}

extern "C" int lrdmc_step_debug(lrdmc_ctx *c, double E0, uint64_t cycle, uint64_t step, double *R_dev, double *scal_dev, int32_t *jstar_dev, void *stream)
{
    if (!c || !R_dev || !scal_dev || !jstar_dev || cycle > 0xFFFFFFFFull || step > 0xFFFFFFFFull) return LRDMC_EINVAL;
    if (!c->bound || !c->state_ok) return LRDMC_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    LRDMC_K_CALL(c->ext, lrdmc_k_step_debug, c->NT, c->ts, grid_for(c), c->wpb * 32, c->smem_bytes, st, c->S, c->W, E0, (uint32_t)cycle, (uint32_t)step, R_dev, scal_dev, jstar_dev);
    ++c->launches;
    CK(cudaGetLastError());
    return LRDMC_OK;
}

extern "C" int lrdmc_launch_count(const lrdmc_ctx *c) { return c ? c->launches : 0; }
extern "C" int lrdmc_listed_sweep(const lrdmc_ctx *c) { return c ? c->listed : 0; }
extern "C" int lrdmc_bound_walkers(const lrdmc_ctx *c) { return (c && c->bound) ? c->W.n_w : 0; }
extern "C" int lrdmc_n_electrons(const lrdmc_ctx *c) { return c ? c->S.N : 0; }
extern "C" const DevSys *lrdmc_devsys(const lrdmc_ctx *c) { return &c->S; }
extern "C" double *lrdmc_positions_ptr(const lrdmc_ctx *c, int which) { return which ? c->W.r_alt : c->W.r; }
extern "C" int lrdmc_launch_config(const lrdmc_ctx *c, int *grid, int *block, int *smem_bytes, int *ctas_per_sm, int *team_warps)
{
    if (!c) return LRDMC_EINVAL;
    if (c->bound && c->team_tw > 1) {            // team mode: one CTA of team_tw warps per walker
        if (grid) *grid = c->W.n_w < c->team_grid_max ? c->W.n_w : c->team_grid_max;
        if (block) *block = c->team_tw * 32; if (smem_bytes) *smem_bytes = c->team_smem; if (ctas_per_sm) *ctas_per_sm = c->team_ctas_per_sm;
        if (team_warps) *team_warps = c->team_tw;
        return LRDMC_OK;
    }
    int pg = c->grid_max, pw = c->wpb; if (c->bound) propagate_shape(c, &pg, &pw);
    if (grid) *grid = pg; if (block) *block = pw * 32; if (smem_bytes) *smem_bytes = c->smem_bytes;
    if (ctas_per_sm) *ctas_per_sm = c->ctas_per_sm; if (team_warps) *team_warps = 1;
    return LRDMC_OK;
}
