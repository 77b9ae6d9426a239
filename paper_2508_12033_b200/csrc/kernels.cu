// kernels.cu -- the walker kernels' launchers.  This one source is compiled TEN times (build.py: -DLRDMC_EXT=0|1|2|3|4 x
// -DLRDMC_TEAM_TU=0|1, in parallel): EXT bit 0 = non-local pseudopotential slots, bit 1 = three-body Jastrow, 4 = listed candidate sweep on stored Bc (lattice-only systems; listed.cuh) (separate code, so
// that every system keeps the register allocation of what it actually has: inlined behind runtime flags the slots cost the
// lattice-only kernel 284 B of spills and 9 % of the C4 throughput; slots and J3 in one instantiation spilled 196 B),
// TEAM_TU = the team kernel / the warp-per-walker kernels.  lrdmc.cu (host logic) calls them through kernels.h.
#include "common.cuh"
#include "philox.cuh"
#include "wavefunction.cuh"
#include "evaluate.cuh"
#include "propagate.cuh"
#include "team.cuh"
#include "kernels.h"

#ifndef LRDMC_EXT
#error "compile with -DLRDMC_EXT=0, 1, 2, 3 or 4"
#endif
#if LRDMC_EXT == 0
#define KFN(name) name##_e0
#elif LRDMC_EXT == 1
#define KFN(name) name##_e1
#elif LRDMC_EXT == 2
#define KFN(name) name##_e2
#elif LRDMC_EXT == 3
#define KFN(name) name##_e3
#else
#define KFN(name) name##_e4
#endif
static constexpr int kNL = LRDMC_EXT;
// The extended warp-per-walker kernels exist twice: compiled for LRDMC_WPB warps per CTA (128 registers) and for LRDMC_WPB_EXT (168 registers, no spills);
// a launch of at most LRDMC_WPB_EXT warps takes the second (systems whose per-walker state leaves room for 6 warps per CTA only).
#if LRDMC_EXT >= 1 && LRDMC_EXT <= 3
#define kWs LRDMC_WPB_EXT
#define KSEL(threads, BIG, SMALL) do { if ((threads) <= 32 * LRDMC_WPB_EXT) { SMALL; } else { BIG; } } while (0)
#define KBOTH(BIG, SMALL) do { BIG; SMALL; } while (0)
#else
#define KSEL(threads, BIG, SMALL) do { BIG; } while (0)
#define KBOTH(BIG, SMALL) do { BIG; } while (0)
#endif

#define FOR_EACH_NT_TS(X) X(1, true) X(2, true) X(4, true) X(1, false) X(2, false) X(4, false)
#define PICK(NT_, TS_, STMT)                                                                   \
    do {                                                                                       \
        if (TS_) { if (NT_ == 1) { STMT(1, true); } else if (NT_ == 2) { STMT(2, true); } else { STMT(4, true); } } \
        else { if (NT_ == 1) { STMT(1, false); } else if (NT_ == 2) { STMT(2, false); } else { STMT(4, false); } }   \
    } while (0)

#if !LRDMC_TEAM_TU
void KFN(lrdmc_k_set_smem)(int smem)
{
#define X(NTV, TSV) KBOTH(cudaFuncSetAttribute(k_propagate<NTV, TSV, kNL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                          cudaFuncSetAttribute(k_step_debug<NTV, TSV, kNL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem), \
                          cudaFuncSetAttribute(k_propagate<NTV, TSV, kNL, kWs>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                          cudaFuncSetAttribute(k_step_debug<NTV, TSV, kNL, kWs>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
    FOR_EACH_NT_TS(X)
#undef X
}
int KFN(lrdmc_k_occupancy)(int NT, int ts, int threads, int smem)
{
    int occ = 0;
#define STMT(NTV, TSV) KSEL(threads, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_propagate<NTV, TSV, kNL>, threads, smem), \
                            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_propagate<NTV, TSV, kNL, kWs>, threads, smem))
    PICK(NT, ts, STMT);
#undef STMT
    return occ;
}
void KFN(lrdmc_k_propagate)(int NT, int ts, int grid, int threads, int smem, cudaStream_t st, const DevSys &S, const DevWalk &W, int mode, int n_moves,
                            double tau, double E0, uint32_t cycle)
{
#define STMT(NTV, TSV) KSEL(threads, (k_propagate<NTV, TSV, kNL><<<grid, threads, smem, st>>>(S, W, mode, n_moves, tau, E0, cycle)), \
                            (k_propagate<NTV, TSV, kNL, kWs><<<grid, threads, smem, st>>>(S, W, mode, n_moves, tau, E0, cycle)))
    PICK(NT, ts, STMT);
#undef STMT
}
void KFN(lrdmc_k_step_debug)(int NT, int ts, int grid, int threads, int smem, cudaStream_t st, const DevSys &S, const DevWalk &W, double E0, uint32_t cycle,
                             uint32_t step, double *R_out, double *scal_out, int *jstar_out)
{
#define STMT(NTV, TSV) KSEL(threads, (k_step_debug<NTV, TSV, kNL><<<grid, threads, smem, st>>>(S, W, E0, cycle, step, R_out, scal_out, jstar_out)), \
                            (k_step_debug<NTV, TSV, kNL, kWs><<<grid, threads, smem, st>>>(S, W, E0, cycle, step, R_out, scal_out, jstar_out)))
    PICK(NT, ts, STMT);
#undef STMT
}
#else
int KFN(lrdmc_k_team_occupancy)(int NT, int ts, int threads, int smem)
{
    int occ = 0;
#define STMT(NTV, TSV) cudaFuncSetAttribute(k_propagate_team<NTV, TSV, kNL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem); \
                       cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_propagate_team<NTV, TSV, kNL>, threads, smem)
    PICK(NT, ts, STMT);
#undef STMT
    return occ;
}
void KFN(lrdmc_k_team)(int NT, int ts, int grid, int threads, int smem, cudaStream_t st, const DevSys &S, const DevWalk &W, const TeamPlan &P, int mode,
                       int n_moves, double tau, double E0, uint32_t cycle)
{
#define STMT(NTV, TSV) k_propagate_team<NTV, TSV, kNL><<<grid, threads, smem, st>>>(S, W, P, mode, n_moves, tau, E0, cycle)
    PICK(NT, ts, STMT);
#undef STMT
}
#endif
