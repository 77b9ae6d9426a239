// kernels.h -- launchers of the walker kernels (kernels.cu, compiled once per {lattice-only, non-local} x {warp-per-walker, team});
// internal to liblrdmc, not part of the C-ABI.
#pragma once
#include "common.cuh"

#define LRDMC_K_DECL(sfx)                                                                                                                     \
    void lrdmc_k_set_smem_##sfx(int smem);                                                                                                    \
    int lrdmc_k_occupancy_##sfx(int NT, int ts, int threads, int smem);                                                                       \
    void lrdmc_k_propagate_##sfx(int NT, int ts, int grid, int threads, int smem, cudaStream_t st, const DevSys &S, const DevWalk &W, int mode, \
                                 int n_moves, double tau, double E0, uint32_t cycle);                                                         \
    void lrdmc_k_step_debug_##sfx(int NT, int ts, int grid, int threads, int smem, cudaStream_t st, const DevSys &S, const DevWalk &W, double E0, \
                                  uint32_t cycle, uint32_t step, double *R_out, double *scal_out, int *jstar_out);                            \
    int lrdmc_k_team_occupancy_##sfx(int NT, int ts, int threads, int smem);                                                                  \
    void lrdmc_k_team_##sfx(int NT, int ts, int grid, int threads, int smem, cudaStream_t st, const DevSys &S, const DevWalk &W,               \
                            const TeamPlan &P, int mode, int n_moves, double tau, double E0, uint32_t cycle);
LRDMC_K_DECL(lat)
LRDMC_K_DECL(nl)
#undef LRDMC_K_DECL
