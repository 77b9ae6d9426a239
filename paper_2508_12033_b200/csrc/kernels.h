// kernels.h -- launchers of the walker kernels (kernels.cu, compiled once per EXT in {0: lattice only, 1: non-local slots, 2: three-body
// Jastrow, 3: both, 4: lattice only as a listed sweep on stored Bc} x {warp-per-walker, team});
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
LRDMC_K_DECL(e0)
LRDMC_K_DECL(e1)
LRDMC_K_DECL(e2)
LRDMC_K_DECL(e3)
LRDMC_K_DECL(e4)
#undef LRDMC_K_DECL
// dispatch on the run-time EXT value of a system
#define LRDMC_K_CALL(ext, name, ...) ((ext) == 0 ? name##_e0(__VA_ARGS__) : (ext) == 1 ? name##_e1(__VA_ARGS__) : (ext) == 2 ? name##_e2(__VA_ARGS__) : (ext) == 3 ? name##_e3(__VA_ARGS__) : name##_e4(__VA_ARGS__))
