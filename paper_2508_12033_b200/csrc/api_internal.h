// api_internal.h -- accessors shared by the two translation units of liblrdmc (not part of the public C-ABI header)
#pragma once
#include "common.cuh"
extern "C" {
int lrdmc_bound_walkers(const lrdmc_ctx *);   // n_w of the bound buffer, 0 if none
int lrdmc_n_electrons(const lrdmc_ctx *);
const DevSys *lrdmc_devsys(const lrdmc_ctx *);
double *lrdmc_positions_ptr(const lrdmc_ctx *, int which); // 0: current positions, 1: gather target / staging
int lrdmc_launch_count(const lrdmc_ctx *);
int lrdmc_launch_config(const lrdmc_ctx *, int *grid, int *block, int *smem_bytes, int *ctas_per_sm);
int lrdmc_debug_draws(const lrdmc_ctx *, uint64_t cycle, uint64_t step, double *out_dev, int n, void *stream);
}
