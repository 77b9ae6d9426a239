// api_internal.h -- accessors shared by the two translation units of liblrdmc (not part of the public C-ABI header)
#pragma once
#include "common.cuh"
extern "C" {
int lrdmc_bound_walkers(const lrdmc_ctx *);   // n_w of the bound buffer, 0 if none
int lrdmc_n_electrons(const lrdmc_ctx *);
const DevSys *lrdmc_devsys(const lrdmc_ctx *);
double *lrdmc_positions_ptr(const lrdmc_ctx *, int which); // 0: current positions, 1: gather target / staging
}
