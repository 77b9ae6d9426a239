// lrdmc_aux.cu -- the parts of the C-ABI that sit beside the walker kernels: host-side estimators over generations
// (Eq.18-19), the end-to-end host-buffer driver and the Philox / draws test hooks.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "philox.cuh"
#include "api_internal.h"

// Eq.18 (L127): G_n^p = prod_{j=1..p} wbar_{n-j};  Eq.19 (L131): E = sum_n G_n^p e_n / sum_n G_n^p, e_n = num_n/den_n
// (Eq.20 L135 / Eq.34).  Error bar: delete-one-block jackknife over blocks of consecutive generations (reading Q9).
extern "C" int lrdmc_energy(const lrdmc_cycle_stats *recs, int n, int p, int n_therm, int n_blocks, double *E, double *sigma)
{
    if (!recs || n < 1 || p < 0 || n_therm < 0 || n_therm >= n || !E) return LRDMC_EINVAL;
    const int m = n - n_therm;
    std::vector<double> G(m), e(m);
    for (int i = 0; i < m; ++i) {
        const int gen = n_therm + i;
        double g = 1.0;
        for (int j = 1; j <= p && gen - j >= 0; ++j) g *= recs[gen - j].wbar;
        G[i] = g; e[i] = recs[gen].num / recs[gen].den;
    }
    double sg = 0.0, sge = 0.0;
    for (int i = 0; i < m; ++i) { sg += G[i]; sge += G[i] * e[i]; }
    *E = sge / sg;
    if (sigma) {
        int nb = n_blocks < 2 ? 2 : n_blocks; if (nb > m) nb = m;
        if (nb < 2) { *sigma = 0.0; return LRDMC_OK; }
        std::vector<double> Ej(nb);
        double mean = 0.0;
        for (int b = 0; b < nb; ++b) {
            const int lo = (int)((long long)m * b / nb), hi = (int)((long long)m * (b + 1) / nb);
            double bg = 0.0, bge = 0.0;
            for (int i = lo; i < hi; ++i) { bg += G[i]; bge += G[i] * e[i]; }
            Ej[b] = (sge - bge) / (sg - bg); mean += Ej[b];
        }
        mean /= nb;
        double v = 0.0;
        for (int b = 0; b < nb; ++b) v += (Ej[b] - mean) * (Ej[b] - mean);
        *sigma = sqrt((double)(nb - 1) / nb * v);
    }
    return LRDMC_OK;
}

// Alg.2 lines 2-13 (L398-L420) / Alg.1 with HOST buffers: the end-to-end path a user without device arrays takes.
extern "C" int lrdmc_run_host(lrdmc_ctx *c, const double *r_in, double *r_out, int mode, int n_moves, double tau, double E0,
                              uint64_t first_cycle, int n_cycles, int n_therm, lrdmc_cycle_stats *stats_out, void *stream)
{
    if (!c || !r_in || n_cycles < 0 || n_therm < 0) return LRDMC_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int n_w = lrdmc_bound_walkers(c); if (n_w <= 0) return LRDMC_ESTATE;
    const size_t bytes = sizeof(double) * (size_t)n_w * 3 * lrdmc_n_electrons(c);
    double *d_r = lrdmc_positions_ptr(c, 1);      // the gather target doubles as the H2D staging area (no allocation here)
    int rc = LRDMC_OK;
    if (cudaMemcpyAsync(d_r, r_in, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = LRDMC_ECUDA;
    if (!rc) rc = lrdmc_set_positions(c, d_r, st);
    double esum = 0.0; int ecnt = 0;
    for (int i = 0; i < n_cycles && !rc; ++i) {
        lrdmc_cycle_stats s;
        rc = lrdmc_propagate(c, mode, n_moves, tau, E0, first_cycle + i, st);
        if (!rc) rc = lrdmc_reconfigure(c, first_cycle + i, NULL, st);
        if (!rc) rc = lrdmc_estimators(c, &s);
        if (rc) break;
        if (stats_out) stats_out[i] = s;
        if (i == n_therm && n_therm > 0) { esum = 0.0; ecnt = 0; } // the running mean restarts once after the equilibration (reading Q8a)
        esum += s.num / s.den; ++ecnt;
        if (mode == LRDMC_BALANCED) E0 = esum / ecnt;             // "Update E_0" (Alg.2 line 12 L418; reading Q8a)
    }
    if (!rc && r_out) {
        if (cudaMemcpyAsync(r_out, lrdmc_positions_ptr(c, 0), bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = LRDMC_ECUDA;
    }
    cudaStreamSynchronize(st);
    return rc;
}

__global__ void k_philox_debug(const uint32_t *ctr, uint32_t k0, uint32_t k1, uint32_t *out, int n)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint4 o = philox4x32_10(make_uint4(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3]), k0, k1);
    out[4 * i] = o.x; out[4 * i + 1] = o.y; out[4 * i + 2] = o.z; out[4 * i + 3] = o.w;
}

extern "C" int lrdmc_debug_philox(const uint32_t *ctr_dev, uint32_t key0, uint32_t key1, uint32_t *out_dev, int n, void *stream)
{
    if (!ctr_dev || !out_dev || n < 1) return LRDMC_EINVAL;
    k_philox_debug<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(ctr_dev, key0, key1, out_dev, n);
    return cudaGetLastError() == cudaSuccess ? LRDMC_OK : LRDMC_ECUDA;
}

// Also expose the frame construction and uniforms for parity tests of row a0: out [n][14] = u1,u2,u3,u_sel,u_tau, U[9]
__global__ void k_draws_debug(DevSys S, uint32_t cycle, uint32_t step, double *out, int n)
{
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    StepDraws d = step_draws(S, (uint32_t)k, cycle, step, true);
    double U[9]; lattice_frame(d.u1, d.u2, d.u3, U);
    double *o = out + 14 * (size_t)k;
    o[0] = d.u1; o[1] = d.u2; o[2] = d.u3; o[3] = d.u_sel; o[4] = d.u_tau;
    for (int i = 0; i < 9; ++i) o[5 + i] = U[i];
}
extern "C" int lrdmc_debug_draws(const lrdmc_ctx *c, uint64_t cycle, uint64_t step, double *out_dev, int n, void *stream)
{
    if (!c || !out_dev || n < 1) return LRDMC_EINVAL;
    k_draws_debug<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(*lrdmc_devsys(c), (uint32_t)cycle, (uint32_t)step, out_dev, n);
    return cudaGetLastError() == cudaSuccess ? LRDMC_OK : LRDMC_ECUDA;
}
