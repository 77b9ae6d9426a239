// lrdmc_aux.cu -- the parts of the C-ABI that sit beside the walker kernels: host-side estimators over generations
// (Eq.18-19), the end-to-end host-buffer driver, the FP64 peak micro-benchmarks and the Philox test hook.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "common.cuh"
#include "philox.cuh"
#include "peaks.cuh"
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
                              uint64_t first_cycle, int n_cycles, lrdmc_cycle_stats *stats_out, void *stream)
{
    if (!c || !r_in || n_cycles < 0) return LRDMC_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int n_w = lrdmc_bound_walkers(c); if (n_w <= 0) return LRDMC_ESTATE;
    const size_t bytes = sizeof(double) * (size_t)n_w * 3 * lrdmc_n_electrons(c);
    double *d_r = lrdmc_positions_ptr(c, 1);      // the gather target doubles as the H2D staging area (no allocation here)
    int rc = LRDMC_OK;
    if (cudaMemcpyAsync(d_r, r_in, bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) rc = LRDMC_ECUDA;
    if (!rc) rc = lrdmc_set_positions(c, d_r, st);
    double esum = 0.0;
    for (int i = 0; i < n_cycles && !rc; ++i) {
        lrdmc_cycle_stats s;
        rc = lrdmc_propagate(c, mode, n_moves, tau, E0, first_cycle + i, st);
        if (!rc) rc = lrdmc_reconfigure(c, first_cycle + i, NULL, st);
        if (!rc) rc = lrdmc_estimators(c, &s);
        if (rc) break;
        if (stats_out) stats_out[i] = s;
        esum += s.num / s.den;
        if (mode == LRDMC_BALANCED) E0 = esum / (i + 1);          // "Update E_0" (Alg.2 line 12 L418; reading Q8a)
    }
    if (!rc && r_out) {
        if (cudaMemcpyAsync(r_out, lrdmc_positions_ptr(c, 0), bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = LRDMC_ECUDA;
    }
    cudaStreamSynchronize(st);
    return rc;
}

extern "C" int lrdmc_measure_fp64_peaks(double *dfma, double *dmma, double *mixed)
{
    int dev = 0; cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return LRDMC_ECUDA;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 8192;
    double *d_out = NULL; if (cudaMalloc((void **)&d_out, sizeof(double) * blocks * threads) != cudaSuccess) return LRDMC_ECUDA;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    double res[3] = { 0, 0, 0 };
    for (int mode = 0; mode < 3; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) k_fp64_peak<0><<<blocks, threads>>>(d_out, iters, 1.000001);
            else if (mode == 1) k_fp64_peak<1><<<blocks, threads>>>(d_out, iters, 1.000001);
            else k_fp64_peak<2><<<blocks, threads>>>(d_out, iters, 1.000001);
            cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double threads_total = (double)blocks * threads, warps = threads_total / 32.0;
        const double fl_fma = threads_total * iters * 8.0 * 2.0, fl_mma = warps * iters * 8.0 * 512.0;
        const double fl = mode == 0 ? fl_fma : (mode == 1 ? fl_mma : fl_fma + fl_mma);
        res[mode] = fl / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (cudaGetLastError() != cudaSuccess) return LRDMC_ECUDA;
    if (dfma) *dfma = res[0]; if (dmma) *dmma = res[1]; if (mixed) *mixed = res[2];
    return LRDMC_OK;
}

extern "C" int lrdmc_measure_fp64_operand_peak(double *dfma3, double *dfma_alu)
{
    int dev = 0; cudaDeviceProp prop;
    if (!dfma3 || cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return LRDMC_ECUDA;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 8192;
    double *d_out = NULL; if (cudaMalloc((void **)&d_out, sizeof(double) * blocks * threads) != cudaSuccess) return LRDMC_ECUDA;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    double res[2] = { 0, 0 };
    for (int mode = 0; mode < 2; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) k_fp64_peak_3reg<<<blocks, threads>>>(d_out, iters, 1.000001);
            else k_fp64_peak_alu<<<blocks, threads>>>(d_out, iters, 1.000001);
            cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        res[mode] = (double)blocks * threads * iters * 8.0 * 2.0 / (best * 1e-3) / 1e12;      // FP64 flop only
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (cudaGetLastError() != cudaSuccess) return LRDMC_ECUDA;
    *dfma3 = res[0]; if (dfma_alu) *dfma_alu = res[1];
    return LRDMC_OK;
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
