// probe.cu -- liblrdmc_probe.so (include/lrdmc_probe.h): FP64 peak micro-benchmarks for bench.py's roofline denominators.
// A library of its own: the product library liblrdmc.so carries no measurement code.
#include <cuda_runtime.h>
#include "peaks.cuh"
#include "../../include/lrdmc_probe.h"

extern "C" int lrdmc_measure_fp64_peaks(double *dfma, double *dmma, double *mixed)
{
    int dev = 0; cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return -4;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 8192;
    double *d_out = NULL; if (cudaMalloc((void **)&d_out, sizeof(double) * blocks * threads) != cudaSuccess) return -4;
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
    if (cudaGetLastError() != cudaSuccess) return -4;
    if (dfma) *dfma = res[0]; if (dmma) *dmma = res[1]; if (mixed) *mixed = res[2];
    return 0;
}

static int operand_peaks(double *dfma3, double *dfma_alu, double *dfma_shared1)
{
    int dev = 0; cudaDeviceProp prop;
    if (!dfma3 || cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return -4;
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 8192;
    double *d_out = NULL; if (cudaMalloc((void **)&d_out, sizeof(double) * blocks * threads) != cudaSuccess) return -4;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    double res[3] = { 0, 0, 0 };
    for (int mode = 0; mode < 3; ++mode) {
        float best = 1e30f;
        for (int rep = 0; rep < 5; ++rep) {
            cudaEventRecord(e0);
            if (mode == 0) k_fp64_peak_3reg<<<blocks, threads>>>(d_out, iters, 1.000001);
            else if (mode == 1) k_fp64_peak_alu<<<blocks, threads>>>(d_out, iters, 1.000001);
            else k_fp64_peak_shared1<<<blocks, threads>>>(d_out, iters, 1.000001);
            cudaEventRecord(e1); cudaEventSynchronize(e1);
            float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        res[mode] = (double)blocks * threads * iters * 8.0 * 2.0 / (best * 1e-3) / 1e12;      // FP64 flop only
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d_out);
    if (cudaGetLastError() != cudaSuccess) return -4;
    *dfma3 = res[0]; if (dfma_alu) *dfma_alu = res[1]; if (dfma_shared1) *dfma_shared1 = res[2];
    return 0;
}
extern "C" int lrdmc_measure_fp64_operand_peak(double *dfma3, double *dfma_alu) { return operand_peaks(dfma3, dfma_alu, NULL); }
extern "C" int lrdmc_measure_fp64_shared_operand_peak(double *dfma_shared1) { double t; return operand_peaks(&t, NULL, dfma_shared1); }

