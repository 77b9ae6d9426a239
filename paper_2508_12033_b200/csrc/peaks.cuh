// peaks.cuh -- FP64 roofline denominators measured on the device itself (MEASURED_PEAKS.json has no FP64 number).
// DFMA: 8 independent FMA chains per thread.  DMMA: 8 independent mma.sync.m8n8k4.f64 accumulator chains per warp.
// MIXED: both interleaved, to see whether the FP64 tensor path and the FP64 ALUs overlap on sm_100a.
#pragma once
#include "wavefunction.cuh"

template <int MODE>   // 0 DFMA, 1 DMMA, 2 both
__global__ void __launch_bounds__(256) k_fp64_peak(double *out, int iters, double seed)
{
    double f[8], c[8][2];
    const double a = seed + threadIdx.x * 1e-9, b = 1.0 - 1e-7;
#pragma unroll
    for (int i = 0; i < 8; ++i) { f[i] = seed * (i + 1); c[i][0] = seed * i; c[i][1] = -seed * i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            if (MODE != 1) f[i] = fma(f[i], b, a);
            if (MODE != 0) dmma884(c[i][0], c[i][1], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += f[i] + c[i][0] + c[i][1];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;   // keep the work alive
}

// DFMA whose three source operands are three DIFFERENT registers in every instruction (no operand-reuse cache hit, no constant
// or immediate operand): the form of most FMAs of a real contraction.  On B200 this issues every 3 cycles per scheduler instead
// of 2 (the register file delivers one 64-bit operand per cycle): 2/3 of the DFMA peak above, whatever the ILP or warp count.
static __global__ void __launch_bounds__(256) k_fp64_peak_3reg(double *out, int iters, double seed)
{
    double f[8], g[8], h[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { f[i] = seed * (i + 1); g[i] = 1.0 - 1e-7 * (i + 1 + threadIdx.x); h[i] = seed * 1e-3 * (i + 2 + threadIdx.x); }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) f[i] = fma(f[i], g[i], h[i]);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += f[i];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// DFMA with ONE source operand shared with the neighbouring DFMAs (acc[i] += g[i] * b: the form of the candidate pass's accumulations, where the
// operand-reuse cache can hold b): between the two cases above -- 2.56 dispatch cycles on B200 against 2.18 (two shared) and 3.11 (none).
static __global__ void __launch_bounds__(256) k_fp64_peak_shared1(double *out, int iters, double seed)
{
    double f[8], g[8];
    const double b = 1.0 - 1e-7 * (1 + threadIdx.x);
#pragma unroll
    for (int i = 0; i < 8; ++i) { f[i] = seed * (i + 1); g[i] = 1e-7 * (i + 1 + threadIdx.x); }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) f[i] = fma(g[i], b, f[i]);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += f[i];
    if (s == 123.456) out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// DFMA (two register operands + a constant: 2 dispatch cycles) interleaved with independent integer ALU work of the same
// warp (an and and an add per DFMA with run-time operands, which the compiler cannot fold): does the other work hide in the FP64 instruction's
// second cycle?  On B200 it does not: the time is the SUM of the dispatch cycles (2 + 1 + 1), see DESIGN.md section 4.
static __global__ void __launch_bounds__(256) k_fp64_peak_alu(double *out, int iters, double seed)
{
    double f[8]; unsigned y[8]; const unsigned m = 0xfff0ff0fu ^ (unsigned)iters, c = 0x9e3779b9u + (unsigned)iters;
    const double a = seed + threadIdx.x * 1e-9, b = 1.0 - 1e-7;
#pragma unroll
    for (int i = 0; i < 8; ++i) { f[i] = seed * (i + 1); y[i] = threadIdx.x * 2654435761u + i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) { f[i] = fma(f[i], b, a); y[i] = (y[i] & m) + c; }
    }
    double s = 0.0; unsigned t = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { s += f[i]; t += y[i]; }
    if (s == 123.456 || t == 77u) out[blockIdx.x * blockDim.x + threadIdx.x] = s + t;
}
