// fastmath.cuh -- short FP64 sequences for the hot loop: exp of a non-positive argument, reciprocal, reciprocal
// square root.  The library versions are IEEE-rounded and cost 30-80 SASS instructions each (slow-path calls, constant
// materialisation); the path needs 1e-10, these deliver <= 2 ulp with 6-20 instructions and no branches.
#pragma once
#include <cuda_runtime.h>

// Taylor coefficients 1/k! (k = 2..11) in constant memory: DFMA takes them as c[bank][offset] operands directly.
static __constant__ double c_exp_poly[10] = {
    2.50521083854417187751e-08,  // 1/11!
    2.75573192239858906526e-07,  // 1/10!
    2.75573192239858906526e-06,  // 1/9!
    2.48015873015873015873e-05,  // 1/8!
    1.98412698412698412698e-04,  // 1/7!
    1.38888888888888888889e-03,  // 1/6!
    8.33333333333333333333e-03,  // 1/5!
    4.16666666666666666667e-02,  // 1/4!
    1.66666666666666666667e-01,  // 1/3!
    5.00000000000000000000e-01,  // 1/2!
};

// exp(x) for x <= 0 (Gaussian / Slater radial factors, -tau*e shifts are NOT routed here).  x < -708 -> 0.
// x = k ln2 + r, |r| <= ln2/2;  e^r by the degree-11 Taylor polynomial (|err| < 2e-17 relative);  2^k by exponent arithmetic.
__device__ __forceinline__ double exp_nonpos(double x)
{
    const double magic = 6755399441055744.0;                       // 1.5 * 2^52: rounds x*log2(e) to an integer in the low word
    double t = fma(x, 1.4426950408889634074, magic);
    int k = __double2loint(t);
    double kd = t - magic;
    double r = fma(kd, -6.93147180369123816490e-01, x);            // ln2 hi
    r = fma(kd, -1.90821492927058770002e-10, r);                   // ln2 lo
    double p = c_exp_poly[0];
#pragma unroll
    for (int i = 1; i < 10; ++i) p = fma(p, r, c_exp_poly[i]);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    int hi = __double2hiint(p) + (k << 20);                        // p in [0.70, 1.42): adding k to the exponent stays normal for k >= -1021
    double res = __hiloint2double(hi, __double2loint(p));
    return (x < -708.0) ? 0.0 : res;
}

// exp(x) for -5e6 < x < 708 through a 256-entry table of 2^(j/256) (shared memory, built at init):
//   x = (256 e + j) ln2/256 + r, |r| <= h = ln2/512 = 1.36e-3;  e^r by a cubic: the Taylor cubic with its r^4/24 term
//   economised onto [-h, h] (r^4 ~ h^2 r^2 - h^4/8), |error| < 1.8e-14 relative;  exp(x) = 2^e * tab[j] * e^r.
//   7 FP64 instructions + 6 integer/LDS ones: the AO exponentials are 1/3 of the FP64 work of the path.
// The reduction uses ln2/256 as one double: |error of r| <= |k| 2^-53 ln2/256, i.e. < 5e-15 relative for results above 1e-20.
// Below x = -707.7 the exponent is clamped: the result is then a correct mantissa times 2^-1021 (1e-308, i.e. zero for
// every sum of the path).  The caller keeps x above -5e6 (the integer conversion of x 256/ln2 must not wrap).
#define LRDMC_EXP_XMIN (-4.0e6)
__device__ __forceinline__ double exp_arg_floor(double x) { return (x < LRDMC_EXP_XMIN) ? LRDMC_EXP_XMIN : x; }   // no NaN handling: 3 instructions
__device__ __forceinline__ double exp_tab(double x, const double *__restrict__ etab)
{
    const double magic = 6755399441055744.0;                       // 1.5 * 2^52
    const double t = fma(x, 369.32993046757463228, magic);         // 256 / ln2
    const int k = __double2loint(t);
    const double kd = t - magic;
    const double r = fma(kd, -2.7076061740622863649e-03, x);       // ln2 / 256
    double p = fma(r, 1.66666666666666666667e-01, 0.5000000763659499);
    p = fma(p, r, 1.0);
    p = fma(p, r, 0.9999999999999825);
    int j; asm("and.b32 %0, %1, 255;" : "=r"(j) : "r"(k));         // opaque to the optimiser, or it re-derives the address from k (2 more instructions)
    double tv;                                                     // explicit shared-space load: one LOP3 (j) serves the address and the exponent
    asm("ld.shared.f64 %0, [%1];" : "=d"(tv) : "r"((unsigned)__cvta_generic_to_shared(etab) + 8u * (unsigned)j));
    const double v = tv * p;                                       // in (0.99, 2.01)
    const int kc = max(k, -1021 * 256);                            // clamped: kc - j is no multiple of 256 then, the value is ~1e-308 anyway
    return __hiloint2double(__double2hiint(v) + ((kc - j) << 12), __double2loint(v));
}

// NX exponentials at once, written stage by stage: the NX dependency chains (8-cycle DFMA latency each) are interleaved in
// program order, which is what lets the FP64 pipe take an instruction every 2.2 cycles from ONE warp (measured on B200:
// independent DFMAs of one warp issue every 2.17 cycles, alternating warps only every 3.0).
template <int NX>
__device__ __forceinline__ void exp_tab_n(const double (&x)[NX], double (&out)[NX], const double *__restrict__ etab)
{
    const double magic = 6755399441055744.0;
    const unsigned base = (unsigned)__cvta_generic_to_shared(etab);
    double t[NX], r[NX], p[NX], tv[NX]; int k[NX], j[NX];
#pragma unroll
    for (int i = 0; i < NX; ++i) t[i] = fma(x[i], 369.32993046757463228, magic);
#pragma unroll
    for (int i = 0; i < NX; ++i) { k[i] = __double2loint(t[i]); asm("and.b32 %0, %1, 255;" : "=r"(j[i]) : "r"(k[i])); }
#pragma unroll
    for (int i = 0; i < NX; ++i) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(tv[i]) : "r"(base + 8u * (unsigned)j[i]) : "memory");
#ifndef LRDMC_NO_EXP_FENCE
    __syncwarp();            // scheduling fence: ptxas otherwise sinks each table load to just before its use (29-cycle LDS latency exposed per exponential)
#endif
#pragma unroll
    for (int i = 0; i < NX; ++i) t[i] -= magic;
#pragma unroll
    for (int i = 0; i < NX; ++i) r[i] = fma(t[i], -2.7076061740622863649e-03, x[i]);
#pragma unroll
    for (int i = 0; i < NX; ++i) p[i] = fma(r[i], 1.66666666666666666667e-01, 0.5000000763659499);
#pragma unroll
    for (int i = 0; i < NX; ++i) p[i] = fma(p[i], r[i], 1.0);
#pragma unroll
    for (int i = 0; i < NX; ++i) p[i] = fma(p[i], r[i], 0.9999999999999825);
#pragma unroll
    for (int i = 0; i < NX; ++i) {
        const double v = tv[i] * p[i];
        const int kc = max(k[i], -1021 * 256);
        out[i] = __hiloint2double(__double2hiint(v) + ((kc - j[i]) << 12), __double2loint(v));
    }
}

// 1/a for ordinary positive a (no denormal / inf handling): hardware seed (about 2^-22) + one cubic step.
__device__ __forceinline__ double fast_rcp(double a)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double e = fma(-a, y, 1.0);
    double e2 = fma(e, e, e);
    return fma(y, e2, y);
}

// 1/sqrt(a) for ordinary positive a: hardware seed + one cubic (Halley) step: y (1 + e/2 + 3e^2/8), e = 1 - a y^2.
__device__ __forceinline__ double fast_rsqrt(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    double ay = a * y;
    double e = fma(-ay, y, 1.0);
    double c = fma(0.375, e, 0.5);
    double ye = y * e;
    return fma(ye, c, y);
}
