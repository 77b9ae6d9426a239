// philox.cuh -- counter-based random numbers and the random lattice frame on the device.
// Philox4x32-10 (Salmon et al., SC'11), written independently of the oracle's copy; the two are compared
// bit for bit in tests (pin P11).  Counter = (walker slot, cycle, step, purpose), key = run seed (readings Q7/Q12).
#pragma once
#include "common.cuh"

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        uint32_t h0 = __umulhi(0xD2511F53u, c.x), l0 = 0xD2511F53u * c.x;
        uint32_t h1 = __umulhi(0xCD9E8D57u, c.z), l1 = 0xCD9E8D57u * c.z;
        c = make_uint4(h1 ^ c.y ^ k0, l1, h0 ^ c.w ^ k1, l0);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}

// top 53 bits of hi:lo, times 2^-53  ->  [0,1)
__device__ __forceinline__ double uniform53(uint32_t lo, uint32_t hi)
{
    unsigned long long v = ((unsigned long long)hi << 32) | lo;
    return (double)(v >> 11) * 1.1102230246251565404e-16;
}

struct StepDraws { double u1, u2, u3, u_sel, u_tau; };

__device__ __forceinline__ StepDraws step_draws(const DevSys &S, uint32_t slot, uint32_t cycle, uint32_t step, bool need_tau)
{
    StepDraws d;
    uint4 o = philox4x32_10(make_uint4(slot, cycle, step, 0u), S.key0, S.key1);
    d.u1 = uniform53(o.x, o.y); d.u2 = uniform53(o.z, o.w);
    o = philox4x32_10(make_uint4(slot, cycle, step, 1u), S.key0, S.key1);
    d.u3 = uniform53(o.x, o.y); d.u_sel = uniform53(o.z, o.w);
    d.u_tau = 0.0;
    if (need_tau) { o = philox4x32_10(make_uint4(slot, cycle, step, 2u), S.key0, S.key1); d.u_tau = uniform53(o.x, o.y); }
    return d;
}

// Haar-uniform rotation from three uniforms through a unit quaternion (L596 "rotate with random angles").
// U row-major, versors = columns.
__device__ __forceinline__ void lattice_frame(double u1, double u2, double u3, double U[9])
{
    double s1 = sqrt(1.0 - u1), s2 = sqrt(u1), sa, ca, sb, cb;
    sincospi(2.0 * u2, &sa, &ca);
    sincospi(2.0 * u3, &sb, &cb);
    double x = s1 * sa, y = s1 * ca, z = s2 * sb, w = s2 * cb;
    U[0] = 1.0 - 2.0 * (y * y + z * z); U[1] = 2.0 * (x * y - z * w);       U[2] = 2.0 * (x * z + y * w);
    U[3] = 2.0 * (x * y + z * w);       U[4] = 1.0 - 2.0 * (x * x + z * z); U[5] = 2.0 * (y * z - x * w);
    U[6] = 2.0 * (x * z - y * w);       U[7] = 2.0 * (y * z + x * w);       U[8] = 1.0 - 2.0 * (x * x + y * y);
}
