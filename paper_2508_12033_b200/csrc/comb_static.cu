// comb_static.cu -- lrdmc_comb_static: the integer comb of the branching step (Eq.15-17, reading Q21) as an entry
// point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that
// forbid it).  A variant of k_comb (reconfigure.cuh): same arithmetic, but the workspace of the prefix sum -- the quantised weights and their
// running totals, which lrdmc_reconfigure keeps in the caller's walker buffer -- is a file-scope device array of a fixed maximum size.
//
// The array lives in every GPU that loads liblrdmc.so, from module load to exit (LRDMC_COMB_STATIC_MAX_WALKERS x 16 bytes = 1 MiB).  All
// calls share it: calls that overlap on the GPU (two streams, two host threads) race.  Nothing in it has to start at zero: each call writes
// entries [0, n_w) of both halves before it reads them and never reads beyond n_w, so what the last call left is harmless.
//
// In host code `g_comb_scratch` is a host-side stand-in, not a device address; the address the kernel gets comes from
// cudaGetSymbolAddress, asked once per device with that device current (comb_scratch_ptr).
#include <cmath>
#include <cstdio>
#include <cstdint>
#include <mutex>

#include <cuda_runtime.h>
#include "../../include/lrdmc.h"

#define CS_THREADS 1024
#define CS_MAX LRDMC_COMB_STATIC_MAX_WALKERS
#define CS_MAX_DEVICES 64

// [0, CS_MAX): u_k = floor(w_k 2^sh); [CS_MAX, 2 CS_MAX): P_k = u_0 + ... + u_k
static __device__ __align__(256) unsigned long long g_comb_scratch[2 * CS_MAX];

// parent[k] = smallest beta with P_beta * (N_w 2^32) > (r32 + k 2^32) * T in 128-bit integers: the comb Z_k = (xi + k)/N_w of Eq.17 against
// the cumulative normalised weights (L121), xi = r32 / 2^32
__device__ __forceinline__ int cs_parent(const unsigned long long *prefix, int n_w, uint32_t r32, unsigned long long T, int k)
{
    const unsigned __int128 scale = (unsigned __int128)(unsigned long long)n_w << 32;
    const unsigned __int128 rhs = ((unsigned __int128)r32 + ((unsigned __int128)(unsigned long long)k << 32)) * T;
    int lo = 0, hi = n_w - 1;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if ((unsigned __int128)prefix[mid] * scale > rhs) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// One CTA: max weight -> shift, quantise, prefix sum in index order, comb search.  `scr` is the device address of g_comb_scratch.
__global__ void __launch_bounds__(CS_THREADS) k_comb_static(const double *__restrict__ w, int n_w, uint32_t r32, unsigned long long *scr,
                                                            int *__restrict__ parents, double *wbar)
{
    __shared__ double s_max[32];
    __shared__ unsigned long long s_part[CS_THREADS];
    __shared__ int s_bad;
    unsigned long long *wq = scr, *prefix = scr + CS_MAX;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_bad = 0;
    __syncthreads();
    double m = 0.0; int bad = 0;
    for (int k = tid; k < n_w; k += CS_THREADS) { const double v = w[k]; if (!(v >= 0.0) || isinf(v)) bad = 1; else m = fmax(m, v); }
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (bad) atomicOr(&s_bad, 1);
    if (lane == 0) s_max[wid] = m;
    __syncthreads();
    m = s_max[0];
    for (int i = 1; i < CS_THREADS / 32; ++i) m = fmax(m, s_max[i]);
    if (s_bad || !(m > 0.0)) {                    // a negative / non-finite weight, or all zero: identity, wbar = 0 (as k_comb)
        for (int k = tid; k < n_w; k += CS_THREADS) parents[k] = k;
        if (tid == 0 && wbar) *wbar = 0.0;
        return;
    }
    int e; (void)frexp(m, &e);
    int L = 1; while ((1 << L) < n_w) ++L;
    const int sh = 62 - L - e;                    // max w = f 2^e: every u_k < 2^(62-L), the total T < 2^62 is exact
    const int chunk = (n_w + CS_THREADS - 1) / CS_THREADS, k0 = tid * chunk, k1 = min(n_w, k0 + chunk);
    unsigned long long local = 0;
    for (int k = k0; k < k1; ++k) { const unsigned long long u = (unsigned long long)floor(ldexp(w[k], sh)); wq[k] = u; local += u; }
    s_part[tid] = local;
    __syncthreads();
    for (int off = 1; off < CS_THREADS; off <<= 1) {          // inclusive scan of the chunk sums (integers: any order is exact)
        const unsigned long long v = (tid >= off) ? s_part[tid - off] : 0ull;
        __syncthreads();
        s_part[tid] += v;
        __syncthreads();
    }
    unsigned long long run = s_part[tid] - local;
    for (int k = k0; k < k1; ++k) { run += wq[k]; prefix[k] = run; }
    __syncthreads();                              // one CTA: the prefix written above is visible to every thread below
    const unsigned long long T = s_part[CS_THREADS - 1];
    for (int k = tid; k < n_w; k += CS_THREADS) parents[k] = cs_parent(prefix, n_w, r32, T, k);
    if (tid == 0 && wbar) *wbar = ldexp((double)T, -sh) / (double)n_w;      // Eq.16
}

static thread_local char t_err[256] = "";

extern "C" const char *lrdmc_comb_static_error(void) { return t_err; }

// device address of g_comb_scratch on the CURRENT device, asked once per device
static unsigned long long *comb_scratch_ptr(void)
{
    static std::mutex mu;
    static unsigned long long *ptr[CS_MAX_DEVICES];
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= CS_MAX_DEVICES) {
        snprintf(t_err, sizeof t_err, "lrdmc_comb_static: cudaGetDevice: %s (device %d)", cudaGetErrorString(e), dev);
        return NULL;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!ptr[dev]) {
        unsigned long long *p = NULL;
        e = cudaGetSymbolAddress((void **)&p, g_comb_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(t_err, sizeof t_err, "lrdmc_comb_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
            return NULL;
        }
        ptr[dev] = p;
    }
    return ptr[dev];
}

extern "C" int lrdmc_comb_static_setup(void)
{
    t_err[0] = 0;
    return comb_scratch_ptr() ? LRDMC_OK : LRDMC_ECUDA;
}

extern "C" int lrdmc_comb_static(const double *w_dev, int n_walkers, uint64_t seed, uint64_t cycle, int32_t *parents_dev, double *wbar_dev,
                                 void *stream)
{
    t_err[0] = 0;
    if (!w_dev || !parents_dev || n_walkers < 1 || cycle > 0xFFFFFFFFull) {
        snprintf(t_err, sizeof t_err, "lrdmc_comb_static: bad argument (w_dev, parents_dev non-NULL; n_walkers >= 1; cycle < 2^32)");
        return LRDMC_EINVAL;
    }
    if (n_walkers > CS_MAX) {
        snprintf(t_err, sizeof t_err, "lrdmc_comb_static: n_walkers = %d exceeds LRDMC_COMB_STATIC_MAX_WALKERS = %d (the static scratch "
                 "array); use lrdmc_reconfigure", n_walkers, CS_MAX);
        return LRDMC_EINVAL;
    }
    unsigned long long *scr = comb_scratch_ptr();
    if (!scr) return LRDMC_ECUDA;
    // comb random number: Philox4x32-10 block of counter (0xFFFFFFFF, cycle, 0, 3) under the run seed, word 0 (as lrdmc_reconfigure)
    uint32_t c[4] = { 0xFFFFFFFFu, (uint32_t)cycle, 0u, 3u }, k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c[0], p1 = (uint64_t)0xCD9E8D57u * c[2];
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0, n1 = (uint32_t)p1, n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1, n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3; k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    k_comb_static<<<1, CS_THREADS, 0, (cudaStream_t)stream>>>(w_dev, n_walkers, c[0], scr, parents_dev, wbar_dev);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { snprintf(t_err, sizeof t_err, "lrdmc_comb_static: launch: %s", cudaGetErrorString(e)); return LRDMC_ECUDA; }
    return LRDMC_OK;
}
