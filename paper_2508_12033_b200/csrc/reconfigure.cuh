// reconfigure.cuh -- branching at fixed N_w (Eq.15-17) as an integer prefix sum + search, the
// gather of the surviving walkers, and the per-generation reductions of Eq.20 / Eq.34.
//
// Integer form (reading Q21): weights are quantised to u_k = floor(w_k 2^sh), sh = 62 - L - e with max w = f 2^e and
// L = max(1, ceil(log2 N_w)), so the total T < 2^62 is exact; parent[k] = min{ b : P_b N_w 2^32 > (r32 + k 2^32) T } is decided
// in 128-bit integers: the comb Z_k = (xi + k)/N_w of Eq.17 against the cumulative normalised weights (L121), bit-exact.
#pragma once
#include "common.cuh"

struct DevStats {
    double wbar, num, den, busy_ns, span_ns;
    long long moves_min, moves_max, moves_sum, n_node, n_nonpos, n_nonfinite;
    long long n_singular;          // walkers found singular by the last k_rebuild (reading Q24)
    int n_warps, comb_degenerate;
    unsigned long long comb_T;     // total of the quantised weights (k_comb -> k_comb_search)
};

#define COMB_THREADS 1024

// parent[k] = smallest beta with prefix[beta] * (N_w 2^32) > (r32 + k 2^32) * T, in 128-bit integers (Eq.17 against the cumulative weights, L121)
__device__ __forceinline__ int comb_parent(const unsigned long long *prefix, int n_w, uint32_t r32, unsigned long long T, int k)
{
    const unsigned __int128 scale = (unsigned __int128)(unsigned long long)n_w << 32;
    const unsigned __int128 rhs = ((unsigned __int128)r32 + ((unsigned __int128)(unsigned long long)k << 32)) * T;
    int lo = 0, hi = n_w - 1;
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if ((unsigned __int128)prefix[mid] * scale > rhs) hi = mid; else lo = mid + 1;
    }
    return lo;
}

// `search_here`: the comb search runs in this CTA (small ensembles: one launch); otherwise k_comb_search does it on the whole device.
__global__ void __launch_bounds__(COMB_THREADS) k_comb(DevWalk W, uint32_t r32, DevStats *st, int *parents_user, int search_here)
{
    __shared__ double s_max[32];
    __shared__ unsigned long long s_part[COMB_THREADS];
    __shared__ int s_bad;
    const int n_w = W.n_w, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_bad = 0;
    __syncthreads();
    // 1. max weight, validity
    double m = 0.0; int bad = 0;
    for (int k = tid; k < n_w; k += COMB_THREADS) { double v = W.w[k]; if (!(v >= 0.0) || isinf(v)) bad = 1; else m = fmax(m, v); }
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (bad) atomicOr(&s_bad, 1);
    if (lane == 0) s_max[wid] = m;
    __syncthreads();
    m = s_max[0];
    for (int i = 1; i < COMB_THREADS / 32; ++i) m = fmax(m, s_max[i]);
    if (s_bad || !(m > 0.0)) {          // degenerate: identity, wbar = 0
        for (int k = tid; k < n_w; k += COMB_THREADS) { W.parents[k] = k; if (parents_user) parents_user[k] = k; }
        if (tid == 0) { st->wbar = 0.0; st->comb_degenerate = 1; }
        return;
    }
    int e; (void)frexp(m, &e);
    int L = 1; while ((1 << L) < n_w) ++L;
    const int sh = 62 - L - e;
    // 2. quantise + per-thread chunk sums (contiguous chunks keep the scan in index order)
    const int chunk = (n_w + COMB_THREADS - 1) / COMB_THREADS, k0 = tid * chunk, k1 = min(n_w, k0 + chunk);
    unsigned long long local = 0;
    for (int k = k0; k < k1; ++k) { unsigned long long u = (unsigned long long)floor(ldexp(W.w[k], sh)); W.wq[k] = u; local += u; }
    s_part[tid] = local;
    __syncthreads();
    // 3. exclusive scan of the 1024 chunk sums (Hillis-Steele in shared memory; integers: any order is exact)
    for (int off = 1; off < COMB_THREADS; off <<= 1) {
        unsigned long long v = (tid >= off) ? s_part[tid - off] : 0ull;
        __syncthreads();
        s_part[tid] += v;
        __syncthreads();
    }
    unsigned long long run = s_part[tid] - local;
    for (int k = k0; k < k1; ++k) { run += W.wq[k]; W.prefix[k] = run; }
    __syncthreads();
    const unsigned long long T = s_part[COMB_THREADS - 1];
    // 4. comb search
    if (search_here) for (int k = tid; k < n_w; k += COMB_THREADS) {
        const int b = comb_parent(W.prefix, n_w, r32, T, k);
        W.parents[k] = b; if (parents_user) parents_user[k] = b;
    }
    if (tid == 0) { st->wbar = ldexp((double)T, -sh) / (double)n_w; st->comb_degenerate = 0; st->comb_T = T; }   // Eq.16
}

// The comb search of large ensembles, one thread per new slot on the whole device (k_comb left prefix, T and the degenerate flag).
__global__ void k_comb_search(DevWalk W, uint32_t r32, const DevStats *st, int *parents_user)
{
    if (st->comb_degenerate) return;                 // k_comb wrote the identity
    const int n_w = W.n_w; const unsigned long long T = st->comb_T;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_w; k += gridDim.x * blockDim.x) {
        const int b = comb_parent(W.prefix, n_w, r32, T, k);
        W.parents[k] = b; if (parents_user) parents_user[k] = b;
    }
}

// new slot k <- positions of parent[k]; weights <- 1 (L129).  Inverses and caches are rebuilt afterwards (reading Q15),
// so the positions are the whole walker record that has to move.
__global__ void k_gather(DevWalk W, int rec, int mocn)
{
    const size_t total = (size_t)W.n_w * rec;
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        int k = (int)(idx / rec), c = (int)(idx - (size_t)k * rec);
        W.r_alt[idx] = W.r[(size_t)W.parents[k] * rec + c];
        if (c == 0) W.w[k] = 1.0;
    }
    // cached MO rows: functions of the electron positions alone, so the parent's rows are the child's, bit for bit (HBM-bound copy)
    const int m2 = mocn >> 1;                                       // mocn = 5 N OS is even; rows are 16-byte aligned
    const size_t total2 = (size_t)W.n_w * m2;
    const double2 *src = reinterpret_cast<const double2 *>(W.moc); double2 *dst = reinterpret_cast<double2 *>(W.moc_alt);
    for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total2; idx += (size_t)gridDim.x * blockDim.x) {
        int k = (int)(idx / m2), c = (int)(idx - (size_t)k * m2);
        dst[idx] = src[(size_t)W.parents[k] * m2 + c];
    }
}

__global__ void k_copy_back(double *dst, const double *src, size_t n)
{
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = src[i];
}

// per-generation sums (row a11): num = sum omega e_L, den = sum omega (Eq.34 L227 / Eq.20), hop statistics, event
// counters, and the measured busy/span times of the persistent warps (branch idle %).
__global__ void __launch_bounds__(1024) k_reduce_obs(DevWalk W, DevStats *st, int n_warps)
{
    __shared__ double s_d[3][32];
    __shared__ long long s_l[6][32];
    __shared__ unsigned long long s_t[2][32];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    double num = 0.0, den = 0.0, busy = 0.0;
    long long mmin = LLONG_MAX, mmax = 0, msum = 0, nn = 0, np = 0, nf = 0;
    unsigned long long t0 = ~0ull, t1 = 0ull;
    for (int k = tid; k < W.n_w; k += blockDim.x) {
        double om = W.omega[k]; num += om * W.eL[k]; den += om;
        long long mv = W.nmoves[k]; mmin = min(mmin, mv); mmax = max(mmax, mv); msum += mv;
        nn += W.flags[3 * k]; np += W.flags[3 * k + 1]; nf += W.flags[3 * k + 2];
    }
    for (int i = tid; i < n_warps; i += blockDim.x) {
        unsigned long long a = W.timing[2 * i], b = W.timing[2 * i + 1];
        t0 = min(t0, a); t1 = max(t1, b); busy += (double)(b - a);
    }
    for (int o = 16; o > 0; o >>= 1) {
        num += __shfl_xor_sync(0xffffffffu, num, o); den += __shfl_xor_sync(0xffffffffu, den, o); busy += __shfl_xor_sync(0xffffffffu, busy, o);
        mmin = min(mmin, __shfl_xor_sync(0xffffffffu, mmin, o)); mmax = max(mmax, __shfl_xor_sync(0xffffffffu, mmax, o));
        msum += __shfl_xor_sync(0xffffffffu, msum, o); nn += __shfl_xor_sync(0xffffffffu, nn, o);
        np += __shfl_xor_sync(0xffffffffu, np, o); nf += __shfl_xor_sync(0xffffffffu, nf, o);
        t0 = min(t0, __shfl_xor_sync(0xffffffffu, t0, o)); t1 = max(t1, __shfl_xor_sync(0xffffffffu, t1, o));
    }
    if (lane == 0) {
        s_d[0][wid] = num; s_d[1][wid] = den; s_d[2][wid] = busy;
        s_l[0][wid] = mmin; s_l[1][wid] = mmax; s_l[2][wid] = msum; s_l[3][wid] = nn; s_l[4][wid] = np; s_l[5][wid] = nf;
        s_t[0][wid] = t0; s_t[1][wid] = t1;
    }
    __syncthreads();
    if (tid == 0) {
        const int nwp = blockDim.x >> 5;
        for (int i = 1; i < nwp; ++i) {
            num += s_d[0][i]; den += s_d[1][i]; busy += s_d[2][i];
            mmin = min(mmin, s_l[0][i]); mmax = max(mmax, s_l[1][i]); msum += s_l[2][i]; nn += s_l[3][i]; np += s_l[4][i]; nf += s_l[5][i];
            t0 = min(t0, s_t[0][i]); t1 = max(t1, s_t[1][i]);
        }
        st->num = num; st->den = den; st->busy_ns = busy; st->span_ns = (t1 > t0) ? (double)(t1 - t0) : 0.0;
        st->moves_min = mmin; st->moves_max = mmax; st->moves_sum = msum; st->n_node = nn; st->n_nonpos = np; st->n_nonfinite = nf;
        st->n_warps = n_warps;
    }
}
