// wavefunction.cuh -- AO evaluation fused with the AO->MO contraction on the FP64 tensor pipe.
//
// Rows a2/a3 of the scope table.  One warp evaluates 8 points at a time:
//   lane = 4*g + t :  g = point (mma row), t = which of 4 concurrently processed shells (mma k slot).
// Each lane computes exp(-zeta |r_g - R_c|^2) of ITS shell at ITS point once (no redundant exponentials) and feeds the
// AO values of that shell straight into mma.sync.m8n8k4.f64 as the A fragment (A[g][t]); the B fragment
// B[t][n] = norm * C[ao(shell t, component)][n] comes pre-swizzled from the table built at init (conflict-free, 256 B per
// warp load).  The contraction index k of the mma is just "which (shell, component)", so shells are sorted by type and
// padded to multiples of 4 -- all four k slots always run the same code.  Accumulator: lane holds MO (2t, 2t+1) of point g.
#pragma once
#include "common.cuh"
#include "fastmath.cuh"
#ifndef LRDMC_COMPACT_COLUMNS
#if defined(LRDMC_EXT) && (LRDMC_EXT == 1 || LRDMC_EXT == 2 || LRDMC_EXT == 3)
#define LRDMC_COMPACT_COLUMNS 1
#else
#define LRDMC_COMPACT_COLUMNS 0
#endif
#endif

// Table element load with an explicit address space.  TS: the tables sit in shared memory (plain load, inferred LDS).
// !TS: global memory -- spelled as ld.global.nc, because nvcc 12.9 otherwise infers "shared" for the fragment pointer of the
// inlined passes (cvta.to.shared + ld.shared on a global address: illegal access; seen in PTX, found by the C5 parity test).
template <bool TS> __device__ __forceinline__ double ldt(const double *p) { return TS ? *p : __ldg(p); }

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Derivative pass: the 8 mma rows of a lane group g = lane / 4 are 8 COMPONENTS of the cartesian primitive x^l y^m z^n e^{-z r^2} at ONE point:
//   g = 0 value, 1..3 d/dx, d/dy, d/dz, 4..6 d2/dx2, d2/dy2, d2/dz2 (their sum is the Laplacian: mo_pass adds rows 5 and 6 to row 4 at the end), 7 zero.
// Every row is ONE product of per-axis factors: the plain monomial v^k on two axes and, on the lane's SPECIAL axis, its first or second
// derivative with the Gaussian's contribution,
//   d/dv [v^k e^{-z v^2}] = (k v^{k-1} - 2 z v^{k+1}) e ,  d2/dv2 = (k(k-1) v^{k-2} - 2 z (2k+1) v^k + 4 z^2 v^{k+2}) e .
// So a lane selects its three factor arrays once per shell and spends two multiplications per AO component -- no per-component selects, and the
// three second derivatives are formed by the otherwise idle rows 4-6 instead of by every lane (round 2: 1.58 k -> 1.0 k instructions per move).
struct DerivSel { int axis, fam; double on; };      // special axis (0 x, 1 y, 2 z; -1 none), family 1 / 2 (first / second derivative), 0 for the zero row
__device__ __forceinline__ DerivSel deriv_sel(int g)
{
    DerivSel d; d.axis = (g >= 1 && g <= 6) ? (g - 1) % 3 : -1; d.fam = g <= 3 ? 1 : 2; d.on = g == 7 ? 0.0 : 1.0;
    return d;
}
template <int KMAX>
__device__ __forceinline__ void deriv_axes(const DerivSel &q, double dx, double dy, double dz, double z, double (&ax)[KMAX + 1], double (&ay)[KMAX + 1],
                                           double (&az)[KMAX + 1])
{
    const double u = q.axis == 1 ? dy : (q.axis == 2 ? dz : dx), u2 = u * u, tz = 2.0 * z, fz2 = tz * tz;
    double sp[KMAX + 1], fx[KMAX + 1], fy[KMAX + 1], fz[KMAX + 1];
    sp[0] = q.fam == 1 ? -tz * u : fma(fz2, u2, -tz);
    fx[0] = 1.0; fy[0] = 1.0; fz[0] = 1.0;
    if (KMAX >= 1) { sp[1] = q.fam == 1 ? fma(-tz, u2, 1.0) : fma(fz2, u2, -3.0 * tz) * u; fx[1] = dx; fy[1] = dy; fz[1] = dz; }
    if (KMAX >= 2) { sp[2] = q.fam == 1 ? u * fma(-tz, u2, 2.0) : fma(u2, fma(fz2, u2, -5.0 * tz), 2.0); fx[2] = dx * dx; fy[2] = dy * dy; fz[2] = dz * dz; }
#pragma unroll
    for (int k = 0; k <= KMAX; ++k) { ax[k] = q.axis == 0 ? sp[k] : fx[k]; ay[k] = q.axis == 1 ? sp[k] : fy[k]; az[k] = q.axis == 2 ? sp[k] : fz[k]; }
}

// One pass over the whole (sorted, padded) shell list for the 8 points held by the warp.
// DERIV = false: A fragment = AO value (candidate evaluation, row a2/a3).
// DERIV = true : the 8 mma rows are 8 COMPONENTS (value, d/dx, d/dy, d/dz, Laplacian, 0,0,0) of ONE point, selector g = lane/4.
// PART (team mode): only the 4-shell iterations [part->lo[g], part->hi[g]) of each group g; the partial sums of the parts add up.
template <int NT, bool DERIV, bool TS, bool PART = false>
__device__ __forceinline__ void mo_pass(const DevSys &S, const double *__restrict__ shells, const double *__restrict__ bf, const double *__restrict__ etab,
                                        double px, double py, double pz, int lane, double (&acc)[NT][2],
                                        const TeamPlan *tp = nullptr, const ShellPart *part = nullptr)
{
#define LRDMC_MO_RANGE(G, NC)                                                                   \
    const int n_ = PART ? part->hi[G] : S.n_it[G]; int it = PART ? part->lo[G] : 0;             \
    if (PART) { sh4 = reinterpret_cast<const double4 *>(shells) + t + 4 * (tp->it_base[G] + it); b = bf + lane + (size_t)(tp->kstep_base[G] + NC * it) * NT * 32; }
    const int t = lane & 3, g = lane >> 2;
    const DerivSel dq = deriv_sel(g);
    const double4 *sh4 = reinterpret_cast<const double4 *>(shells) + t;
    const double *b = bf + lane;
#pragma unroll
    for (int nt = 0; nt < NT; ++nt) { acc[nt][0] = 0.0; acc[nt][1] = 0.0; }
#define LRDMC_FEED(aval)                                                                        \
    {                                                                                           \
        double a_ = (aval);                                                                     \
        _Pragma("unroll") for (int nt = 0; nt < NT; ++nt) dmma884(acc[nt][0], acc[nt][1], a_, ldt<TS>(b + nt * 32)); \
        b += NT * 32;                                                                           \
    }
    // ---- group 0: Slater-type s, chi = exp(-z r); grad = -z chi rhat; lap = chi (z^2 - 2 z / r)
    { LRDMC_MO_RANGE(0, 1) for (; it < n_; ++it, sh4 += 4) {
        double4 s = *sh4; double dx = px - s.x, dy = py - s.y, dz = pz - s.z, z = s.w;
        double r = sqrt(dx * dx + dy * dy + dz * dz), e = exp_tab(exp_arg_floor(-z * r), etab);
        if (!DERIV) { LRDMC_FEED(e); }
        else {
            double ir = 1.0 / r, d = (g == 1) ? dx : ((g == 2) ? dy : dz);
            double v = (g == 0) ? e : ((g == 4) ? e * (z * z - 2.0 * z * ir) : -z * e * d * ir);
            LRDMC_FEED((g > 4) ? 0.0 : v);
        }
    } }
    // ---- group 1: s Gaussians
    { LRDMC_MO_RANGE(1, 1) for (; it < n_; ++it, sh4 += 4) {
        double4 s = *sh4; double dx = px - s.x, dy = py - s.y, dz = pz - s.z, z = s.w;
        double e = exp_tab(exp_arg_floor(-z * (dx * dx + dy * dy + dz * dz)), etab);
        if (!DERIV) { LRDMC_FEED(e); }
        else { double ax[1], ay[1], az[1]; deriv_axes<0>(dq, dx, dy, dz, z, ax, ay, az); LRDMC_FEED(ax[0] * ay[0] * (az[0] * (e * dq.on))); }
    } }
    // ---- group 2: p Gaussians (x, y, z)
    { LRDMC_MO_RANGE(2, 3) for (; it < n_; ++it, sh4 += 4) {
        double4 s = *sh4; double dx = px - s.x, dy = py - s.y, dz = pz - s.z, z = s.w;
        double e = exp_tab(exp_arg_floor(-z * (dx * dx + dy * dy + dz * dz)), etab);
        if (!DERIV) { LRDMC_FEED(dx * e); LRDMC_FEED(dy * e); LRDMC_FEED(dz * e); }
        else {
            double ax[2], ay[2], az[2]; deriv_axes<1>(dq, dx, dy, dz, z, ax, ay, az);
            const double eo = e * dq.on, yz = ay[0] * az[0] * eo;
            LRDMC_FEED(ax[1] * yz); LRDMC_FEED(ax[0] * (ay[1] * (az[0] * eo))); LRDMC_FEED(ax[0] * (ay[0] * (az[1] * eo)));
        }
    } }
    // ---- group 3: d Gaussians (xx, xy, xz, yy, yz, zz)
    { LRDMC_MO_RANGE(3, 6) for (; it < n_; ++it, sh4 += 4) {
        double4 s = *sh4; double dx = px - s.x, dy = py - s.y, dz = pz - s.z, z = s.w;
        double e = exp_tab(exp_arg_floor(-z * (dx * dx + dy * dy + dz * dz)), etab);
        if (!DERIV) {
            double xe = dx * e, ye = dy * e, ze = dz * e;
            LRDMC_FEED(dx * xe); LRDMC_FEED(dx * ye); LRDMC_FEED(dx * ze); LRDMC_FEED(dy * ye); LRDMC_FEED(dy * ze); LRDMC_FEED(dz * ze);
        } else {
            double ax[3], ay[3], az[3]; deriv_axes<2>(dq, dx, dy, dz, z, ax, ay, az);
            const double eo = e * dq.on, x0 = ax[0] * eo, x1 = ax[1] * eo;
            LRDMC_FEED(ax[2] * eo * (ay[0] * az[0])); LRDMC_FEED(x1 * (ay[1] * az[0])); LRDMC_FEED(x1 * (ay[0] * az[1]));
            LRDMC_FEED(x0 * (ay[2] * az[0])); LRDMC_FEED(x0 * (ay[1] * az[1])); LRDMC_FEED(x0 * (ay[0] * az[2]));
        }
    } }
    if (DERIV) {                          // rows 4, 5, 6 hold the three second derivatives: their sum, the Laplacian, goes to row 4
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
            for (int c = 0; c < 2; ++c) {
                const double s2 = __shfl_down_sync(0xffffffffu, acc[nt][c], 4) + __shfl_down_sync(0xffffffffu, acc[nt][c], 8);
                if (g == 4) acc[nt][c] += s2;
            }
        }
    }
#undef LRDMC_MO_RANGE
#undef LRDMC_FEED
}

// ---- candidate ratios in column form (rows a2-a4 fused) -----------------------------------------------------------
// The determinant ratio of candidate p (electron i moved to r'_p) needs ONE linear combination of the MOs at r'_p:
//     sum_m phi_m(r'_p) Dinv[m][i]  =  sum_mu chi_mu(r'_p) Bc[mu][i],      Bc = C Dinv   (A x n_s),
// so the warp forms the entries of Bc it needs once per evaluation (2 A n_s^2 flop per spin) and contracts every AO value
// with one number (2 P A flop) instead of with n_s MO coefficients (2 P A n_s flop through the MOs).
// Lane = 4 g + t: row g = electron il of the current block of 8 same-spin electrons, t = shell slot of the current
// 4-shell group.  The lane builds Bc[ao(shell t, component c)][electron g] from the same fragment table the tensor-core
// pass uses -- exactly the entries it consumes, nothing is exchanged between lanes -- and handles all six displaced
// points r_i +- a e_k of its electron:  |r_i +- a e_k - R|^2 = |d0|^2 + a^2 +- 2 a e_k.d0  (d0 = r_i - R) shares the
// centre distance and three dot products between the six exponent arguments.
//   av[k] = a e_k (displacement of direction +k), a2 = a^2;  acc[d], d = 2k (+), 2k+1 (-): this lane's share (its
//   shells) of the determinant ratio of candidate (i, d); the caller adds the four lanes of a quad.
// Bc on the FP64 tensor pipe: one mma.m8n8k4 row = electron g, k = 4 MOs, columns = (k-step parity, shell slot), so the
// lane's two accumulators are exactly its own entries Bc[ao(slot t)][electron g] of two consecutive k-steps:
// 2 NT DMMA + 2 NT LDS per pair of entries instead of 16 NT DFMA + 16 NT LDS (same FP64-pipe time, 1/8 of the issue slots).
// A operand = column il of Dinv (2 NT registers per lane); B operand = the pair table `cf` built at init.  Each shell
// group is padded to an even number of k-steps; s and p iterations are taken two at a time with a one-iteration tail.
// PART (team mode): only the iterations [part->lo[g], part->hi[g]) of each shell group (lo even in groups 0-2, so that a part
// starts on a k-step pair); acc is then the part's share of the ratio.
// BCS (team kernel of the large systems, where the C Dinv product is the largest share): the Bc entries of a block depend on the
// inverse of ITS spin only, and not on the mesh.  BCS = 1: compute them (2 NT DMMA per k-step pair) and park them in a global
// scratch `bcs0` [pair][lane] -- lane-private: the lane that parks an entry is the lane that takes it back; BCS = 2: take them from
// there (blocks of the spin that did not hop since the last evaluation; the second mesh).  Results are bit-identical to BCS = 0.
template <int NT, bool TS, bool PART = false, int BCS = 0>
__device__ __forceinline__ void ao_columns(const DevSys &S, const double *__restrict__ shells, const double *__restrict__ cf, const double *__restrict__ etab,
                                           const double *__restrict__ dinv, int ns, int il, double x0, double y0, double z0,
                                           const double (&av)[3][3], double a2, int lane, double (&acc)[6],
                                           const TeamPlan *tp = nullptr, const ShellPart *part = nullptr, double2 *bcs0 = nullptr)
{
    double2 *bcs = bcs0;
#define LRDMC_COL_RANGE(G, PAIRS)                                                               \
    const int n = PART ? part->hi[G] : S.n_it[G]; int it = PART ? part->lo[G] : 0;              \
    if (PART) { sh4 = reinterpret_cast<const double4 *>(shells) + t + 4 * (tp->it_base[G] + it); b = cf + lane + (size_t)(tp->pair_base[G] + (PAIRS)) * NA * 32; \
                if (BCS) bcs = bcs0 + (size_t)(tp->pair_base[G] + (PAIRS)) * 32; }
    const int t = lane & 3;
    const double4 *sh4 = reinterpret_cast<const double4 *>(shells) + t;
    const double *b = cf + lane;
    constexpr int NA = 2 * NT;
    double aop[NA];                                  // A fragments: Dinv[4 j + t][il] (rows >= n_s are zero padded)
#pragma unroll
    for (int j = 0; j < NA; ++j) aop[j] = (BCS == 2) ? 0.0 : dinv[(4 * j + t) * ns + il];
#pragma unroll
    for (int d = 0; d < 6; ++d) acc[d] = 0.0;
#define LRDMC_BPAIR(v0, v1)                                                                     \
    {                                                                                           \
        if (BCS == 2) { const double2 q_ = __ldcg(bcs); v0 = q_.x; v1 = q_.y; }                 \
        else {                                                                                  \
            v0 = 0.0; v1 = 0.0;                                                                 \
            _Pragma("unroll") for (int j = 0; j < NA; ++j) dmma884(v0, v1, aop[j], ldt<TS>(b + j * 32));  \
            if (BCS == 1) __stcg(bcs, make_double2(v0, v1));                                    \
            b += NA * 32;                                                                       \
        }                                                                                       \
        if (BCS) bcs += 32;                                                                     \
    }
#define LRDMC_GEOM                                                                              \
        const double4 s = *sh4; const double z = s.w;                                           \
        const double dx0 = x0 - s.x, dy0 = y0 - s.y, dz0 = z0 - s.z;                            \
        const double q0 = fma(dx0, dx0, fma(dy0, dy0, fma(dz0, dz0, a2)));                      \
        double sk[3];                                                                           \
        _Pragma("unroll") for (int k = 0; k < 3; ++k) sk[k] = fma(av[k][0], dx0, fma(av[k][1], dy0, av[k][2] * dz0));
#define LRDMC_EXPS                                                                              \
        const double zq0 = -z * q0; const bool far_ = zq0 < 0.5 * LRDMC_EXP_XMIN;   /* |2 z sk| <= z q0: the six arguments lie in [2 zq, 0] */ \
        const double zq = far_ ? 0.5 * LRDMC_EXP_XMIN : zq0, tz = far_ ? 0.0 : -2.0 * z;        \
        double ex_[6], e[6];                                                                    \
        _Pragma("unroll") for (int k = 0; k < 3; ++k) { ex_[2 * k] = fma(tz, sk[k], zq); ex_[2 * k + 1] = fma(-tz, sk[k], zq); } \
        exp_tab_n<6>(ex_, e, etab);
    auto slater_body = [&](double bc) {              // Slater s: exp(-z r)
        LRDMC_GEOM
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            const double q = fma((d & 1) ? -2.0 : 2.0, sk[d >> 1], q0);
            acc[d] = fma(exp_tab(exp_arg_floor(-z * (q * fast_rsqrt(q))), etab), bc, acc[d]);
        }
        sh4 += 4;
    };
    auto s_body = [&](double bc) {
        LRDMC_GEOM
        LRDMC_EXPS
#pragma unroll
        for (int d = 0; d < 6; ++d) acc[d] = fma(e[d], bc, acc[d]);
        sh4 += 4;
    };
    auto p_body = [&](double bcx, double bcy, double bcz) {       // x y z  ->  e (bc . d); the shift adds bc . (a e_k)
        LRDMC_GEOM
        LRDMC_EXPS
        const double l0 = fma(bcx, dx0, fma(bcy, dy0, bcz * dz0));
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double lk = fma(bcx, av[k][0], fma(bcy, av[k][1], bcz * av[k][2]));
            acc[2 * k] = fma(e[2 * k], l0 + lk, acc[2 * k]);
            acc[2 * k + 1] = fma(e[2 * k + 1], l0 - lk, acc[2 * k + 1]);
        }
        sh4 += 4;
    };
    // LRDMC_COMPACT_COLUMNS (extended kernels): ONE copy of each shell body (the second iteration of a k-step pair goes round a two-trip loop) instead of
    // three (pair loop + tail): the extended kernels' hot loop did not fit the instruction cache (ncu: `no_instruction` 0.9 - 1.2 stall cycles per issue
    // at 11.4 k - 11.8 k SASS instructions against 0.06 for the lattice-only kernel's 10.0 k).
#if LRDMC_COMPACT_COLUMNS
    {
        LRDMC_COL_RANGE(0, it / 2) double b0, sv = 0.0;
        for (const int i0 = it; it < n; ++it) { if (!((it - i0) & 1)) { LRDMC_BPAIR(b0, sv) } else b0 = sv; slater_body(b0); }
    }
    {
        LRDMC_COL_RANGE(1, it / 2) double b0, sv = 0.0;
        for (const int i0 = it; it < n; ++it) { if (!((it - i0) & 1)) { LRDMC_BPAIR(b0, sv) } else b0 = sv; s_body(b0); }
    }
    {
        LRDMC_COL_RANGE(2, 3 * it / 2) double b0, b1, b2, sv = 0.0;        // k-steps of two iterations: (0 1 2)(3 4 5) = pairs (0 1)(2 3)(4 5)
        for (const int i0 = it; it < n; ++it) {
            if (!((it - i0) & 1)) { LRDMC_BPAIR(b0, b1) LRDMC_BPAIR(b2, sv) } else { b0 = sv; LRDMC_BPAIR(b1, b2) }
            p_body(b0, b1, b2);
        }
    }
#else
    {
        LRDMC_COL_RANGE(0, it / 2) double b0, b1;
        for (; it + 1 < n; it += 2) { LRDMC_BPAIR(b0, b1) slater_body(b0); slater_body(b1); }
        if (it < n) { LRDMC_BPAIR(b0, b1) slater_body(b0); }
    }
    {
        LRDMC_COL_RANGE(1, it / 2) double b0, b1;
        for (; it + 1 < n; it += 2) { LRDMC_BPAIR(b0, b1) s_body(b0); s_body(b1); }
        if (it < n) { LRDMC_BPAIR(b0, b1) s_body(b0); }
    }
    {
        LRDMC_COL_RANGE(2, 3 * it / 2) double b0, b1, b2, b3, b4, b5;
        for (; it + 1 < n; it += 2) { LRDMC_BPAIR(b0, b1) LRDMC_BPAIR(b2, b3) LRDMC_BPAIR(b4, b5) p_body(b0, b1, b2); p_body(b3, b4, b5); }
        if (it < n) { LRDMC_BPAIR(b0, b1) LRDMC_BPAIR(b2, b3) p_body(b0, b1, b2); }
    }
#endif
    { LRDMC_COL_RANGE(3, 3 * it) for (; it < n; ++it, sh4 += 4) {   // d: xx xy xz yy yz zz  ->  e Q(d),  Q(d0 +- v) = Q(d0) +- v.grad Q(d0) + Q(v)
        double bc[6]; LRDMC_BPAIR(bc[0], bc[1]) LRDMC_BPAIR(bc[2], bc[3]) LRDMC_BPAIR(bc[4], bc[5])
        LRDMC_GEOM
        LRDMC_EXPS
        const double gx = fma(2.0 * bc[0], dx0, fma(bc[1], dy0, bc[2] * dz0));
        const double gy = fma(bc[1], dx0, fma(2.0 * bc[3], dy0, bc[4] * dz0));
        const double gz = fma(bc[2], dx0, fma(bc[4], dy0, 2.0 * bc[5] * dz0));
        const double Q0 = 0.5 * fma(gx, dx0, fma(gy, dy0, gz * dz0));
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double vx = av[k][0], vy = av[k][1], vz = av[k][2];
            const double lin = fma(gx, vx, fma(gy, vy, gz * vz));
            const double Qv = fma(vx, fma(bc[0], vx, fma(bc[1], vy, bc[2] * vz)), fma(vy, fma(bc[3], vy, bc[4] * vz), bc[5] * vz * vz));
            const double Qs = Q0 + Qv;
            acc[2 * k] = fma(e[2 * k], Qs + lin, acc[2 * k]);
            acc[2 * k + 1] = fma(e[2 * k + 1], Qs - lin, acc[2 * k + 1]);
        }
    } }
#undef LRDMC_EXPS
#undef LRDMC_GEOM
#undef LRDMC_BPAIR
#undef LRDMC_COL_RANGE
}

// Refresh the cached MO rows (value, gradient, Laplacian) of electron i at position (px,py,pz): moc[i][comp][m].
template <int NT, bool TS>
__device__ __forceinline__ void refresh_mo_cache(const DevSys &S, const double *shells, const double *bf, const double *etab, double *moc_i,
                                                 double px, double py, double pz, int lane)
{
    double acc[NT][2];
    mo_pass<NT, true, TS>(S, shells, bf, etab, px, py, pz, lane, acc);
    const int t = lane & 3, g = lane >> 2;
    if (g < 5) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
            moc_i[g * S.OS + 8 * nt + 2 * t] = acc[nt][0];
            moc_i[g * S.OS + 8 * nt + 2 * t + 1] = acc[nt][1];
        }
    }
}

// In-place Gauss-Jordan inversion with partial (row) pivoting of the n x n matrix A (row stride ld) by one warp.
// On entry A[i][m] = D[i][m]; on exit A[m][i] = Dinv[m][i] (sum_m D[i][m] Dinv[m][k] = delta_ik).  Returns false when a pivot
// is not above 2^-44 max|A_ij| (reading Q24: "|D| = 0" in FP64 -- two identical rows leave a pivot of rounding size, not a zero).
__device__ __forceinline__ bool warp_invert(double *A, int n, int ld, int *perm, int lane)
{
    bool ok = true;
    double amax = 0.0;
    for (int idx = lane; idx < n * n; idx += 32) amax = fmax(amax, fabs(A[(idx / n) * ld + idx % n]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = fmax(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const double tiny = ldexp(amax, -44);
    for (int c = 0; c < n; ++c) {
        // pivot search over rows i >= c
        double best = -1.0; int bi = c;
        for (int i = c + lane; i < n; i += 32) { double v = fabs(A[i * ld + c]); if (v > best) { best = v; bi = i; } }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double ob = __shfl_xor_sync(0xffffffffu, best, o); int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if (!(best > tiny) || isinf(best)) { ok = false; break; }
        if (lane == 0) perm[c] = bi;
        if (bi != c) for (int j = lane; j < n; j += 32) { double tmp = A[c * ld + j]; A[c * ld + j] = A[bi * ld + j]; A[bi * ld + j] = tmp; }
        __syncwarp();
        double ip = 1.0 / A[c * ld + c];
        __syncwarp();
        for (int j = lane; j < n; j += 32) A[c * ld + j] = (j == c) ? ip : A[c * ld + j] * ip;
        __syncwarp();
        for (int idx = lane; idx < n * n; idx += 32) {
            int i = idx / n, j = idx - i * n;
            if (i == c) continue;
            double f = A[i * ld + c];
            // column c of row i must be read by every lane of that row before it is overwritten: do it in two sweeps
            if (j != c) A[i * ld + j] -= f * A[c * ld + j];
        }
        __syncwarp();
        for (int i = lane; i < n; i += 32) if (i != c) A[i * ld + c] = -A[i * ld + c] * A[c * ld + c];
        __syncwarp();
    }
    if (ok) {
        for (int c = n - 1; c >= 0; --c) {
            int p = perm[c];
            if (p != c) for (int i = lane; i < n; i += 32) { double tmp = A[i * ld + c]; A[i * ld + c] = A[i * ld + p]; A[i * ld + p] = tmp; }
            __syncwarp();
        }
    }
    return ok;
}
