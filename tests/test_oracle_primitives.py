"""Pins of the oracle's primitives (CPU only): Philox, uniforms, frame, AOs, inverse, comb.

Each test checks the oracle against something that is NOT the oracle: published known-answer vectors,
closed forms / quadrature, numpy's LAPACK, exact rational arithmetic, invariants.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import lrdmc_ref as ref
from paper_2508_12033_b200 import workloads as wl
from conftest import read_golden


# ----------------------------------------------------------------------------- RNG (pin P11)
def test_philox_known_answers():
    for name, v in read_golden("philox4x32_10_kat.txt").items():
        x = [int(t, 16) for t in v]
        assert ref.philox4x32_10(x[0:4], x[4:6]) == tuple(x[6:10]), name


def _philox_python(ctr, key):
    """Independent re-statement with Python integers (no C): pins the oracle's round structure."""
    c = list(ctr); k = list(key)
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]; p1 = 0xCD9E8D57 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xFFFFFFFF, p1 & 0xFFFFFFFF, ((p0 >> 32) ^ c[3] ^ k[1]) & 0xFFFFFFFF, p0 & 0xFFFFFFFF]
        k = [(k[0] + 0x9E3779B9) & 0xFFFFFFFF, (k[1] + 0xBB67AE85) & 0xFFFFFFFF]
    return tuple(c)


def test_philox_random_counters_match_python_integers():
    rng = np.random.default_rng(0)
    for _ in range(200):
        ctr = [int(v) for v in rng.integers(0, 2**32, 4)]; key = [int(v) for v in rng.integers(0, 2**32, 2)]
        assert ref.philox4x32_10(ctr, key) == _philox_python(ctr, key)


def test_uniform53_range_and_exact_values():
    assert ref.uniform53(0, 0) == 0.0
    assert ref.uniform53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0**-53
    assert ref.uniform53(0, 0x80000000) == 0.5
    assert ref.uniform53(0x7FF, 0) == 0.0          # the low 11 bits are dropped
    assert ref.uniform53(0x800, 0) == 2.0**-53


def test_draws_use_the_documented_counters():
    s = wl.hydrogen(); o = ref.Ref(s)
    seed = s["seed"]; key = (seed & 0xFFFFFFFF, seed >> 32)
    u = o.draws(7, 3, 11)
    b0 = _philox_python((7, 3, 11, 0), key); b1 = _philox_python((7, 3, 11, 1), key); b2 = _philox_python((7, 3, 11, 2), key)
    f = lambda lo, hi: ((hi << 32 | lo) >> 11) * 2.0**-53
    assert list(u) == [f(b0[0], b0[1]), f(b0[2], b0[3]), f(b1[0], b1[1]), f(b1[2], b1[3]), f(b2[0], b2[1])]
    assert o.comb_r32(5) == _philox_python((0xFFFFFFFF, 5, 0, 3), key)[0]


def test_uniforms_are_uniform():
    s = wl.hydrogen(); o = ref.Ref(s)
    u = np.array([o.draws(k, 0, st) for k in range(400) for st in range(10)])
    assert u.min() >= 0.0 and u.max() < 1.0
    for col in range(5):        # mean 1/2 +- 1/sqrt(12 n), 5 sigma
        assert abs(u[:, col].mean() - 0.5) < 5.0 / math.sqrt(12 * len(u))
    assert abs(np.corrcoef(u[:, 0], u[:, 3])[0, 1]) < 0.08


# ----------------------------------------------------------------------------- frame (L596, Q7)
def test_frame_is_a_rotation_and_haar_distributed():
    rng = np.random.default_rng(1)
    us = rng.random((4000, 3))
    Us = np.array([ref.frame(*u) for u in us])
    eye = np.einsum("nij,nkj->nik", Us, Us)
    assert np.abs(eye - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(Us) - 1.0).max() < 1e-13
    # Haar: every column is uniform on the sphere -> each component has mean 0 and variance 1/3,
    # and each matrix element is uniform on [-1,1] (Archimedes): check first two moments and a KS distance
    assert np.abs(Us.mean(axis=0)).max() < 5.0 / math.sqrt(3 * len(Us))
    assert np.abs((Us**2).mean(axis=0) - 1.0 / 3.0).max() < 0.02
    for (i, j) in ((0, 0), (1, 2), (2, 1)):
        v = np.sort(Us[:, i, j]); cdf = (v + 1.0) / 2.0
        ks = np.abs(cdf - (np.arange(len(v)) + 0.5) / len(v)).max()
        assert ks < 1.95 / math.sqrt(len(v))
    # special values: u1=1,u2=u3=0 -> quaternion (0,0,0,1) -> identity; u1 = 0, u2 = 0 -> q = (0,1,0,0): rotation by pi about y
    assert np.allclose(ref.frame(1.0, 0.0, 0.0), np.eye(3), atol=1e-15)
    assert np.allclose(ref.frame(0.0, 0.0, 0.0), np.diag([-1.0, 1.0, -1.0]), atol=1e-15)


# ----------------------------------------------------------------------------- AOs (pin P4)
def _one_shell(stype, zeta, center=(0.1, -0.2, 0.3)):
    n = {0: 1, 1: 3, 2: 6, 10: 1}[stype]
    return wl._system("one-shell", [1.0], [list(center)], 1, 0, [0], [stype], [zeta], np.ones((n, 1)), np.zeros((n, 0)), {}, 0.2)


@pytest.mark.parametrize("stype", [0, 1, 2])
@pytest.mark.parametrize("zeta", [0.37, 2.9])
def test_gaussian_ao_unit_self_overlap_and_d_shell_metric(stype, zeta):
    """N_lmn gives <chi|chi> = 1; for d shells <xx|yy> = 1/3 (the cartesian metric) and <xx|xy> = 0.
    Gauss-Hermite quadrature with weight exp(-2 zeta v^2) is exact for these polynomials."""
    o = ref.Ref(_one_shell(stype, zeta)); c = np.array([0.1, -0.2, 0.3])
    t, wq = np.polynomial.hermite.hermgauss(12)
    v = t / math.sqrt(2 * zeta); wv = wq / math.sqrt(2 * zeta)
    S = 0.0
    for ix, x in enumerate(v):
        for iy, y in enumerate(v):
            for iz, z in enumerate(v):
                val, _, _ = o.ao(c + np.array([x, y, z]))
                g = val * math.exp(zeta * (x * x + y * y + z * z))      # strip the Gaussian: quadrature carries exp(-2 zeta r^2)
                S = S + wv[ix] * wv[iy] * wv[iz] * np.outer(g, g)
    assert np.allclose(np.diag(S), 1.0, atol=1e-12)
    if stype == 1:
        assert np.allclose(S, np.eye(3), atol=1e-12)
    if stype == 2:      # order xx xy xz yy yz zz
        assert abs(S[0, 3] - 1.0 / 3.0) < 1e-12 and abs(S[0, 5] - 1.0 / 3.0) < 1e-12 and abs(S[3, 5] - 1.0 / 3.0) < 1e-12
        assert abs(S[0, 1]) < 1e-12 and abs(S[1, 2]) < 1e-12 and abs(S[1, 4]) < 1e-12


def test_ao_angular_order_and_slater_type():
    """p shell = (x, y, z) times the s-like radial part; d shell order xx xy xz yy yz zz; type 10 = exp(-zeta r)."""
    z = 0.8; c = np.array([0.1, -0.2, 0.3]); d = np.array([0.7, -0.4, 0.25])
    vp, _, _ = ref.Ref(_one_shell(1, z)).ao(c + d)
    assert np.allclose(vp / vp[0], d / d[0], rtol=1e-13)
    vd, _, _ = ref.Ref(_one_shell(2, z)).ao(c + d)
    mono = np.array([d[0] * d[0] / math.sqrt(3), d[0] * d[1], d[0] * d[2], d[1] * d[1] / math.sqrt(3), d[1] * d[2], d[2] * d[2] / math.sqrt(3)])
    assert np.allclose(vd / vd[1], mono / mono[1], rtol=1e-13)
    vs, gs, ls = ref.Ref(_one_shell(10, z)).ao(c + d)
    r = np.linalg.norm(d)
    assert abs(vs[0] - math.exp(-z * r)) < 1e-15
    assert np.allclose(gs[0], -z * math.exp(-z * r) * d / r, rtol=1e-13)
    assert abs(ls[0] - math.exp(-z * r) * (z * z - 2 * z / r)) < 1e-13


@pytest.mark.parametrize("stype", [0, 1, 2, 10])
def test_ao_gradient_and_laplacian_match_finite_differences(stype):
    o = ref.Ref(_one_shell(stype, 0.9)); r0 = np.array([0.55, 0.3, -0.45]); h = 1e-3
    _, g, l = o.ao(r0)
    f = lambda r: o.ao(r)[0]
    lap_fd = 0.0
    for ax in range(3):
        e = np.zeros(3); e[ax] = h
        # 4th-order central differences
        g_fd = (-f(r0 + 2 * e) + 8 * f(r0 + e) - 8 * f(r0 - e) + f(r0 - 2 * e)) / (12 * h)
        assert np.allclose(g[:, ax], g_fd, atol=1e-9)
        lap_fd = lap_fd + (-f(r0 + 2 * e) + 16 * f(r0 + e) - 30 * f(r0) + 16 * f(r0 - e) - f(r0 - 2 * e)) / (12 * h * h)
    assert np.allclose(l, lap_fd, atol=2e-7)


def _contracted_d(zetas, coefs, sph, centre=(0.1, -0.2, 0.3), extra_s=None):
    """One contracted d shell (and optionally one s primitive as a second contracted shell) on one centre."""
    n = len(zetas); types = [wl.SHELL_D] * n; z = list(zetas); co = list(coefs); first = [0, n]; sp = [1 if sph else 0]
    if extra_s is not None:
        types.append(wl.SHELL_S); z.append(extra_s); co.append(1.0); first.append(n + 1); sp.append(0)
    nao = wl.n_ao_contracted(types, first, sp)
    return wl._system("contracted-d", [1.0], [list(centre)], 1, 0, [0] * len(types), types, z, np.eye(nao)[:, :1], np.zeros((nao, 0)), {}, 0.2,
                      contraction=(first, co, sp))


def test_solid_harmonic_d_shell_is_orthonormal_and_has_no_s_component():
    """Scope row f2 (L242 "spherical (solid) harmonics").  For one primitive the five functions z2, xz, yz, x2-y2, xy are
    orthonormal and orthogonal to an s Gaussian on the same centre, while the cartesian xx + yy + zz overlaps it: 3-D
    Gauss-Hermite quadrature, exact for these polynomials.  Their polynomial parts are harmonic and homogeneous of degree 2."""
    zeta = 0.8; c = np.array([0.1, -0.2, 0.3])
    t, wq = np.polynomial.hermite.hermgauss(14)

    def overlap(ctx):
        S = 0.0
        for ix, x in enumerate(v):
            for iy, y in enumerate(v):
                for iz, z in enumerate(v):
                    val, _, _ = ctx.ao(c + np.array([x, y, z]))
                    S = S + wv[ix] * wv[iy] * wv[iz] * np.outer(val, val) * math.exp(2 * zq * (x * x + y * y + z * z))
        return S
    # the s function takes the same exponent, so that every product is polynomial x exp(-2 zeta r^2): the rule is then exact
    o = ref.Ref(_contracted_d([zeta], [1.0], True, extra_s=zeta)); oc = ref.Ref(_contracted_d([zeta], [1.0], False, extra_s=zeta))
    zq = zeta; v = t / math.sqrt(2 * zq); wv = wq / math.sqrt(2 * zq)
    S = overlap(o)
    assert S.shape == (6, 6) and np.allclose(S, np.eye(6), atol=1e-12)        # 5 solid harmonics + s: orthonormal, no s contaminant
    Sc = overlap(oc)
    assert abs(Sc[0, 6] - Sc[3, 6]) < 1e-12 and Sc[0, 6] > 0.5                # cartesian xx, yy, zz each overlap the s function
    # harmonic and homogeneous of degree 2: strip the Gaussian, check f(2 d) = 4 f(d) and the values against the explicit polynomials
    d = np.array([0.7, -0.4, 0.25]); val, _, _ = o.ao(c + d); val2, _, _ = o.ao(c + 2 * d)
    r2 = d @ d
    f = val[:5] * math.exp(zeta * r2); f2 = val2[:5] * math.exp(zeta * 4 * r2)
    assert np.allclose(f2, 4 * f, rtol=1e-12)
    poly = np.array([(2 * d[2]**2 - d[0]**2 - d[1]**2) / (2 * math.sqrt(3)), d[0] * d[2], d[1] * d[2], (d[0]**2 - d[1]**2) / 2, d[0] * d[1]])
    assert np.allclose(f / f[4], poly / poly[4], rtol=1e-12)


def test_contracted_shell_is_the_stated_sum_of_normalised_primitives_with_correct_derivatives():
    """chi = sum_k d_k chi_k^prim: value against the closed form of the normalised primitives written out here; gradient and
    Laplacian against 4th-order finite differences."""
    zs = [0.4, 1.1, 3.0]; ds = [0.7, -0.35, 0.2]; c = np.array([0.1, -0.2, 0.3])
    o = ref.Ref(_contracted_d(zs, ds, True)); r0 = c + np.array([0.45, 0.3, -0.35]); d = r0 - c
    val, g, l = o.ao(r0)
    N110 = lambda z: (2 * z / math.pi) ** 0.75 * (4 * z)            # norm of the xy-type d primitive (unit self-overlap)
    want_xy = sum(dk * N110(z) * d[0] * d[1] * math.exp(-z * (d @ d)) for z, dk in zip(zs, ds))
    want_z2 = sum(dk * N110(z) * (2 * d[2]**2 - d[0]**2 - d[1]**2) / (2 * math.sqrt(3)) * math.exp(-z * (d @ d)) for z, dk in zip(zs, ds))
    assert abs(val[4] - want_xy) < 1e-14 and abs(val[0] - want_z2) < 1e-14
    h = 1e-3; f = lambda r: o.ao(r)[0]; lap_fd = 0.0
    for ax in range(3):
        e = np.zeros(3); e[ax] = h
        g_fd = (-f(r0 + 2 * e) + 8 * f(r0 + e) - 8 * f(r0 - e) + f(r0 - 2 * e)) / (12 * h)
        assert np.allclose(g[:, ax], g_fd, atol=1e-9)
        lap_fd = lap_fd + (-f(r0 + 2 * e) + 16 * f(r0 + e) - 30 * f(r0) + 16 * f(r0 - e) - f(r0 - 2 * e)) / (12 * h * h)
    assert np.allclose(l, lap_fd, atol=2e-7)


def test_contracted_slater_shell_is_the_stated_sum_with_correct_derivatives():
    """Scope row f2, contracted Slater shells: chi = sum_k d_k exp(-zeta_k |r - R|) written out; gradient and Laplacian against
    the closed forms grad = -sum d_k zeta_k e^{-zeta_k r} rhat, lap = sum d_k e^{-zeta_k r} (zeta_k^2 - 2 zeta_k / r) and against finite
    differences; the Gaussian p / solid-harmonic d shells beside them keep their own pins (same code path as before)."""
    s = wl.contracted_slater_molecule(); o = ref.Ref(s)
    assert s["n_ao"] == 4 + 3 + 5 and s["n_shell"] == 10
    rng = np.random.default_rng(2)
    prim = [(0, [(2.6, 0.5), (1.4, 0.4), (0.9, 0.2)]), (1, [(3.1, 0.7), (1.1, -0.3)]), (0, [(0.7, 1.0)]), (1, [(0.8, 1.0)])]
    for _ in range(5):
        r = rng.normal(size=3) * 1.2; v, g, l = o.ao(r)
        for mu, (I, terms) in enumerate(prim):
            d = r - s["R"][I]; rr = np.linalg.norm(d)
            val = sum(c * math.exp(-z * rr) for z, c in terms)
            grad = -sum(c * z * math.exp(-z * rr) for z, c in terms) * d / rr
            lap = sum(c * math.exp(-z * rr) * (z * z - 2 * z / rr) for z, c in terms)
            assert abs(v[mu] - val) < 1e-15 and np.abs(g[mu] - grad).max() < 1e-14 and abs(l[mu] - lap) < 1e-13
        h = 1e-3                                          # 4th-order finite differences of every function (incl. the p and d shells)
        lap_fd = np.zeros(s["n_ao"])
        for ax in range(3):
            e = np.zeros(3); e[ax] = h
            fp, fm, fpp, fmm = o.ao(r + e)[0], o.ao(r - e)[0], o.ao(r + 2 * e)[0], o.ao(r - 2 * e)[0]
            assert np.abs(g[:, ax] - (-fpp + 8 * fp - 8 * fm + fmm) / (12 * h)).max() < 1e-9
            lap_fd += (-fpp + 16 * fp - 30 * v + 16 * fm - fmm) / (12 * h * h)
        assert np.abs(l - lap_fd).max() < 2e-6


def test_mo_is_ao_times_coefficients():
    s = wl.synthetic10(); o = ref.Ref(s); r = np.array([0.3, -0.8, 0.5])
    av, ag, al = o.ao(r); mv, mg, ml = o.mo(0, r)
    assert np.allclose(mv, av @ s["C_up"], rtol=1e-12, atol=1e-14)
    assert np.allclose(mg, (ag.T @ s["C_up"]).T, rtol=1e-12, atol=1e-14)
    assert np.allclose(ml, al @ s["C_up"], rtol=1e-12, atol=1e-13)


# ----------------------------------------------------------------------------- inverse (a13) vs LAPACK
def test_build_inverse_matches_numpy_and_reports_singular():
    s = wl.synthetic10(); o = ref.Ref(s)
    x = wl.initial_walkers(s, 3, 11)
    for k in range(3):
        rc, du, dd = o.build_inverse(x[k]); assert rc == 0
        D = np.array([o.mo(0, x[k, i])[0] for i in range(5)])          # D[i][m]
        assert np.allclose(D @ du, np.eye(5), atol=1e-9)
        assert np.allclose(du, np.linalg.inv(D), rtol=1e-8, atol=1e-10)
        la, sg = o.logpsi(x[k])
        Dd = np.array([o.mo(1, x[k, 5 + i])[0] for i in range(5)])
        s1, l1 = np.linalg.slogdet(D); s2, l2 = np.linalg.slogdet(Dd)
        assert sg == int(s1 * s2)
    xs = x[0].copy(); xs[1] = xs[0]                                     # two same-spin electrons at one point
    rc, du, _ = o.build_inverse(xs)                                     # exact zero pivot is not guaranteed in FP:
    assert rc == -2 or np.abs(du).max() > 1e10                          # either flagged, or visibly ill-conditioned


# ----------------------------------------------------------------------------- comb (pin P10)
def _comb_exact(w, r32):
    """Eq.17 with exact rationals ON THE QUANTISED WEIGHTS' DEFINITION: parent_k = min{beta: cum_beta/T > (xi+k)/N}."""
    n = len(w); m = max(w); e = math.frexp(m)[1]; L = max(1, math.ceil(math.log2(n))); sh = 62 - L - e
    u = [int(math.floor(math.ldexp(x, sh))) for x in w]; T = sum(u)
    xi = Fraction(r32, 2**32); out = []; cum = 0; beta = -1
    for k in range(n):
        z = (xi + k) / n
        while True:
            if beta >= 0 and Fraction(cum, T) > z:
                break
            beta += 1; cum += u[beta]
        out.append(beta)
    return out, u, T, sh


def test_comb_worked_example():
    g = read_golden("comb_worked_example.txt")
    w = [float(v) for v in g["w"]]
    rc, par, wbar, u, T, sh = ref.comb(w, 0)
    assert rc == 0 and sh == int(g["sh"][0]) and T == int(g["T"][0]) and [int(v) for v in u] == [int(v) for v in g["u"]]
    assert abs(wbar - sum(w) / 5) < 1e-13
    for r32 in (0x00000000, 0x80000000, 0xFFFFFFFF):
        rc, par, *_ = ref.comb(w, r32)
        assert list(par) == [int(v) for v in g["parents_r32_%08x" % r32]]


def test_comb_matches_exact_rationals_and_invariants():
    rng = np.random.default_rng(4)
    for trial in range(120):
        n = int(rng.integers(1, 90))
        w = rng.random(n) ** 3 * 10.0 ** rng.integers(-6, 6)
        if trial % 5 == 0:
            w[rng.integers(0, n, size=max(1, n // 3))] = 0.0
            if w.max() == 0.0:
                w[0] = 1.0
        r32 = int(rng.integers(0, 2**32))
        rc, par, wbar, u, T, sh = ref.comb(w, r32)
        exact, ue, Te, she = _comb_exact(list(w), r32)
        assert rc == 0 and list(par) == exact and T == Te and sh == she
        assert np.all(np.diff(par) >= 0)                                    # sorted
        assert abs(wbar - w.mean()) <= 2.0**-44 * w.mean()                 # Eq.16 up to the quantisation
        counts = np.bincount(par, minlength=n)
        ideal = n * u.astype(np.float64) / T
        assert np.all(counts >= np.floor(ideal) - 1e-9) and np.all(counts <= np.ceil(ideal) + 1e-9)
        assert np.all(counts[w == 0.0] == 0)                                # dead walkers never survive


def test_comb_preserves_the_weighted_average():
    """Reconfiguration 'does not change their statistical average' (L117): E_xi[copies of beta] = N_w w_beta / sum w."""
    g = read_golden("comb_worked_example.txt"); w = np.array([float(v) for v in g["w"]])
    M = 4096; acc = np.zeros(5)
    for q in range(M):
        _, par, *_ = ref.comb(w, int((q + 0.5) / M * 2**32))
        acc += np.bincount(par, minlength=5)
    assert np.allclose(acc / M, 5 * w / w.sum(), atol=2.0 / M * 5)


def test_comb_degenerate_inputs():
    rc, par, wbar, *_ = ref.comb(np.zeros(4), 123)
    assert rc == 0 and list(par) == [0, 1, 2, 3] and wbar == 0.0
    rc, par, wbar, *_ = ref.comb(np.array([1.0, np.nan, 2.0]), 5)
    assert rc == -1 and list(par) == [0, 1, 2]
    rc, par, wbar, *_ = ref.comb(np.array([3.5]), 0xFFFFFFFF)
    assert rc == 0 and list(par) == [0] and wbar == 3.5
