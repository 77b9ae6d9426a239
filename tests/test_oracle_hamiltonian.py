"""Pins of the oracle's one-evaluation routine (Appendix D), the ratios, Sherman-Morrison and the
heat-bath selection -- CPU only.  Checked against closed forms (H atom), brute force (full determinants
through LAPACK-free pivoted elimination AND numpy's slogdet, full re-inversion), the identity Eq.D7, and
finite differences of log|Psi_G|.
"""
import math

import numpy as np
import pytest

from oracle import lrdmc_ref as ref
from paper_2508_12033_b200 import workloads as wl
from conftest import read_golden


def _rand_frame(rng):
    return ref.frame(*rng.random(3))


# ----------------------------------------------------------------------------- H atom closed forms (pin P1)
def test_h_atom_worked_example_against_closed_forms():
    g = read_golden("h_atom_worked_example.txt"); alpha, a = 0.9, 0.2
    o = ref.Ref(wl.hydrogen(alpha=alpha, a=a)); x = np.array([[0.3, 0.4, 1.2]])
    R, sc, per, cand = o.evaluate(x, np.eye(3))
    # closed forms re-derived here, independent of the oracle's code path
    r = np.linalg.norm(x[0]); disp = a * np.array([[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], float)
    R_cf = np.exp(-alpha * (np.linalg.norm(x[0] + disp, axis=1) - r))
    assert np.allclose(cand, x[0] + disp, atol=1e-15)
    assert np.allclose(R, R_cf, rtol=1e-14)
    assert np.allclose(R, [float(v) for v in g["R"]], rtol=1e-14)
    lap = alpha**2 - 2 * alpha / r; T = (R_cf.sum() - 6) / a**2
    for key, val, cf in (("bbar", sc["bbar"], R_cf.sum() / (2 * a * a)), ("T", per[0, 0], T), ("lap", per[0, 1], lap),
                         ("v_zv", per[0, 3], -1 / r + 0.5 * (T - lap)), ("W", sc["W"], 3 / a**2 - 1 / r + 0.5 * (T - lap)),
                         ("e_L", sc["e_L"], -alpha**2 / 2 + (alpha - 1) / r)):
        assert abs(val - cf) < 2e-12 * max(1.0, abs(cf)), key
        assert abs(val - float(g[key][0])) < 2e-12 * max(1.0, abs(cf)), key
    assert abs(sc["bbar"] / (sc["W"] + 0.5) - float(g["b_x"][0])) < 1e-13
    cum = np.cumsum(R) / R.sum()
    assert np.allclose(cum, [float(v) for v in g["cum_p"]], atol=1e-10)
    for u, j in ((0.0, 0), (0.158, 0), (0.159, 1), (0.5, 3), (0.999999, 5)):
        assert o.select(R, u)[0] == j
    # second point: close to the nucleus, v_zv < v^a_ei, but no node flag -> the max branch (D11) stays off
    x2 = np.array([[0.05, 0.0, 0.1]]); R2, sc2, per2, _ = o.evaluate(x2, np.eye(3))
    assert abs(per2[0, 3] - float(g["v_zv_close"][0])) < 1e-11 and per2[0, 4] == -5.0 and sc2["n_vmax"] == 0
    assert abs(sc2["e_L"] - float(g["e_L_close"][0])) < 1e-11


def test_h_atom_exact_trial_function_has_zero_variance():
    """Psi_G = exp(-r) is the exact ground state: e_L = -1/2 and b_x = 1 for E_0 = -1/2 at every x, a and frame (pin P5)."""
    rng = np.random.default_rng(3)
    for a in (0.05, 0.2, 0.5):
        o = ref.Ref(wl.hydrogen(alpha=1.0, a=a))
        for _ in range(20):
            x = rng.normal(size=(1, 3)) * 1.5
            R, sc, per, _ = o.evaluate(x, _rand_frame(rng))
            assert abs(sc["e_L"] + 0.5) < 2e-11 / a**2 * 1e-2 + 1e-12
            assert abs(sc["bbar"] / (sc["W"] + 0.5) - 1.0) < 1e-13


# ----------------------------------------------------------------------------- Eq.D7 identity (pin P2)
SYSTEMS = {
    "tiny-2u1d": lambda: wl.tiny_molecule(2, 1, 2, 6, seed=7),
    "tiny-3u3d-pp": lambda: wl.tiny_molecule(3, 3, 3, 9, seed=8, with_pp=True),
    "tiny-2u2d-doublemesh": lambda: wl.tiny_molecule(2, 2, 2, 7, seed=9, a=0.15, a2=0.3),
    "C2": wl.synthetic10,
    "C3": lambda: wl.water_methane(n_walkers=4),
    "tiny-j3": lambda: wl.with_jastrow3(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 4, 2),   # three-body Jastrow (scope row f2)
    "tiny-j3-spd": lambda: wl.with_jastrow3(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 5, 4, n_max=12, poly=True),   # s/p/d functions, 12 of them
    "contracted-sph": lambda: wl.contracted_molecule(3, 2, 3, 9, seed=31, spherical=True, with_pp=True),   # scope row f2
    "contracted-slater": wl.contracted_slater_molecule,                                                      # scope row f2: contracted Slater shells
}


@pytest.mark.parametrize("name", list(SYSTEMS))
def test_regularised_local_energy_equals_continuum_local_energy(name):
    """e_L^a(x) = e_L(x) (Eq.D7): -bbar + W must equal sum_i[-lap_i/2 + v_ei] + V_ee + V_ii whenever the
    max branch of D11 did not fire.  This closes the bookkeeping of K_diag, T_i, v_zv, V_sf and every sign."""
    s = SYSTEMS[name](); o = ref.Ref(s); rng = np.random.default_rng(5)
    xs = wl.initial_walkers(s, 6, 21); N = s["n_up"] + s["n_dn"]; amin = s["a"]
    checked = 0
    for x in xs:
        try:
            R, sc, per, _ = o.evaluate(x, _rand_frame(rng))
        except FloatingPointError:
            continue
        if s["a2"] == 0:
            assert abs(sc["K_diag"] - 3 * N / s["a"]**2) < 1e-9 * sc["K_diag"]      # K^a_{x,x} = 3 N_e / a^2 (Eq.D5)
        if sc["n_vmax"] == 0:
            scale = 3 * N / amin**2
            assert abs(sc["e_L"] - sc["e_L_continuum"]) < 1e-9 * scale
            checked += 1
        else:   # the max branch only ever raises W
            assert sc["e_L"] >= sc["e_L_continuum"] - 1e-9
        assert sc["V_sf"] >= 0.0 and (sc["node"] == 1.0) == bool((R < 0).any())
        if s["a2"] > 0:
            assert abs(sc["K_diag"] - 3 * N * (0.5 / s["a"]**2 + 0.5 / s["a2"]**2)) < 1e-9 * sc["K_diag"]
    assert checked >= 1     # random-MO trial functions have nodes everywhere: the D11 branch fires often on C3


@pytest.mark.parametrize("name", ["tiny-2u1d", "tiny-3u3d-pp", "C2", "contracted-sph", "tiny-j3", "tiny-j3-spd", "contracted-slater"])
def test_continuum_laplacian_matches_finite_differences_of_logpsi(name):
    """lap_i Psi/Psi = lap_i log|Psi| + |grad_i log|Psi||^2, by 4th-order central differences of the brute-force log|Psi|."""
    s = SYSTEMS[name](); o = ref.Ref(s); x = wl.initial_walkers(s, 1, 33)[0]
    R, sc, per, _ = o.evaluate(x, np.eye(3)); h = 2e-3
    for i in range(x.shape[0]):
        lap = 0.0; g2 = 0.0
        f0 = o.logpsi(x)[0]
        for ax in range(3):
            def f(t):
                y = x.copy(); y[i, ax] += t; return o.logpsi(y)[0]
            fp, fm, fpp, fmm = f(h), f(-h), f(2 * h), f(-2 * h)
            g = (-fpp + 8 * fp - 8 * fm + fmm) / (12 * h)
            lap += (-fpp + 16 * fp - 30 * f0 + 16 * fm - fmm) / (12 * h * h); g2 += g * g
        assert abs(per[i, 1] - (lap + g2)) < 2e-5 * max(1.0, abs(per[i, 1])), i


# ----------------------------------------------------------------------------- ratios vs brute force (pin P3)
@pytest.mark.parametrize("name", ["tiny-2u1d", "tiny-3u3d-pp", "tiny-2u2d-doublemesh", "C2", "contracted-sph", "tiny-j3", "tiny-j3-spd", "contracted-slater"])
def test_candidate_ratios_match_full_wavefunction_recomputation(name):
    s = SYSTEMS[name](); o = ref.Ref(s); rng = np.random.default_rng(6)
    x = wl.initial_walkers(s, 1, 44)[0]; U = _rand_frame(rng)
    R, sc, per, cand = o.evaluate(x, U)
    l0, s0 = o.logpsi(x); N = x.shape[0]
    assert len(R) == 6 * N * (2 if s["a2"] > 0 else 1)
    for j in range(len(R)):
        i = (j % (6 * N)) // 6; d = j % 6; am = s["a2"] if j >= 6 * N else s["a"]
        y = x.copy(); y[i] = x[i] + (1 if d % 2 == 0 else -1) * am * U[:, d // 2]
        assert np.allclose(cand[j], y[i], atol=1e-15)
        l1, s1 = o.logpsi(y)
        assert abs(R[j] - s0 * s1 * math.exp(l1 - l0)) < 1e-10 * max(1.0, abs(R[j])), j


def test_logpsi_matches_numpy_slogdet_and_explicit_jastrow():
    s = wl.tiny_molecule(3, 2, 2, 7, seed=12); o = ref.Ref(s); x = wl.initial_walkers(s, 1, 2)[0]
    Du = np.array([o.mo(0, x[i])[0] for i in range(3)]); Dd = np.array([o.mo(1, x[3 + i])[0] for i in range(2)])
    su, lu = np.linalg.slogdet(Du); sd, ld = np.linalg.slogdet(Dd)
    J = 0.0
    for i in range(5):
        for I in range(s["n_nuc"]):
            r = np.linalg.norm(x[i] - s["R"][I]); J -= s["c1"][I] * r / (1 + s["b1"][I] * r)
        for j in range(i + 1, 5):
            r = np.linalg.norm(x[i] - x[j]); aij = s["a_par"] if (i < 3) == (j < 3) else s["a_anti"]
            J += aij * r / (1 + s["b2"] * r)
    la, sg = o.logpsi(x)
    assert sg == int(su * sd) and abs(la - (lu + ld + J)) < 1e-11
    # three-body Jastrow: J3 = sum_{i<j} sum_ab g_ab chi_a(r_i) chi_b(r_j), chi_a = exp(-zeta_a |r - R_a|^2), written out with numpy
    s3 = wl.with_jastrow3(s, 4, 2); o3 = ref.Ref(s3)
    chi = np.exp(-s3["j3_zeta"][None, :] * np.sum((x[:, None, :] - s["R"][s3["j3_center"]][None, :, :]) ** 2, axis=2))    # [electron][a]
    M = chi @ s3["j3_g"] @ chi.T
    J3 = np.sum(np.triu(M, 1))
    la3, sg3 = o3.logpsi(x)
    assert sg3 == sg and abs(la3 - (la + J3)) < 1e-12 and abs(J3) > 1e-3
    # the same with p and cartesian d functions and more than 8 of them: chi_a = dx^l dy^m dz^n exp(-zeta_a |d|^2), d = r - R_a
    sp = wl.with_jastrow3(s, 5, 6, n_max=12, poly=True); op = ref.Ref(sp)
    assert len(sp["j3_zeta"]) == 12 and set(map(int, sp["j3_lmn"].sum(axis=1))) == {0, 1, 2}
    d = x[:, None, :] - s["R"][sp["j3_center"]][None, :, :]                                                              # [electron][a][3]
    chi = np.prod(d ** sp["j3_lmn"][None, :, :], axis=2) * np.exp(-sp["j3_zeta"][None, :] * np.sum(d * d, axis=2))
    J3p = np.sum(np.triu(chi @ sp["j3_g"] @ chi.T, 1))
    lap_, sgp = op.logpsi(x)
    assert sgp == sg and abs(lap_ - (la + J3p)) < 1e-12 and abs(J3p) > 1e-3


@pytest.mark.parametrize("name", ["tiny-2u1d", "tiny-3u3d-pp", "C2"])
def test_sherman_morrison_tracks_full_reinversion(name):
    """After a whole branching interval of accepted moves the stored inverses equal the inverses rebuilt from the positions."""
    s = SYSTEMS[name](); o = ref.Ref(s)
    assert o.set_positions(wl.initial_walkers(s, 8, 55)) == 0
    assert o.propagate(ref.BALANCED, 25, 0.0, -100.0, 0) == 0
    r, du, dd, w = o.get_state(); _, _, _, nm = o.get_obs()
    assert nm.min() == 25
    for k in range(8):
        rc, du2, dd2 = o.build_inverse(r[k]); assert rc == 0
        assert np.allclose(du[k], du2, rtol=1e-7, atol=1e-9 * np.abs(du2).max())
        assert np.allclose(dd[k], dd2, rtol=1e-7, atol=1e-9 * max(1e-300, np.abs(dd2).max()))


# ----------------------------------------------------------------------------- fixed node + selection (pin P8)
def test_fixed_node_split_and_heat_bath_frequencies():
    """Two same-spin electrons, D = det[exp(-2r), exp(-0.6 r)] (nodal surface r1 = r2).  Put them at nearly equal radii:
    some hops cross the node (R_j < 0).  Those go to V_sf, never to bbar, and are never selected; selected-move
    frequencies over a fine u grid equal kappa R_j / bbar."""
    s = wl.slater_atom(2.0, [2.0, 0.6], 2, 0, np.eye(2), np.zeros((2, 0)), 0.2)
    o = ref.Ref(s); x = np.array([[0.5, 0.1, 0.0], [0.0, -0.1, 0.56]])
    R, sc, per, _ = o.evaluate(x, np.eye(3))
    assert (R < 0).any() and (R > 0).any() and sc["node"] == 1.0
    kap = 1 / (2 * 0.2**2)
    assert abs(sc["bbar"] - kap * R[R > 0].sum()) < 1e-12 * sc["bbar"]
    assert abs(sc["V_sf"] + kap * R[R < 0].sum()) < 1e-12 * max(1.0, sc["V_sf"])
    # W and e_L re-assembled from the per-electron pieces with the D9/D11 max branch active
    vopt = np.maximum(per[:, 3], per[:, 4])
    W = 3 * 2 / 0.2**2 + vopt.sum() + sc["V_ee"] + sc["V_ii"] + sc["V_sf"]
    assert abs(sc["W"] - W) < 1e-11 * abs(W) and abs(sc["e_L"] - (W - sc["bbar"])) < 1e-11 * abs(W)
    M = 20000; counts = np.zeros(len(R))
    for q in range(M):
        j, _ = o.select(R, (q + 0.5) / M); counts[j] += 1
    p = np.where(R > 0, R, 0.0); p /= p.sum()
    assert np.all(counts[R <= 0] == 0)
    assert np.abs(counts / M - p).max() < 1.5 / M
    # all moves forbidden -> no selection
    assert o.select(-np.abs(R), 0.3)[0] == -1


def test_selection_margin_and_fallback():
    o = ref.Ref(wl.hydrogen()); R = np.array([1.0, 0.0, -2.0, 3.0, 0.0, 0.0])
    assert o.select(R, 0.0)[0] == 0 and o.select(R, 0.2499999)[0] == 0 and o.select(R, 0.25)[0] == 3
    j, mg = o.select(R, 0.25 + 1e-12); assert j == 3 and abs(mg - 1e-12) < 1e-15
    assert o.select(R, 1.0 - 2.0**-53)[0] == 3          # largest u still lands on the last allowed move


# ----------------------------------------------------------------------------- pseudopotential form (reading Q14)
def test_local_pseudopotential_limits():
    """v(r) is finite at the nucleus (-> gamma), tends to -Z/r far away; a bare nucleus is exactly -Z/r."""
    s = wl.tiny_molecule(1, 0, 1, 1, seed=3, with_pp=True); o = ref.Ref(s)
    Z = s["Z"][0]; al, be, ga, de = s["pp"][0]; R0 = s["R"][0]
    for r, want in ((1e-6, ga), (8.0, -Z / 8.0)):
        x = (R0 + np.array([r, 0, 0]))[None, :]
        _, _, per, _ = o.evaluate(x, np.eye(3))
        assert abs(per[0, 2] - want) < 1e-5 * max(1.0, abs(want))
        assert abs(per[0, 4] + Z / r) < 1e-9 * Z / r          # ECP bound of L623: -Z_eff/r, no cutoff
    s2 = wl.tiny_molecule(1, 0, 1, 1, seed=3); o2 = ref.Ref(s2)
    x = (R0 + np.array([0.05, 0, 0]))[None, :]
    _, _, per, _ = o2.evaluate(x, np.eye(3))
    assert abs(per[0, 2] + Z / 0.05) < 1e-10 and abs(per[0, 4] + Z / 0.2) < 1e-12     # D10: -Z/max(r,a)


def test_local_pseudopotential_mid_range_formula():
    """The local-PP branch of v_ei at mid-range radii against the formula of include/lrdmc.h (lrdmc_system.pp, reading Q14)
    written out here: v(r) = -(Z/r)(1 - e^{-alpha r^2}) + Z alpha r e^{-beta r^2} + gamma e^{-delta r^2}.  At r = 0.3 / 0.7 / 1.5 the
    middle term is of order one: a wrong sign on it, a beta <-> delta swap or an alpha <-> beta swap fails this pin (each is
    shown to change the value by far more than the tolerance), while the r -> 0 and r -> infinity limits would not notice."""
    for seed in (3, 4):
        s = wl.tiny_molecule(1, 0, 1, 1, seed=seed, with_pp=True); o = ref.Ref(s)
        Z = float(s["Z"][0]); al, be, ga, de = (float(v) for v in s["pp"][0]); R0 = s["R"][0]
        for r in (0.3, 0.7, 1.5):
            want = -(Z / r) * (-math.expm1(-al * r * r)) + Z * al * r * math.exp(-be * r * r) + ga * math.exp(-de * r * r)
            for direction in (np.array([1.0, 0, 0]), np.array([0.6, 0.0, -0.8])):
                _, _, per, _ = o.evaluate((R0 + r * direction)[None, :], np.eye(3))
                assert abs(per[0, 2] - want) < 1e-13 * max(1.0, abs(want)), (seed, r)
                assert abs(per[0, 4] + Z / r) < 1e-13 * Z / r                     # L623: the bound of an ECP nucleus has no cutoff
            # the pin has teeth: the plausible mistakes move the value well beyond the tolerance at these radii
            wrong_sign = -(Z / r) * (-math.expm1(-al * r * r)) - Z * al * r * math.exp(-be * r * r) + ga * math.exp(-de * r * r)
            swap_bd = -(Z / r) * (-math.expm1(-al * r * r)) + Z * al * r * math.exp(-de * r * r) + ga * math.exp(-be * r * r)
            if r < 1.0:
                assert abs(wrong_sign - want) > 1e-6 and abs(swap_bd - want) > 1e-9
    # two PP nuclei: v_ei is the plain sum over nuclei of the same formula
    s = wl.tiny_molecule(2, 1, 2, 6, seed=8, with_pp=True); o = ref.Ref(s)
    x = wl.initial_walkers(s, 1, 3)[0]
    _, _, per, _ = o.evaluate(x, np.eye(3))
    for i in range(3):
        want = 0.0
        for I in range(2):
            r = float(np.linalg.norm(x[i] - s["R"][I])); Z = float(s["Z"][I]); al, be, ga, de = (float(v) for v in s["pp"][I])
            want += -(Z / r) * (-math.expm1(-al * r * r)) + Z * al * r * math.exp(-be * r * r) + ga * math.exp(-de * r * r)
        assert abs(per[i, 2] - want) < 1e-12 * max(1.0, abs(want))


def test_double_mesh_selection_weights_and_sums():
    """Double mesh (reading Q13, g = 1/2): the heat-bath selection draws candidate j with probability kappa_j max(R_j, 0) / bbar,
    kappa = (1/2)/(2 a^2) for the first 6N candidates (spacing a) and (1/2)/(2 a'^2) for the second 6N (spacing a').  Frequencies
    over a 20 000-point u grid against those weights written out here; a kappa that ignored the mesh (or swapped a and a') is
    shown to differ by far more than the grid resolution.  Also bbar, V_sf, K_diag and T_i re-assembled from R with the same kappas."""
    s = wl.tiny_molecule(2, 2, 2, 7, seed=9, a=0.15, a2=0.3); o = ref.Ref(s); N = 4
    rng = np.random.default_rng(17)
    x = wl.initial_walkers(s, 1, 21)[0]; U = _rand_frame(rng)
    R, sc, per, _ = o.evaluate(x, U)
    assert len(R) == 12 * N
    kap = np.concatenate([np.full(6 * N, 0.5 / (2 * 0.15**2)), np.full(6 * N, 0.5 / (2 * 0.3**2))])
    q = kap * np.maximum(R, 0.0)
    assert q[:6 * N].sum() > 0 and q[6 * N:].sum() > 0
    assert abs(sc["bbar"] - q.sum()) < 1e-12 * q.sum()
    assert abs(sc["V_sf"] - (kap * np.maximum(-R, 0.0)).sum()) < 1e-12 * max(1.0, sc["V_sf"])
    assert abs(sc["K_diag"] - kap.sum()) < 1e-12 * kap.sum()
    for i in range(N):          # T_i = g T_i(a) + (1-g) T_i(a'), T_i(a) = (sum_d R - 6)/a^2
        T = 0.5 * (R[6 * i:6 * i + 6].sum() - 6) / 0.15**2 + 0.5 * (R[6 * N + 6 * i:6 * N + 6 * i + 6].sum() - 6) / 0.3**2
        assert abs(per[i, 0] - T) < 1e-10 * max(1.0, abs(T))
    M = 20000; counts = np.zeros(len(R))
    for k in range(M):
        j, _ = o.select(R, (k + 0.5) / M); counts[j] += 1
    p = q / q.sum()
    assert np.all(counts[R <= 0] == 0)
    assert np.abs(counts / M - p).max() < 1.5 / M
    p_flat = np.maximum(R, 0.0) / np.maximum(R, 0.0).sum()           # the mistakes this pin must catch
    p_swap = kap[::-1] * np.maximum(R, 0.0); p_swap /= p_swap.sum()
    assert np.abs(p_flat - p).max() > 20 / M and np.abs(p_swap - p).max() > 20 / M
    # share of the coarse mesh among the selected moves = its share of bbar
    assert abs(counts[6 * N:].sum() / M - q[6 * N:].sum() / q.sum()) < 12 * N * 1.5 / M
