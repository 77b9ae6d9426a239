"""Whole-run pins of the oracle (CPU only, seconds each): exact energies the projection must reach,
balanced == conventional, branching invariants, the estimators of Eq.18-19, the Poisson trip-count law.
"""
import math

import numpy as np
import pytest

from oracle import lrdmc_ref as ref, ref_driver as drv
from paper_2508_12033_b200 import workloads as wl


def _fit_a2(a, E, sg):
    A = np.stack([np.ones_like(a), a**2], 1) / sg[:, None]
    cov = np.linalg.inv(A.T @ A); coef = cov @ A.T @ (E / sg)
    return coef[0], math.sqrt(cov[0, 0])


def test_zero_variance_run_keeps_unit_weights_and_exact_energy():
    """Psi_G = exact ground state (pin P5; Appendix B Eq.B2-B6): with E_0 = -1/2 every b_x = 1, weights stay 1,
    every generation gives e = -1/2 and wbar = 1, in both modes."""
    o = ref.Ref(wl.hydrogen(alpha=1.0, a=0.2))
    o.set_positions(wl.hydrogen_walkers(64, 1))
    out = drv.run(o, ref.BALANCED, 5, n_moves=30, E0=-0.5, feedback=False)
    assert np.abs(out["e"] + 0.5).max() < 1e-11 and np.abs(out["wbar"] - 1.0).max() < 1e-11
    assert out["moves_min"].min() == 30 and out["moves_max"].max() == 30 and out["lockstep_idle_frac"].max() == 0.0
    o.set_positions(wl.hydrogen_walkers(64, 1))
    out = drv.run(o, ref.CONVENTIONAL, 5, tau=0.4, E_ref=-0.5)
    assert np.abs(out["e"] + 0.5).max() < 1e-11 and np.abs(out["wbar"] - 1.0).max() < 1e-10
    assert out["moves_max"].max() > out["moves_min"].min()          # stochastic trip count (L168)


def test_hydrogen_energy_extrapolates_to_minus_half():
    """Config C1 (alpha = 0.9, variational energy alpha^2/2 - alpha = -0.495): LRDMC must project to
    E(a) = -1/2 + c a^2 (L23, L140); intercept within 3 sigma of the exact -0.5 (pin P6)."""
    a = np.array([0.15, 0.25, 0.35, 0.45]); E = []; sg = []
    for ai in a:
        o = ref.Ref(wl.hydrogen(alpha=0.9, a=float(ai))); o.set_positions(wl.hydrogen_walkers(256, 1))
        out = drv.run(o, ref.BALANCED, 300, n_moves=max(4, int(round(40 * (0.2 / ai) ** 2))), E0=-0.495)
        e, s = drv.energy(out["wbar"], out["num"], out["den"], p=10, n_therm=60); E.append(e); sg.append(s)
        assert out["n_nonpos_diag"].sum() == 0 and out["n_nonfinite"].sum() == 0 and out["n_node_flag"].sum() == 0
    E0, s0 = _fit_a2(a, np.array(E), np.array(sg))
    assert abs(E0 + 0.5) < 3 * s0 and s0 < 2e-3
    assert np.all(np.array(E) < -0.495 + 3 * np.array(sg))           # below the variational energy: it really projects


def test_helium_singlet_reaches_the_exact_nonrelativistic_energy():
    """Nodeless two-electron ground state (pin P7): FN is exact, so E(a -> 0) = -2.903724 Ha (textbook value).
    Exercises two spins, e-e repulsion, the two-body Jastrow and its gradient cross terms in the run."""
    a = np.array([0.15, 0.25, 0.35]); E = []; sg = []; rng = np.random.default_rng(0)
    for ai in a:
        s = wl.slater_atom(2.0, [1.85], 1, 1, np.ones((1, 1)), np.ones((1, 1)), float(ai), jastrow=dict(a_anti=0.5, a_par=0.25, b2=0.5))
        o = ref.Ref(s); assert o.set_positions(rng.normal(size=(512, 2, 3)) * 0.7) == 0
        out = drv.run(o, ref.BALANCED, 400, n_moves=int(round(20 * (0.2 / ai) ** 2)), E0=-2.9)
        e, sgm = drv.energy(out["wbar"], out["num"], out["den"], p=10, n_therm=80); E.append(e); sg.append(sgm)
    E0, s0 = _fit_a2(a, np.array(E), np.array(sg))
    assert abs(E0 + 2.903724) < 3 * s0 and s0 < 4e-3


def test_helium_triplet_fixed_node_energy():
    """He 2^3S with D = det[exp(-2r), exp(-0.6r)]: the node r1 = r2 is exact, so fixed-node LRDMC gives -2.175229 Ha as
    a -> 0 (pin P8).  Exercises V_sf, the node flag and the D9/D11 max branch inside a run."""
    # The lattice bias of this system is below the noise already at a = 0.2 (a longer oracle run gave -2.17542(34) at
    # a = 0.2 and -2.17518(60) at a = 0.12), so one a suffices; 5e-4 of slack covers it.  10 blocks: generations are correlated.
    rng = np.random.default_rng(1)
    s = wl.slater_atom(2.0, [2.0, 0.6], 2, 0, np.eye(2), np.zeros((2, 0)), 0.2, jastrow=dict(a_par=0.25, a_anti=0.5, b2=0.5))
    o = ref.Ref(s)
    x = rng.normal(size=(1024, 2, 3)); x[:, 0] *= 0.4; x[:, 1] *= 2.0
    assert o.set_positions(x) == 0
    out = drv.run(o, ref.BALANCED, 600, n_moves=30, E0=-2.17)
    E, sg = drv.energy(out["wbar"], out["num"], out["den"], p=10, n_therm=100, n_blocks=10)
    assert out["n_node_flag"].sum() > 0 and out["n_nonpos_diag"].sum() == 0
    assert abs(E + 2.175229) < 3 * sg + 5e-4 and sg < 2e-3


@pytest.mark.parametrize("system", ["C1", "tiny"])
def test_balanced_and_conventional_agree(system):
    """'both algorithms sample the same fixed-node ground state at fixed a' (L244, Table I; pin P12):
    energies within 3 combined sigma when the mean number of moves per branching is the same (L234)."""
    if system == "C1":
        s = wl.hydrogen(alpha=0.9, a=0.2); x0 = wl.hydrogen_walkers(256, 1); n_moves, cycles, E0 = 40, 300, -0.495
    else:
        s = wl.slater_atom(2.0, [1.85], 1, 1, np.ones((1, 1)), np.ones((1, 1)), 0.25, jastrow=dict(a_anti=0.5, a_par=0.25, b2=0.5))
        x0 = np.random.default_rng(2).normal(size=(256, 2, 3)) * 0.7; n_moves, cycles, E0 = 16, 300, -2.9
    o = ref.Ref(s); o.set_positions(x0)
    ob = drv.run(o, ref.BALANCED, cycles, n_moves=n_moves, E0=E0)
    Eb, sb = drv.energy(ob["wbar"], ob["num"], ob["den"], p=10, n_therm=60)
    N = s["n_up"] + s["n_dn"]
    tau = n_moves * s["a"] ** 2 / (3 * N)                      # first guess of reading Q19: mean rate bbar ~ 3N/a^2
    o.set_positions(x0)
    oc = drv.run(o, ref.CONVENTIONAL, cycles, tau=tau, E_ref=E0)
    Ec, sc = drv.energy(oc["wbar"], oc["num"], oc["den"], p=10, n_therm=60)
    mean_moves = oc["moves_sum"].mean() / len(x0)
    assert abs(mean_moves - n_moves) < 0.15 * n_moves
    assert abs(Eb - Ec) < 3 * math.hypot(sb, sc)
    assert ob["lockstep_idle_frac"].max() == 0.0 and oc["lockstep_idle_frac"].mean() > 0.1   # the paper's point (L168)


def test_conventional_trip_counts_follow_the_poisson_law():
    """Appendix C (L552): at a constant rate b the number of hops in time tau is Poisson(tau b).  With Psi_G = exp(-r)
    sampled far from the nucleus the rate bbar ~ 3/a^2 is nearly constant; mean and variance of the counts must match."""
    o = ref.Ref(wl.hydrogen(alpha=1.0, a=0.1)); o.set_positions(wl.hydrogen_walkers(2000, 3))
    tau = 0.5; assert o.propagate(ref.CONVENTIONAL, 0, tau, -0.5, 0) == 0
    _, _, _, nm = o.get_obs()
    lam = tau * 3 / 0.1**2
    assert abs(nm.mean() - lam) < 0.03 * lam and abs(nm.var() / nm.mean() - 1.0) < 0.25


def test_reconfiguration_in_a_run_copies_whole_walkers_and_resets_weights():
    s = wl.tiny_molecule(2, 1, 2, 6, seed=7); o = ref.Ref(s); x0 = wl.initial_walkers(s, 32, 3)
    assert o.set_positions(x0) == 0 and o.propagate(ref.BALANCED, 10, 0.0, -50.0, 4) == 0
    r1, du1, dd1, w1 = o.get_state()
    rc, par = o.reconfigure(4); assert rc == 0
    r2, du2, dd2, w2 = o.get_state()
    rc_, par_direct, wbar, *_ = ref.comb(w1, o.comb_r32(4))
    assert list(par) == list(par_direct) and np.array_equal(r2, r1[par]) and np.all(w2 == 1.0)
    assert abs(o.estimators()["wbar"] - w1.mean()) < 1e-12 * w1.mean()
    for k in range(32):                                           # inverses rebuilt from the copied positions (Q15)
        rc, du, dd = o.build_inverse(r2[k]); assert np.array_equal(du, du2[k]) and np.array_equal(dd, dd2[k])


def test_population_factor_and_energy_estimator():
    """Eq.18-19 on a hand-made series: G_n^p = product of the p previous wbar; constant e -> E = e, sigma = 0;
    p = 0 -> plain mean of e_n."""
    wbar = np.array([2.0, 0.5, 3.0, 1.0, 4.0])
    assert list(drv.population_factors(wbar, 2)) == [1.0, 2.0, 1.0, 1.5, 3.0]
    num = np.array([1.0, 2.0, 3.0, 4.0, 5.0]); den = np.ones(5)
    E, sg = drv.energy(wbar, num, den, p=2, n_therm=1, n_blocks=4)
    assert abs(E - (2 * 2 + 1 * 3 + 1.5 * 4 + 3 * 5) / 7.5) < 1e-14
    E, sg = drv.energy(wbar, num, den, p=0, n_therm=0)
    assert abs(E - 3.0) < 1e-14
    E, sg = drv.energy(wbar, -0.5 * np.ones(5), den, p=3)
    assert E == -0.5 and sg < 1e-15


def test_singular_walkers_are_dead_until_the_next_branching():
    """Reading Q24: a walker whose Slater matrix is singular (here: two same-spin electrons at one point, and a matrix with a pivot
    of rounding size) is reported by set_positions (ESINGULAR), gets zero inverses, is never evaluated, leaves propagate with
    w = omega = 0 and no moves, is never chosen as a parent, and is gone after the branching."""
    s = wl.tiny_molecule(2, 1, 2, 6, seed=7); o = ref.Ref(s)
    x = wl.initial_walkers(s, 6, 3); x[2, 1] = x[2, 0]; x[4, 1] = x[4, 0]        # coincident same-spin pairs in walkers 2 and 4
    assert o.set_positions(x) == -2
    r, du, dd, w = o.get_state()
    assert np.all(du[[2, 4]] == 0.0) and np.all(dd[[2, 4]] == 0.0) and np.abs(du[0]).max() > 0
    rc, du1, dd1 = o.build_inverse(x[2]); assert rc == -2
    # the live walkers are untouched by their dead neighbours: same trajectories as in an ensemble without them
    o2 = ref.Ref(s); keep = [0, 1, 3, 5]
    assert o.propagate(ref.BALANCED, 7, 0.0, -5.0, 0) == 0
    eL, W, om, nm = o.get_obs(); r1, _, _, w1 = o.get_state()
    assert np.all(w1[[2, 4]] == 0.0) and np.all(om[[2, 4]] == 0.0) and np.all(nm[[2, 4]] == 0) and np.all(nm[keep] == 7)
    assert np.array_equal(r1[[2, 4]], x[[2, 4]])
    for k in keep:
        o2.set_slot_offset(k); assert o2.set_positions(x[k:k + 1]) == 0
        assert o2.propagate(ref.BALANCED, 7, 0.0, -5.0, 0) == 0
        assert np.array_equal(o2.get_state()[0][0], r1[k]) and o2.get_state()[3][0] == w1[k]
    st = o.estimators(); assert st["n_singular"] == 2 and st["moves_sum"] == 28
    rc, par = o.reconfigure(0); assert rc == 0
    assert 2 not in par and 4 not in par
    assert o.estimators()["n_singular"] == 0 and abs(o.estimators()["wbar"] - w1.sum() / 6) < 1e-12
    # a matrix with two rows equal up to rounding noise is singular by the 2^-44 rule, a well-conditioned one is not
    A = np.random.default_rng(0).normal(size=(5, 5)); B_ = A.copy(); B_[3] = A[1] * (1 + 2e-16)
    import ctypes as C
    inv = np.zeros((5, 5))
    f = ref.lib().ref_invert; f.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    assert f(5, A.ctypes.data, inv.ctypes.data, None, None) == 0 and np.allclose(inv @ A, np.eye(5), atol=1e-12)
    assert f(5, B_.ctypes.data, inv.ctypes.data, None, None) == -2


def test_a_scan_fit_closed_forms_and_independent_runs():
    """oracle.ref_driver.a_scan / fit_even_powers (the oracle side of scope row f3).  The fit against closed forms: exact data
    E = E_0 + c a^2 are reproduced; for equal error bars sigma(E_0) equals the textbook intercept error of a straight line in
    a^2; a four-point, three-term fit of exact quartic data returns its intercept.  The scan: every (a, mode) run has its own
    Philox key (first generations differ between runs that share a and the walkers), rows carry (E, sigma) per mode."""
    a = np.array([0.1, 0.2, 0.3, 0.4]); x = a**2; sg = np.full(4, 2e-3)
    E0, s0 = drv.fit_even_powers(a, -0.5 + 0.3 * x, sg)
    assert abs(E0 + 0.5) < 1e-13
    assert abs(s0 - 2e-3 * np.sqrt(np.sum(x**2) / (4 * np.sum(x**2) - np.sum(x)**2))) < 1e-15
    E0, _ = drv.fit_even_powers(a, 1.25 - 2 * x + 7 * x**2, sg, n_terms=3)
    assert abs(E0 - 1.25) < 1e-11
    # a point with a tiny error bar pins the curve
    E0, _ = drv.fit_even_powers([0.0, 0.2, 0.4], [3.0, 9.0, -4.0], [1e-9, 1.0, 1.0])
    assert abs(E0 - 3.0) < 1e-8
    mk = lambda a_: wl.hydrogen(alpha=0.9, a=a_); mw = lambda s, n: wl.hydrogen_walkers(n, 1)
    out = drv.a_scan(mk, mw, [0.2, 0.4], n_walkers=48, cycles=12, moves=8, E0=-0.5, n_blocks=4)
    assert [r["a"] for r in out["rows"]] == [0.2, 0.4]
    for r in out["rows"]:
        for mode in ("balanced", "conventional"):
            E, s = r[mode]; assert -0.8 < E < -0.3 and s > 0
    # run q = 0 is what ref_driver.run gives with key seed + 1000003, and differs from a run with the unshifted key
    s = dict(mk(0.2)); s["seed"] += 1000003
    o = ref.Ref(s); o.set_positions(mw(s, 48)); e_shift = drv.run(o, ref.BALANCED, 3, n_moves=8, E0=-0.5)["e"]
    o = ref.Ref(mk(0.2)); o.set_positions(mw(s, 48)); e_plain = drv.run(o, ref.BALANCED, 3, n_moves=8, E0=-0.5)["e"]
    assert np.array_equal(out["rows"][0]["balanced_first_e"], e_shift) and not np.array_equal(e_shift, e_plain)
    assert len(out["balanced"]) == 2 and out["balanced"][1] > 0
