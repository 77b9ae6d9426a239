"""Parity of the CUDA path (through the C-ABI binding) with the CPU oracle on identical seeded inputs.  -m gpu.

Tolerances: FP64 quantities within 1e-10 relative to max(|value|, natural scale) where
the natural scale is the size of the summands the value is assembled from (1 for a wavefunction ratio, K_diag = 3N/a^2
for W and e_L, max|Dinv| for an inverse); selected moves, trip counts and reconfiguration indices bit-exact.
"""
import numpy as np
import pytest

from oracle import lrdmc_ref as ref, ref_driver as rdrv
from paper_2508_12033_b200 import workloads as wl
from conftest import read_golden

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2508_12033_b200 import binding
    binding.load_library()
    return binding


def np_(t):
    return t.cpu().numpy()


def relerr(a, b, scale=0.0):
    a = np.asarray(a, float); b = np.asarray(b, float)
    return float(np.max(np.abs(a - b) / np.maximum(np.maximum(np.abs(a), np.abs(b)), max(scale, 1e-300)))) if a.size else 0.0


SYSTEMS = {
    "C1-hydrogen": lambda: (wl.hydrogen(), wl.hydrogen_walkers(256, 1)),
    "tiny-2u1d": lambda: _with_walkers(wl.tiny_molecule(2, 1, 2, 6, seed=7), 37),
    "tiny-3u3d-pp": lambda: _with_walkers(wl.tiny_molecule(3, 3, 3, 9, seed=8, with_pp=True), 37),
    "tiny-2u2d-doublemesh": lambda: _with_walkers(wl.tiny_molecule(2, 2, 2, 7, seed=9, a=0.15, a2=0.3), 41),
    "ragged-5u2d": lambda: _with_walkers(wl.tiny_molecule(5, 2, 3, 11, seed=10), 19),
    "ragged-9u4d-NT2": lambda: _with_walkers(wl.tiny_molecule(9, 4, 4, 20, seed=11), 13),
    "ragged-17u3d-NT4": lambda: _with_walkers(wl.tiny_molecule(17, 3, 5, 30, seed=12), 9),
    "he-triplet-slater": lambda: _with_walkers(wl.slater_atom(2.0, [2.0, 0.6], 2, 0, np.eye(2), np.zeros((2, 0)), 0.2, jastrow=dict(a_par=0.25, a_anti=0.5, b2=0.5)), 64),
    "C2-synthetic10": lambda: _with_walkers(wl.synthetic10(), 1024),          # BASELINE configs[1] at its full N_w
    "C3-water-methane-shaped": lambda: _with_walkers(wl.water_methane(n_walkers=100), 100),
    "C5-cluster64-doublemesh": lambda: _with_walkers(wl.cluster64(n_walkers=10), 10),   # 64 e, 600 AOs, a/a' (NT = 4, tables in global memory)
    # scope row f1: non-local pseudopotential channels (synthetic), determinant locality (DLA) and full-ratio (T-move) forms
    "hydrogen-nl-s-channel": lambda: (wl.with_nonlocal(wl.hydrogen(alpha=1.1), [[2.2, -0.8, 1.5, 0, 1, 0, 1]]), wl.hydrogen_walkers(100, 3)),
    "tiny-3u2d-nlDLA-K2": lambda: _with_walkers(wl.random_nonlocal(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 5, 1.6, 2, True), 37),
    "tiny-3u2d-nlTM-K2": lambda: _with_walkers(wl.random_nonlocal(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 5, 1.6, 2, False), 37),
    "tiny-3u2d-nlDLA-strong": lambda: _with_walkers(wl.random_nonlocal(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 5, 1.6, 2, True, scale=200.0), 37),
    "tiny-2u1d-nlTM-strong": lambda: _with_walkers(wl.random_nonlocal(wl.tiny_molecule(2, 1, 2, 6, seed=7), 8, 1.4, 1, False, scale=600.0), 41),
    "tiny-2u2d-doublemesh-nlTM": lambda: _with_walkers(wl.random_nonlocal(wl.tiny_molecule(2, 2, 2, 7, seed=9, a=0.15, a2=0.3), 4, 1.5, 2, False, scale=150.0), 33),
    "ragged-9u4d-nlDLA": lambda: _with_walkers(wl.random_nonlocal(wl.tiny_molecule(9, 4, 4, 20, seed=11), 6, 1.2, 2, True), 13),
    "C3-water-methane-nlDLA": lambda: _with_walkers(wl.water_methane_nonlocal(n_walkers=100), 100),
    "C3-water-methane-nlTM": lambda: _with_walkers(wl.water_methane_nonlocal(n_walkers=50, dla=False), 50),
    # scope row f2: contracted shells and real solid-harmonic d shells (the oracle evaluates the contracted functions themselves,
    # lrdmc_init folds the contraction into its primitive coefficient tables)
    "contracted-3u2d-sph-pp": lambda: _with_walkers(wl.contracted_molecule(3, 2, 3, 9, seed=31, spherical=True, with_pp=True), 37),
    "contracted-9u7d-cart": lambda: _with_walkers(wl.contracted_molecule(9, 7, 4, 21, seed=32, spherical=False), 21),
    "contracted-slater-spd": lambda: _with_walkers(wl.contracted_slater_molecule(), 45),                # contracted Slater shells + Gaussian p / solid-harmonic d
    "contracted-slater-only": lambda: _with_walkers(wl.contracted_slater_molecule(with_gaussians=False), 33),
    # scope row f2: three-body Jastrow (s Gaussians at the nuclei), alone, with non-local slots in the full-ratio form, on C3
    "tiny-3u2d-pp-J3": lambda: _with_walkers(wl.with_jastrow3(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 4, 2), 37),
    "tiny-3u2d-J3-nlTM": lambda: _with_walkers(wl.with_jastrow3(wl.random_nonlocal(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 5, 1.6, 2, False, scale=200.0), 4, 2), 37),
    "ragged-9u4d-J3": lambda: _with_walkers(wl.with_jastrow3(wl.tiny_molecule(9, 4, 4, 20, seed=11), 6, 2, strength=0.1), 13),
    # scope row f2 (remainder): p and cartesian d functions in the three-body Jastrow, more than 8 functions (12, 12, 24)
    "tiny-3u2d-pp-J3spd": lambda: _with_walkers(wl.with_jastrow3(wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True), 5, 4, n_max=12, poly=True), 37),
    "ragged-9u4d-J3spd-nlTM": lambda: _with_walkers(wl.with_jastrow3(wl.random_nonlocal(wl.tiny_molecule(9, 4, 4, 20, seed=11), 5, 1.6, 2, False, scale=50.0), 6, 3, strength=0.1, n_max=12, poly=True), 13),
    "C3-water-methane-J3spd": lambda: _with_walkers(wl.with_jastrow3(wl.water_methane(n_walkers=100), 8, 3, strength=0.03, n_max=24, poly=True), 100),
    "C3-water-methane-J3": lambda: _with_walkers(wl.with_jastrow3(wl.water_methane(n_walkers=100), 7, 1, strength=0.05), 100),
    "contracted-4u4d-sph-nlDLA": lambda: _with_walkers(wl.random_nonlocal(wl.contracted_molecule(4, 4, 3, 12, seed=33, spherical=True, with_pp=True), 9, 1.5, 2, True, scale=100.0), 29),
}


def _with_walkers(s, n):
    return s, wl.initial_walkers(s, n, 5)


def _pair(B, name, options=None):
    s, x0 = SYSTEMS[name]()
    o = ref.Ref(s); rc = o.set_positions(x0); assert rc == 0, rc
    g = B.Lrdmc(s, options=options); g.lrdmc_set_positions(x0)
    return s, x0, o, g


# ------------------------------------------------------------------------------------------ a0: RNG + frame
def test_philox_device_matches_oracle_and_known_answers(B):
    g = B.Lrdmc(wl.hydrogen())
    kat = read_golden("philox4x32_10_kat.txt")
    for name, v in kat.items():
        x = [int(t, 16) for t in v]
        out = g.debug_philox(np.array([x[0:4]], dtype=np.uint32), (x[4], x[5]))
        assert [int(t) for t in out[0]] == x[6:10], name
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2**32, size=(1000, 4), dtype=np.uint64).astype(np.uint32)
    out = g.debug_philox(ctr, (0xDEADBEEF, 0x12345678))
    for i in range(0, 1000, 7):
        assert tuple(int(t) for t in out[i]) == ref.philox4x32_10([int(t) for t in ctr[i]], (0xDEADBEEF, 0x12345678))


def test_draws_and_frames_match_oracle(B):
    s = wl.synthetic10(); g = B.Lrdmc(s); o = ref.Ref(s)
    out = np_(g.debug_draws(9, 4, 500))
    for k in range(0, 500, 3):
        u = o.draws(k, 9, 4)
        assert np.array_equal(out[k, :5], u)                      # uniforms are integer arithmetic: bit-exact
        assert np.abs(out[k, 5:].reshape(3, 3) - ref.frame(u[0], u[1], u[2])).max() < 2e-15   # sincospi vs sin(2 pi u): a few ulp


# ------------------------------------------------------------------------------------------ a13: inverse build
@pytest.mark.parametrize("name", list(SYSTEMS))
def test_set_positions_builds_the_same_inverse(B, name):
    s, x0, o, g = _pair(B, name)
    r, du, dd, w = o.get_state(); gr, gdu, gdd, gw = [np_(t) for t in g.lrdmc_get_walkers()]
    assert np.array_equal(gr, r) and np.all(gw == 1.0)
    for a, b in ((gdu, du), (gdd, dd)):
        if b.size:
            sc = np.abs(b).max(axis=(1, 2), keepdims=True)
            assert np.max(np.abs(a - b) / sc) < 1e-8          # conditioning of random Slater matrices, not arithmetic


# ------------------------------------------------------------------------------------------ a1-a9: one step
@pytest.mark.parametrize("name", list(SYSTEMS))
def test_one_evaluation_and_selection_from_the_oracle_state(B, name):
    s, x0, o, g = _pair(B, name)
    N = s["n_up"] + s["n_dn"]
    r, du, dd, w = o.get_state(); g.lrdmc_set_state(r, du, dd, w)
    for (E0, cycle, step) in ((-3.0, 0, 0), (0.5, 7, 3)):
        R, scal, js = o.step_debug(E0, cycle, step)
        gR, gscal, gjs = [np_(t) for t in g.lrdmc_step_debug(E0, cycle, step)]
        assert gR.shape == R.shape == (len(x0), 6 * N * ((2 if s["a2"] > 0 else 1) + s["nl_K"]))
        if s["nl_K"]:
            assert np.count_nonzero(R[:, 6 * N * (2 if s["a2"] > 0 else 1):]) > 0        # the non-local slots are exercised
        Kdiag = scal[:, 2:3] * 0 + 3 * N * ((1 / s["a"]**2) if s["a2"] == 0 else (0.5 / s["a"]**2 + 0.5 / s["a2"]**2))
        assert relerr(gR, R, 1.0) < TOL                                                  # ratios
        for col, nm in ((0, "bbar"), (1, "V_sf"), (2, "W"), (3, "e_L")):
            assert np.max(np.abs(gscal[:, col] - scal[:, col]) / np.maximum(np.abs(scal[:, col]), Kdiag[:, 0])) < TOL, nm
        ok = np.abs(scal[:, 2] - E0) > 1e-6 * Kdiag[:, 0]
        assert relerr(gscal[ok, 4], scal[ok, 4]) < 1e-9                                   # b_x = bbar/(W-E0)
        assert relerr(gscal[:, 5], scal[:, 5]) < TOL and np.array_equal(gscal[:, 6], scal[:, 6])   # tau_xi, node flag
        near_tie = scal[:, 7] < 1e-9
        assert np.array_equal(gjs[~near_tie], js[~near_tie]) and near_tie.sum() == 0      # selected moves: bit-exact
    g.close()


# ------------------------------------------------------------------------------------------ whole cycles
@pytest.mark.parametrize("name", list(SYSTEMS))
@pytest.mark.parametrize("mode", ["balanced", "conventional"])
@pytest.mark.parametrize("kernel", ["warp-per-walker", "auto"])
def test_whole_cycle_trajectories_weights_and_branching(B, name, mode, kernel):
    """kernel = warp-per-walker forces k_propagate (lrdmc_set_option LRDMC_OPT_TEAM_WARPS = 1); auto lets lrdmc_bind_walkers pick
    the team size (k_propagate_team for these small ensembles and for the 64-electron system), as bench.py and a user get it."""
    g = _whole_cycles(B, name, mode, keep=True, options={B.OPT_TEAM_WARPS: 1} if kernel == "warp-per-walker" else None)
    if kernel == "warp-per-walker":
        assert g.launch_config()["kernel"] == "k_propagate"
    g.close()


@pytest.mark.parametrize("tw", [2, 4, 8, 16])
@pytest.mark.parametrize("name,mode", [("tiny-3u3d-pp", "balanced"), ("tiny-2u2d-doublemesh", "conventional"), ("ragged-9u4d-NT2", "balanced"),
                                       ("ragged-17u3d-NT4", "conventional"), ("he-triplet-slater", "balanced"), ("C3-water-methane-shaped", "balanced"),
                                       ("C3-water-methane-shaped", "conventional"), ("C5-cluster64-doublemesh", "balanced"),
                                       ("tiny-3u2d-nlDLA-strong", "balanced"), ("tiny-2u1d-nlTM-strong", "conventional"), ("C3-water-methane-nlDLA", "balanced"),
                                       ("C3-water-methane-nlTM", "balanced"), ("contracted-4u4d-sph-nlDLA", "balanced"), ("tiny-2u2d-doublemesh-nlTM", "conventional"),
                                       ("tiny-3u2d-pp-J3", "balanced"), ("tiny-3u2d-J3-nlTM", "conventional"), ("C3-water-methane-J3", "balanced"),
                                       ("tiny-3u2d-pp-J3spd", "balanced"), ("ragged-9u4d-J3spd-nlTM", "conventional"), ("C3-water-methane-J3spd", "balanced")])
def test_team_kernel_every_team_size(B, name, mode, tw):
    """k_propagate_team with TW = 2, 4, 8, 16 warps per walker (work units = electron blocks x shell parts, partial sums
    in shared memory): same trajectories, weights and indices as the oracle."""
    g = _whole_cycles(B, name, mode, n_cycles=1, keep=True, options={B.OPT_TEAM_WARPS: tw})
    cfg = g.launch_config()
    assert cfg["block"] == 32 * tw and cfg["team_warps"] == tw and cfg["kernel"] == "k_propagate_team"
    g.close()


@pytest.mark.parametrize("name", ["C3-water-methane-shaped", "tiny-3u2d-nlDLA-strong", "C5-cluster64-doublemesh"])
def test_team_kernel_is_bitwise_reproducible(B, name):
    """compute-sanitizer is not available on the GPU pool; a shared-memory race between the warps of a team would show as
    run-to-run differences.  Three runs of the same cycle from the same state must agree bit for bit (positions, inverses,
    weights, local energies), for the largest team."""
    s, x0 = SYSTEMS[name]()
    outs = []
    for rep in range(3):
        g = B.Lrdmc(s, options={B.OPT_TEAM_WARPS: 16}); g.lrdmc_set_positions(x0)
        g.lrdmc_propagate(B.BALANCED, 25, 0.0, -5.0, 3)
        outs.append([np_(t).copy() for t in g.lrdmc_get_walkers()] + [np_(t).copy() for t in g.lrdmc_get_obs()])
        assert g.launch_config()["block"] == 512
        g.close()
    for other in outs[1:]:
        for a, b in zip(outs[0], other):
            assert np.array_equal(a, b)


def _whole_cycles(B, name, mode, n_cycles=2, keep=False, options=None):
    s, x0, o, g = _pair(B, name, options)
    N = s["n_up"] + s["n_dn"]; n_moves = 30
    for cycle in range(n_cycles):
        if mode == "balanced":
            assert o.propagate(ref.BALANCED, n_moves, 0.0, -5.0, cycle) == 0
            g.lrdmc_propagate(B.BALANCED, n_moves, 0.0, -5.0, cycle)
        else:
            tau = n_moves * s["a"]**2 / (3 * N)
            assert o.propagate(ref.CONVENTIONAL, 0, tau, -1.0, cycle) == 0
            g.lrdmc_propagate(B.CONVENTIONAL, 0, tau, -1.0, cycle)
        r, du, dd, w = o.get_state(); gr, gdu, gdd, gw = [np_(t) for t in g.lrdmc_get_walkers()]
        eL, W, om, nm = o.get_obs(); geL, gW, gom, gnm = [np_(t) for t in g.lrdmc_get_obs()]
        assert np.array_equal(gnm, nm)                                                    # trip counts bit-exact
        assert np.abs(gr - r).max() < 1e-11                                               # same trajectory
        assert relerr(gw, w) < 1e-9 and relerr(gom, om) < 1e-9                            # products of ~30 factors
        Kd = 3 * N / s["a"]**2
        assert np.max(np.abs(geL - eL) / np.maximum(np.abs(eL), Kd)) < TOL and relerr(gW, W) < TOL
        rc, par = o.reconfigure(cycle); gpar = np_(g.lrdmc_reconfigure(cycle, want_parents=True))
        so, sg = o.estimators(), g.lrdmc_estimators()
        assert np.array_equal(gpar, par)                                                  # reconfiguration indices bit-exact
        assert abs(sg.wbar - so["wbar"]) <= 1e-9 * so["wbar"]
        assert abs(sg.num - so["num"]) <= 1e-9 * max(abs(so["num"]), Kd * so["den"]) and abs(sg.den - so["den"]) <= 1e-9 * so["den"]
        assert (sg.moves_min, sg.moves_max, sg.moves_sum) == (so["moves_min"], so["moves_max"], so["moves_sum"])
        assert (sg.n_node_flag, sg.n_nonpos_diag, sg.n_nonfinite) == (so["n_node_flag"], so["n_nonpos_diag"], so["n_nonfinite"])
        assert abs(sg.lockstep_idle_frac - so["lockstep_idle_frac"]) < 1e-12
        r2, *_ = o.get_state(); gr2 = np_(g.lrdmc_get_walkers()[0])
        assert np.abs(gr2 - r2).max() < 1e-11 and np.all(np_(g.lrdmc_get_walkers()[3]) == 1.0)
    if keep:
        return g
    g.close()


LATTICE_ONLY = ["C1-hydrogen", "tiny-2u1d", "tiny-3u3d-pp", "tiny-2u2d-doublemesh", "ragged-5u2d", "ragged-9u4d-NT2", "ragged-17u3d-NT4", "he-triplet-slater",
                "C2-synthetic10", "C3-water-methane-shaped", "contracted-3u2d-sph-pp", "contracted-9u7d-cart", "contracted-slater-spd"]


@pytest.mark.parametrize("name", LATTICE_ONLY)
@pytest.mark.parametrize("mode", ["balanced", "conventional"])
@pytest.mark.parametrize("tw", [1, 4])
def test_listed_sweep_forced_on_small_systems(B, name, mode, tw):
    """lrdmc_set_option(LRDMC_OPT_LISTED, 1): per-electron shell lists + Bc = C Dinv as rank-1-updated state (the candidate pass of the 64-electron
    configuration) forced on every lattice-only system, with tables in shared memory, in the warp-per-walker and the team kernel: one evaluation and
    whole cycles against the oracle (which never screens)."""
    s, x0, o, g = _pair(B, name, {B.OPT_LISTED: 1, B.OPT_TEAM_WARPS: tw})
    N = s["n_up"] + s["n_dn"]; Kd = 3 * N / s["a"]**2
    r, du, dd, w = o.get_state(); g.lrdmc_set_state(r, du, dd, w)
    R, scal, js = o.step_debug(-3.0, 2, 1)
    gR, gscal, gjs = [np_(t) for t in g.lrdmc_step_debug(-3.0, 2, 1)]
    assert relerr(gR, R, 1.0) < TOL and np.array_equal(gjs, js)
    assert np.max(np.abs(gscal[:, :4] - scal[:, :4]) / np.maximum(np.abs(scal[:, :4]), Kd)) < TOL
    g.close()
    g = _whole_cycles(B, name, mode, keep=True, options={B.OPT_LISTED: 1, B.OPT_TEAM_WARPS: tw})
    assert g.launch_config()["kernel"] == ("k_propagate" if tw == 1 else "k_propagate_team")
    g.close()


@pytest.mark.parametrize("name", ["C1-hydrogen", "tiny-3u3d-pp", "C3-water-methane-shaped"])
def test_large_system_path_tables_in_global_memory(B, name):
    """The kernels of systems whose tables do not fit shared memory (C5) read fragments and MO cache from global memory;
    lrdmc_set_option(LRDMC_OPT_GLOBAL_TABLES) forces that path on small systems so that it is compared with the oracle on every run."""
    s, x0, o, g = _pair(B, name, {B.OPT_GLOBAL_TABLES: 1})
    N = s["n_up"] + s["n_dn"]; Kd = 3 * N / s["a"]**2
    r, du, dd, w = o.get_state(); g.lrdmc_set_state(r, du, dd, w)
    R, scal, js = o.step_debug(-3.0, 2, 1)
    gR, gscal, gjs = [np_(t) for t in g.lrdmc_step_debug(-3.0, 2, 1)]
    assert relerr(gR, R, 1.0) < TOL and np.array_equal(gjs, js)
    assert np.max(np.abs(gscal[:, :4] - scal[:, :4]) / np.maximum(np.abs(scal[:, :4]), Kd)) < TOL
    assert o.propagate(ref.BALANCED, 12, 0.0, -5.0, 4) == 0
    g.lrdmc_propagate(B.BALANCED, 12, 0.0, -5.0, 4)
    assert np.abs(np_(g.lrdmc_get_walkers()[0]) - o.get_state()[0]).max() < 1e-11
    assert relerr(np_(g.lrdmc_get_walkers()[3]), o.get_state()[3]) < 1e-9
    rc, par = o.reconfigure(4)
    assert np.array_equal(np_(g.lrdmc_reconfigure(4, want_parents=True)), par)
    g.close()


# ------------------------------------------------------------------------------------------ a12: reconfiguration alone
@pytest.mark.parametrize("n_w", [1, 2, 5, 33, 1024, 1025, 4099, 8192, 8193, 70001])      # above 8192 the comb search is a kernel of its own (k_comb_search)
def test_reconfigure_indices_bit_exact_for_adversarial_weights(B, n_w):
    s = wl.hydrogen(); g = B.Lrdmc(s); o = ref.Ref(s); rng = np.random.default_rng(n_w)
    x0 = wl.hydrogen_walkers(n_w, 2)
    cases = [rng.random(n_w), rng.random(n_w) ** 8 * 1e-200, np.exp(rng.normal(size=n_w) * 20), np.ones(n_w)]
    sparse = np.zeros(n_w); sparse[rng.integers(0, n_w, size=max(1, n_w // 50))] = rng.random(max(1, n_w // 50)) + 0.1; cases.append(sparse)
    for ci, w in enumerate(cases):
        g.lrdmc_set_state(x0, None, None, w)
        gpar = np_(g.lrdmc_reconfigure(100 + ci, want_parents=True))
        rc, par, wbar, *_ = ref.comb(w, o.comb_r32(100 + ci))
        assert np.array_equal(gpar, par), ci
        gr = np_(g.lrdmc_get_walkers()[0]); assert np.array_equal(gr, x0[par])
    # degenerate: all weights zero -> identity, wbar = 0
    g.lrdmc_set_state(x0, None, None, np.zeros(n_w))
    assert np.array_equal(np_(g.lrdmc_reconfigure(3, want_parents=True)), np.arange(n_w))
    g.close()


def test_reconfigure_worked_example(B):
    gold = read_golden("comb_worked_example.txt"); w = np.array([float(v) for v in gold["w"]])
    s = wl.hydrogen(); g = B.Lrdmc(s); o = ref.Ref(s); x0 = wl.hydrogen_walkers(5, 2)
    for cycle in range(6):
        g.lrdmc_set_state(x0, None, None, w)
        gpar = np_(g.lrdmc_reconfigure(cycle, want_parents=True))
        assert list(gpar) == list(ref.comb(w, o.comb_r32(cycle))[1])


# ------------------------------------------------------------------------------------------ full size, bench launch configuration
def test_full_size_c4_sampled_walkers_match_oracle(B):
    """N_w = 25600 (BASELINE configs[3]) in the launch configuration bench.py times; the oracle recomputes sampled walkers one by one."""
    n_w = 25600
    s = wl.water_methane(n_walkers=n_w); x0 = wl.initial_walkers(s, n_w, 5)
    g = B.Lrdmc(s); g.lrdmc_set_positions(x0, allow_singular=True)
    g.lrdmc_propagate(B.BALANCED, 5, 0.0, 0.0, 0)
    gr, gdu, gdd, gw = [np_(t) for t in g.lrdmc_get_walkers()]
    gR, gscal, gjs = [np_(t) for t in g.lrdmc_step_debug(0.0, 1, 0)]
    o = ref.Ref(s); rng = np.random.default_rng(1); pick = np.sort(rng.choice(n_w, 24, replace=False))
    for k in pick:
        u = o.draws(int(k), 1, 0)
        R, sc, per, _ = o.evaluate(gr[k], ref.frame(u[0], u[1], u[2]), gdu[k], gdd[k])
        assert relerr(gR[k], R, 1.0) < TOL
        assert abs(gscal[k, 2] - sc["W"]) < TOL * 1200 and abs(gscal[k, 3] - sc["e_L"]) < TOL * 1200 and abs(gscal[k, 0] - sc["bbar"]) < TOL * 1200
        assert gjs[k] == o.select(R, u[3])[0]
    # properties that hold at any size: parents sorted, copies within floor/ceil of N_w w/sum(w), weights reset
    g.lrdmc_propagate(B.BALANCED, 3, 0.0, 0.0, 2)
    w = np_(g.lrdmc_get_walkers()[3]); par = np_(g.lrdmc_reconfigure(2, want_parents=True))
    assert np.array_equal(par, ref.comb(w, o.comb_r32(2))[1])
    assert np.all(np.diff(par) >= 0)
    st = g.lrdmc_estimators(); assert abs(st.wbar - w.mean()) < 1e-9 * w.mean() and st.moves_sum == 3 * n_w
    g.close()


@pytest.mark.parametrize("cfg,mode", [("C4", "balanced"), ("C4", "conventional"), ("C5", "balanced"), ("C5", "conventional"), ("C3nl", "balanced")])
def test_full_size_trajectories_of_sampled_walkers(B, cfg, mode):
    """Whole branching intervals at the full BASELINE sizes in the launch configuration bench.py times (C4: 25600 walkers,
    warp-per-walker; C5: 4096 walkers, team kernel with parked Bc entries; C3 + non-local slots: 25600): groups of walkers from
    the start, the middle and the end of the ensemble are replayed by the oracle on their own random streams."""
    s, n_w, n_moves, per = {"C4": (wl.water_methane(n_walkers=25600), 25600, 20, 6), "C5": (wl.cluster64(), 4096, 12, 2),
                            "C3nl": (wl.water_methane_nonlocal(n_walkers=25600), 25600, 20, 6)}[cfg]
    N = s["n_up"] + s["n_dn"]; x0 = wl.initial_walkers(s, n_w, 5)
    g = B.Lrdmc(s); g.lrdmc_set_positions(x0, allow_singular=True)
    cycle = 3
    if mode == "balanced":
        g.lrdmc_propagate(B.BALANCED, n_moves, 0.0, -5.0, cycle)
    else:
        tau = n_moves * s["a"]**2 / (3 * N) * (0.5 if s["a2"] > 0 else 1.0); g.lrdmc_propagate(B.CONVENTIONAL, 0, tau, -1.0, cycle)
    gr, _, _, gw = [np_(t) for t in g.lrdmc_get_walkers()]; geL, gW, gom, gnm = [np_(t) for t in g.lrdmc_get_obs()]
    for k0 in (0, n_w // 2 - 37, n_w - per):
        o = ref.Ref(s); o.set_slot_offset(k0)
        rc = o.set_positions(x0[k0:k0 + per]); assert rc in (0, -2)
        if mode == "balanced":
            assert o.propagate(ref.BALANCED, n_moves, 0.0, -5.0, cycle) == 0
        else:
            assert o.propagate(ref.CONVENTIONAL, 0, tau, -1.0, cycle) == 0
        r, _, _, w = o.get_state(); eL, W, om, nm = o.get_obs()
        sl = slice(k0, k0 + per); Kd = 3 * N / s["a"]**2
        assert np.array_equal(gnm[sl], nm) and np.abs(gr[sl] - r).max() < 1e-11
        assert relerr(gw[sl], w) < 1e-9 and relerr(gom[sl], om) < 1e-9
        assert np.max(np.abs(geL[sl] - eL) / np.maximum(np.abs(eL), Kd)) < TOL
    g.close()


# ------------------------------------------------------------------------------------------ runs: energies within 3 sigma
def test_hydrogen_run_energy_matches_oracle_and_exact(B):
    from paper_2508_12033_b200 import driver as drv
    s = wl.hydrogen(alpha=0.9, a=0.2); x0 = wl.hydrogen_walkers(256, 1)
    g = B.Lrdmc(s); g.lrdmc_set_positions(x0)
    recs = drv.run(g, B.BALANCED, 200, n_moves=40, E0=-0.495)
    Eg, sg = B.lrdmc_energy(recs, p=10, n_therm=40, n_blocks=10)
    o = ref.Ref(s); o.set_positions(x0)
    out = rdrv.run(o, ref.BALANCED, 200, n_moves=40, E0=-0.495)
    Eo, so = rdrv.energy(out["wbar"], out["num"], out["den"], p=10, n_therm=40, n_blocks=10)
    assert abs(Eg - Eo) < 3 * np.hypot(sg, so) and abs(Eg + 0.5) < 3 * sg + 2e-3
    # same seed, same RNG stream: the first generations are identical to rounding
    for n in range(5):
        assert abs(recs[n].num / recs[n].den - out["e"][n]) < 1e-9 and abs(recs[n].wbar - out["wbar"][n]) < 1e-9
    recs_c = drv.run(g, B.CONVENTIONAL, 200, tau=40 * 0.04 / 3, E0=-0.5, first_cycle=1000)
    Ec, sc = B.lrdmc_energy(recs_c, p=10, n_therm=40, n_blocks=10)
    assert abs(Ec - Eg) < 3 * np.hypot(sc, sg) + 1e-3                                     # balanced == conventional (L244)
    g.close()


def test_c2_full_run_energy_matches_the_oracle_run(B):
    """north_star: "mean energies over full runs within 3 combined standard errors".  BASELINE configs[1] at its full size (C2:
    1024 walkers x 100 branchings x 50 moves, Alg.2 with the E_0 feedback of L232 / L418), the whole run on the CUDA path and the
    whole run through the oracle (5.1 M walker-moves on the host cores): the first generations agree to rounding (same seeds, same
    streams), the run energies within 3 combined sigma."""
    from paper_2508_12033_b200 import driver as drv
    s = wl.synthetic10(); x0 = wl.initial_walkers(s, 1024, 5); Kd = 3 * 10 / s["a"]**2
    g = B.Lrdmc(s); g.lrdmc_set_positions(x0)
    recs = drv.run(g, B.BALANCED, 100, n_moves=50, E0=0.0, n_therm=20)
    Eg, sg = B.lrdmc_energy(recs, p=5, n_therm=20, n_blocks=10)
    ref.set_threads(0)
    o = ref.Ref(s); assert o.set_positions(x0) == 0
    out = rdrv.run(o, ref.BALANCED, 100, n_moves=50, E0=0.0, n_therm=20)
    Eo, so = rdrv.energy(out["wbar"], out["num"], out["den"], p=5, n_therm=20, n_blocks=10)
    for n in range(5):
        assert abs(recs[n].num / recs[n].den - out["e"][n]) < 1e-9 * Kd and abs(recs[n].wbar - out["wbar"][n]) < 1e-9 * out["wbar"][n], n
        assert recs[n].moves_sum == out["moves_sum"][n]
    assert sum(r.n_nonfinite + r.n_nonpos_diag + r.n_singular for r in recs) == 0 and out["n_nonfinite"].sum() == 0
    assert abs(Eg - Eo) < 3 * np.hypot(sg, so), (Eg, sg, Eo, so)
    # how long the two runs stay on one trajectory (reported, not asserted: the first near-tie or 1e-16 difference in a weight separates them)
    same = 0
    while same < 100 and abs(recs[same].num / recs[same].den - out["e"][same]) < 1e-6 * Kd:
        same += 1
    print(f"C2 full run: GPU {Eg:.5f} +- {sg:.5f}, oracle {Eo:.5f} +- {so:.5f}, generations on one trajectory: {same}")
    g.close()


def test_nonlocal_s_channel_energy_on_the_cuda_path(B):
    """Scope row f1 through the CUDA path: one electron in -1/r plus an attractive non-local s channel.  The exact ground-state
    energy comes from the radial eigen-solver of tests/test_oracle_nonlocal.py (independent of both implementations); LRDMC with the
    non-local hops must reach it as a -> 0 in both modes, and the first generations must equal the oracle's to rounding."""
    from paper_2508_12033_b200 import driver as drv
    from test_oracle_nonlocal import _radial_ground_state
    A0, B0, rc = -0.8, 1.5, 2.2
    E_exact = _radial_ground_state(A0, B0, rc)
    mk = lambda a: wl.with_nonlocal(wl.hydrogen(alpha=1.1, a=a), [[rc, A0, B0, 0, 1, 0, 1]])
    out = drv.a_scan(mk, lambda s, n: wl.hydrogen_walkers(n, 3), [0.2, 0.3, 0.4], n_walkers=2048, cycles=150, moves=30, E0=-0.6)
    for mode in ("balanced", "conventional"):
        E0, s0, coef, chi2 = out[mode]
        assert abs(E0 - E_exact) < 3 * s0 + 5e-4 and s0 < 1.5e-3, (mode, E0, s0, E_exact)
    s = mk(0.3); x0 = wl.hydrogen_walkers(256, 3)
    g = B.Lrdmc(s); g.lrdmc_set_positions(x0); o = ref.Ref(s); o.set_positions(x0)
    recs = drv.run(g, B.BALANCED, 5, n_moves=18, E0=-0.6); outo = rdrv.run(o, ref.BALANCED, 5, n_moves=18, E0=-0.6)
    for n in range(5):
        assert abs(recs[n].num / recs[n].den - outo["e"][n]) < 1e-9 and abs(recs[n].wbar - outo["wbar"][n]) < 1e-9
    g.close()


def test_a_to_zero_scan_balanced_vs_conventional_table_shape(B):
    """SURVEY 8(f) f3, the shape of Table I (L254-L265): several a and both algorithms in ONE batch (8 contexts on 8 streams in
    flight together).  At every a the two modes agree within 3 combined sigma, both E(a) extrapolate to the exact -1/2 Ha of the
    hydrogen atom (L23, L140), and the batch equals the same runs made one after the other bit for bit (the runs are independent:
    concurrency changes nothing but the wall time)."""
    from paper_2508_12033_b200 import driver as drv
    mk = lambda a: wl.hydrogen(alpha=0.9, a=a); mw = lambda s, n: wl.hydrogen_walkers(n, 1); a_list = [0.15, 0.25, 0.35, 0.45]
    out = drv.a_scan(mk, mw, a_list, n_walkers=2048, cycles=150, moves=30, E0=-0.5)
    for r in out["rows"]:
        (Eb, sb), (Ec, sc) = r["balanced"], r["conventional"]
        assert abs(Eb - Ec) < 3 * np.hypot(sb, sc) + 2e-4, r
        assert Eb < -0.495 + 3 * sb                                                       # below the variational energy
    for mode in ("balanced", "conventional"):
        E0, s0, coef, chi2 = out[mode]
        assert abs(E0 + 0.5) < 3 * s0 + 2e-4 and s0 < 1e-3, (mode, E0, s0)
    seq = drv.a_scan(mk, mw, a_list[:2], n_walkers=2048, cycles=40, moves=30, E0=-0.5, concurrent=False)
    con = drv.a_scan(mk, mw, a_list[:2], n_walkers=2048, cycles=40, moves=30, E0=-0.5, concurrent=True)
    for rs, rc in zip(seq["rows"], con["rows"]):
        assert rs["balanced"] == rc["balanced"] and rs["conventional"] == rc["conventional"]


def test_a_to_zero_scan_matches_the_oracle_scan_row_by_row(B):
    """f3 against the oracle: the same a-scan (same systems, same per-run Philox keys) through oracle.ref_driver.a_scan; every row
    and both extrapolations within 3 combined sigma, and the first generations of every run equal to rounding."""
    from paper_2508_12033_b200 import driver as drv
    mk = lambda a: wl.hydrogen(alpha=0.9, a=a); mw = lambda s, n: wl.hydrogen_walkers(n, 1); a_list = [0.2, 0.3, 0.4]
    kw = dict(n_walkers=1024, cycles=120, moves=30, E0=-0.5, n_therm=24, p=10, n_blocks=10)
    ref.set_threads(0)
    oo = rdrv.a_scan(mk, mw, a_list, **kw)
    gg = drv.a_scan(mk, mw, a_list, **kw)
    for ro, rg in zip(oo["rows"], gg["rows"]):
        for mode in ("balanced", "conventional"):
            (Eo, so), (Eg, sg) = ro[mode], rg[mode]
            assert abs(Eo - Eg) < 3 * np.hypot(so, sg) + 1e-12, (ro["a"], mode, Eo, so, Eg, sg)
            assert 0.3 < sg / so < 3.0                                                    # same statistics, same error bars
    for mode in ("balanced", "conventional"):
        assert abs(oo[mode][0] - gg[mode][0]) < 3 * np.hypot(oo[mode][1], gg[mode][1])
        assert abs(oo[mode][1] - gg[mode][1]) < 0.5 * oo[mode][1]
    # first generations of one run of the batch against the oracle's run with the same key (q = 3: a = 0.3, conventional)
    s = dict(mk(0.3)); s["seed"] += 1000003 * 4
    g = B.Lrdmc(s); g.lrdmc_set_positions(mw(s, 1024))
    recs = drv.run(g, B.CONVENTIONAL, 3, tau=30 * 0.09 / 3, E0=-0.5)
    for n in range(3):
        assert abs(recs[n].num / recs[n].den - oo["rows"][1]["conventional_first_e"][n]) < 1e-9
    g.close()


def test_helium_energies_on_the_cuda_path(B):
    """Pins P7/P8 through the CUDA path: nodeless He 1S -> -2.903724 Ha as a -> 0; He 2 3S with its exact node -> -2.175229 Ha."""
    from paper_2508_12033_b200 import driver as drv
    rng = np.random.default_rng(0); a = [0.15, 0.25, 0.35]; E = []; sg = []
    for ai in a:
        s = wl.slater_atom(2.0, [1.85], 1, 1, np.ones((1, 1)), np.ones((1, 1)), ai, jastrow=dict(a_anti=0.5, a_par=0.25, b2=0.5))
        g = B.Lrdmc(s); g.lrdmc_set_positions(rng.normal(size=(4096, 2, 3)) * 0.7)
        recs = drv.run(g, B.BALANCED, 300, n_moves=int(round(20 * (0.2 / ai) ** 2)), E0=-2.9)
        e, sd = B.lrdmc_energy(recs, p=10, n_therm=60, n_blocks=10); E.append(e); sg.append(sd); g.close()
    E0, s0, *_ = drv.fit_a_to_zero(a, E, sg)
    assert abs(E0 + 2.903724) < 3 * s0 + 3e-4 and s0 < 2e-3, (E0, s0)
    s = wl.slater_atom(2.0, [2.0, 0.6], 2, 0, np.eye(2), np.zeros((2, 0)), 0.2, jastrow=dict(a_par=0.25, a_anti=0.5, b2=0.5))
    x = rng.normal(size=(4096, 2, 3)); x[:, 0] *= 0.4; x[:, 1] *= 2.0
    g = B.Lrdmc(s); g.lrdmc_set_positions(x)
    recs = drv.run(g, B.BALANCED, 400, n_moves=30, E0=-2.17)
    Et, st = B.lrdmc_energy(recs, p=10, n_therm=80, n_blocks=10)
    assert sum(r.n_node_flag for r in recs) > 0 and sum(r.n_nonpos_diag for r in recs) == 0
    assert abs(Et + 2.175229) < 3 * st + 5e-4 and st < 1e-3, (Et, st)
    g.close()


def test_balanced_equals_conventional_on_the_synthetic_molecule(B):
    """Pin P12 on config C2 (10 electrons, s/p/d GTOs, Jastrow, nodes): the two modes sample the same fixed-node state (L234, L244)."""
    from paper_2508_12033_b200 import driver as drv
    s = wl.synthetic10(); x0 = wl.initial_walkers(s, 4096, 5); N = 10
    g = B.Lrdmc(s); g.lrdmc_set_positions(x0, allow_singular=True)
    pilot = drv.run(g, B.BALANCED, 30, n_moves=50, E0=0.0, feedback=False)
    Eref = float(np.mean([r.num / r.den for r in pilot[10:]]))
    # the balanced Green's function projects onto the ground state only for E_0 = E (Eq.28, "E_0 is updated after each
    # branching step" L232): run it with the feedback of Alg.2 line 12, first a thermalising leg, then the measured one
    rt = drv.run(g, B.BALANCED, 60, n_moves=50, E0=Eref, first_cycle=100)
    rb = drv.run(g, B.BALANCED, 200, n_moves=50, E0=float(np.mean([r.num / r.den for r in rt[20:]])), first_cycle=200)
    Eb, sb = B.lrdmc_energy(rb, p=5, n_therm=30, n_blocks=10)
    rc = drv.run(g, B.CONVENTIONAL, 260, tau=50 * s["a"]**2 / (3 * N), E0=Eref, first_cycle=1000)
    Ec, sc = B.lrdmc_energy(rc, p=5, n_therm=90, n_blocks=10)
    mean_moves = np.mean([r.moves_sum for r in rc]) / 4096
    assert 35 < mean_moves < 65
    assert sum(r.n_nonfinite for r in rb + rc) == 0
    assert abs(Eb - Ec) < 3 * np.hypot(sb, sc), (Eb, sb, Ec, sc)
    g.close()


@pytest.mark.parametrize("dla", [True, False])
def test_balanced_equals_conventional_with_nonlocal_slots(B, dla):
    """Pin P12 with non-local hops in the Green's function (row f1; L244 / Table I shape: "both algorithms sample the same
    fixed-node ground state"): helium-like atom, Slater orbital x Jastrow (so the determinant-locality and the full-ratio forms
    differ), attractive s and repulsive p channel: about 1.5 % of the hops are non-local and a third of the non-local amplitudes
    are sign-forbidden (they go to V_sf).  Error bars ~1e-3 Ha."""
    from paper_2508_12033_b200 import driver as drv
    rng = np.random.default_rng(0)
    base = wl.slater_atom(2.0, [1.85], 1, 1, np.ones((1, 1)), np.ones((1, 1)), 0.25, jastrow=dict(a_anti=0.5, a_par=0.25, b2=0.5))
    s = wl.with_nonlocal(base, [[2.0, -1.0, 1.2, 0.8, 0.9, 0.0, 1.0]], dla)
    g = B.Lrdmc(s); g.lrdmc_set_positions(rng.normal(size=(4096, 2, 3)) * 0.7)
    rb = drv.run(g, B.BALANCED, 300, n_moves=20, E0=-3.2)
    Eb, sb = B.lrdmc_energy(rb, p=10, n_therm=60, n_blocks=10)
    rc = drv.run(g, B.CONVENTIONAL, 300, tau=20 * 0.25**2 / 6, E0=-3.2, first_cycle=1000)
    Ec, sc = B.lrdmc_energy(rc, p=10, n_therm=60, n_blocks=10)
    R, scal, js = [np_(t) for t in g.lrdmc_step_debug(-3.2, 5000, 0)]
    assert (js >= 12).sum() > 10 and (R[:, 12:] < 0).mean() > 0.1          # non-local hops are taken; forbidden ones exist
    assert sum(r.n_nonfinite for r in rb + rc) == 0 and sc < 3e-3
    assert abs(Eb - Ec) < 3 * np.hypot(sb, sc), (Eb, sb, Ec, sc)
    assert Eb < -3.5                                                       # far below the channel-free helium energy (-2.90): the s channel binds
    g.close()


def test_helium_with_three_body_jastrow_still_reaches_the_exact_energy(B):
    """Row f2 in whole runs: the nodeless He ground-state energy does not depend on the Jastrow factor, so with a three-body term
    switched on E(a -> 0) must still be the textbook -2.903724 Ha, and the two modes must agree at fixed a (L234)."""
    from paper_2508_12033_b200 import driver as drv
    rng = np.random.default_rng(0); a = [0.15, 0.25, 0.35]; E = []; sg = []

    def he(ai):
        s = dict(wl.slater_atom(2.0, [1.85], 1, 1, np.ones((1, 1)), np.ones((1, 1)), ai, jastrow=dict(a_anti=0.5, a_par=0.25, b2=0.5)))
        s.update(j3_center=np.array([0, 0], dtype=np.int32), j3_zeta=np.array([0.8, 2.0]), j3_g=np.array([[0.05, -0.03], [-0.03, 0.06]]), name="he-J3")
        return s
    for ai in a:
        g = B.Lrdmc(he(ai)); g.lrdmc_set_positions(rng.normal(size=(4096, 2, 3)) * 0.7)
        recs = drv.run(g, B.BALANCED, 300, n_moves=int(round(20 * (0.2 / ai) ** 2)), E0=-2.9)
        e, sd = B.lrdmc_energy(recs, p=10, n_therm=60, n_blocks=10); E.append(e); sg.append(sd)
        if ai == 0.25:
            rc = drv.run(g, B.CONVENTIONAL, 300, tau=int(round(20 * (0.2 / ai) ** 2)) * ai**2 / 6, E0=-2.9, first_cycle=1000)
            Ec, sc = B.lrdmc_energy(rc, p=10, n_therm=60, n_blocks=10)
            assert abs(e - Ec) < 3 * np.hypot(sd, sc), (e, sd, Ec, sc)
        g.close()
    E0, s0, *_ = drv.fit_a_to_zero(a, E, sg)
    assert abs(E0 + 2.903724) < 3 * s0 + 3e-4 and s0 < 3e-3, (E0, s0)


# ------------------------------------------------------------------------------------------ the host-buffer entry point (bench.py's e2e number)
@pytest.mark.parametrize("n_therm", [0, 2])
def test_run_host_end_to_end_matches_the_oracle_driver(B, n_therm):
    """lrdmc_run_host (HOST positions in, Alg.2 lines 2-13 with the E_0 feedback of L232 / L418 inside the library, HOST positions
    out) on C3 with 100 walkers against oracle.ref_driver.run: every generation's num/den and wbar to 1e-9 (a wrong feedback rule --
    no update, or a mean that does not restart at n_therm -- changes the weights of the following generation), the positions handed
    back equal lrdmc_get_walkers() bit for bit, the hop counts are exact."""
    s = wl.water_methane(n_walkers=100); x0 = wl.initial_walkers(s, 100, 5); n_cyc = 4; Kd = 3 * 16 / s["a"]**2
    g = B.Lrdmc(s)
    stats, r_out = g.lrdmc_run_host(x0, B.BALANCED, 20, 0.0, 3.0, 11, n_cyc, n_therm=n_therm)
    o = ref.Ref(s); assert o.set_positions(x0) == 0
    out = rdrv.run(o, ref.BALANCED, n_cyc, n_moves=20, E0=3.0, first_cycle=11, n_therm=n_therm)
    assert len(stats) == n_cyc
    for n in range(n_cyc):
        assert abs(stats[n].num / stats[n].den - out["e"][n]) < 1e-9 * Kd, n
        assert abs(stats[n].wbar - out["wbar"][n]) < 1e-9 * out["wbar"][n], n
        assert abs(stats[n].den - out["den"][n]) < 1e-9 * out["den"][n], n
        assert stats[n].moves_sum == out["moves_sum"][n] == 20 * 100 and stats[n].n_singular == 0
    # the feedback really changed E_0 between generations (otherwise the comparison above would not test it)
    assert len(set(np.round(out["E0_used"], 9))) == n_cyc
    if n_therm:
        assert abs(out["E0_used"][3] - out["e"][2]) < 1e-12         # generation 2 restarted the mean
    gr = np_(g.lrdmc_get_walkers()[0])
    assert np.array_equal(r_out.numpy(), gr) and np.abs(gr - o.get_state()[0]).max() < 1e-11
    # conventional mode keeps the shift (Q8b)
    stats_c, _ = g.lrdmc_run_host(x0, B.CONVENTIONAL, 0, 20 * s["a"]**2 / 48, 5.0, 40, 2)
    o.set_positions(x0); out_c = rdrv.run(o, ref.CONVENTIONAL, 2, tau=20 * s["a"]**2 / 48, E_ref=5.0, first_cycle=40)
    for n in range(2):
        assert abs(stats_c[n].num / stats_c[n].den - out_c["e"][n]) < 1e-9 * Kd and stats_c[n].moves_sum == out_c["moves_sum"][n]
    g.close()


def test_run_host_errors(B):
    s = wl.tiny_molecule(2, 1, 2, 6, seed=7); g = B.Lrdmc(s)
    xs = wl.initial_walkers(s, 4, 3)
    L = g.L; import ctypes as C
    st = (B.CycleStats * 2)()
    assert L.lrdmc_run_host(g.h, xs.ctypes.data, None, B.BALANCED, 5, 0.0, 0.0, 0, 2, 0, st, None) == B.ESTATE      # nothing bound
    g.lrdmc_bind_walkers(4)
    assert L.lrdmc_run_host(g.h, None, None, B.BALANCED, 5, 0.0, 0.0, 0, 2, 0, st, None) == B.EINVAL
    assert L.lrdmc_run_host(g.h, xs.ctypes.data, None, B.BALANCED, 5, 0.0, 0.0, 0, 2, -1, st, None) == B.EINVAL
    bad = xs.copy(); bad[2, 1] = bad[2, 0]                                                # coincident same-spin electrons
    out = np.full_like(bad, 7.0)
    assert L.lrdmc_run_host(g.h, bad.ctypes.data, out.ctypes.data, B.BALANCED, 5, 0.0, 0.0, 0, 2, 0, st, None) == B.ESINGULAR
    assert np.all(out == 7.0)                                                             # nothing propagated, r_out untouched
    assert L.lrdmc_run_host(g.h, xs.ctypes.data, out.ctypes.data, B.BALANCED, 5, 0.0, -5.0, 0, 2, 0, st, None) == 0
    assert st[1].moves_sum == 20 and np.array_equal(out, np_(g.lrdmc_get_walkers()[0]))
    g.close()


@pytest.mark.parametrize("tw", [1, 4])
def test_singular_walkers_are_dead_until_the_next_branching(B, tw):
    """Reading Q24 on the CUDA path, both kernels, against the oracle: walkers with coincident same-spin electrons are reported
    (ESINGULAR, n_singular), get zero inverses, leave propagate with w = omega = 0 and no moves, are never parents, and the live
    walkers beside them follow the oracle's trajectories."""
    s = wl.tiny_molecule(2, 1, 2, 6, seed=7)
    x = wl.initial_walkers(s, 70, 3); deadk = [2, 4, 33, 69]
    for k in deadk:
        x[k, 1] = x[k, 0]
    g = B.Lrdmc(s, options={B.OPT_TEAM_WARPS: tw}); o = ref.Ref(s)
    assert g.lrdmc_set_positions(x, allow_singular=True) == B.ESINGULAR and o.set_positions(x) == -2
    gr, gdu, gdd, gw = [np_(t) for t in g.lrdmc_get_walkers()]; r, du, dd, w = o.get_state()
    assert np.all(gdu[deadk] == 0.0) and np.all(gdd[deadk] == 0.0)
    live = np.setdiff1d(np.arange(70), deadk)
    assert np.max(np.abs(gdu[live] - du[live]) / np.abs(du[live]).max(axis=(1, 2), keepdims=True)) < 1e-8
    g.lrdmc_propagate(B.BALANCED, 9, 0.0, -5.0, 0); assert o.propagate(ref.BALANCED, 9, 0.0, -5.0, 0) == 0
    gr, _, _, gw = [np_(t) for t in g.lrdmc_get_walkers()]; r, _, _, w = o.get_state()
    geL, gW, gom, gnm = [np_(t) for t in g.lrdmc_get_obs()]; eL, W, om, nm = o.get_obs()
    assert np.all(gw[deadk] == 0.0) and np.all(gom[deadk] == 0.0) and np.all(gnm[deadk] == 0) and np.array_equal(gnm, nm)
    assert np.abs(gr - r).max() < 1e-11 and relerr(gw, w) < 1e-9 and relerr(gom, om) < 1e-9
    par = np_(g.lrdmc_reconfigure(0, want_parents=True)); rc, opar = o.reconfigure(0)
    assert np.array_equal(par, opar) and not set(deadk) & set(par.tolist())
    st = g.lrdmc_estimators(); so = o.estimators()
    assert st.n_singular == so["n_singular"] == 0 and st.moves_sum == so["moves_sum"] == 9 * 66
    assert abs(st.wbar - so["wbar"]) < 1e-9 * so["wbar"]
    # before the branching the count of the last rebuild (set_positions) is what the stats carry
    g.lrdmc_set_positions(x, allow_singular=True); g.lrdmc_propagate(B.BALANCED, 1, 0.0, -5.0, 1)
    assert g.lrdmc_estimators().n_singular == 4
    g.close()


# ------------------------------------------------------------------------------------------ edge cases and error behaviour
def test_edge_cases_and_errors(B):
    s = wl.tiny_molecule(2, 1, 2, 6, seed=7); g = B.Lrdmc(s)
    with pytest.raises(B.LrdmcError) as e:
        g.lrdmc_propagate(B.BALANCED, 5, 0.0, 0.0, 0)                                    # nothing bound
    assert e.value.code == B.ESTATE
    x0 = wl.initial_walkers(s, 1, 3); g.lrdmc_set_positions(x0)                          # a single walker
    o = ref.Ref(s); o.set_positions(x0)
    g.lrdmc_propagate(B.BALANCED, 0, 0.0, -5.0, 0); o.propagate(ref.BALANCED, 0, 0.0, -5.0, 0)   # zero moves: measurement only
    assert np_(g.lrdmc_get_obs()[3])[0] == 0 and relerr(np_(g.lrdmc_get_obs()[0]), o.get_obs()[0], 100.0) < TOL
    for bad in (dict(mode=7, n_moves=1, tau=0.0), dict(mode=B.CONVENTIONAL, n_moves=0, tau=0.0), dict(mode=B.BALANCED, n_moves=-1, tau=0.0)):
        with pytest.raises(B.LrdmcError) as e:
            g.lrdmc_propagate(bad["mode"], bad["n_moves"], bad["tau"], 0.0, 0)
        assert e.value.code == B.EINVAL
    xs = wl.initial_walkers(s, 4, 3); xs[2, 1] = xs[2, 0]                                 # coincident same-spin electrons
    assert g.lrdmc_set_positions(xs, allow_singular=True) == B.ESINGULAR                 # reading Q24: pivot <= 2^-44 max|D|
    with pytest.raises(B.LrdmcError) as e:
        g.lrdmc_set_option(B.OPT_TEAM_WARPS, 4)                                          # options come before the walkers are bound
    assert e.value.code == B.ESTATE
    # W - E0 <= 0 is counted and kills the weight (reading Q16)
    g.lrdmc_set_positions(wl.initial_walkers(s, 8, 3)); o.set_positions(wl.initial_walkers(s, 8, 3))
    g.lrdmc_propagate(B.BALANCED, 3, 0.0, 1e6, 0); o.propagate(ref.BALANCED, 3, 0.0, 1e6, 0)
    g.lrdmc_reconfigure(0); o.reconfigure(0)
    st = g.lrdmc_estimators(); so = o.estimators()
    assert st.n_nonpos_diag == so["n_nonpos_diag"] == 8 * 4 and st.wbar == 0.0 == so["wbar"]
    g.close()


def test_malformed_nonlocal_and_contraction_inputs_are_rejected(B):
    """lrdmc_init validates the f1 / f2 inputs: too many slots per electron, contracted shells that mix centres or types, ranges that
    do not tile the primitive list, an MO matrix whose row count is not the contracted function count -> LRDMC_EINVAL."""
    s = wl.random_nonlocal(wl.tiny_molecule(2, 1, 2, 6, seed=7), 8, 1.4, 1, True); s["nl_K"] = 5
    with pytest.raises(B.LrdmcError) as e:
        B.Lrdmc(s)
    assert e.value.code == B.EINVAL
    good = wl.contracted_molecule(3, 2, 3, 9, seed=31, spherical=True)
    for breakit in ("first", "mixed", "nao"):
        c = dict(good)
        if breakit == "first":
            f = good["cs_first"].copy(); f[-1] -= 1; c["cs_first"] = f                   # ranges do not end at n_shell
        elif breakit == "mixed":
            t = good["shell_type"].copy(); k = int(good["cs_first"][1]) - 1
            if int(good["cs_first"][1]) - int(good["cs_first"][0]) < 2:
                f = good["cs_first"].copy(); f[1] += 1; c["cs_first"] = f                # merge a p primitive into the first (s) shell
            else:
                t[k] = wl.SHELL_P; c["shell_type"] = t
        else:
            c["n_ao"] = good["n_ao"] + 1; c["C_up"] = np.vstack([good["C_up"], np.zeros((1, 3))]); c["C_dn"] = np.vstack([good["C_dn"], np.zeros((1, 2))])
        with pytest.raises(B.LrdmcError) as e:
            B.Lrdmc(c)
        assert e.value.code == B.EINVAL, breakit


# ------------------------------------------------------------------------------------------ random shapes x random options
def _random_case(case):
    """A seeded random system (electron counts 1..19 / 0..n_up, 1..6 nuclei, 3..39 shells; primitive or contracted basis; optionally a
    second mesh, a local pseudopotential, non-local slots, a three-body Jastrow) with a random kernel choice (team size, global tables,
    listed sweep), mode and ensemble size.  A sweep of 1000 such cases ran green on the B200 before these 24 were fixed as tests."""
    rng = np.random.default_rng([2026, case])
    while True:
        n_up = int(rng.integers(1, 20)); n_dn = int(rng.integers(0, n_up + 1)); n_nuc = int(rng.integers(1, 7))
        n_shell = int(rng.integers(max(3, (n_up + 3) // 2), 40)); seed = int(rng.integers(1, 10**6)); a2 = 0.0 if rng.random() < 0.7 else 0.3
        try:
            if rng.random() < 0.6:
                s = wl.tiny_molecule(n_up, n_dn, n_nuc, n_shell, seed=seed, a=0.15 if a2 else 0.2, a2=a2, with_pp=bool(rng.integers(0, 2)))
            else:
                s = wl.contracted_molecule(n_up, n_dn, n_nuc, max(n_shell // 2, (n_up + 1) // 2 + 2), seed=seed, spherical=bool(rng.integers(0, 2)), with_pp=bool(rng.integers(0, 2)))
        except Exception:
            continue                                    # fewer basis functions than orbitals: draw again
        break
    ext = int(rng.integers(0, 4))
    if ext & 1:
        args = (int(rng.integers(2, 9)), int(rng.integers(1, 3)), bool(rng.integers(0, 2))); scale = float(rng.choice([1.0, 50.0, 200.0]))
        s1 = wl.random_nonlocal(s, args[0], float(rng.uniform(0.5, 1.0)), args[1], args[2], scale=scale)
        s = s1 if s1["nl_K"] <= 4 else wl.random_nonlocal(s, args[0], 0.5, args[1], args[2], scale=scale)      # disjoint spheres: one slot per electron
    if ext & 2:
        s = wl.with_jastrow3(s, int(rng.integers(2, 9)), int(rng.integers(1, 4)), strength=0.1, n_max=int(rng.choice([8, 12, 24])), poly=bool(rng.integers(0, 2)))
    n_w = int(rng.integers(1, 60)); x0 = wl.initial_walkers(s, n_w, int(rng.integers(1, 100)))
    opts = {}; tw = int(rng.choice([0, 1, 2, 4, 8, 16]))
    if tw:
        opts["OPT_TEAM_WARPS"] = tw
    if rng.random() < 0.3:
        opts["OPT_GLOBAL_TABLES"] = 1
    if ext == 0 and rng.random() < 0.5:
        opts["OPT_LISTED"] = 1
    return s, x0, opts, ("balanced" if rng.random() < 0.5 else "conventional")


@pytest.mark.parametrize("case", range(24))
def test_random_shapes_and_options(B, case):
    """One evaluation from the oracle's state and two whole cycles, as the fixed systems above.  Ratios are sums of phi x Dinv products, so their
    scale is max(1, max|Dinv|) of the walker (random orbitals give near-singular Slater matrices now and then: conditioning, not arithmetic)."""
    s, x0, opts, mode = _random_case(case)
    N = s["n_up"] + s["n_dn"]; Kd = 3 * N * ((1 / s["a"]**2) if s["a2"] == 0 else (0.5 / s["a"]**2 + 0.5 / s["a2"]**2))
    o = ref.Ref(s)
    if o.set_positions(x0) != 0:
        pytest.skip("a singular Slater matrix among the random walkers")
    g = B.Lrdmc(s, options={getattr(B, k): v for k, v in opts.items()}); g.lrdmc_set_positions(x0)
    r, du, dd, w = o.get_state(); g.lrdmc_set_state(r, du, dd, w)
    cond = np.maximum(1.0, np.maximum(np.abs(du).max(axis=(1, 2)), np.abs(dd).max(axis=(1, 2)) if dd.size else 0.0))[:, None]
    R, scal, js = o.step_debug(-3.0, 2, 1); gR, gscal, gjs = [np_(t) for t in g.lrdmc_step_debug(-3.0, 2, 1)]
    assert np.max(np.abs(gR - R) / np.maximum(np.abs(R), cond)) < TOL
    near_tie = scal[:, 7] < 1e-9
    assert np.array_equal(gjs[~near_tie], js[~near_tie])
    assert np.max(np.abs(gscal[:, :4] - scal[:, :4]) / np.maximum(np.abs(scal[:, :4]), Kd * cond)) < TOL
    for cycle in range(2):
        if mode == "balanced":
            assert o.propagate(ref.BALANCED, 20, 0.0, -5.0, cycle) == 0; g.lrdmc_propagate(B.BALANCED, 20, 0.0, -5.0, cycle)
        else:
            tau = 20 * s["a"]**2 / (3 * N)
            assert o.propagate(ref.CONVENTIONAL, 0, tau, -1.0, cycle) == 0; g.lrdmc_propagate(B.CONVENTIONAL, 0, tau, -1.0, cycle)
        gr, gdu, gdd, gw = [np_(t) for t in g.lrdmc_get_walkers()]; geL, gW, gom, gnm = [np_(t) for t in g.lrdmc_get_obs()]
        r, du, dd, w = o.get_state(); eL, W, om, nm = o.get_obs()
        assert np.array_equal(gnm, nm) and np.abs(gr - r).max() < 1e-11
        assert relerr(gw, w) < 1e-9 and relerr(gom, om) < 1e-9
        rc, par = o.reconfigure(cycle); gpar = np_(g.lrdmc_reconfigure(cycle, want_parents=True))
        assert np.array_equal(gpar, par)
        so, sg = o.estimators(), g.lrdmc_estimators()
        assert abs(sg.wbar - so["wbar"]) <= 1e-9 * so["wbar"]
        assert (sg.n_node_flag, sg.n_nonpos_diag, sg.n_nonfinite) == (so["n_node_flag"], so["n_nonpos_diag"], so["n_nonfinite"])
    g.close()
