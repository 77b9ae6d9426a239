"""lrdmc_comb_static (include/lrdmc.h): the comb of the branching step with no allocation inside the library -- its scratch is a static
device array -- against the existing path (lrdmc_reconfigure on a bound ctx), two calls in a row.  -m gpu.

Collected last on purpose (file name): the suite runs with pytest -x, a failure here must not hide another test.  Indices bit-exact, wbar
within the tolerance of tests/test_gpu_parity.py.  The oracle is not involved: both sides are the CUDA path.
"""
import numpy as np
import pytest

from paper_2508_12033_b200 import workloads as wl

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2508_12033_b200 import binding
    binding.load_library()
    return binding


def _walkers(s, n_w):
    return wl.initial_walkers(s, n_w, 5) if s["n_up"] + s["n_dn"] > 1 else wl.hydrogen_walkers(n_w, 2)


def _existing_path(B, s, n_w, cycle, n_moves):
    """(weights, parents, wbar) of lrdmc_reconfigure after a real branching interval (lrdmc_estimators, the source of wbar, wants one)."""
    g = B.Lrdmc(s)
    g.lrdmc_set_positions(_walkers(s, n_w))
    g.lrdmc_propagate(B.BALANCED, n_moves, 0.0, -3.0, cycle)
    wt = g.lrdmc_get_walkers()[3].clone()
    par = g.lrdmc_reconfigure(cycle, want_parents=True)
    wbar = g.lrdmc_estimators().wbar
    out = wt, par.cpu().numpy(), wbar
    g.close()
    return out


def test_comb_static_matches_reconfigure_on_two_calls_in_a_row(B):
    import torch
    s1 = wl.synthetic10(); s2 = wl.tiny_molecule(3, 3, 3, 9, seed=8, with_pp=True); s2["seed"] = 0x1234567890ABCDEF
    # call 1 fills 5000 entries of the static scratch; call 2 (fewer walkers, other weights, other seed and cycle) runs over what it left
    w1, par1, wbar1 = _existing_path(B, s1, 5000, 7, 6)
    w2, par2, wbar2 = _existing_path(B, s2, 777, 3, 40)
    assert not np.array_equal(par1, np.arange(5000)) and not np.array_equal(par2, np.arange(777)) and wbar1 > 0 and wbar2 > 0
    a1, ab1 = B.lrdmc_comb_static(w1, s1["seed"], 7)
    a2, ab2 = B.lrdmc_comb_static(w2, s2["seed"], 3)
    torch.cuda.synchronize()
    for got, gotbar, par, wbar in ((a1, ab1, par1, wbar1), (a2, ab2, par2, wbar2)):
        assert got.dtype == torch.int32 and np.array_equal(got.cpu().numpy(), par)
        assert abs(float(gotbar.item()) - wbar) <= TOL * abs(wbar)
    # the first result again after the second call: nothing of call 2 survives into it
    a3, ab3 = B.lrdmc_comb_static(w1, s1["seed"], 7)
    assert np.array_equal(a3.cpu().numpy(), par1) and float(ab3.item()) == float(ab1.item())


def test_comb_static_matches_reconfigure_for_adversarial_weights(B):
    """Weights set as state (sixteen decades apart, tiny, sparse): indices only -- without a propagate the existing path reports no wbar."""
    rng = np.random.default_rng(12); n_w = 4099
    s = wl.hydrogen(); g = B.Lrdmc(s); x0 = _walkers(s, n_w)
    sparse = np.zeros(n_w); sparse[rng.integers(0, n_w, size=80)] = rng.random(80) + 0.1
    for ci, w in enumerate([np.exp(rng.normal(size=n_w) * 20), rng.random(n_w) ** 8 * 1e-200, sparse, np.ones(n_w)]):
        g.lrdmc_set_state(x0, None, None, w)
        par = g.lrdmc_reconfigure(50 + ci, want_parents=True).cpu().numpy()
        got, wbar = B.lrdmc_comb_static(g._dev(w, np.float64), s["seed"], 50 + ci)
        assert np.array_equal(got.cpu().numpy(), par), ci
        assert abs(float(wbar.item()) - w.mean()) <= 1e-9 * w.mean(), ci      # Eq.16 up to the quantisation of reading Q21
    g.close()


def test_comb_static_degenerate_weights_and_size_limit(B):
    import torch
    z = torch.zeros(100, dtype=torch.float64, device="cuda:0")
    par, wbar = B.lrdmc_comb_static(z, 1, 0)
    assert np.array_equal(par.cpu().numpy(), np.arange(100)) and float(wbar.item()) == 0.0
    # the largest ensemble the scratch holds runs; one more walker is refused with a text that names the limit, and nothing is launched
    n = B.COMB_STATIC_MAX_WALKERS
    w = torch.rand(n + 1, dtype=torch.float64, device="cuda:0", generator=torch.Generator(device="cuda:0").manual_seed(5)) + 0.05
    par, wbar = B.lrdmc_comb_static(w[:n].contiguous(), 9, 4)
    p = par.cpu().numpy(); cnt = np.bincount(p, minlength=n); expect = (w[:n] / w[:n].mean()).cpu().numpy()
    assert np.all(np.diff(p) >= 0) and np.all(np.abs(cnt - expect) < 1.0 + 1e-9)        # copies within floor/ceil of N_w w_k / sum w (Eq.17)
    assert abs(float(wbar.item()) - float(w[:n].mean().item())) <= 1e-9 * float(wbar.item())
    with pytest.raises(RuntimeError, match="LRDMC_COMB_STATIC_MAX_WALKERS = %d" % n):
        B.lrdmc_comb_static(w, 9, 4)
