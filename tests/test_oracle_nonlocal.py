"""Pins of the oracle's non-local pseudopotential candidates (scope row f1: "DLA", Eq.D1).
CPU only.  The oracle is checked against what the mathematics fixes, not against itself:
  * closed form: a pure-l orbital about the centre is an eigenfunction of the projector, V_nl psi / psi = v_l(r), whatever the frame;
  * the projector integral written out in Python on a 50-point Lebedev rule (scipy), with Psi from the brute-force log|Psi|;
  * brute-force wavefunction / determinant ratios at the quadrature points;
  * the exact ground-state energy of  -1/2 lap - 1/r + v_0(r)|s><s|  from a radial finite-difference eigen-solver.
"""
import math

import numpy as np
import pytest
from scipy.integrate import lebedev_rule
from scipy.linalg import eigh_tridiagonal

from oracle import lrdmc_ref as ref, ref_driver as drv
from paper_2508_12033_b200 import workloads as wl

RNG = np.random.default_rng(11)


def _haar(rng):
    q, r = np.linalg.qr(rng.standard_normal((3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


def _one_centre(stypes, zetas, C_up, C_dn, centre, nl_row, dla=True, jastrow=None, a=0.2, Z=1.0):
    n_up, n_dn = C_up.shape[1], C_dn.shape[1]
    s = wl._system("nl-one-centre", [Z], [centre], n_up, n_dn, [0] * len(stypes), stypes, zetas, C_up, C_dn, jastrow or {}, a)
    return wl.with_nonlocal(s, [nl_row], dla)


NL_ROW = [2.5, -0.7, 1.3, 0.9, 0.8, 0.6, 1.1]      # r_c, (A_l, B_l) for l = 0, 1, 2


@pytest.mark.parametrize("l", [0, 1])
def test_pure_l_orbital_is_an_eigenfunction_of_the_projector(l):
    """One electron in a pure s (l=0) or pure p (l=1) orbital centred on the nucleus: sum_q nu_q rho_q = v_l(r) exactly
    (octahedral rule exact to degree 3 >= l + l_channel for l_channel <= 2), for any position and any frame; all three
    channels are switched on, only channel l may contribute."""
    centre = [0.3, -0.2, 0.5]
    if l == 0:
        s = _one_centre([wl.SHELL_S], [0.7], np.ones((1, 1)), np.zeros((1, 0)), centre, NL_ROW)
    else:
        c = RNG.standard_normal((3, 1))
        s = _one_centre([wl.SHELL_P], [0.7], c, np.zeros((3, 0)), centre, NL_ROW)
    o = ref.Ref(s); assert s["nl_K"] == 1 and o.P == 12
    for _ in range(20):
        x = np.array(centre) + RNG.standard_normal(3) * 0.6
        r = np.linalg.norm(x - centre)
        U = _haar(RNG)
        rc, du, dd = o.build_inverse(x[None]); assert rc == 0
        nu, rho, cand = o.nl_info(x[None], U, du, dd)
        inside = r < NL_ROW[0]
        want = NL_ROW[1 + 2 * l] * math.exp(-NL_ROW[2 + 2 * l] * r * r) if inside else 0.0
        assert abs(np.sum(nu * rho) - want) < 1e-13
        if inside:
            assert np.allclose(np.linalg.norm(cand - centre, axis=1), r, atol=1e-13)       # points on the sphere |r' - R| = r
            assert np.allclose(cand[0::2] + cand[1::2], 2 * np.array(centre), atol=1e-13)   # antipodal pairs +-e_k
            assert np.allclose((cand[0::2] - centre) / r, U.T, atol=1e-13)                  # along the versors = columns of U
        R, sc, per, _ = o.evaluate(x[None], U)
        assert np.allclose(R[6:], -nu * rho, atol=1e-15)                                    # slot value = -nu_q rho_q
        if sc["n_vmax"] == 0:                                                               # (a p orbital has a node: D9/D11 may fire)
            assert abs(sc["e_L"] - sc["e_L_continuum"]) < 1e-9 * sc["K_diag"]               # Eq.D7 with V_nl on both sides


def test_projector_matches_lebedev_integration_of_its_definition():
    """V_nl Psi/Psi = sum_i sum_l v_l(r_i) (2l+1)/(4 pi) int P_l(rhat.rhat') Psi(.., R + r_i Omega', ..)/Psi dOmega' written out on
    a 50-point Lebedev rule with Psi from the brute-force log|Psi| (2 electrons, s+p basis on one centre, no Jastrow so Psi = D):
    the 6-point rule of the oracle is exact here (degree <= 3), so the two must agree to rounding."""
    stypes = [wl.SHELL_S, wl.SHELL_P, wl.SHELL_S, wl.SHELL_P]; zetas = [0.5, 0.6, 1.4, 1.7]
    C_up = RNG.standard_normal((8, 1)); C_dn = RNG.standard_normal((8, 1)); centre = np.array([0.1, 0.2, -0.3])
    s = _one_centre(stypes, zetas, C_up, C_dn, centre, NL_ROW)
    o = ref.Ref(s)
    pts, wts = lebedev_rule(11); pts = pts.T
    for _ in range(5):
        x = centre + RNG.standard_normal((2, 3)) * 0.7
        U = _haar(RNG)
        la0, sg0 = o.logpsi(x)
        want = 0.0
        for i in range(2):
            d = x[i] - centre; r = np.linalg.norm(d)
            if r >= NL_ROW[0]:
                continue
            for om, w in zip(pts, wts):
                xq = x.copy(); xq[i] = centre + r * om
                la, sg = o.logpsi(xq)
                ratio = sg * sg0 * math.exp(la - la0)
                ct = float(om @ d) / r
                P = [1.0, ct, 0.5 * (3 * ct * ct - 1)]
                want += sum(NL_ROW[1 + 2 * l] * math.exp(-NL_ROW[2 + 2 * l] * r * r) * (2 * l + 1) / (4 * math.pi) * P[l] for l in range(3)) * w * ratio
        rc, du, dd = o.build_inverse(x); assert rc == 0
        nu, rho, _ = o.nl_info(x, U, du, dd)
        assert abs(np.sum(nu * rho) - want) < 1e-12 * max(1.0, abs(want))


@pytest.mark.parametrize("dla", [True, False])
def test_nonlocal_ratios_slots_and_fixed_node_bookkeeping(dla):
    """Many-electron system, several overlapping cutoff spheres (K > 1), Jastrow on: rho_q against a full recomputation of
    D(x')/D(x) (dla, Jastrow-free clone) or Psi_G(x')/Psi_G(x); nu_q against the Legendre formula; slot order (electron, rank of
    the centre in range, q); R = -nu rho; bbar / V_sf split by sign; node flag from rho < 0; e_L = -bbar + W = continuum + sum nu rho."""
    base = wl.tiny_molecule(3, 2, 3, 9, seed=21, with_pp=True)
    s = wl.random_nonlocal(base, 5, 1.6, 2, dla)
    assert s["nl_K"] >= 2
    o = ref.Ref(s); N = 5; K = s["nl_K"]; P_lat = 6 * N
    nojas = dict(base); nojas.update(a_par=0.0, a_anti=0.0, c1=None, b1=None)
    o_det = ref.Ref(nojas)                                           # Psi = D: brute-force determinant ratios for the DLA case
    o_full = ref.Ref(base)
    seen_active = seen_neg = 0
    for trial in range(12):
        x = base["R"][RNG.integers(0, 3, size=N)] + RNG.standard_normal((N, 3)) * 0.7
        U = _haar(RNG)
        R, sc, per, cand = o.evaluate(x, U)
        rc, du, dd = o.build_inverse(x); assert rc == 0
        nu, rho, cq = o.nl_info(x, U, du, dd)
        brute = o_det if dla else o_full
        la0, sg0 = brute.logpsi(x)
        for i in range(N):
            inr = [I for I in range(3) if s["nl"][I, 0] > 0 and np.linalg.norm(x[i] - base["R"][I]) < s["nl"][I, 0]]
            assert len(inr) <= K
            for kk in range(K):
                for q in range(6):
                    o_ = 6 * (i * K + kk) + q
                    if kk >= len(inr):
                        assert nu[o_] == 0.0 and rho[o_] == 0.0 and R[P_lat + o_] == 0.0
                        continue
                    I = inr[kk]; d = x[i] - base["R"][I]; r = np.linalg.norm(d)
                    e = U[:, q // 2] * (1.0 if q % 2 == 0 else -1.0)
                    assert np.allclose(cq[o_], base["R"][I] + r * e, atol=1e-13) and np.allclose(cand[P_lat + o_], cq[o_])
                    ct = float(e @ d) / r; P = [1.0, ct, 0.5 * (3 * ct * ct - 1)]
                    want_nu = sum((2 * l + 1) * s["nl"][I, 1 + 2 * l] * math.exp(-s["nl"][I, 2 + 2 * l] * r * r) * P[l] for l in range(3)) / 6.0
                    assert abs(nu[o_] - want_nu) < 1e-14 * max(1.0, abs(want_nu))
                    xq = x.copy(); xq[i] = cq[o_]
                    la, sg = brute.logpsi(xq)
                    assert abs(rho[o_] - sg * sg0 * math.exp(la - la0)) < 1e-10 * max(1.0, abs(rho[o_]))
                    seen_active += 1
        A = -nu * rho
        assert np.allclose(R[P_lat:], A, rtol=0, atol=1e-15)
        seen_neg += int((A < 0).sum())
        kap = 1.0 / (2 * s["a"] ** 2)
        bbar = kap * R[:P_lat][R[:P_lat] > 0].sum() + A[A > 0].sum()
        vsf = -kap * R[:P_lat][R[:P_lat] < 0].sum() - A[A < 0].sum()
        assert abs(sc["bbar"] - bbar) < 1e-10 * bbar and abs(sc["V_sf"] - vsf) < 1e-10 * max(1.0, vsf)
        assert sc["node"] == float((R[:P_lat] < 0).any() or (rho < 0).any())
        assert abs(sc["e_L"] - (sc["W"] - sc["bbar"])) < 1e-9 * sc["K_diag"]
        # continuum local energy of the Jastrow-Slater function + the non-local energy on the quadrature (Eq.D7), when no v_max fired
        if sc["n_vmax"] == 0:
            Rl, scl, *_ = o_full.evaluate(x, U)
            assert abs(sc["e_L_continuum"] - (scl["e_L_continuum"] + np.sum(nu * rho))) < 1e-9 * sc["K_diag"]
            assert abs(sc["e_L"] - sc["e_L_continuum"]) < 1e-9 * sc["K_diag"]
        # selection never takes an empty or sign-forbidden slot; the cumulative sums run over lattice then non-local slots
        for u in np.linspace(0.0, 0.999999, 41):
            j, _ = o.select(R, float(u))
            assert R[j] > 0.0
        q = np.concatenate([kap * np.maximum(R[:P_lat], 0), np.maximum(A, 0)]); C = np.cumsum(q)
        for u in (0.03, 0.5, 0.97):
            assert o.select(R, u)[0] == int(np.searchsorted(C, u * C[-1], side="right"))
    assert seen_active > 100 and seen_neg > 5


def test_too_many_centres_in_range_is_an_error():
    base = wl.tiny_molecule(2, 1, 3, 6, seed=22)
    s = wl.random_nonlocal(base, 5, 3.0, 1); s["nl_K"] = 1           # spheres overlap, but only one slot per electron declared
    o = ref.Ref(s)
    x = np.tile(base["R"].mean(0), (3, 1)) + RNG.standard_normal((3, 3)) * 0.1
    with pytest.raises(FloatingPointError):
        o.evaluate(x, np.eye(3))


def _radial_ground_state(A0, B0, rc, Z=1.0, rmax=40.0, h=0.004):
    """Lowest eigenvalue of -1/2 u'' + (-Z/r + v_0(r) [r < r_c]) u = E u, u(0) = u(rmax) = 0: the s-wave sector of
    -1/2 lap - Z/r + v_0(r)|s><s| (the projector is the identity on s functions).  Richardson-extrapolated in h."""
    def solve(hh):
        r = np.arange(1, int(rmax / hh)) * hh
        v = -Z / r + np.where(r < rc, A0 * np.exp(-B0 * r * r), 0.0)
        return eigh_tridiagonal(1.0 / hh**2 + v, np.full(len(r) - 1, -0.5 / hh**2), select="i", select_range=(0, 0))[0][0]
    e1, e2 = solve(h), solve(h / 2)
    return e2 + (e2 - e1) / 3.0


def test_hydrogen_with_an_s_channel_projects_to_the_radial_solver_energy():
    """One electron, -1/r plus an attractive non-local s channel: the ground state is an s state whose exact energy comes from
    the radial equation; LRDMC with the non-local hops must reach it as a -> 0 (O(a^2) bias, L23/L140), in both modes, and lie
    below the energy without the channel (-0.5)."""
    A0, B0, rc = -0.8, 1.5, 2.2
    E_exact = _radial_ground_state(A0, B0, rc)
    assert -0.75 < E_exact < -0.55
    a = np.array([0.2, 0.3, 0.4]); E = []; sg = []
    for ai in a:
        s = wl.with_nonlocal(wl.hydrogen(alpha=1.1, a=float(ai)), [[rc, A0, B0, 0, 1, 0, 1]])
        o = ref.Ref(s); o.set_positions(wl.hydrogen_walkers(256, 3))
        out = drv.run(o, ref.BALANCED, 300, n_moves=max(4, int(round(40 * (0.2 / ai) ** 2))), E0=-0.6)
        e, sgm = drv.energy(out["wbar"], out["num"], out["den"], p=10, n_therm=60); E.append(e); sg.append(sgm)
        assert out["n_nonpos_diag"].sum() == 0 and out["n_nonfinite"].sum() == 0
    E = np.array(E); sg = np.array(sg)
    Amat = np.stack([np.ones_like(a), a**2], 1) / sg[:, None]
    cov = np.linalg.inv(Amat.T @ Amat); coef = cov @ Amat.T @ (E / sg)
    assert abs(coef[0] - E_exact) < 3 * math.sqrt(cov[0, 0]) + 5e-4 and math.sqrt(cov[0, 0]) < 3e-3
    # conventional mode at one spacing agrees with the balanced one (L234)
    s = wl.with_nonlocal(wl.hydrogen(alpha=1.1, a=0.3), [[rc, A0, B0, 0, 1, 0, 1]])
    o = ref.Ref(s); o.set_positions(wl.hydrogen_walkers(256, 3))
    out = drv.run(o, ref.CONVENTIONAL, 300, tau=18 * 0.09 / 3, E_ref=-0.6)
    ec, sc_ = drv.energy(out["wbar"], out["num"], out["den"], p=10, n_therm=60)
    assert abs(ec - E[1]) < 3 * math.hypot(sc_, sg[1])
