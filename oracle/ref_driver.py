"""ORACLE (test infrastructure): the outer loops of Alg.1 / Alg.2 and the estimators of Eq.18-19.

Plain numpy, written from PAPER.md:
  * Alg.2 lines 2-13 (L398-L420): for each generation: propagate all walkers, average, branch, update E_0.
  * Eq.18 (L127): G_n^p = prod_{j=1..p} wbar_{n-j};  Eq.19 (L131): E_0 ~ sum_n G_n^p e_n / sum_n G_n^p.
  * Eq.20 (L135) / Eq.34 (L227): e_n = num_n / den_n, evaluated just before each reconfiguration (L138).
Readings: Q8a E_0 policy = running mean of e_n over the generations so far, Q9 p = 10,
n_therm = 20 % of the run, jackknife over blocks of generations.
"""
from __future__ import annotations

import numpy as np

from . import lrdmc_ref as ref


def population_factors(wbar, p):
    """Eq.18: G[n] = wbar[n-1] * ... * wbar[n-p] (factors with n-j < 0 are left out)."""
    wbar = np.asarray(wbar, dtype=np.float64)
    G = np.ones(len(wbar))
    for n in range(len(wbar)):
        for j in range(1, p + 1):
            if n - j >= 0:
                G[n] *= wbar[n - j]
    return G


def energy(wbar, num, den, p=10, n_therm=0, n_blocks=20):
    """Eq.19 over generations n >= n_therm, and a delete-one-block jackknife error bar."""
    wbar = np.asarray(wbar, float); num = np.asarray(num, float); den = np.asarray(den, float)
    G = population_factors(wbar, p)[n_therm:]
    e = (num / den)[n_therm:]
    n = len(e)
    E = float(np.sum(G * e) / np.sum(G))
    nb = max(2, min(n_blocks, n))
    edges = np.linspace(0, n, nb + 1).astype(int)
    Ej = []
    for b in range(nb):
        keep = np.ones(n, bool); keep[edges[b]:edges[b + 1]] = False
        Ej.append(np.sum(G[keep] * e[keep]) / np.sum(G[keep]))
    Ej = np.array(Ej)
    sigma = float(np.sqrt((nb - 1) / nb * np.sum((Ej - Ej.mean()) ** 2)))
    return E, sigma


def run(o: "ref.Ref", mode, cycles, n_moves=0, tau=0.0, E0=None, E_ref=None, first_cycle=0, feedback=True, n_therm=0):
    """Alg.2 (balanced) / Alg.1 (conventional) outer loop on an oracle context whose walkers are set.

    Returns a dict of per-generation arrays (wbar, num, den, e, moves_*, flags).  `E0`: initial guess
    for the balanced Green's function (Eq.28); updated after each branching (L232) as the running mean
    of e_n when `feedback`; the mean restarts once at generation `n_therm` (reading Q8a: "after n_therm: restart the mean").
    Conventional mode passes the fixed shift E_ref (Q8b)."""
    rec = {k: [] for k in ("wbar", "num", "den", "moves_min", "moves_max", "moves_sum", "n_node_flag",
                           "n_nonpos_diag", "n_nonfinite", "lockstep_idle_frac", "E0_used")}
    e_hist = []
    for c in range(first_cycle, first_cycle + cycles):
        shift = E0 if mode == ref.BALANCED else (E_ref if E_ref is not None else 0.0)
        rc = o.propagate(mode, n_moves, tau, shift, c); assert rc == 0, rc
        rc, _ = o.reconfigure(c); assert rc == 0, rc
        s = o.estimators()
        for k in rec:
            if k != "E0_used":
                rec[k].append(s[k])
        rec["E0_used"].append(shift)
        e_hist.append(s["num"] / s["den"])
        if mode == ref.BALANCED and feedback:    # "Update E_0" (Alg.2 line 12, L418; reading Q8a)
            i = len(e_hist) - 1
            E0 = float(np.mean(e_hist[n_therm:] if (n_therm > 0 and i >= n_therm) else e_hist))
    out = {k: np.array(v) for k, v in rec.items()}
    out["e"] = np.array(e_hist)
    return out


def fit_even_powers(a_list, energies, sigmas, n_terms=2):
    """E(a) = E_0 + c_2 a^2 (+ c_4 a^4): the lattice bias is even in a and vanishes as a -> 0 (L23, L140).  Weighted least squares
    through the normal equations, written out; returns (E_0, sigma(E_0))."""
    a = np.asarray(a_list, float); E = np.asarray(energies, float); w = 1.0 / np.asarray(sigmas, float) ** 2
    M = np.zeros((n_terms, n_terms)); v = np.zeros(n_terms)
    for k in range(n_terms):
        for l in range(n_terms):
            M[k, l] = np.sum(w * a ** (2 * k) * a ** (2 * l))
        v[k] = np.sum(w * a ** (2 * k) * E)
    cov = np.linalg.inv(M)
    return float((cov @ v)[0]), float(np.sqrt(cov[0, 0]))


def a_scan(make_system, make_walkers, a_list, n_walkers, cycles, moves, modes=("balanced", "conventional"), E0=0.0, n_therm=None,
           p=10, n_blocks=10):
    """The a -> 0 validation in the shape of Table I (L254-L265): one run per lattice spacing and algorithm, one after the other;
    E(a) per row, then the a -> 0 fit per algorithm (L140).  Run number q (a-major, mode-minor) uses the Philox key
    seed + 1000003 (q + 1): independent points.  Conventional runs take tau = moves a^2 / (3N) (same mean move count, Q19)."""
    rows = []
    for ia, a in enumerate(a_list):
        row = {"a": a}
        for im, mode in enumerate(modes):
            q = ia * len(modes) + im
            s = dict(make_system(a)); s["seed"] = int(s["seed"]) + 1000003 * (q + 1)
            N = s["n_up"] + s["n_dn"]
            o = ref.Ref(s); rc = o.set_positions(make_walkers(s, n_walkers)); assert rc == 0, rc
            if mode == "balanced":
                out = run(o, ref.BALANCED, cycles, n_moves=moves, E0=E0)
            else:
                out = run(o, ref.CONVENTIONAL, cycles, tau=moves * a * a / (3 * N), E_ref=E0)
            row[mode] = energy(out["wbar"], out["num"], out["den"], p=p, n_therm=cycles // 5 if n_therm is None else n_therm, n_blocks=n_blocks)
            row[mode + "_first_e"] = out["e"][:3].copy()
        rows.append(row)
    res = {"rows": rows}
    for mode in modes:
        res[mode] = fit_even_powers([r["a"] for r in rows], [r[mode][0] for r in rows], [r[mode][1] for r in rows])
    return res
