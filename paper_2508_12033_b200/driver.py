"""Outer loop of Alg.2 / Alg.1 on the CUDA path (PAPER.md L389-L423 / L311-L387): per generation
propagate -> reconfigure -> estimators, E_0 fed back after each branching (L232, Alg.2 line 12 L418).

Host-side control only; every numerical step is a call into liblrdmc.so (binding.Lrdmc).  The energy over
generations (Eq.18-19) is computed by the library's `lrdmc_energy`.
"""
from __future__ import annotations

from . import binding as B


def work_per_walker_move(sysd):
    """FP64 flop per walker-move, two counts.

    `total` -- the ALGORITHMIC count of SURVEY.md 8(d) (every candidate through the MOs; exp = 25 flop):
        2PAO + P(8S+2A) + 25PS + 12P(N-1+M) + 2PO + [8S+10A+10AO] + 4O^2.
    `executed` -- what the kernels actually run (column form): the candidates never go through the MOs;
        per evaluation Bc = C Dinv costs sum_spin 2 A O n_spin = 2AON and every AO value meets ONE number (2PA), so the terms
        2PAO + 2PO become 2PA + 2AON; everything else is counted as in `total`.  `total / executed` is the algorithmic saving of
        the column form; `executed / time` is what the FP64 pipe really delivers (compare ncu sm__pipe_fp64_cycles_active)."""
    N = sysd["n_up"] + sysd["n_dn"]; M = sysd["n_nuc"]; A = sysd["n_ao"]; S = sysd["n_shell"]
    O = max(sysd["n_up"], sysd["n_dn"]); P = 6 * N * (2 if sysd["a2"] > 0 else 1)
    parts = dict(gemm=2 * P * A * O, ao_poly=P * (8 * S + 2 * A), exps=25 * P * S, jastrow=12 * P * (N - 1 + M),
                 ratios=2 * P * O, refresh=8 * S + 10 * A + 10 * A * O, sherman_morrison=4 * O * O)
    parts["total"] = sum(parts.values())
    parts["column_form"] = 2 * P * A + 2 * A * O * N
    parts["executed"] = parts["total"] - parts["gemm"] - parts["ratios"] + parts["column_form"]
    return parts


def state_bytes_per_walker(sysd):
    """Walker record in HBM: positions 3N, two inverses, cached MO rows N x 5 x OS (OS = MO count padded to 8)."""
    N = sysd["n_up"] + sysd["n_dn"]; O = max(sysd["n_up"], sysd["n_dn"]); OS = 8 * (1 if O <= 8 else (2 if O <= 16 else 4))
    return 8 * (3 * N + sysd["n_up"] ** 2 + sysd["n_dn"] ** 2 + N * 5 * OS)


def run(g: "B.Lrdmc", mode, cycles, n_moves=0, tau=0.0, E0=0.0, first_cycle=0, feedback=True, n_therm=0):
    """Returns the list of per-generation CycleStats.  Balanced: E0 is the Green's-function energy of Eq.28,
    updated after each branching (L232, Alg.2 line 12 L418) to the running mean of e_n; the mean restarts once, when
    generation n_therm is reached, so that the equilibration transient does not stay in it (reading Q8a).
    Conventional: E0 is the fixed reference shift (Q8b)."""
    recs = []; esum = 0.0; ecnt = 0
    for i, c in enumerate(range(first_cycle, first_cycle + cycles)):
        g.lrdmc_propagate(mode, n_moves, tau, E0, c)
        g.lrdmc_reconfigure(c)
        s = g.lrdmc_estimators()
        recs.append(s)
        if i == n_therm and n_therm > 0:
            esum = 0.0; ecnt = 0
        esum += s.num / s.den; ecnt += 1
        if mode == B.BALANCED and feedback:
            E0 = esum / ecnt
    return recs


# ---- a -> 0 driver ("extrapolated to a -> 0", Table I L254-L265 shape) -----------------
def fit_a_to_zero(a_list, energies, sigmas, n_terms=2):
    """Weighted least squares of E(a) = E_0 + c_2 a^2 (+ c_4 a^4 for n_terms = 3): the lattice bias is even in a (L23, L140).
    Returns (E_0, sigma(E_0), coefficients, chi2).  Host arithmetic on a handful of numbers; no device work."""
    import numpy as np
    a = np.asarray(a_list, float); E = np.asarray(energies, float); s = np.asarray(sigmas, float)
    if not (len(a) == len(E) == len(s)) or len(a) < n_terms or np.any(s <= 0):
        raise ValueError("need at least n_terms points with positive error bars")
    X = np.stack([a ** (2 * k) for k in range(n_terms)], axis=1) / s[:, None]
    cov = np.linalg.inv(X.T @ X)
    coef = cov @ (X.T @ (E / s))
    chi2 = float(np.sum((X @ coef - E / s) ** 2))
    return float(coef[0]), float(np.sqrt(cov[0, 0])), coef, chi2


def a_scan(make_system, make_walkers, a_list, n_walkers, cycles, moves, modes=("balanced", "conventional"), E0=0.0, n_therm=None,
           p=10, n_blocks=10, device="cuda:0", concurrent=True, feedback_therm=0):
    """SURVEY 8(f) f3 "several a in one batch": one LRDMC run per (lattice spacing, mode), ALL of them in flight together on the CUDA
    path -- every run is a context of its own on a CUDA stream of its own; each run's next generation is enqueued as soon as its own
    estimators have been read and its E_0 updated (pipelined, no barrier across the runs), so the small ensembles of an a-scan share the
    device instead of leaving most SMs idle one after the other (`concurrent=False`: one run after the other, same numbers).
    Rows shaped like Table I (a, E_balanced, E_conventional; L254-L265), then the E(a) = E_0 + c a^2 fits (L140).
    make_system(a) -> system dict; make_walkers(system, n_walkers) -> positions.  Run number q (a-major, mode-minor) draws from its
    own random streams: Philox key = the system's seed + 1000003 (q + 1), so the points of the fit are statistically independent.
    Conventional mode uses the projection time with the same mean move count, tau = moves a^2 / (3N) (reading Q19)."""
    import torch
    runs = []
    for ia, a in enumerate(a_list):
        for im, mode in enumerate(modes):
            q = ia * len(modes) + im
            sysd = dict(make_system(a)); sysd["seed"] = int(sysd["seed"]) + 1000003 * (q + 1)
            N = sysd["n_up"] + sysd["n_dn"]
            g = B.Lrdmc(sysd, device=device)
            st = torch.cuda.Stream(device=device) if concurrent else torch.cuda.current_stream(device)
            with torch.cuda.stream(st):
                g.lrdmc_set_positions(make_walkers(sysd, n_walkers))
            runs.append(dict(a=a, mode=mode, g=g, stream=st, E0=E0, esum=0.0, ecnt=0, recs=[],
                             kind=B.BALANCED if mode == "balanced" else B.CONVENTIONAL,
                             n_moves=moves if mode == "balanced" else 0, tau=0.0 if mode == "balanced" else moves * a * a / (3 * N)))

    def enqueue(r, c):                                             # nothing here waits for the device
        with torch.cuda.stream(r["stream"]):
            r["g"].lrdmc_propagate(r["kind"], r["n_moves"], r["tau"], r["E0"], c)
            r["g"].lrdmc_reconfigure(c)

    def collect(r):                                                # waits for the run's own stream only
        s = r["g"].lrdmc_estimators(); r["recs"].append(s)
        if len(r["recs"]) - 1 == feedback_therm and feedback_therm > 0:
            r["esum"] = 0.0; r["ecnt"] = 0
        r["esum"] += s.num / s.den; r["ecnt"] += 1
        if r["kind"] == B.BALANCED:
            r["E0"] = r["esum"] / r["ecnt"]                        # "Update E_0" (Alg.2 line 12 L418; reading Q8a)
    if concurrent:
        # Pipelined: a run's generation c is enqueued as soon as ITS generation c - 1 has been read (E_0 feedback), while the other runs'
        # kernels are still queued or running -- no barrier across the runs between generations, so the device always has every run's
        # CTAs to fill its SMs with (a generation of all runs together does not fit the resident slots: lock-stepped generations ran in two waves).
        for c in range(cycles):
            for r in runs:
                if c > 0:
                    collect(r)
                enqueue(r, c)
        for r in runs:
            collect(r)
    else:
        for r in runs:
            for c in range(cycles):
                enqueue(r, c); collect(r)
    rows = []
    for a in a_list:
        row = {"a": a}
        for r in runs:
            if r["a"] == a:
                row[r["mode"]] = B.lrdmc_energy(r["recs"], p=p, n_therm=cycles // 5 if n_therm is None else n_therm, n_blocks=n_blocks)
        rows.append(row)
    for r in runs:
        r["g"].close()
    out = {"rows": rows}
    for mode in modes:
        out[mode] = fit_a_to_zero([r["a"] for r in rows], [r[mode][0] for r in rows], [r[mode][1] for r in rows])
    return out
