"""Outer loop of Alg.2 / Alg.1 on the CUDA path (PAPER.md L389-L423 / L311-L387): per generation
propagate -> reconfigure -> estimators, E_0 fed back after each branching (L232, Alg.2 line 12 L418).

Host-side control only; every numerical step is a call into liblrdmc.so (binding.Lrdmc).  The energy over
generations (Eq.18-19) is computed by the library's `lrdmc_energy`.
"""
from __future__ import annotations

from . import binding as B


def work_per_walker_move(sysd):
    """Algorithmic FP64 flop per walker-move (SURVEY.md 8(d) count; exp = 25 flop):
    2PAO + P(8S+2A) + 25PS + 12P(N-1+M) + 2PO + [8S+10A+10AO] + 4O^2."""
    N = sysd["n_up"] + sysd["n_dn"]; M = sysd["n_nuc"]; A = sysd["n_ao"]; S = sysd["n_shell"]
    O = max(sysd["n_up"], sysd["n_dn"]); P = 6 * N * (2 if sysd["a2"] > 0 else 1)
    parts = dict(gemm=2 * P * A * O, ao_poly=P * (8 * S + 2 * A), exps=25 * P * S, jastrow=12 * P * (N - 1 + M),
                 ratios=2 * P * O, refresh=8 * S + 10 * A + 10 * A * O, sherman_morrison=4 * O * O)
    parts["total"] = sum(parts.values())
    return parts


def state_bytes_per_walker(sysd):
    """Walker record in HBM: positions 3N, two inverses, cached MO rows N x 5 x OS (OS = MO count padded to 8)."""
    N = sysd["n_up"] + sysd["n_dn"]; O = max(sysd["n_up"], sysd["n_dn"]); OS = 8 * (1 if O <= 8 else (2 if O <= 16 else 4))
    return 8 * (3 * N + sysd["n_up"] ** 2 + sysd["n_dn"] ** 2 + N * 5 * OS)


def run(g: "B.Lrdmc", mode, cycles, n_moves=0, tau=0.0, E0=0.0, first_cycle=0, feedback=True):
    """Returns the list of per-generation CycleStats.  Balanced: E0 is the Green's-function energy of Eq.28,
    updated to the running mean of e_n (reading Q8a).  Conventional: E0 is the fixed reference shift (Q8b)."""
    recs = []; esum = 0.0
    for c in range(first_cycle, first_cycle + cycles):
        g.lrdmc_propagate(mode, n_moves, tau, E0, c)
        g.lrdmc_reconfigure(c)
        s = g.lrdmc_estimators()
        recs.append(s)
        esum += s.num / s.den
        if mode == B.BALANCED and feedback:
            E0 = esum / len(recs)
    return recs
