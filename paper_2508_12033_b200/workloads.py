"""Seeded synthetic input generators shared by the oracle, the CUDA path, the tests and bench.py.

This module holds NONE of the method's arithmetic: it only draws the arrays that describe a
system (nuclei, shells, MO coefficients, Jastrow / pseudopotential parameters, lattice spacing) and
the initial walker positions, with numpy only.  Both `oracle/` and the CUDA binding consume the
plain dict it returns; neither imports the other.

The five configurations are the ones listed in BASELINE.json `configs` (SURVEY.md section 8, table
"Config shorthand", and section 8(d) "Inputs").  The paper's own workloads (water-methane with ccECP /
cc-pVTZ and PySCF trial wavefunctions; benzene, L279-L285) are not available; these
synthetic systems take their shapes (electron count, nuclei count, basis size, N_w, a, moves per
branching) and nothing else.
"""
from __future__ import annotations

import numpy as np

# shell type codes (the C-ABI and the oracle use the same integers; PAPER.md names the basis only,
# L242/L285 -- the functional forms are DESIGN.md reading Q14)
SHELL_S, SHELL_P, SHELL_D, SHELL_SLATER_S = 0, 1, 2, 10
_AO_PER_SHELL = {SHELL_S: 1, SHELL_P: 3, SHELL_D: 6, SHELL_SLATER_S: 1}

PHILOX_RUN_SEED = 12345


def n_ao_of(types) -> int:
    return int(sum(_AO_PER_SHELL[int(t)] for t in types))


def n_ao_contracted(types, first, sph) -> int:
    """AO count of contracted shells: run cs of primitive shells first[cs]..first[cs+1]-1; a solid-harmonic d shell has 5 functions."""
    return int(sum(5 if (int(types[first[cs]]) == SHELL_D and sph[cs]) else _AO_PER_SHELL[int(types[first[cs]])] for cs in range(len(sph))))


def _system(name, Z, R, n_up, n_dn, center, stype, zeta, C_up, C_dn, jastrow, a, a2=0.0, pp=None,
            n_walkers=0, cycles=0, moves=0, seed=PHILOX_RUN_SEED, contraction=None):
    Z = np.ascontiguousarray(Z, dtype=np.float64)
    R = np.ascontiguousarray(R, dtype=np.float64).reshape(-1, 3)
    d = dict(
        name=name,
        Z=Z, R=R, n_nuc=int(Z.shape[0]), n_up=int(n_up), n_dn=int(n_dn),
        pp=None if pp is None else np.ascontiguousarray(pp, dtype=np.float64).reshape(-1, 4),
        shell_center=np.ascontiguousarray(center, dtype=np.int32),
        shell_type=np.ascontiguousarray(stype, dtype=np.int32),
        shell_zeta=np.ascontiguousarray(zeta, dtype=np.float64),
        n_shell=int(len(center)), n_ao=n_ao_of(stype) if contraction is None else n_ao_contracted(stype, contraction[0], contraction[2]),
        # contracted / solid-harmonic shells (scope row f2): the shells above are then primitives, the MOs refer to the contracted AOs
        cs_first=None if contraction is None else np.ascontiguousarray(contraction[0], dtype=np.int32),
        prim_coef=None if contraction is None else np.ascontiguousarray(contraction[1], dtype=np.float64),
        cs_sph=None if contraction is None else np.ascontiguousarray(contraction[2], dtype=np.int32),
        C_up=np.ascontiguousarray(C_up, dtype=np.float64),
        C_dn=np.ascontiguousarray(C_dn, dtype=np.float64),
        a_par=float(jastrow.get("a_par", 0.0)), a_anti=float(jastrow.get("a_anti", 0.0)),
        b2=float(jastrow.get("b2", 1.0)),
        c1=None if jastrow.get("c1") is None else np.ascontiguousarray(jastrow["c1"], dtype=np.float64),
        b1=None if jastrow.get("b1") is None else np.ascontiguousarray(jastrow["b1"], dtype=np.float64),
        a=float(a), a2=float(a2), seed=int(seed),
        n_walkers=int(n_walkers), cycles=int(cycles), moves=int(moves),
        nl=None, nl_K=0, nl_dla=1,      # non-local pseudopotential channels (scope row f1): see with_nonlocal
        j3_center=None, j3_zeta=None, j3_g=None, j3_lmn=None,   # three-body Jastrow (scope row f2): see with_jastrow3
    )
    assert d["C_up"].shape == (d["n_ao"], d["n_up"])
    assert d["C_dn"].shape == (d["n_ao"], d["n_dn"])
    return d


def _round_robin_shells(rng, n_nuc, n_shell):
    center = np.arange(n_shell) % n_nuc
    stype = np.array([(SHELL_S, SHELL_P, SHELL_D)[k % 3] for k in range(n_shell)])
    zeta = np.exp(rng.uniform(np.log(0.1), np.log(20.0), size=n_shell))
    return center, stype, zeta


def _orthonormal_mos(rng, n_ao, n_occ):
    q, _ = np.linalg.qr(rng.standard_normal((n_ao, n_occ)))
    return np.ascontiguousarray(q[:, :n_occ])


def _separated_points(rng, n, draw, min_sep):
    pts = []
    while len(pts) < n:
        p = draw()
        if all(np.linalg.norm(p - q) >= min_sep for q in pts):
            pts.append(p)
    return np.array(pts)


def initial_walkers(sysd, n_walkers, seed):
    """Q18: each electron starts at a nucleus chosen with probability ~ Z plus a
    N(0, 1 bohr) offset.  Config C1 overrides this (uniform cube).  Returns [n_w][N][3] float64."""
    rng = np.random.default_rng(seed)
    N = sysd["n_up"] + sysd["n_dn"]
    p = sysd["Z"] / sysd["Z"].sum()
    which = rng.choice(sysd["n_nuc"], size=(n_walkers, N), p=p)
    return np.ascontiguousarray(sysd["R"][which] + rng.standard_normal((n_walkers, N, 3)))


def hydrogen(alpha=0.9, a=0.2, n_walkers=256, cycles=200, moves=40, seed=PHILOX_RUN_SEED):
    """C1: H atom, one electron, Z=1 at the origin, psi = exp(-alpha r), no Jastrow."""
    return _system("C1-hydrogen", [1.0], [[0.0, 0.0, 0.0]], 1, 0, [0], [SHELL_SLATER_S], [alpha],
                   np.ones((1, 1)), np.zeros((1, 0)), {}, a,
                   n_walkers=n_walkers, cycles=cycles, moves=moves, seed=seed)


def hydrogen_walkers(n_walkers=256, seed=1):
    """C1 start: uniform in the 2-bohr cube [-1, 1]^3 (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    return np.ascontiguousarray(rng.uniform(-1.0, 1.0, size=(n_walkers, 1, 3)))


def slater_atom(Z, zetas, n_up, n_dn, C_up, C_dn, a, jastrow=None, name="slater-atom"):
    """Small all-electron atom on Slater-type s orbitals at the origin (pins P7/P8: He singlet and
    He 2^3S).  Not one of the BASELINE configs; used by the oracle's physics pins and GPU parity."""
    ns = len(zetas)
    return _system(name, [float(Z)], [[0.0, 0.0, 0.0]], n_up, n_dn, [0] * ns, [SHELL_SLATER_S] * ns,
                   zetas, C_up, C_dn, jastrow or {}, a)


def slater_molecule(Z, R, zetas, centers, n_up, n_dn, C_up, C_dn, a, jastrow=None, name="slater-mol"):
    """Small all-electron molecule on Slater-type s orbitals (pin P7: H2)."""
    return _system(name, Z, R, n_up, n_dn, centers, [SHELL_SLATER_S] * len(zetas), zetas, C_up, C_dn,
                   jastrow or {}, a)


def synthetic10(a=0.2, n_walkers=1024, cycles=100, moves=50, seed=PHILOX_RUN_SEED):
    """C2: 10 electrons (5/5), nuclei Z = 6, 2, 2 inside a 3-bohr ball, 60 s/p/d GTOs (18 shells),
    random orthonormal MOs, one- and two-body Pade Jastrow with b = 1."""
    rng = np.random.default_rng(2)

    def draw():
        while True:
            p = rng.uniform(-3.0, 3.0, size=3)
            if np.linalg.norm(p) <= 3.0:
                return p
    R = _separated_points(rng, 3, draw, 1.0)
    Z = np.array([6.0, 2.0, 2.0])
    center, stype, zeta = _round_robin_shells(rng, 3, 18)
    C = _orthonormal_mos(rng, n_ao_of(stype), 5)
    jas = dict(a_par=0.25, a_anti=0.5, b2=1.0, c1=Z.copy(), b1=np.ones(3))
    return _system("C2-synthetic10", Z, R, 5, 5, center, stype, zeta, C, C.copy(), jas, a,
                   n_walkers=n_walkers, cycles=cycles, moves=moves, seed=seed)


def _water_methane_geometry(rng):
    # equilibrium-LIKE template (generic bond lengths/angles), jittered; not a published geometry
    oh, hoh = 1.81, np.deg2rad(104.5)
    O = np.zeros(3)
    H1 = oh * np.array([np.sin(hoh / 2), 0.0, np.cos(hoh / 2)])
    H2 = oh * np.array([-np.sin(hoh / 2), 0.0, np.cos(hoh / 2)])
    Cc = np.array([0.0, 0.0, -6.5])
    ch = 2.05
    t = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], dtype=float) / np.sqrt(3.0)
    Hc = Cc + ch * t
    R = np.vstack([O, Cc, H1, H2, Hc])
    return R + rng.normal(0.0, 0.05, size=R.shape)


def water_methane(a=0.2, n_walkers=400, cycles=200, moves=100, seed=PHILOX_RUN_SEED, name=None):
    """C3/C4: water-methane-SHAPED complex: 16 valence electrons (8/8); O, C, 6 H with effective
    charges 6, 4, 1 and a local Gaussian pseudopotential per nucleus; 200 s/p/d GTOs (60 shells)."""
    rng = np.random.default_rng(3)
    R = _water_methane_geometry(rng)
    Z = np.array([6.0, 4.0] + [1.0] * 6)
    center, stype, zeta = _round_robin_shells(rng, 8, 60)
    C = _orthonormal_mos(rng, n_ao_of(stype), 8)
    # local PP parameters (alpha, beta, gamma, delta) per nucleus, reading Q14
    alpha = np.exp(rng.uniform(0.0, np.log(10.0), size=8))
    beta = np.exp(rng.uniform(0.0, np.log(10.0), size=8))
    delta = np.exp(rng.uniform(0.0, np.log(10.0), size=8))
    gamma = rng.uniform(0.0, 2.0 * Z)
    pp = np.stack([alpha, beta, gamma, delta], axis=1)
    jas = dict(a_par=0.25, a_anti=0.5, b2=1.0, c1=np.full(8, 0.5), b1=np.ones(8))
    return _system(name or f"C3-water-methane-shaped-Nw{n_walkers}", Z, R, 8, 8, center, stype, zeta,
                   C, C.copy(), jas, a, pp=pp, n_walkers=n_walkers, cycles=cycles, moves=moves, seed=seed)


def water_methane_full(a=0.2, seed=PHILOX_RUN_SEED):
    """C4: the C3 system scaled to fill one B200: N_w = 25600, 500 cycles x 100 moves."""
    return water_methane(a=a, n_walkers=25600, cycles=500, moves=100, seed=seed,
                         name="C4-water-methane-shaped-Nw25600")


def cluster64(a=0.2, a2=0.4, n_walkers=4096, cycles=200, moves=200, seed=PHILOX_RUN_SEED):
    """C5: 64 electrons (32/32), 24 all-electron nuclei with Z in {1, 4, 6} (sum 64) in a 12-bohr
    box, 600 s/p/d GTOs (180 shells), double lattice spacing a / a'."""
    rng = np.random.default_rng(5)
    R = _separated_points(rng, 24, lambda: rng.uniform(0.0, 12.0, size=3), 1.5)
    while True:
        Z = rng.choice([1.0, 4.0, 6.0], size=24)
        if Z.sum() == 64.0:
            break
    center, stype, zeta = _round_robin_shells(rng, 24, 180)
    C = _orthonormal_mos(rng, n_ao_of(stype), 32)
    jas = dict(a_par=0.25, a_anti=0.5, b2=1.0, c1=Z.copy(), b1=np.ones(24))
    return _system("C5-cluster64", Z, R, 32, 32, center, stype, zeta, C, C.copy(), jas, a, a2=a2,
                   n_walkers=n_walkers, cycles=cycles, moves=moves, seed=seed)


def tiny_molecule(n_up=2, n_dn=1, n_nuc=2, n_shell=6, seed=7, a=0.2, a2=0.0, with_pp=False):
    """A few-electron s/p/d system for brute-force pins (P3) and ragged-shape parity cases."""
    rng = np.random.default_rng(seed)
    R = _separated_points(rng, n_nuc, lambda: rng.uniform(-1.5, 1.5, size=3), 1.0)
    Z = rng.choice([1.0, 2.0, 3.0], size=n_nuc)
    center, stype, zeta = _round_robin_shells(rng, n_nuc, n_shell)
    zeta = np.exp(rng.uniform(np.log(0.2), np.log(3.0), size=n_shell))
    n_ao = n_ao_of(stype)
    C_up = _orthonormal_mos(rng, n_ao, n_up)
    C_dn = _orthonormal_mos(rng, n_ao, n_dn) if n_dn else np.zeros((n_ao, 0))
    pp = None
    c1 = Z.copy()
    if with_pp:
        pp = np.stack([np.exp(rng.uniform(0.0, np.log(10.0), size=n_nuc)),
                       np.exp(rng.uniform(0.0, np.log(10.0), size=n_nuc)),
                       rng.uniform(0.0, 2.0 * Z),
                       np.exp(rng.uniform(0.0, np.log(10.0), size=n_nuc))], axis=1)
        c1 = np.full(n_nuc, 0.5)
    jas = dict(a_par=0.25, a_anti=0.5, b2=0.8, c1=c1, b1=rng.uniform(0.5, 1.5, size=n_nuc))
    return _system(f"tiny-{n_up}u{n_dn}d", Z, R, n_up, n_dn, center, stype, zeta, C_up, C_dn, jas, a,
                   a2=a2, pp=pp)


def contracted_molecule(n_up=3, n_dn=2, n_nuc=3, n_cshell=9, seed=31, a=0.2, spherical=True, with_pp=False):
    """Scope row f2: a small molecule on CONTRACTED shells (1-3 primitives each, seeded coefficients) with real solid-harmonic d
    shells -- the shape of the paper's cc-pVTZ / spherical-harmonics basis (L242); exponents and coefficients are synthetic."""
    rng = np.random.default_rng(seed)
    R = _separated_points(rng, n_nuc, lambda: rng.uniform(-1.5, 1.5, size=3), 1.0)
    Z = rng.choice([1.0, 2.0, 3.0], size=n_nuc)
    center, stype, zeta, coef, first, sph = [], [], [], [], [0], []
    for cs in range(n_cshell):
        t = (SHELL_S, SHELL_P, SHELL_D)[cs % 3]; nprim = int(rng.integers(1, 4))
        z0 = np.exp(rng.uniform(np.log(0.2), np.log(1.0)))
        for k in range(nprim):
            center.append(cs % n_nuc); stype.append(t); zeta.append(z0 * 2.5 ** k); coef.append(rng.uniform(0.2, 1.0) * (1 if k % 2 == 0 else -0.5))
        first.append(len(center)); sph.append(1 if (t == SHELL_D and spherical) else 0)
    n_ao = n_ao_contracted(stype, first, sph)
    C_up = _orthonormal_mos(rng, n_ao, n_up)
    C_dn = _orthonormal_mos(rng, n_ao, n_dn) if n_dn else np.zeros((n_ao, 0))
    pp = None; c1 = Z.copy()
    if with_pp:
        pp = np.stack([np.exp(rng.uniform(0.0, np.log(10.0), size=n_nuc)), np.exp(rng.uniform(0.0, np.log(10.0), size=n_nuc)),
                       rng.uniform(0.0, 2.0 * Z), np.exp(rng.uniform(0.0, np.log(10.0), size=n_nuc))], axis=1)
        c1 = np.full(n_nuc, 0.5)
    jas = dict(a_par=0.25, a_anti=0.5, b2=0.8, c1=c1, b1=rng.uniform(0.5, 1.5, size=n_nuc))
    return _system(f"contracted-{n_up}u{n_dn}d" + ("-sph" if spherical else "-cart"), Z, R, n_up, n_dn, center, stype, zeta, C_up, C_dn, jas, a,
                   pp=pp, contraction=(first, coef, sph))


def contracted_slater_molecule(a=0.2, with_gaussians=True):
    """Scope row f2: CONTRACTED SLATER shells (L242 names the Slater-type basis of the TurboRVB runs): a two-centre, four-electron
    (2/2) molecule whose s functions are fixed sums of 2-3 Slater primitives exp(-zeta r), optionally next to Gaussian p/d shells
    (one contracted p, one solid-harmonic d) so that all shell groups of the kernels meet in one system.  Seeded, synthetic."""
    rng = np.random.default_rng(41)
    R = np.array([[0.0, 0.0, -0.7], [0.1, 0.0, 0.75]]); Z = np.array([2.0, 2.0])
    center = [0, 0, 0, 1, 1, 0, 1]; stype = [SHELL_SLATER_S] * 7; zeta = [2.6, 1.4, 0.9, 3.1, 1.1, 0.7, 0.8]
    coef = [0.5, 0.4, 0.2, 0.7, -0.3, 1.0, 1.0]; first = [0, 3, 5, 6, 7]; sph = [0, 0, 0, 0]
    if with_gaussians:
        center += [0, 0, 1]; stype += [SHELL_P, SHELL_P, SHELL_D]; zeta += [1.3, 0.5, 0.9]; coef += [0.6, 0.5, 1.0]
        first += [9, 10]; sph += [0, 1]
    n_ao = n_ao_contracted(stype, first, sph)
    C_up = _orthonormal_mos(rng, n_ao, 2); C_dn = _orthonormal_mos(rng, n_ao, 2)
    jas = dict(a_par=0.25, a_anti=0.5, b2=0.8, c1=Z.copy(), b1=np.array([1.1, 0.9]))
    return _system("contracted-slater-2u2d" + ("-spd" if with_gaussians else ""), Z, R, 2, 2, center, stype, zeta, C_up, C_dn, jas, a,
                   contraction=(first, coef, sph))


def with_jastrow3(sysd, seed, n_per_nucleus=1, strength=0.3, n_max=8, poly=False):
    """Attach a synthetic three-body Jastrow J3 = sum_{i<j} sum_ab g_ab chi_a(r_i) chi_b(r_j) on Gaussians centred on the nuclei,
    chi_a = dx^l dy^m dz^n exp(-zeta_a |r - R_a|^2) (at most n_max functions): zeta log-uniform in [0.3, 2], g symmetric, uniform in
    [-strength, strength].  poly = False: s functions only (j3_lmn None); poly = True: the monomials cycle through s, the three p and
    the six cartesian d functions.  The paper's runs use the TurboRVB 3-body Jastrow with optimised parameters (L242, L285): not in
    the container."""
    rng = np.random.default_rng(seed)
    centers = [I for I in range(sysd["n_nuc"]) for _ in range(n_per_nucleus)][:n_max]
    n = len(centers)
    zeta = np.exp(rng.uniform(np.log(0.3), np.log(2.0), size=n))
    g = rng.uniform(-strength, strength, size=(n, n)); g = 0.5 * (g + g.T)
    d = dict(sysd)
    d.update(j3_center=np.ascontiguousarray(centers, dtype=np.int32), j3_zeta=zeta, j3_g=np.ascontiguousarray(g), name=sysd["name"] + "-J3")
    if poly:
        mono = [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (2, 0, 0), (1, 1, 0), (1, 0, 1), (0, 2, 0), (0, 1, 1), (0, 0, 2)]
        d.update(j3_lmn=np.ascontiguousarray([mono[(3 * k + seed) % 10] for k in range(n)], dtype=np.int32), name=sysd["name"] + "-J3spd")
    return d


def with_nonlocal(sysd, nl, dla=True):
    """Attach non-local (semi-local) pseudopotential channels to a system (scope row f1).
    nl [n_nuc][7] = (r_c, A_0, B_0, A_1, B_1, A_2, B_2): v_l(r) = A_l exp(-B_l r^2) inside r < r_c, r_c <= 0 = none.
    nl_K = how many cutoff spheres can contain one point: the largest number of centres J (itself included) whose sphere
    overlaps that of a centre I -- a property of the geometry, counted here, used as the slot count per electron."""
    d = dict(sysd)
    nl = np.ascontiguousarray(nl, dtype=np.float64).reshape(sysd["n_nuc"], 7)
    rc = np.maximum(nl[:, 0], 0.0); R = sysd["R"]
    K = 0
    for I in range(sysd["n_nuc"]):
        if rc[I] > 0.0:
            K = max(K, int(sum(1 for J in range(sysd["n_nuc"]) if rc[J] > 0.0 and np.linalg.norm(R[I] - R[J]) < rc[I] + rc[J])))
    d.update(nl=nl, nl_K=K, nl_dla=1 if dla else 0, name=sysd["name"] + ("-nlDLA" if dla else "-nlTM"))
    return d


def random_nonlocal(sysd, seed, r_c, l_max=2, dla=True, nuclei=None, scale=1.0):
    """Seeded synthetic channels: A_l uniform in [-Z, Z] x scale, B_l log-uniform in [2, 8], cutoff r_c on the chosen nuclei
    (default all).  scale >> 1 makes the non-local hops as likely as the lattice ones (kappa = 1/2a^2): test systems only."""
    rng = np.random.default_rng(seed)
    n = sysd["n_nuc"]; nl = np.zeros((n, 7))
    for I in (range(n) if nuclei is None else nuclei):
        nl[I, 0] = r_c
        for l in range(l_max + 1):
            nl[I, 1 + 2 * l] = rng.uniform(-1.0, 1.0) * sysd["Z"][I] * scale
            nl[I, 2 + 2 * l] = np.exp(rng.uniform(np.log(2.0), np.log(8.0)))
    return with_nonlocal(sysd, nl, dla)


def water_methane_nonlocal(n_walkers=400, moves=100, dla=True, seed=PHILOX_RUN_SEED, a=0.2):
    """C3 with s/p/d non-local channels of range 0.8 bohr on every nucleus (spheres disjoint: one slot per electron) -- the
    shape of the paper's ccECP + DLA runs (L242); the channels themselves are synthetic."""
    return random_nonlocal(water_methane(a=a, n_walkers=n_walkers, moves=moves, seed=seed), 33, 0.8, 2, dla)


CONFIGS = {
    "C1": hydrogen,
    "C2": synthetic10,
    "C3": water_methane,
    "C4": water_methane_full,
    "C5": cluster64,
}
