"""ctypes front-end of the CPU FP64 ORACLE (oracle/*.c).

TEST INFRASTRUCTURE, NOT PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this.  It imports nothing from paper_2508_12033_b200 except being
handed the plain dict of arrays that `workloads.py` (no arithmetic of the method) produces.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = ["ref_rng.c", "ref_wf.c", "ref_ham.c", "ref_run.c"]
_LIB_PATH = os.path.join(_HERE, "liblrdmc_ref.so")
_lib = None

BALANCED, CONVENTIONAL = 0, 1


def build(force: bool = False) -> str:
    """gcc -O2, no fast-math, no FMA contraction, OpenMP over walkers."""
    srcs = [os.path.join(_HERE, s) for s in _SRC]
    deps = srcs + [os.path.join(_HERE, "lrdmc_ref.h"), os.path.join(_HERE, "ref_internal.h")]
    if force or not os.path.exists(_LIB_PATH) or any(os.path.getmtime(d) > os.path.getmtime(_LIB_PATH) for d in deps):
        cmd = ["gcc", "-std=gnu11", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wno-misleading-indentation",
               "-o", _LIB_PATH] + srcs + ["-lm"]
        subprocess.run(cmd, check=True)
    return _LIB_PATH


class Stats(C.Structure):
    _fields_ = [("wbar", C.c_double), ("num", C.c_double), ("den", C.c_double),
                ("moves_min", C.c_int64), ("moves_max", C.c_int64), ("moves_sum", C.c_int64),
                ("n_node_flag", C.c_int64), ("n_nonpos_diag", C.c_int64), ("n_nonfinite", C.c_int64),
                ("lockstep_idle_frac", C.c_double), ("n_singular", C.c_int64)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _ip(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_int32))


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB_PATH)
        _lib.lrdmc_ref_uniform53.restype = C.c_double
        _lib.lrdmc_ref_comb_r32.restype = C.c_uint32
        _lib.lrdmc_ref_uniform53.argtypes = [C.c_uint32, C.c_uint32]
        _lib.lrdmc_ref_frame.argtypes = [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]
        _lib.lrdmc_ref_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int,
                                          C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_void_p,
                                          C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p, C.c_double, C.c_double,
                                          C.c_uint64]
        _lib.lrdmc_ref_destroy.argtypes = [C.c_void_p]
        vp = C.c_void_p      # every pointer argument is declared: a bare Python int would be passed as a 32-bit C int
        _lib.lrdmc_ref_set_positions.argtypes = [vp, C.c_int, vp]
        _lib.lrdmc_ref_get_state.argtypes = [vp, vp, vp, vp, vp]
        _lib.lrdmc_ref_set_state.argtypes = [vp, C.c_int, vp, vp, vp, vp]
        _lib.lrdmc_ref_get_obs.argtypes = [vp, vp, vp, vp, vp]
        _lib.lrdmc_ref_estimators.argtypes = [vp, vp]
        _lib.lrdmc_ref_ao.argtypes = [vp, vp, vp, vp, vp]
        _lib.lrdmc_ref_mo.argtypes = [vp, C.c_int, vp, vp, vp, vp]
        _lib.lrdmc_ref_logpsi.argtypes = [vp, vp, vp, vp]
        _lib.lrdmc_ref_build_inverse.argtypes = [vp, vp, vp, vp]
        _lib.lrdmc_ref_evaluate.argtypes = [vp] * 9
        _lib.lrdmc_ref_philox4x32_10.argtypes = [vp, vp, vp]
        _lib.lrdmc_ref_set_threads.argtypes = [C.c_int]
        _lib.lrdmc_ref_set_slot_offset.argtypes = [vp, C.c_uint32]
        _lib.lrdmc_ref_set_contraction.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.lrdmc_ref_set_jastrow3.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.lrdmc_ref_set_nonlocal.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p]
        _lib.lrdmc_ref_nl_info.argtypes = [C.c_void_p] + [C.c_void_p] * 7
        _lib.lrdmc_ref_n_candidates.argtypes = [C.c_void_p]
        _lib.lrdmc_ref_propagate.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_uint64]
        _lib.lrdmc_ref_reconfigure.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p]
        _lib.lrdmc_ref_step_debug.argtypes = [C.c_void_p, C.c_double, C.c_uint64, C.c_uint64, C.c_void_p, C.c_void_p, C.c_void_p]
        _lib.lrdmc_ref_comb_r32.argtypes = [C.c_void_p, C.c_uint64]
        _lib.lrdmc_ref_draws.argtypes = [C.c_void_p, C.c_uint32, C.c_uint64, C.c_uint64, C.c_void_p]
        _lib.lrdmc_ref_select.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        _lib.lrdmc_ref_comb.argtypes = [C.c_int, C.c_void_p, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    return _lib


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    lib().lrdmc_ref_philox4x32_10(c, k, o)
    return tuple(int(v) for v in o)


def uniform53(lo, hi):
    return float(lib().lrdmc_ref_uniform53(lo, hi))


def frame(u1, u2, u3):
    U = np.zeros(9)
    lib().lrdmc_ref_frame(u1, u2, u3, _dp(U))
    return U.reshape(3, 3)


def comb(w, r32):
    """Eq.15-17 in integers.  Returns parents, wbar, u (quantised weights), T, sh."""
    w = np.ascontiguousarray(w, dtype=np.float64); n = w.shape[0]
    par = np.zeros(n, dtype=np.int32); u = np.zeros(n, dtype=np.uint64)
    wbar = C.c_double(); T = C.c_uint64(); sh = C.c_int()
    rc = lib().lrdmc_ref_comb(n, w.ctypes.data, r32, par.ctypes.data, C.byref(wbar), u.ctypes.data, C.byref(T), C.byref(sh))
    return rc, par, wbar.value, u, int(T.value), sh.value


class Ref:
    """One oracle context = one system (+ its walkers).  `sysd` is a dict from workloads.py."""

    def __init__(self, sysd):
        L = lib()
        self.sysd = sysd
        self.N = sysd["n_up"] + sysd["n_dn"]; self.n_up = sysd["n_up"]; self.n_dn = sysd["n_dn"]; self.n_ao = sysd["n_ao"]
        h = C.c_void_p()
        keep = [np.ascontiguousarray(sysd[k]) if sysd.get(k) is not None else None
                for k in ("Z", "R", "pp", "shell_center", "shell_type", "shell_zeta", "C_up", "C_dn", "c1", "b1")]
        ptr = [None if a is None else a.ctypes.data for a in keep]
        rc = L.lrdmc_ref_create(C.byref(h), sysd["n_nuc"], ptr[0], ptr[1], ptr[2], sysd["n_up"], sysd["n_dn"], sysd["n_shell"],
                                ptr[3], ptr[4], ptr[5], sysd["n_ao"], ptr[6], ptr[7], sysd["a_par"], sysd["a_anti"], sysd["b2"],
                                ptr[8], ptr[9], sysd["a"], sysd["a2"], sysd["seed"])
        if rc:
            raise ValueError(f"lrdmc_ref_create failed: {rc}")
        self.h = h
        if sysd.get("cs_first") is not None:                           # contracted / solid-harmonic shells (scope row f2)
            cf = np.ascontiguousarray(sysd["cs_first"], dtype=np.int32); pc = np.ascontiguousarray(sysd["prim_coef"], dtype=np.float64)
            sp = np.ascontiguousarray(sysd["cs_sph"], dtype=np.int32)
            rc = L.lrdmc_ref_set_contraction(h, len(sp), cf.ctypes.data, pc.ctypes.data, sp.ctypes.data)
            if rc:
                raise ValueError(f"lrdmc_ref_set_contraction failed: {rc}")
        if sysd.get("j3_zeta") is not None:                            # three-body Jastrow (scope row f2)
            jc = np.ascontiguousarray(sysd["j3_center"], dtype=np.int32); jz = np.ascontiguousarray(sysd["j3_zeta"], dtype=np.float64)
            jg = np.ascontiguousarray(sysd["j3_g"], dtype=np.float64)
            jl = None if sysd.get("j3_lmn") is None else np.ascontiguousarray(sysd["j3_lmn"], dtype=np.int32)
            rc = L.lrdmc_ref_set_jastrow3(h, len(jz), jc.ctypes.data, jz.ctypes.data, jg.ctypes.data, None if jl is None else jl.ctypes.data)
            if rc:
                raise ValueError(f"lrdmc_ref_set_jastrow3 failed: {rc}")
        self.nl_slots = 0
        if sysd.get("nl") is not None and sysd.get("nl_K", 0) > 0:      # non-local pseudopotential channels (scope row f1)
            nl = np.ascontiguousarray(sysd["nl"], dtype=np.float64)
            rc = L.lrdmc_ref_set_nonlocal(h, int(sysd["nl_K"]), int(sysd["nl_dla"]), nl.ctypes.data)
            if rc:
                raise ValueError(f"lrdmc_ref_set_nonlocal failed: {rc}")
            self.nl_slots = 6 * self.N * int(sysd["nl_K"])
        self.P = L.lrdmc_ref_n_candidates(h)
        self.n_w = 0

    def __del__(self):
        if getattr(self, "h", None) and _lib is not None:
            try:
                _lib.lrdmc_ref_destroy(self.h)
            except Exception:       # interpreter shutdown
                pass
            self.h = None

    def set_slot_offset(self, offset):
        """walker k draws from the random streams of slot offset + k"""
        return lib().lrdmc_ref_set_slot_offset(self.h, offset)

    # ---- walkers ----
    def set_positions(self, r):
        r = np.ascontiguousarray(r, dtype=np.float64); self.n_w = r.shape[0]
        assert r.shape == (self.n_w, self.N, 3)
        return lib().lrdmc_ref_set_positions(self.h, self.n_w, r.ctypes.data)

    def get_state(self):
        r = np.zeros((self.n_w, self.N, 3)); du = np.zeros((self.n_w, self.n_up, self.n_up))
        dd = np.zeros((self.n_w, self.n_dn, self.n_dn)); w = np.zeros(self.n_w)
        rc = lib().lrdmc_ref_get_state(self.h, _dp(r), _dp(du), _dp(dd), _dp(w)); assert rc == 0
        return r, du, dd, w

    def set_state(self, r, du=None, dd=None, w=None):
        r = np.ascontiguousarray(r, dtype=np.float64); self.n_w = r.shape[0]
        du = None if du is None else np.ascontiguousarray(du); dd = None if dd is None else np.ascontiguousarray(dd)
        w = None if w is None else np.ascontiguousarray(w, dtype=np.float64)
        return lib().lrdmc_ref_set_state(self.h, self.n_w, _dp(r), _dp(du), _dp(dd), _dp(w))

    def get_obs(self):
        eL = np.zeros(self.n_w); W = np.zeros(self.n_w); om = np.zeros(self.n_w); nm = np.zeros(self.n_w, dtype=np.int64)
        rc = lib().lrdmc_ref_get_obs(self.h, _dp(eL), _dp(W), _dp(om), nm.ctypes.data_as(C.POINTER(C.c_int64))); assert rc == 0
        return eL, W, om, nm

    # ---- the path ----
    def propagate(self, mode, n_moves, tau, E0, cycle):
        return lib().lrdmc_ref_propagate(self.h, mode, n_moves, tau, E0, cycle)

    def reconfigure(self, cycle):
        par = np.zeros(self.n_w, dtype=np.int32)
        rc = lib().lrdmc_ref_reconfigure(self.h, cycle, par.ctypes.data)
        return rc, par

    def estimators(self):
        s = Stats(); rc = lib().lrdmc_ref_estimators(self.h, C.byref(s)); assert rc == 0
        return s.asdict()

    def step_debug(self, E0, cycle, step):
        R = np.zeros((self.n_w, self.P)); scal = np.zeros((self.n_w, 8)); js = np.zeros(self.n_w, dtype=np.int32)
        rc = lib().lrdmc_ref_step_debug(self.h, E0, cycle, step, R.ctypes.data, scal.ctypes.data, js.ctypes.data); assert rc == 0
        return R, scal, js

    # ---- primitives for the pins ----
    def draws(self, slot, cycle, step):
        u = np.zeros(5); lib().lrdmc_ref_draws(self.h, slot, cycle, step, u.ctypes.data); return u

    def comb_r32(self, cycle):
        return int(lib().lrdmc_ref_comb_r32(self.h, cycle))

    def ao(self, r):
        r = np.ascontiguousarray(r, dtype=np.float64); v = np.zeros(self.n_ao); g = np.zeros((self.n_ao, 3)); l = np.zeros(self.n_ao)
        rc = lib().lrdmc_ref_ao(self.h, _dp(r), _dp(v), _dp(g), _dp(l)); assert rc == 0
        return v, g, l

    def mo(self, spin, r):
        O = self.n_dn if spin else self.n_up
        r = np.ascontiguousarray(r, dtype=np.float64); v = np.zeros(O); g = np.zeros((O, 3)); l = np.zeros(O)
        rc = lib().lrdmc_ref_mo(self.h, spin, _dp(r), _dp(v), _dp(g), _dp(l)); assert rc == 0
        return v, g, l

    def logpsi(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64); la = C.c_double(); sg = C.c_int()
        rc = lib().lrdmc_ref_logpsi(self.h, _dp(x), C.byref(la), C.byref(sg))
        if rc:
            raise FloatingPointError("singular Slater matrix")
        return la.value, sg.value

    def build_inverse(self, x):
        x = np.ascontiguousarray(x, dtype=np.float64); du = np.zeros((self.n_up, self.n_up)); dd = np.zeros((self.n_dn, self.n_dn))
        rc = lib().lrdmc_ref_build_inverse(self.h, _dp(x), _dp(du), _dp(dd))
        return rc, du, dd

    def evaluate(self, x, U, du=None, dd=None):
        """returns R[P], scal dict, per[N][5] = (T_i, lap_i, v_ei, v_zv, v^a_ei), cand[P][3]"""
        x = np.ascontiguousarray(x, dtype=np.float64); U = np.ascontiguousarray(U, dtype=np.float64)
        R = np.zeros(self.P); scal = np.zeros(10); per = np.zeros((self.N, 5)); cand = np.zeros((self.P, 3))
        du = None if du is None else np.ascontiguousarray(du); dd = None if dd is None else np.ascontiguousarray(dd)
        if du is not None and dd is None:
            dd = np.zeros((0, 0))
        rc = lib().lrdmc_ref_evaluate(self.h, _dp(x), _dp(du), _dp(dd) if du is not None else None, _dp(U), _dp(R), _dp(scal), _dp(per), _dp(cand))
        if rc:
            raise FloatingPointError(f"evaluate failed: {rc}")
        keys = ("bbar", "V_sf", "W", "e_L", "node", "V_ee", "V_ii", "K_diag", "n_vmax", "e_L_continuum")
        return R, dict(zip(keys, scal)), per, cand

    def nl_info(self, x, U, du, dd):
        """nu_q = V^nl_{x_q,x}, rho_q (determinant or wavefunction ratio) and the quadrature points of every non-local slot"""
        x = np.ascontiguousarray(x, dtype=np.float64); U = np.ascontiguousarray(U, dtype=np.float64)
        du = np.ascontiguousarray(du); dd = np.ascontiguousarray(dd) if dd is not None and dd.size else np.zeros(1)
        n = self.nl_slots; nu = np.zeros(n); rho = np.zeros(n); cand = np.zeros((n, 3))
        rc = lib().lrdmc_ref_nl_info(self.h, x.ctypes.data, du.ctypes.data, dd.ctypes.data, U.ctypes.data, nu.ctypes.data, rho.ctypes.data, cand.ctypes.data)
        assert rc == 0
        return nu, rho, cand

    def select(self, R, u_sel):
        R = np.ascontiguousarray(R, dtype=np.float64); mg = C.c_double()
        j = lib().lrdmc_ref_select(self.h, R.ctypes.data, u_sel, C.byref(mg))
        return j, mg.value


def set_threads(n):
    return lib().lrdmc_ref_set_threads(n)
