"""Thin ctypes binding of liblrdmc.so: same names as include/lrdmc.h, argument marshalling only.

PyTorch supplies device memory (tensors) and streams; every step of the path runs in the CUDA kernels.
There is NO CPU fallback: importing works anywhere, but `Lrdmc(...)` raises if the library or a CUDA device is missing.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("LRDMC_LIB", os.path.join(_HERE, "liblrdmc.so"))    # override: kernel experiments only
BALANCED, CONVENTIONAL = 0, 1
OK, EINVAL, ESINGULAR, ESTATE, ECUDA, ENOMEM = 0, -1, -2, -3, -4, -5

PROBE_LIB_PATH = os.path.join(_HERE, "liblrdmc_probe.so")                     # include/lrdmc_probe.h (bench.py's roofline denominators)
OPT_TEAM_WARPS, OPT_GLOBAL_TABLES, OPT_LISTED = 1, 2, 3
COMB_STATIC_MAX_WALKERS = 65536                                               # LRDMC_COMB_STATIC_MAX_WALKERS

# every symbol this module touches; tests check that include/lrdmc.h (resp. lrdmc_probe.h) declares each and the libraries export each
EXPORTS = ["lrdmc_init", "lrdmc_free", "lrdmc_strerror", "lrdmc_last_error", "lrdmc_set_option", "lrdmc_n_candidates", "lrdmc_walker_bytes",
           "lrdmc_bind_walkers", "lrdmc_set_positions", "lrdmc_propagate", "lrdmc_reconfigure", "lrdmc_estimators", "lrdmc_energy",
           "lrdmc_step_debug", "lrdmc_get_walkers", "lrdmc_set_state", "lrdmc_get_obs", "lrdmc_run_host", "lrdmc_debug_philox",
           "lrdmc_debug_draws", "lrdmc_launch_count", "lrdmc_launch_config", "lrdmc_listed_sweep",
           "lrdmc_comb_static", "lrdmc_comb_static_setup", "lrdmc_comb_static_error"]
PROBE_EXPORTS = ["lrdmc_measure_fp64_peaks", "lrdmc_measure_fp64_operand_peak", "lrdmc_measure_fp64_shared_operand_peak"]


class System(C.Structure):
    _fields_ = [("n_nuc", C.c_int), ("Z", C.c_void_p), ("R", C.c_void_p), ("n_up", C.c_int), ("n_dn", C.c_int), ("pp", C.c_void_p),
                ("nl", C.c_void_p), ("nl_K", C.c_int), ("nl_dla", C.c_int)]


class Basis(C.Structure):
    _fields_ = [("n_shell", C.c_int), ("center", C.c_void_p), ("type", C.c_void_p), ("zeta", C.c_void_p),
                ("n_cshell", C.c_int), ("cs_first", C.c_void_p), ("prim_coef", C.c_void_p), ("cs_sph", C.c_void_p)]


class Mo(C.Structure):
    _fields_ = [("n_ao", C.c_int), ("C_up", C.c_void_p), ("C_dn", C.c_void_p)]


class Jastrow(C.Structure):
    _fields_ = [("a_par", C.c_double), ("a_anti", C.c_double), ("b2", C.c_double), ("c1", C.c_void_p), ("b1", C.c_void_p),
                ("n_j3", C.c_int), ("j3_center", C.c_void_p), ("j3_zeta", C.c_void_p), ("j3_g", C.c_void_p), ("j3_lmn", C.c_void_p)]


class Lattice(C.Structure):
    _fields_ = [("a", C.c_double), ("a2", C.c_double), ("seed", C.c_uint64)]


class CycleStats(C.Structure):
    _fields_ = [("wbar", C.c_double), ("num", C.c_double), ("den", C.c_double),
                ("moves_min", C.c_int64), ("moves_max", C.c_int64), ("moves_sum", C.c_int64),
                ("n_node_flag", C.c_int64), ("n_nonpos_diag", C.c_int64), ("n_nonfinite", C.c_int64), ("n_singular", C.c_int64),
                ("lockstep_idle_frac", C.c_double), ("barrier_idle_frac", C.c_double),
                ("propagate_ms", C.c_float), ("reconfigure_ms", C.c_float)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None


def load_library():
    """dlopen liblrdmc.so (built in-tree by `python -m paper_2508_12033_b200.build`); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2508_12033_b200.build` (nvcc, sm_100a). "
                               "There is no CPU fallback.")
        L = C.CDLL(LIB_PATH)
        vp, i32, u64, dbl = C.c_void_p, C.c_int, C.c_uint64, C.c_double
        L.lrdmc_init.argtypes = [C.POINTER(vp), C.POINTER(System), C.POINTER(Basis), C.POINTER(Mo), C.POINTER(Jastrow), C.POINTER(Lattice)]
        L.lrdmc_free.argtypes = [vp]; L.lrdmc_free.restype = None
        L.lrdmc_strerror.argtypes = [i32]; L.lrdmc_strerror.restype = C.c_char_p
        L.lrdmc_n_candidates.argtypes = [vp]
        L.lrdmc_walker_bytes.argtypes = [vp, i32]; L.lrdmc_walker_bytes.restype = C.c_size_t
        L.lrdmc_bind_walkers.argtypes = [vp, vp, C.c_size_t, i32]
        L.lrdmc_set_positions.argtypes = [vp, vp, vp]
        L.lrdmc_propagate.argtypes = [vp, i32, i32, dbl, dbl, u64, vp]
        L.lrdmc_reconfigure.argtypes = [vp, u64, vp, vp]
        L.lrdmc_estimators.argtypes = [vp, C.POINTER(CycleStats)]
        L.lrdmc_energy.argtypes = [C.POINTER(CycleStats), i32, i32, i32, i32, C.POINTER(dbl), C.POINTER(dbl)]
        L.lrdmc_step_debug.argtypes = [vp, dbl, u64, u64, vp, vp, vp, vp]
        L.lrdmc_get_walkers.argtypes = [vp, vp, vp, vp, vp, vp]
        L.lrdmc_set_state.argtypes = [vp, vp, vp, vp, vp, vp]
        L.lrdmc_get_obs.argtypes = [vp, vp, vp, vp, vp, vp]
        L.lrdmc_run_host.argtypes = [vp, vp, vp, i32, i32, dbl, dbl, u64, i32, i32, C.POINTER(CycleStats), vp]
        L.lrdmc_last_error.argtypes = [vp]; L.lrdmc_last_error.restype = C.c_char_p
        L.lrdmc_set_option.argtypes = [vp, i32, i32]
        L.lrdmc_debug_philox.argtypes = [vp, C.c_uint32, C.c_uint32, vp, i32, vp]
        L.lrdmc_debug_draws.argtypes = [vp, u64, u64, vp, i32, vp]
        L.lrdmc_launch_count.argtypes = [vp]
        L.lrdmc_launch_config.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
        L.lrdmc_listed_sweep.argtypes = [vp]
        L.lrdmc_comb_static.argtypes = [vp, i32, u64, u64, vp, vp, vp]
        L.lrdmc_comb_static_setup.argtypes = []
        L.lrdmc_comb_static_error.argtypes = []; L.lrdmc_comb_static_error.restype = C.c_char_p
        _lib = L
    return _lib


class LrdmcError(RuntimeError):
    def __init__(self, code, where, ctx=None):
        self.code = code
        L = load_library(); text = L.lrdmc_strerror(code).decode()
        if code == ECUDA:
            text += ": " + L.lrdmc_last_error(ctx).decode()
        super().__init__(f"{where}: {text} ({code})")


def _check(rc, where, allow=(), ctx=None):
    if rc != 0 and rc not in allow:
        raise LrdmcError(rc, where, ctx)
    return rc


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def lrdmc_energy(records, p=10, n_therm=0, n_blocks=20):
    """Eq.18-19 over a list of CycleStats (host)."""
    arr = (CycleStats * len(records))(*records)
    E, sg = C.c_double(), C.c_double()
    _check(load_library().lrdmc_energy(arr, len(records), p, n_therm, n_blocks, C.byref(E), C.byref(sg)), "lrdmc_energy")
    return E.value, sg.value


def lrdmc_comb_static(w, seed, cycle, want_wbar=True):
    """include/lrdmc.h lrdmc_comb_static: the comb of the branching step with NO allocation inside the library (static device scratch,
    at most COMB_STATIC_MAX_WALKERS walkers).  `w`: float64 CUDA tensor [n_w]; the two outputs are allocated HERE, by the caller's side.
    Returns (parents int32 [n_w], wbar float64 [1] or None), both on w's device, asynchronous on torch's current stream."""
    import torch
    L = load_library()
    if not (isinstance(w, torch.Tensor) and w.is_cuda and w.dtype == torch.float64 and w.dim() == 1 and w.is_contiguous()):
        raise ValueError("lrdmc_comb_static: w must be a contiguous 1-d float64 CUDA tensor")
    with torch.cuda.device(w.device):
        par = torch.empty(w.shape[0], dtype=torch.int32, device=w.device)
        wbar = torch.empty(1, dtype=torch.float64, device=w.device) if want_wbar else None
        rc = L.lrdmc_comb_static(_ptr(w), int(w.shape[0]), int(seed), int(cycle), _ptr(par), _ptr(wbar),
                                 C.c_void_p(torch.cuda.current_stream(w.device).cuda_stream))
    if rc != 0:
        raise RuntimeError(f"{L.lrdmc_comb_static_error().decode()} ({rc})")
    return par, wbar


_probe = None


def lrdmc_measure_fp64_peaks():
    """include/lrdmc_probe.h: FP64 peaks measured on the current device (liblrdmc_probe.so, not the product library)."""
    global _probe
    if _probe is None:
        if not os.path.exists(PROBE_LIB_PATH):
            raise RuntimeError(f"{PROBE_LIB_PATH} is missing: run `python -m paper_2508_12033_b200.build`")
        _probe = C.CDLL(PROBE_LIB_PATH)
        dp = C.POINTER(C.c_double)
        _probe.lrdmc_measure_fp64_peaks.argtypes = [dp, dp, dp]; _probe.lrdmc_measure_fp64_operand_peak.argtypes = [dp, dp]; _probe.lrdmc_measure_fp64_shared_operand_peak.argtypes = [dp]
    a, b, m, t, u, v = (C.c_double() for _ in range(6))
    if (_probe.lrdmc_measure_fp64_peaks(C.byref(a), C.byref(b), C.byref(m)) or _probe.lrdmc_measure_fp64_operand_peak(C.byref(t), C.byref(u))
            or _probe.lrdmc_measure_fp64_shared_operand_peak(C.byref(v))):
        raise RuntimeError("FP64 peak probe failed (CUDA error)")
    return dict(dfma_tflops=a.value, dmma_tflops=b.value, mixed_tflops=m.value, dfma_3reg_tflops=t.value, dfma_alu_tflops=u.value, dfma_shared1_tflops=v.value)


class Lrdmc:
    """One context = one system on the current CUDA device; walkers live in a torch uint8 tensor owned by this object."""

    def __init__(self, sysd, device="cuda:0", options=None):
        """options: {OPT_TEAM_WARPS: tw, OPT_GLOBAL_TABLES: 0/1} applied with lrdmc_set_option before any walker is bound."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("liblrdmc needs a CUDA device (B200, sm_100a); there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        L = load_library()
        self.L = L
        self.sysd = sysd
        self.N = sysd["n_up"] + sysd["n_dn"]; self.n_up = sysd["n_up"]; self.n_dn = sysd["n_dn"]
        k = {n: (None if sysd.get(n) is None else np.ascontiguousarray(sysd[n])) for n in
             ("Z", "R", "pp", "shell_center", "shell_type", "shell_zeta", "C_up", "C_dn", "c1", "b1", "nl", "cs_first", "prim_coef", "cs_sph", "j3_center", "j3_zeta", "j3_g", "j3_lmn")}
        self._keep = k
        p = lambda a: None if a is None else a.ctypes.data
        s = System(sysd["n_nuc"], p(k["Z"]), p(k["R"]), sysd["n_up"], sysd["n_dn"], p(k["pp"]),
                   p(k["nl"]), int(sysd.get("nl_K", 0) or 0), int(sysd.get("nl_dla", 1)))
        b = Basis(sysd["n_shell"], p(k["shell_center"]), p(k["shell_type"]), p(k["shell_zeta"]),
                  0 if k["cs_sph"] is None else len(k["cs_sph"]), p(k["cs_first"]), p(k["prim_coef"]), p(k["cs_sph"]))
        m = Mo(sysd["n_ao"], p(k["C_up"]), p(k["C_dn"]))
        j = Jastrow(sysd["a_par"], sysd["a_anti"], sysd["b2"], p(k["c1"]), p(k["b1"]),
                    0 if k["j3_zeta"] is None else len(k["j3_zeta"]), p(k["j3_center"]), p(k["j3_zeta"]), p(k["j3_g"]), p(k["j3_lmn"]))
        la = Lattice(sysd["a"], sysd["a2"], sysd["seed"])
        h = C.c_void_p()
        _check(L.lrdmc_init(C.byref(h), C.byref(s), C.byref(b), C.byref(m), C.byref(j), C.byref(la)), "lrdmc_init")
        self.h = h
        for opt, val in (options or {}).items():
            self.lrdmc_set_option(opt, val)
        self.P = L.lrdmc_n_candidates(h)
        self.n_w = 0
        self.buf = None

    def close(self):
        if getattr(self, "h", None):
            self.L.lrdmc_free(self.h); self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def _dev(self, a, dtype=None):
        t = self.torch
        if isinstance(a, t.Tensor):
            return a.to(self.device).contiguous()
        return t.from_numpy(np.ascontiguousarray(a, dtype=dtype)).to(self.device)

    def lrdmc_set_option(self, option, value):
        _check(self.L.lrdmc_set_option(self.h, int(option), int(value)), "lrdmc_set_option", ctx=self.h)

    def lrdmc_last_error(self):
        return self.L.lrdmc_last_error(self.h).decode()

    # ---- storage ----
    def lrdmc_walker_bytes(self, n_w):
        return int(self.L.lrdmc_walker_bytes(self.h, n_w))

    def lrdmc_bind_walkers(self, n_w):
        nbytes = self.lrdmc_walker_bytes(n_w)
        self.buf = self.torch.zeros(nbytes, dtype=self.torch.uint8, device=self.device)
        _check(self.L.lrdmc_bind_walkers(self.h, _ptr(self.buf), nbytes, n_w), "lrdmc_bind_walkers", ctx=self.h)
        self.n_w = n_w

    # ---- the path ----
    def lrdmc_set_positions(self, r, allow_singular=False):
        r = self._dev(r, np.float64)
        if self.n_w != r.shape[0]:
            self.lrdmc_bind_walkers(int(r.shape[0]))
        assert tuple(r.shape) == (self.n_w, self.N, 3)
        return _check(self.L.lrdmc_set_positions(self.h, _ptr(r), self._stream()), "lrdmc_set_positions", ctx=self.h,
                      allow=(ESINGULAR,) if allow_singular else ())

    def lrdmc_propagate(self, mode, n_moves, tau, E0, cycle):
        _check(self.L.lrdmc_propagate(self.h, mode, n_moves, tau, E0, cycle, self._stream()), "lrdmc_propagate", ctx=self.h)

    def lrdmc_reconfigure(self, cycle, want_parents=False):
        par = self.torch.empty(self.n_w, dtype=self.torch.int32, device=self.device) if want_parents else None
        _check(self.L.lrdmc_reconfigure(self.h, cycle, _ptr(par), self._stream()), "lrdmc_reconfigure", ctx=self.h)
        return par

    def lrdmc_estimators(self):
        s = CycleStats()
        _check(self.L.lrdmc_estimators(self.h, C.byref(s)), "lrdmc_estimators", ctx=self.h)
        return s

    def lrdmc_step_debug(self, E0, cycle, step):
        t = self.torch
        R = t.empty((self.n_w, self.P), dtype=t.float64, device=self.device)
        scal = t.empty((self.n_w, 8), dtype=t.float64, device=self.device)
        js = t.empty(self.n_w, dtype=t.int32, device=self.device)
        _check(self.L.lrdmc_step_debug(self.h, E0, cycle, step, _ptr(R), _ptr(scal), _ptr(js), self._stream()), "lrdmc_step_debug", ctx=self.h)
        return R, scal, js

    def lrdmc_get_walkers(self):
        t = self.torch; f = dict(dtype=t.float64, device=self.device)
        r = t.empty((self.n_w, self.N, 3), **f); du = t.empty((self.n_w, self.n_up, self.n_up), **f)
        dd = t.empty((self.n_w, self.n_dn, self.n_dn), **f); w = t.empty(self.n_w, **f)
        _check(self.L.lrdmc_get_walkers(self.h, _ptr(r), _ptr(du), _ptr(dd) if self.n_dn else None, _ptr(w), self._stream()), "lrdmc_get_walkers", ctx=self.h)
        return r, du, dd, w

    def lrdmc_set_state(self, r, du=None, dd=None, w=None):
        r = self._dev(r, np.float64)
        if self.n_w != r.shape[0]:
            self.lrdmc_bind_walkers(int(r.shape[0]))
        du = None if du is None else self._dev(du, np.float64); dd = None if dd is None or self.n_dn == 0 else self._dev(dd, np.float64)
        w = None if w is None else self._dev(w, np.float64)
        _check(self.L.lrdmc_set_state(self.h, _ptr(r), _ptr(du), _ptr(dd), _ptr(w), self._stream()), "lrdmc_set_state", ctx=self.h)
        self._hold = (r, du, dd, w)

    def lrdmc_get_obs(self):
        t = self.torch; f = dict(dtype=t.float64, device=self.device)
        eL = t.empty(self.n_w, **f); W = t.empty(self.n_w, **f); om = t.empty(self.n_w, **f)
        nm = t.empty(self.n_w, dtype=t.int64, device=self.device)
        _check(self.L.lrdmc_get_obs(self.h, _ptr(eL), _ptr(W), _ptr(om), _ptr(nm), self._stream()), "lrdmc_get_obs", ctx=self.h)
        return eL, W, om, nm

    def lrdmc_run_host(self, r_host, mode, n_moves, tau, E0, first_cycle, n_cycles, want_positions=True, n_therm=0):
        """HOST buffers in and out (numpy / pinned torch CPU tensors): copies are inside the call."""
        r_in = np.ascontiguousarray(r_host, dtype=np.float64) if not isinstance(r_host, self.torch.Tensor) else r_host
        n_w = int(r_in.shape[0])
        if self.n_w != n_w:
            self.lrdmc_bind_walkers(n_w)
        r_out = None
        if want_positions:      # pinned result buffer, allocated once per walker count
            if getattr(self, "_pinned_out", None) is None or self._pinned_out.shape[0] != n_w:
                self._pinned_out = self.torch.empty((n_w, self.N, 3), dtype=self.torch.float64).pin_memory()
            r_out = self._pinned_out
        stats = (CycleStats * max(1, n_cycles))()
        pin = r_in.data_ptr() if isinstance(r_in, self.torch.Tensor) else r_in.ctypes.data
        _check(self.L.lrdmc_run_host(self.h, pin, None if r_out is None else r_out.data_ptr(), mode, n_moves, tau, E0, first_cycle, n_cycles,
                                     n_therm, stats, self._stream()), "lrdmc_run_host", ctx=self.h)
        return [stats[i] for i in range(n_cycles)], r_out

    # ---- diagnostics ----
    def launch_count(self):
        return int(self.L.lrdmc_launch_count(self.h))

    def launch_config(self):
        g, b, s, c, t = C.c_int(), C.c_int(), C.c_int(), C.c_int(), C.c_int()
        self.L.lrdmc_launch_config(self.h, C.byref(g), C.byref(b), C.byref(s), C.byref(c), C.byref(t))
        return dict(grid=g.value, block=b.value, smem_bytes=s.value, ctas_per_sm=c.value, team_warps=t.value,
                    kernel="k_propagate" if t.value <= 1 else "k_propagate_team", listed_sweep=bool(self.L.lrdmc_listed_sweep(self.h)))

    def debug_draws(self, cycle, step, n):
        out = self.torch.empty((n, 14), dtype=self.torch.float64, device=self.device)
        _check(self.L.lrdmc_debug_draws(self.h, cycle, step, _ptr(out), n, self._stream()), "lrdmc_debug_draws", ctx=self.h)
        return out

    def debug_philox(self, ctr, key):
        t = self.torch
        c = t.from_numpy(np.ascontiguousarray(ctr, dtype=np.uint32).view(np.int32)).to(self.device)
        out = t.empty_like(c)
        _check(self.L.lrdmc_debug_philox(_ptr(c), key[0], key[1], _ptr(out), c.shape[0], self._stream()), "lrdmc_debug_philox")
        return out.cpu().numpy().view(np.uint32)
