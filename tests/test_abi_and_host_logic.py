"""CPU-only checks of the product's boundary and host logic: the shared library loads and exports every symbol
include/lrdmc.h declares, the binding refuses to run without CUDA (no CPU fallback), the host-side estimator of
Eq.18-19 agrees with the oracle's, bench.py's rank aggregation works under a 2-rank gloo group."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

from paper_2508_12033_b200 import binding as B, driver as drv, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    if not os.path.exists(B.LIB_PATH):
        from paper_2508_12033_b200 import build
        build.build()
    return B.load_library()


def _declared(header):
    hdr = open(os.path.join(ROOT, "include", header)).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return set(re.findall(r"\b(lrdmc_[a-z0-9_]+)\s*\(", hdr))


def test_library_exports_every_declared_symbol(lib):
    names = _declared("lrdmc.h")
    assert {"lrdmc_init", "lrdmc_propagate", "lrdmc_reconfigure", "lrdmc_estimators", "lrdmc_set_option", "lrdmc_last_error"} <= names and len(names) >= 20
    for n in sorted(names):
        assert hasattr(lib, n), n
    assert set(B.EXPORTS) == names               # the binding's list IS the header's list
    # every library symbol binding.py touches (L.lrdmc_x / self.L.lrdmc_x / load_library().lrdmc_x) is declared in the header
    src = open(os.path.join(ROOT, "paper_2508_12033_b200", "binding.py")).read()
    used = set(re.findall(r"(?:\bL|self\.L|load_library\(\))\.(lrdmc_[a-z0-9_]+)", src))
    assert used and used <= names, used - names
    probe_names = _declared("lrdmc_probe.h")
    assert probe_names == set(B.PROBE_EXPORTS) and not (probe_names & names)
    assert set(re.findall(r"_probe\.(lrdmc_[a-z0-9_]+)", src)) <= probe_names
    probe = C.CDLL(B.PROBE_LIB_PATH)
    for n in probe_names:
        assert hasattr(probe, n), n
        assert not hasattr(lib, n), n            # the product library carries no measurement probes
    # no environment variable steers the product library
    csrc = os.path.join(ROOT, "paper_2508_12033_b200", "csrc")
    for f in os.listdir(csrc):
        if os.path.isfile(os.path.join(csrc, f)):
            assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_header_declares_only_c_types():
    hdr = open(os.path.join(ROOT, "include", "lrdmc.h")).read()
    assert 'extern "C"' in hdr
    code = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    assert "torch" not in code.lower() and "at::" not in code and "std::" not in code and "template" not in code


def test_strerror_and_struct_layout(lib):
    assert lib.lrdmc_strerror(0) == b"ok" and b"singular" in lib.lrdmc_strerror(-2)
    assert lib.lrdmc_last_error(None) is not None      # per-thread slot of a failed lrdmc_init; "" or the CUDA text
    assert lib.lrdmc_set_option(None, 1, 4) == B.EINVAL
    assert C.sizeof(B.CycleStats) == 104         # 3 doubles, 7 int64, 2 doubles, 2 floats


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.Lrdmc(wl.hydrogen())
    src = open(os.path.join(ROOT, "paper_2508_12033_b200", "binding.py")).read() + open(os.path.join(ROOT, "paper_2508_12033_b200", "driver.py")).read()
    assert "oracle" not in src                   # the product path never touches the oracle


def test_host_energy_estimator_matches_oracle_estimator(lib):
    from oracle import ref_driver as rdrv
    rng = np.random.default_rng(0); n = 137
    wbar = np.exp(rng.normal(size=n) * 0.05); den = rng.random(n) + 5.0; e = -0.5 + 0.01 * rng.normal(size=n); num = e * den
    recs = []
    for i in range(n):
        s = B.CycleStats(); s.wbar = wbar[i]; s.num = num[i]; s.den = den[i]; recs.append(s)
    for (p, nth, nb) in ((0, 0, 20), (10, 27, 20), (3, 100, 7), (50, 0, 2)):
        E, sg = B.lrdmc_energy(recs, p=p, n_therm=nth, n_blocks=nb)
        Eo, so = rdrv.energy(wbar, num, den, p=p, n_therm=nth, n_blocks=nb)
        assert abs(E - Eo) < 1e-13 and abs(sg - so) < 1e-12 * max(1.0, so) + 1e-15
    with pytest.raises(B.LrdmcError):
        B.lrdmc_energy(recs, p=1, n_therm=n)


def test_algorithmic_work_count_matches_survey_table():
    # C2 ~ 0.092 MFLOP, C3/C4 ~ 0.582 MFLOP, C5 single mesh ~ 18.1 MFLOP per walker-move
    assert abs(drv.work_per_walker_move(wl.synthetic10())["total"] - 0.092e6) < 0.002e6
    w = drv.work_per_walker_move(wl.water_methane()); assert w["total"] == 582448 and w["gemm"] == 307200
    c5 = wl.cluster64(); c5["a2"] = 0.0
    assert abs(drv.work_per_walker_move(c5)["total"] - 18.1e6) < 0.2e6
    assert drv.state_bytes_per_walker(wl.water_methane()) == 8 * (48 + 128 + 640)


def test_a_to_zero_fit_closed_forms():
    """f3 host logic: two points reduce to the textbook Richardson formula with its error propagation; exact data are recovered."""
    from paper_2508_12033_b200 import driver as drv
    a1, a2, E1, E2, s1, s2 = 0.2, 0.4, -0.49, -0.46, 1e-3, 2e-3
    E0, sg, coef, chi2 = drv.fit_a_to_zero([a1, a2], [E1, E2], [s1, s2])
    d = a2**2 - a1**2
    assert abs(E0 - (E1 * a2**2 - E2 * a1**2) / d) < 1e-14 and abs(sg - np.hypot(s1 * a2**2, s2 * a1**2) / d) < 1e-14 and chi2 < 1e-20
    a = np.array([0.1, 0.2, 0.3, 0.4]); E = -0.5 + 0.07 * a**2 - 0.3 * a**4
    E0, sg, coef, chi2 = drv.fit_a_to_zero(a, E, np.full(4, 1e-4), n_terms=3)
    assert abs(E0 + 0.5) < 1e-12 and abs(coef[1] - 0.07) < 1e-10 and abs(coef[2] + 0.3) < 1e-9
    E0, sg, *_ = drv.fit_a_to_zero(a, E, np.full(4, 1e-4), n_terms=2)      # a^4 term left out: biased, and chi2 says so
    assert abs(E0 + 0.5) > 3 * sg
    with pytest.raises(ValueError):
        drv.fit_a_to_zero([0.1], [0.0], [1.0])


def test_workload_generators_are_seeded_and_shaped():
    a, b = wl.water_methane(), wl.water_methane()
    assert np.array_equal(a["C_up"], b["C_up"]) and np.array_equal(a["R"], b["R"]) and a["n_ao"] == 200 and a["n_shell"] == 60
    assert (a["n_up"], a["n_dn"], a["n_nuc"]) == (8, 8, 8) and a["pp"].shape == (8, 4) and list(a["Z"]) == [6, 4, 1, 1, 1, 1, 1, 1]
    c2 = wl.synthetic10(); assert c2["n_ao"] == 60 and c2["n_shell"] == 18 and (c2["n_up"], c2["n_dn"]) == (5, 5)
    c5 = wl.cluster64(); assert c5["n_ao"] == 600 and c5["Z"].sum() == 64 and c5["a2"] == 0.4
    assert np.allclose(a["C_up"].T @ a["C_up"], np.eye(8), atol=1e-12)
    x = wl.initial_walkers(a, 7, 5); assert x.shape == (7, 16, 3) and np.array_equal(x, wl.initial_walkers(a, 7, 5))


_GLOO = r"""
import os, sys, torch, torch.distributed as dist
sys.path.insert(0, %r)
import bench
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=2)
rank = dist.get_rank()
def red(op):
    def f(v):
        t = torch.tensor([float(v)], dtype=torch.float64); dist.all_reduce(t, op=op); return t.item()
    return f
units, secs = (1000.0, 2.0) if rank == 0 else (3000.0, 4.0)       # independent replicas of different speed
value, tmax = bench.aggregate_over_ranks(units, secs, 2, red(dist.ReduceOp.MAX), red(dist.ReduceOp.SUM))
assert tmax == 4.0 and value == 1000.0, (value, tmax)               # (1000 + 3000) / max(2, 4)
dist.barrier(); dist.destroy_process_group()
print("rank", rank, "ok")
"""


def test_rank_aggregation_world_size_2_gloo(tmp_path):
    script = tmp_path / "gloo_agg.py"; script.write_text(_GLOO % ROOT)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE, stderr=subprocess.STDOUT) for r in range(2)]
    outs = [p.communicate(timeout=180)[0].decode() for p in procs]
    assert all(p.returncode == 0 for p in procs), outs
    assert "rank 0 ok" in outs[0] and "rank 1 ok" in outs[1]


def test_reference_arm_prints_one_json_line():
    import json
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--steps", "1", "--warmup", "0", "--ref-nw", "8", "--moves", "5"],
                         capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "walker-moves/s" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["higher_is_better"] is True


def test_ctypes_structures_match_the_c_header(tmp_path):
    """The binding's ctypes mirrors of lrdmc_system / lrdmc_basis / lrdmc_mo / lrdmc_jastrow / lrdmc_lattice / lrdmc_cycle_stats have
    the sizes and field offsets gcc gives the structs of include/lrdmc.h (guards the f1 / f2 extensions of the problem statement)."""
    import subprocess
    names = {"lrdmc_system": B.System, "lrdmc_basis": B.Basis, "lrdmc_mo": B.Mo, "lrdmc_jastrow": B.Jastrow, "lrdmc_lattice": B.Lattice,
             "lrdmc_cycle_stats": B.CycleStats}
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "lrdmc.h"', 'int main(void) {']
    for cname, cls in names.items():
        lines.append(f'printf("{cname} %zu\\n", sizeof({cname}));')
        for fname, _ in cls._fields_:
            lines.append(f'printf("{cname}.{fname} %zu\\n", offsetof({cname}, {fname}));')
    lines += ['return 0; }']
    src = tmp_path / "layout.c"; exe = tmp_path / "layout"
    src.write_text("\n".join(lines))
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), "-o", str(exe), str(src)], check=True)
    out = dict(l.split() for l in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.splitlines())
    for cname, cls in names.items():
        assert int(out[cname]) == C.sizeof(cls), cname
        for fname, _ in cls._fields_:
            assert int(out[f"{cname}.{fname}"]) == getattr(cls, fname).offset, (cname, fname)
