#!/usr/bin/env python
"""bench.py -- walker-moves/s of load-balanced LRDMC on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--nw N_w] [--moves N_proj]

A step = one whole branching interval of the hot path: lrdmc_propagate (N_proj moves of all N_w walkers + the
measurement evaluation) -> lrdmc_reconfigure (comb, gather, inverse rebuild) -> lrdmc_estimators, on the
water-methane-shaped config C4 (BASELINE.json configs[3]: N_w = 25600, 100 moves per branching, the config the metric is
quoted on).  Multi-GPU (torchrun): independent replicas, no data-path collective (north_star: "no collectives").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2508_12033_b200 import workloads as wl  # noqa: E402
from paper_2508_12033_b200 import driver as drv    # noqa: E402

METRIC = "walker-moves/s on 1 B200 (balanced vs conventional); roofline %; branch idle %"
UNIT = "walker-moves/s"


def aggregate_over_ranks(units_this_rank, seconds_this_rank, world_size, all_reduce_max=None, all_reduce_sum=None):
    """Whole-job throughput for independent replicas: sum of units / MAX over ranks of the time (host logic, gloo-tested)."""
    t = seconds_this_rank if all_reduce_max is None else all_reduce_max(seconds_this_rank)
    u = units_this_rank * world_size if all_reduce_sum is None else all_reduce_sum(units_this_rank)
    return u / t, t


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.rows = []; self.stop = False; self.index = index; self.th = None

    def _loop(self):
        while not self.stop:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            time.sleep(0.2)

    def __enter__(self):
        self.th = threading.Thread(target=self._loop, daemon=True); self.th.start(); return self

    def __exit__(self, *a):
        self.stop = True; self.th.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": float(self.rows[0][1]) if self.rows[0][1].replace(".", "").isdigit() else None,
                "reasons": reasons, "samples": len(self.rows)}


def oracle_sample(sysd, n_w, cycles, moves, seed=5, min_seconds=0.0):
    """The oracle as it stands, timed on the host cores on a bounded sample of the same workload."""
    from oracle import lrdmc_ref as ref
    o = ref.Ref(sysd)
    cores = ref.set_threads(0)
    x0 = wl.initial_walkers(sysd, n_w, seed)
    rc = o.set_positions(x0)
    if rc not in (0, -2):
        raise RuntimeError(f"oracle set_positions failed: {rc}")
    t0 = time.perf_counter(); n = 0; c = 0
    while c < cycles or (min_seconds > 0 and time.perf_counter() - t0 < min_seconds and c < 50 * cycles):
        o.propagate(ref.BALANCED, moves, 0.0, 0.0, c); o.reconfigure(c); n += int(o.estimators()["moves_sum"]); c += 1
    dt = time.perf_counter() - t0
    return n / dt, cores, dt, n


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle (there is no reference code).  Rank 0 only."""
    if rank != 0:
        return
    sysd = wl.water_methane(n_walkers=args.ref_nw, moves=args.moves)
    for c in range(args.warmup):
        oracle_sample(sysd, args.ref_nw, 1, max(1, args.moves // 10))
    vals = []; t_tot = 0.0; cores = 0
    for s in range(args.steps):
        v, cores, dt, n = oracle_sample(sysd, args.ref_nw, 1, args.moves, seed=5 + s); vals.append(n); t_tot += dt
    value = sum(vals) / t_tot
    sample = f"C4 system (water-methane-shaped, 16 e, 200 AO), N_w={args.ref_nw} walkers x 1 cycle x {args.moves} moves per step, balanced mode, incl. reconfiguration"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_tot / max(1, args.steps), "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": "C4 water-methane-shaped (bounded sample)", "n_walkers": args.ref_nw, "moves_per_cycle": args.moves, "mode": "balanced"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1); ap.add_argument("--steps", type=int, default=10); ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours"); ap.add_argument("--nw", type=int, default=25600); ap.add_argument("--moves", type=int, default=100)
    ap.add_argument("--ref-nw", type=int, default=64); ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-conventional", action="store_true"); ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C4", "C5", "C3nl", "C3j3"],
                    help="C4 (default) is the configuration the metric is quoted on; C2 / C5 are the other BASELINE.json systems, C3nl adds non-local pseudopotential channels (use with --nw/--moves)")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1")); local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world); return
    args.warmup = max(3, args.warmup)

    import torch
    from paper_2508_12033_b200 import binding as B
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path has no CPU fallback (use --impl reference for the oracle)")
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = f"cuda:{local}"; torch.cuda.set_device(dev)

    if args.workload == "C4":
        sysd = wl.water_methane(n_walkers=args.nw, moves=args.moves, seed=wl.PHILOX_RUN_SEED + rank, name="C4-water-methane-shaped")
        wname = "C4 water-methane-shaped: 16 e (8/8), 8 nuclei, 200 s/p/d GTOs, local PP, 1b+2b Jastrow, a=0.2 (BASELINE.json configs[3])"
    elif args.workload == "C1":
        sysd = wl.hydrogen(n_walkers=args.nw, moves=args.moves, seed=wl.PHILOX_RUN_SEED + rank)
        wname = "C1 hydrogen atom: 1 e, psi = exp(-0.9 r), a=0.2 (BASELINE.json configs[0])"
    elif args.workload == "C2":
        sysd = wl.synthetic10(n_walkers=args.nw, moves=args.moves, seed=wl.PHILOX_RUN_SEED + rank)
        wname = "C2 synthetic 10-electron molecule: 5/5, 3 nuclei, 60 s/p/d GTOs, 1b+2b Jastrow, a=0.2 (BASELINE.json configs[1])"
    elif args.workload == "C3j3":
        sysd = wl.with_jastrow3(wl.water_methane(n_walkers=args.nw, moves=args.moves, seed=wl.PHILOX_RUN_SEED + rank), 7, 1, strength=0.05)
        wname = "C3/C4 water-methane-shaped system + synthetic three-body Jastrow (8 s Gaussians at the nuclei): scope row f2; flop count = without the J3 part"
    elif args.workload == "C3nl":
        sysd = wl.water_methane_nonlocal(n_walkers=args.nw, moves=args.moves, seed=wl.PHILOX_RUN_SEED + rank)
        wname = "C3/C4 water-methane-shaped system + synthetic non-local s/p/d pseudopotential channels (r_c = 0.8 bohr, DLA): scope row f1; flop count = lattice part only"
    else:
        sysd = wl.cluster64(n_walkers=args.nw, moves=args.moves, seed=wl.PHILOX_RUN_SEED + rank)
        wname = "C5 64-electron cluster: 32/32, 24 nuclei, 600 s/p/d GTOs, 1b+2b Jastrow, double mesh a=0.2/a'=0.4 (BASELINE.json configs[4])"
    x0 = wl.hydrogen_walkers(args.nw, 1 + rank) if args.workload == "C1" else wl.initial_walkers(sysd, args.nw, 5 + rank)
    g = B.Lrdmc(sysd, device=dev)
    g.lrdmc_set_positions(x0, allow_singular=True)
    E0 = 0.0          # fixed Green's-function energy for the timing runs (W ~ 3N/a^2 = 1200 >> e_L; nonpos events are reported)
    N = sysd["n_up"] + sysd["n_dn"]
    tau = args.moves * sysd["a"] ** 2 / (3 * N)       # reading Q19 first guess; refined from a pilot below

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(mode, steps, first_cycle, tau_):
        """K steps bracketed by barrier+sync, CUDA events on the launching (current torch) stream."""
        barrier()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        l0 = g.launch_count(); recs = []
        e0.record()
        for c in range(first_cycle, first_cycle + steps):
            g.lrdmc_propagate(mode, args.moves if mode == B.BALANCED else 0, tau_, E0 if mode == B.BALANCED else 0.0, c)
            g.lrdmc_reconfigure(c)
            recs.append(g.lrdmc_estimators())
        e1.record(); barrier()
        return e0.elapsed_time(e1) * 1e-3, recs, g.launch_count() - l0

    # ---- warm-up + pilot for tau (conventional mode with the same mean move count, L283-L285)
    _, wrecs, _ = timed(B.BALANCED, args.warmup, 0, 0.0)
    cyc = args.warmup
    with ClockSampler(local) as clk:
        secs, recs, launches = timed(B.BALANCED, args.steps, cyc, 0.0)
    cyc += args.steps
    moves = sum(r.moves_sum for r in recs)
    fmax = (lambda v: float(_allreduce(dist, torch, v, "max", dev))) if dist is not None else None
    fsum = (lambda v: float(_allreduce(dist, torch, v, "sum", dev))) if dist is not None else None
    value, tmax = aggregate_over_ranks(moves, secs, world, fmax, fsum)

    prop_ms = float(np.mean([r.propagate_ms for r in recs])); rec_ms = float(np.mean([r.reconfigure_ms for r in recs]))
    flop = drv.work_per_walker_move(sysd)
    peaks = B.lrdmc_measure_fp64_peaks()
    achieved = flop["total"] * (moves / len(recs)) / (prop_ms * 1e-3) / 1e12
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_propagate_traffic.txt")) as f:     # last ncu --set full capture (text)
            for ln in f:
                if ln.startswith("dram_bytes_per_launch"):
                    traffic = float(ln.split()[1])
    except Exception:
        pass
    roofline = {"bound": "alu", "kernel": "k_propagate", "achieved": achieved, "peak": peaks["dfma_tflops"], "unit": "TFLOP/s", "frac": achieved / peaks["dfma_tflops"],
                "traffic": traffic, "peak_source": "measured live: lrdmc_measure_fp64_peaks (independent DFMA chains, all SMs)",
                "dmma_peak": peaks["dmma_tflops"], "dfma_dmma_mixed": peaks["mixed_tflops"], "dfma_3reg_peak": peaks["dfma_3reg_tflops"], "dfma_with_2_alu_peak": peaks["dfma_alu_tflops"], "flop_per_walker_move": flop["total"],
                "kernel_ms": prop_ms, "kernel_share_of_step": prop_ms * len(recs) / (secs * 1e3),
                "hbm_bytes_per_launch_algorithmic": 2 * drv.state_bytes_per_walker(sysd) * args.nw}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tmax / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wname,
                       "n_walkers": args.nw, "moves_per_cycle": args.moves, "mode": "balanced", "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2: walker state %.0f MB per replica" % (drv.state_bytes_per_walker(sysd) * args.nw / 1e6),
                       "launch": g.launch_config()},
            "roofline": roofline, "gpu_launches": launches, "reconfigure_ms": rec_ms,
            "branch_idle": {"balanced_device": float(np.mean([r.barrier_idle_frac for r in recs])), "balanced_lockstep": float(np.mean([r.lockstep_idle_frac for r in recs]))}}

    # ---- conventional mode at equal N_w and equal mean move count
    if not args.no_conventional:
        _, pil, _ = timed(B.CONVENTIONAL, 1, cyc, tau); cyc += 1
        mean_moves = pil[0].moves_sum / args.nw
        tau *= args.moves / max(1.0, mean_moves)
        timed(B.CONVENTIONAL, 1, cyc, tau); cyc += 1
        csecs, crecs, _ = timed(B.CONVENTIONAL, args.steps, cyc, tau); cyc += args.steps
        cmoves = sum(r.moves_sum for r in crecs)
        cval, _ = aggregate_over_ranks(cmoves, csecs, world, fmax, fsum)
        line["conventional"] = {"value": cval, "unit": UNIT, "tau": tau, "mean_moves_per_cycle": cmoves / len(crecs) / args.nw,
                                "moves_max": int(max(r.moves_max for r in crecs)), "ms_per_step": 1e3 * csecs / args.steps,
                                "balanced_over_conventional": value / cval}
        line["branch_idle"]["conventional_device"] = float(np.mean([r.barrier_idle_frac for r in crecs]))
        line["branch_idle"]["conventional_lockstep"] = float(np.mean([r.lockstep_idle_frac for r in crecs]))

    # ---- end to end through the host-buffer C-ABI call (H2D of the positions, D2H of positions + stats inside the timed region)
    if not args.no_e2e:
        xin = torch.from_numpy(x0).pin_memory()
        g.lrdmc_run_host(xin, B.BALANCED, args.moves, 0.0, E0, cyc, 1); cyc += 1
        barrier(); t0 = time.perf_counter(); emoves = 0
        for s in range(args.steps):
            st, xout = g.lrdmc_run_host(xin, B.BALANCED, args.moves, 0.0, E0, cyc, 1); cyc += 1
            emoves += st[0].moves_sum
        barrier(); esecs = time.perf_counter() - t0
        eval_, _ = aggregate_over_ranks(emoves, esecs, world, fmax, fsum)
        nbytes = int(x0.nbytes)
        line["e2e"] = {"value": eval_, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 104,
                       "note": "lrdmc_run_host: pinned host positions in, set_positions (inverse rebuild), propagate, reconfigure, estimators, host positions out"}
    line["clocks"] = clk.summary()

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        ref_sys = sysd if args.workload != "C4" else wl.water_methane(n_walkers=args.ref_nw)
        v, cores, dt, n = oracle_sample(ref_sys, args.ref_nw, 2, args.moves, min_seconds=12.0)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"same {args.workload} system, N_w={args.ref_nw} walkers x {n // (args.ref_nw * args.moves)} cycles x {args.moves} moves ({n} walker-moves, {dt:.1f} s), balanced, incl. reconfiguration"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    g.close()
    if dist is not None:
        dist.destroy_process_group()


def _allreduce(dist, torch, v, op, dev):
    t = torch.tensor([float(v)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return t.item()


if __name__ == "__main__":
    main()
