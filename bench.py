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


def oracle_sample(sysd, n_w, cycles, moves, seed=5, min_seconds=0.0, threads=0):
    """The oracle as it stands, timed on the host cores on a bounded sample of the same workload."""
    from oracle import lrdmc_ref as ref
    o = ref.Ref(sysd)
    cores = ref.set_threads(threads)           # 0 = all host cores (OpenMP over walkers)
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


def make_workload(args, rank, seed_shift=0):
    seed = wl.PHILOX_RUN_SEED + rank + 1000 * seed_shift
    if args.workload == "C4":
        sysd = wl.water_methane(n_walkers=args.nw, moves=args.moves, seed=seed, name="C4-water-methane-shaped")
        wname = "C4 water-methane-shaped: 16 e (8/8), 8 nuclei, 200 s/p/d GTOs, local PP, 1b+2b Jastrow, a=0.2 (BASELINE.json configs[3]; with --nw 100/400: configs[2])"
    elif args.workload == "C1":
        sysd = wl.hydrogen(n_walkers=args.nw, moves=args.moves, seed=seed)
        wname = "C1 hydrogen atom: 1 e, psi = exp(-0.9 r), a=0.2 (BASELINE.json configs[0])"
    elif args.workload == "C2":
        sysd = wl.synthetic10(n_walkers=args.nw, moves=args.moves, seed=seed)
        wname = "C2 synthetic 10-electron molecule: 5/5, 3 nuclei, 60 s/p/d GTOs, 1b+2b Jastrow, a=0.2 (BASELINE.json configs[1])"
    elif args.workload == "C3j3":
        sysd = wl.with_jastrow3(wl.water_methane(n_walkers=args.nw, moves=args.moves, seed=seed), 7, 1, strength=0.05)
        wname = "C3/C4 water-methane-shaped system + synthetic three-body Jastrow (8 s Gaussians at the nuclei): scope row f2; flop count = without the J3 part"
    elif args.workload == "C3j3spd":
        sysd = wl.with_jastrow3(wl.water_methane(n_walkers=args.nw, moves=args.moves, seed=seed), 8, 3, strength=0.03, n_max=24, poly=True)
        wname = "C3/C4 water-methane-shaped system + synthetic three-body Jastrow (24 s/p/d Gaussians at the nuclei): scope row f2; flop count = without the J3 part"
    elif args.workload == "C3nl":
        sysd = wl.water_methane_nonlocal(n_walkers=args.nw, moves=args.moves, seed=seed)
        wname = "C3/C4 water-methane-shaped system + synthetic non-local s/p/d pseudopotential channels (r_c = 0.8 bohr, DLA): scope row f1; flop count = lattice part only"
    else:
        sysd = wl.cluster64(n_walkers=args.nw, moves=args.moves, seed=seed)
        wname = "C5 64-electron cluster: 32/32, 24 nuclei, 600 s/p/d GTOs, 1b+2b Jastrow, double mesh a=0.2/a'=0.4 (BASELINE.json configs[4])"
    x0 = wl.hydrogen_walkers(args.nw, 1 + rank + 100 * seed_shift) if args.workload == "C1" else wl.initial_walkers(sysd, args.nw, 5 + rank + 100 * seed_shift)
    return sysd, wname, x0


def measured_traffic(workload, n_w, kernel, moves):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the propagate kernel from an `ncu --set full` capture of THIS
    workload (profiles/ncu_traffic_by_workload.md: one table row per captured workload); None if that workload was never captured."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic_by_workload.md")) as f:
            for ln in f:
                c = [t.strip() for t in ln.strip().strip("|").split("|")]
                if len(c) >= 5 and c[0] == workload and c[1] == str(n_w) and c[2] == kernel and c[4] == str(moves):
                    return float(c[3])
    except Exception:
        pass
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1); ap.add_argument("--steps", type=int, default=10); ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours"); ap.add_argument("--nw", type=int, default=25600); ap.add_argument("--moves", type=int, default=100)
    ap.add_argument("--ref-nw", type=int, default=64); ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-conventional", action="store_true"); ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--workload", default="C4", choices=["C1", "C2", "C4", "C5", "C3nl", "C3j3", "C3j3spd"],
                    help="C4 (default) is the configuration the metric is quoted on; C2 / C5 are the other BASELINE.json systems, C3nl adds non-local pseudopotential channels (use with --nw/--moves)")
    ap.add_argument("--contexts", type=int, default=1,
                    help="K independent ensembles of --nw walkers each (own context, own CUDA stream, own seed) in flight together: the paper's "
                         "small-ensemble regime (100 walkers per GPU, L289) and the several-a batch of SURVEY 8(f) f3; value = aggregate over the K")
    ap.add_argument("--team", type=int, default=0, help="lrdmc_set_option(LRDMC_OPT_TEAM_WARPS): 0 = automatic")
    ap.add_argument("--listed", type=int, default=-1, help="lrdmc_set_option(LRDMC_OPT_LISTED): -1 = automatic, 0 = dense candidate sweep, 1 = listed sweep on stored Bc")
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

    K = max(1, args.contexts)
    ctxs = []
    for q in range(K):
        sysd, wname, x0 = make_workload(args, rank, q)
        opts = {}
        if args.team: opts[B.OPT_TEAM_WARPS] = args.team
        if args.listed >= 0: opts[B.OPT_LISTED] = args.listed
        g = B.Lrdmc(sysd, device=dev, options=opts or None)
        g.stream = torch.cuda.Stream(device=dev) if K > 1 else torch.cuda.current_stream(dev)
        with torch.cuda.stream(g.stream):
            g.lrdmc_set_positions(x0, allow_singular=True)
        ctxs.append((g, sysd, x0))
    g, sysd, x0 = ctxs[0]
    N = sysd["n_up"] + sysd["n_dn"]
    tau = args.moves * sysd["a"] ** 2 / (3 * N)       # reading Q19 first guess; refined from a pilot below
    E0 = [0.0] * K; esum = [0.0] * K; ecnt = [0] * K  # Green's-function energy per ensemble, fed back after each branching (L232)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(mode, steps, first_cycle, tau_, feedback=True):
        """K steps bracketed by barrier+sync, CUDA events on the launching stream.  Per step and ensemble: read the estimators of its last
        interval (E_0 feedback), enqueue propagate + reconfigure on its own stream; the region ends when all results are on the host."""
        barrier()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        l0 = sum(c[0].launch_count() for c in ctxs); recs = [[] for _ in ctxs]
        main_stream = torch.cuda.current_stream(dev)
        e0.record(main_stream)
        if K > 1:
            for c in ctxs:
                c[0].stream.wait_event(e0)
        def collect(q, c):
            st = c[0].lrdmc_estimators(); recs[q].append(st)
            if mode == B.BALANCED and feedback and st.den > 0:
                esum[q] += st.num / st.den; ecnt[q] += 1; E0[q] = esum[q] / ecnt[q]   # "Update E_0" (Alg.2 line 12 L418)
        # pipelined over the ensembles (driver.a_scan does the same): ensemble q's next interval is enqueued as soon as ITS last one has been read
        for cyc_ in range(first_cycle, first_cycle + steps):
            for q, c in enumerate(ctxs):
                if cyc_ > first_cycle:
                    collect(q, c)
                with torch.cuda.stream(c[0].stream):
                    c[0].lrdmc_propagate(mode, args.moves if mode == B.BALANCED else 0, tau_, E0[q] if mode == B.BALANCED else 0.0, cyc_)
                    c[0].lrdmc_reconfigure(cyc_)
        for q, c in enumerate(ctxs):
            collect(q, c)
        if K > 1:
            for c in ctxs:
                main_stream.wait_stream(c[0].stream)
        e1.record(main_stream); barrier()
        return e0.elapsed_time(e1) * 1e-3, recs, sum(c[0].launch_count() for c in ctxs) - l0

    # ---- warm-up (it also seeds E_0) + timed balanced steps
    timed(B.BALANCED, args.warmup, 0, 0.0)
    cyc = args.warmup
    with ClockSampler(local) as clk:
        secs, recs_all, launches = timed(B.BALANCED, args.steps, cyc, 0.0)
    cyc += args.steps
    recs = recs_all[0]
    moves = sum(r.moves_sum for rr in recs_all for r in rr)
    fmax = (lambda v: float(_allreduce(dist, torch, v, "max", dev))) if dist is not None else None
    fsum = (lambda v: float(_allreduce(dist, torch, v, "sum", dev))) if dist is not None else None
    value, tmax = aggregate_over_ranks(moves, secs, world, fmax, fsum)

    prop_ms = float(np.mean([r.propagate_ms for r in recs])); rec_ms = float(np.mean([r.reconfigure_ms for r in recs]))
    flop = drv.work_per_walker_move(sysd)
    peaks = B.lrdmc_measure_fp64_peaks()
    cfg = g.launch_config()
    per_launch_moves = sum(r.moves_sum for r in recs) / len(recs)
    achieved = flop["total"] * per_launch_moves / (prop_ms * 1e-3) / 1e12
    executed = flop["executed"] * per_launch_moves / (prop_ms * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": cfg["kernel"], "achieved": achieved, "peak": peaks["dfma_tflops"], "unit": "TFLOP/s", "frac": achieved / peaks["dfma_tflops"], "frac_vs_dmma_peak": achieved / peaks["dmma_tflops"],
                "traffic": measured_traffic(args.workload, args.nw, cfg["kernel"], args.moves) if K == 1 else None,
                "frac_note": "frac = ALGORITHMIC flop (SURVEY 8(d) count, every candidate through the MOs) / kernel time / peak: speed relative to the naive algorithm "
                             "at peak, may exceed 1; frac_executed = flop the column-form kernel executes / kernel time / peak: FP64-pipe utilisation (compare ncu sm__pipe_fp64_cycles_active)",
                "achieved_executed": executed, "frac_executed": executed / peaks["dfma_tflops"],
                "flop_per_walker_move": flop["total"], "flop_executed_per_walker_move": flop["executed"],
                "peak_source": "measured live: liblrdmc_probe lrdmc_measure_fp64_peaks (independent DFMA chains, all SMs)",
                "dmma_peak": peaks["dmma_tflops"], "dfma_dmma_mixed": peaks["mixed_tflops"], "dfma_3reg_peak": peaks["dfma_3reg_tflops"], "dfma_1shared_peak": peaks["dfma_shared1_tflops"], "dfma_with_2_alu_peak": peaks["dfma_alu_tflops"],
                "kernel_ms": prop_ms, "kernel_share_of_step": prop_ms * len(recs) / (secs * 1e3),
                "hbm_bytes_per_launch_algorithmic": 2 * drv.state_bytes_per_walker(sysd) * args.nw}
    if cfg.get("listed_sweep"):      # the executed count assumes the dense sweep; the listed sweep skips the unlisted (electron, shell) pairs and keeps Bc as state
        roofline["frac_executed"] = None; roofline["achieved_executed"] = None
        roofline["frac_executed_note"] = ("listed sweep: the flop executed depend on the walkers' shell lists (DESIGN.md section 4: 58 percent of the pairs are skipped at C5, 41 percent at C4); "
                                          f"the dense column-form count would give {executed / peaks['dfma_tflops']:.3f}")
    if K > 1:
        roofline["note"] = f"{K} contexts in flight: kernel_ms is one launch of context 0 while the others run beside it; achieved/frac describe that launch, not the device"

    evals = sum(r.moves_sum + args.nw for rr in recs_all for r in rr)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tmax / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wname,
                       "n_walkers": args.nw, "contexts": K, "moves_per_cycle": args.moves, "mode": "balanced", "parallelism": f"replicas x{world}",
                       "l2": "inputs larger than L2: walker state %.0f MB per replica" % (drv.state_bytes_per_walker(sysd) * args.nw * K / 1e6)
                             if drv.state_bytes_per_walker(sysd) * args.nw * K > 126e6 else
                             "walker state %.1f MB fits L2 (the path re-reads 2 x state per step from wherever it lives; HBM is not the bound)" % (drv.state_bytes_per_walker(sysd) * args.nw * K / 1e6),
                       "launch": cfg},
            "roofline": roofline, "gpu_launches": launches, "reconfigure_ms": rec_ms,
            "result_check": {"E0_feedback": True, "e_mean_last_step": float(np.mean([rr[-1].num / rr[-1].den for rr in recs_all])),
                             "E0_last": float(np.mean(E0)), "n_nonpos_diag": int(sum(r.n_nonpos_diag for rr in recs_all for r in rr)),
                             "n_nonfinite": int(sum(r.n_nonfinite for rr in recs_all for r in rr)),
                             "node_flag_share_of_evaluations": float(sum(r.n_node_flag for rr in recs_all for r in rr)) / max(1, evals),
                             "wbar_last_step": float(np.mean([rr[-1].wbar for rr in recs_all]))},
            "branch_idle": {"balanced_device": float(np.mean([r.barrier_idle_frac for r in recs])), "balanced_lockstep": float(np.mean([r.lockstep_idle_frac for r in recs]))}}

    # ---- conventional mode at equal N_w and equal mean move count
    if not args.no_conventional:
        _, pil, _ = timed(B.CONVENTIONAL, 1, cyc, tau); cyc += 1
        mean_moves = pil[0][0].moves_sum / args.nw
        tau *= args.moves / max(1.0, mean_moves)
        timed(B.CONVENTIONAL, 1, cyc, tau); cyc += 1
        csecs, crecs_all, _ = timed(B.CONVENTIONAL, args.steps, cyc, tau); cyc += args.steps
        crecs = crecs_all[0]
        cmoves = sum(r.moves_sum for rr in crecs_all for r in rr)
        cval, _ = aggregate_over_ranks(cmoves, csecs, world, fmax, fsum)
        line["conventional"] = {"value": cval, "unit": UNIT, "tau": tau, "mean_moves_per_cycle": cmoves / len(crecs) / args.nw / K,
                                "moves_max": int(max(r.moves_max for r in crecs)), "ms_per_step": 1e3 * csecs / args.steps,
                                "balanced_over_conventional": value / cval, "n_nonfinite": int(sum(r.n_nonfinite for rr in crecs_all for r in rr))}
        line["branch_idle"]["conventional_device"] = float(np.mean([r.barrier_idle_frac for r in crecs]))
        line["branch_idle"]["conventional_lockstep"] = float(np.mean([r.lockstep_idle_frac for r in crecs]))

    # ---- end to end through the host-buffer C-ABI call (H2D of the positions, D2H of positions + stats inside the timed region)
    if not args.no_e2e:
        xin = [torch.from_numpy(c[2]).pin_memory() for c in ctxs]
        for q, c in enumerate(ctxs):
            c[0].lrdmc_run_host(xin[q], B.BALANCED, args.moves, 0.0, E0[q], cyc, 1)
        cyc += 1
        barrier(); t0 = time.perf_counter(); emoves = 0
        for s_ in range(args.steps):
            for q, c in enumerate(ctxs):        # the host-buffer call is synchronous: with K contexts they run one after the other
                st, xout = c[0].lrdmc_run_host(xin[q], B.BALANCED, args.moves, 0.0, E0[q], cyc, 1)
                emoves += st[0].moves_sum
            cyc += 1
        barrier(); esecs = time.perf_counter() - t0
        eval_, _ = aggregate_over_ranks(emoves, esecs, world, fmax, fsum)
        nbytes = int(x0.nbytes) * K
        line["e2e"] = {"value": eval_, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes + 104 * K,
                       "note": "lrdmc_run_host: pinned host positions in, set_positions (inverse rebuild), propagate, reconfigure, estimators, host positions out"}
    line["clocks"] = clk.summary()

    if rank == 0 and not args.no_cpu_baseline and world == 1:
        ref_sys = sysd if args.workload != "C4" else wl.water_methane(n_walkers=args.ref_nw)
        v, cores, dt, n = oracle_sample(ref_sys, args.ref_nw, 2, args.moves, min_seconds=12.0)
        # also on ONE core (after the all-core sample: the oracle's thread count stays at what was set last)
        v1, _, dt1, n1 = oracle_sample(ref_sys, 8, 1, args.moves, min_seconds=3.0, threads=1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "value_1core": v1,
                                "sample_1core": f"N_w=8 walkers x {n1 // (8 * args.moves)} cycles x {args.moves} moves, 1 thread ({dt1:.1f} s)",
                                "sample": f"same {args.workload} system, N_w={args.ref_nw} walkers x {n // (args.ref_nw * args.moves)} cycles x {args.moves} moves ({n} walker-moves, {dt:.1f} s), balanced, incl. reconfiguration"}
    if rank == 0:
        print(json.dumps(line), flush=True)
    for c in ctxs:
        c[0].close()
    if dist is not None:
        dist.destroy_process_group()


def _allreduce(dist, torch, v, op, dev):
    t = torch.tensor([float(v)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX if op == "max" else dist.ReduceOp.SUM)
    return t.item()


if __name__ == "__main__":
    main()
