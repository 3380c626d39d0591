#!/usr/bin/env python
"""bench.py -- one JSON line for the exact-exchange hot path (BASELINE.json metric: Poisson solves/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--nc n_c] [--impl reference]

A "step" is one full exchange apply (all SURVEY 8(a) rows: pair density, 3+3 mode products with the
eigen-space multiply, accumulate, energy) of one BASELINE.json config over synthetic orbitals.
Default workload: BASELINE.json configs[1] (48^3 HSE bulk, 64 orbitals, 4,096 pair solves).
N > 1 (torchrun): targets are sharded across ranks, orbitals replicated, no data-path collective
(weak scaling: every rank applies Vx to its own block of n_tgt targets); rank 0 prints the line.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

from paper_2501_16572_b200 import workloads as wl  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum per k_mode_t launch (average over the six passes of a batch) from the
# `ncu --set full` captures summarised in profiles/r1_final2_summary.md and r1_final_summary.md, keyed by (config, n_c); other shapes: null.
NCU_TRAFFIC_BYTES = {(2, 128): 167.9e6, (2, 1024): 1.739e9, (5, 128): 3.545e9}

METRIC = "poisson_pair_solves_per_s"
UNIT = "solves/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-based); default 2 = configs[1]")
    ap.add_argument("--nc", type=int, default=0, help="right-hand sides per batch (0 = workload default)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--variant", type=int, default=0, help="0 = DMMA path (default), 1 = plain-kernel cross-check variant")
    ap.add_argument("--n-orb", type=int, default=0, help="override orbital count (debug; invalidates the headline)")
    ap.add_argument("--n-tgt", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--solver-sweep", action="store_true",
                    help="bare exx_poisson_solve over n_c = 1..512 on the config's grid (the paper's Figs. 1-2 in shape)")
    ap.add_argument("--bloch", action="store_true",
                    help="measure the Bloch-periodic complex variant (SURVEY 8(f) NEXT-3) on the config's grid instead")
    ap.add_argument("--nc-sym", type=int, default=0,
                    help="batch size of the pair-symmetric apply (0 = min(n_c, 4 n_orb): larger rectangles waste more "
                         "j > k pairs inside their diagonal blocks)")
    ap.add_argument("--no-ace", action="store_true", help="skip the ACE tail/apply measurement (SURVEY 8(f) NEXT-1)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def workload_from_args(args) -> wl.Workload:
    w = wl.WORKLOADS[args.config]
    if args.n_orb or args.n_tgt:
        n_orb = args.n_orb or w.n_orb
        w = wl.scaled(w, n_orb, args.n_tgt or min(w.n_tgt, n_orb))
    return w


def config_dict(w: wl.Workload, n_c: int, extra=None) -> dict:
    bcs = "".join("P" if b == wl.PERIODIC else "D" for b in w.bc)
    d = {"workload": f"BASELINE.json configs[{w.cfg - 1}]: {w.name}", "grid": [w.nx, w.ny, w.nz], "h_bohr": w.h,
         "bc_xyz": bcs, "fd_order": w.order, "omega": w.omega, "n_occ": w.n_orb, "n_tgt": w.n_tgt,
         "tgt_start": w.tgt_start, "pair_solves_per_step": w.pair_solves, "n_c": n_c,
         "flops_per_solve": w.flops_per_solve, "l2": "flushed between timed steps (256 MiB write)"}
    if extra:
        d.update(extra)
    return d


# ---------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------

def _oracle_threads() -> int:
    try:
        from threadpoolctl import threadpool_info
        n = [p.get("num_threads", 1) for p in threadpool_info() if p.get("user_api") == "blas"]
        if n:
            return int(max(n))
    except Exception:
        pass
    return len(os.sched_getaffinity(0))


def time_oracle(w: wl.Workload, psi, occ, tgt, occ_t, budget_s: float, steps: int = 1, warmup: int = 0):
    """Oracle exx_apply on a bounded sample of the workload's targets (all occupied orbitals, the first
    n_s targets, n_s sized from a one-target calibration so a step takes about `budget_s`)."""
    from oracle import exx_oracle as orc   # the one place bench.py executes oracle/ (cpu_baseline / --impl reference)
    plan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    psi_n, occ_n, tgt_n, occ_t_n = psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy()
    t0 = time.perf_counter()
    orc.exx_apply(plan, psi_n, occ_n, tgt_n[:1], occ_t_n[:1])
    t1 = time.perf_counter() - t0
    n_s = int(max(1, min(w.n_tgt, budget_s / max(t1, 1e-6))))
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        orc.exx_apply(plan, psi_n, occ_n, tgt_n[:n_s], occ_t_n[:n_s])
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
    dt = sum(times) / len(times)
    solves = w.n_orb * n_s
    return {"value": solves / dt, "unit": UNIT, "cores": _oracle_threads(), "kind": "oracle",
            "sample": f"oracle/exx_oracle.exx_apply (numpy FP64) on {n_s} of {w.n_tgt} targets x {w.n_orb} occupied "
                      f"= {solves} pair solves, {dt:.2f} s per step"}, dt, solves


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload_from_args(args)
    psi, occ, tgt, occ_t = wl.make_inputs(w, "cpu")
    steps = max(1, min(args.steps, 3))
    budget = min(args.cpu_seconds, 120.0 / (steps + 1))
    cb, dt, solves = time_oracle(w, psi, occ, tgt, occ_t, budget, steps=steps, warmup=min(args.warmup, 1))
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": min(args.warmup, 1), "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, args.nc or w.default_nc, {"l2": "n/a (CPU)"}),
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# B200 arm
# ---------------------------------------------------------------------------------------------------

class ClockSampler:
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            text, _ = self.proc.communicate(timeout=5)
        except Exception:
            return out
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in text.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 8:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                power.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[4:8]):
                if v.lower() == "active":
                    reasons.add(nm)
        if sm:
            busy = [s for s, p in zip(sm, power) if p > 0.5 * max(power)] or sm
            out.update({"sm_mhz": statistics.median(busy), "sm_max_mhz": max(mx), "reasons": sorted(reasons),
                        "samples": len(sm), "power_w_max": max(power)})
        return out


def run_b200(args):
    import torch.distributed as dist
    from paper_2501_16572_b200 import exx

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        dist.barrier()

    w = workload_from_args(args)
    n_c = args.nc or w.default_nc
    # inputs: generated on the GPU for the large configs, on the host (numpy) for configs 1-3
    gen_dev = dev if w.cfg >= 4 else "cpu"
    psi, occ, tgt, occ_t = wl.make_inputs(w, gen_dev)
    d_psi, d_occ = psi.to(dev), occ.to(dev)
    # weak scaling: rank r applies Vx to n_tgt targets starting at tgt_start + r*n_tgt (wrapping)
    from paper_2501_16572_b200 import sharding
    idx = sharding.weak_scaling_targets(w.tgt_start, w.n_tgt, w.n_orb, rank)
    if world == 1:
        d_tgt = d_psi[w.tgt_start:w.tgt_start + w.n_tgt]
        d_occ_t = d_occ[w.tgt_start:w.tgt_start + w.n_tgt]
    else:
        d_tgt = d_psi[idx.to(dev)].contiguous()
        d_occ_t = d_occ[idx.to(dev)].contiguous()

    plan = exx.Plan.for_workload(w, max_batch=max(128, n_c), device=local)
    plan.set_variant(args.variant)
    vx = torch.empty((w.n_tgt, w.nz, w.ny, w.nx), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def step():
        return plan.apply(d_psi, d_occ, d_tgt, d_occ_t, vx=vx, n_c=n_c, stream=stream)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    launches_per_step = plan.last_launch_count

    sampler = ClockSampler(local) if rank == 0 else None
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for e0, e1 in ev:
        flush.fill_(1)             # evict L2 between timed steps (outside the event pair)
        e0.record(stream)
        _, e_k, ex = step()
        e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    total_ms = sum(e0.elapsed_time(e1) for e0, e1 in ev)
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    clocks = sampler.stop() if sampler else None
    ms_per_step = total_ms / args.steps
    value = world * w.pair_solves / (ms_per_step * 1e-3)
    ex_val = float(ex.item())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class (mode products on the FP64 tensor pipe) -----------------
    peak_dmma = exx.probe_fp64_peak(1, local, 1.5)
    peak_dfma = exx.probe_fp64_peak(0, local, 0.5)
    plan.set_profiling(True)
    prof_steps = min(2, args.steps)
    for _ in range(prof_steps):
        flush.fill_(1)
        step()
    prof = plan.get_profile()
    plan.set_profiling(False)
    mp_ms, mp_cnt = prof["mode_product"]
    all_ms = sum(v[0] for v in prof.values())
    flops_step = w.pair_solves * w.flops_per_solve
    achieved = flops_step * prof_steps / (mp_ms * 1e-3) / 1e12 if mp_ms > 0 else 0.0
    roofline = {"bound": "tensor", "kernel": "k_mode_dmma (six mode products per batch, FP64 mma.sync -> DMMA.8x8x4)",
                "achieved": achieved, "peak": peak_dmma, "unit": "TFLOP/s", "frac": achieved / peak_dmma,
                "traffic": NCU_TRAFFIC_BYTES.get((w.cfg, n_c)),
                "traffic_note": "bytes per k_mode_t launch, profiles/r1_final2_summary.md / r1_final_summary.md (cold-cache ncu replay); "
                                f"algorithmic bytes per launch = {2 * 8 * w.N * min(n_c, w.pair_solves):.4g} (batch read + written in place)",
                "peak_source": "measured live: exx_probe_fp64_peak DMMA issue loop (MEASURED_PEAKS.json has no FP64 entry); "
                               f"DFMA loop {peak_dfma:.2f} TF",
                "avg_launch_ms": mp_ms / max(mp_cnt, 1), "launches": mp_cnt // prof_steps,
                "share_of_step": mp_ms / all_ms if all_ms > 0 else None,
                "step_frac": flops_step / (ms_per_step * 1e-3) / 1e12 / peak_dmma,
                "class_ms_per_step": {k: v[0] / prof_steps for k, v in prof.items()},
                "measured": "separate instrumented steps (CUDA-event pair around every launch, caller's stream)"}

    # ---- end to end through the C-ABI with host buffers (H2D + D2H inside the timed region) ------------
    e2e = None
    if not args.no_e2e and world == 1 and w.n_orb * w.N * 8 <= (24 << 30):
        h_psi = torch.empty(psi.shape, dtype=torch.float64, pin_memory=True)
        h_psi.copy_(psi)
        h_occ = occ.cpu().contiguous()
        h_occ_t = occ_t.cpu().contiguous()
        h_vx = torch.empty((w.n_tgt, w.nz, w.ny, w.nx), dtype=torch.float64, pin_memory=True)
        k = max(3, min(args.steps, 5))
        for _ in range(2):
            plan.apply_host(h_psi, h_occ, tgt_start=w.tgt_start, n_tgt=w.n_tgt, occ_tgt=h_occ_t, vx=h_vx, n_c=n_c)
        t0 = time.perf_counter()
        for _ in range(k):
            _, _, ex_h = plan.apply_host(h_psi, h_occ, tgt_start=w.tgt_start, n_tgt=w.n_tgt, occ_tgt=h_occ_t,
                                         vx=h_vx, n_c=n_c)
        dt = (time.perf_counter() - t0) / k
        e2e = {"value": w.pair_solves / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(h_psi.numel() * 8 + h_occ.numel() * 8 + h_occ_t.numel() * 8),
               "d2h_bytes_per_step": int(h_vx.numel() * 8 + w.n_tgt * 8 + 8), "ms_per_step": dt * 1e3,
               "api": "exx_apply_host (pinned host buffers; synchronous; wall clock)", "ex": ex_h}

    # ---- ACE tail and application, when the targets are the orbitals themselves ---
    ace = None
    if not args.no_ace and world == 1 and w.n_tgt == w.n_orb and w.tgt_start == 0:
        n = w.n_orb
        xi = torch.empty_like(vx)
        out = torch.empty_like(vx)

        def timed(fn, reps=5):
            for _ in range(2):
                fn()
            ts = []
            for _ in range(reps):
                flush.fill_(1)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream)
                fn()
                b.record(stream)
                torch.cuda.synchronize()
                ts.append(a.elapsed_time(b))
            return statistics.median(ts)

        info_box = []
        ms_build = timed(lambda: info_box.append(plan.ace_build(d_psi, vx, xi=xi, want_M=False, stream=stream)[2]))
        n_launch_build = plan.last_launch_count
        ms_apply = timed(lambda: plan.ace_apply(xi, d_psi, out=out, stream=stream))
        n_launch_apply = plan.last_launch_count
        fl_build = 2.0 * n * n * w.N + sum(2.0 * min(64, n - kb) * (kb + min(64, n - kb)) * w.N
                                           for kb in range(0, n, 64)) + n ** 3 / 3.0
        fl_apply = 4.0 * n * n * w.N
        ace = {"build_ms": ms_build, "apply_ms": ms_apply, "info": int(info_box[-1].item()),
               "build_tflops": fl_build / ms_build / 1e9, "apply_tflops": fl_apply / ms_apply / 1e9,
               "build_frac_of_dmma_peak": fl_build / ms_build / 1e9 / peak_dmma,
               "apply_frac_of_dmma_peak": fl_apply / ms_apply / 1e9 / peak_dmma,
               "apply_columns_per_s": n / (ms_apply * 1e-3), "launches": [int(n_launch_build), int(n_launch_apply)],
               "max_abs_err_ace_psi_minus_vx": float((out - vx).abs().max().item()),
               "max_abs_vx": float(vx.abs().max().item()),
               "what": "exx_ace_build(psi, W=vx) and exx_ace_apply(xi, psi): median of 5, L2 flushed, CUDA events; "
                       "share of the exchange step = (build_ms) / ms_per_step"}

    # ---- pair-symmetric apply: same result from about half the solves --------------
    symmetric = None
    if not args.no_ace and world == 1 and w.n_tgt == w.n_orb and w.tgt_start == 0:
        vx_s = torch.empty_like(vx)
        n_c_sym = args.nc_sym or min(n_c, 4 * w.n_orb)
        for _ in range(2):
            plan.apply_symmetric(d_psi, d_occ, vx=vx_s, n_c=n_c_sym, stream=stream)
        ts = []
        for _ in range(min(args.steps, 5)):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            _, _, ex_s = plan.apply_symmetric(d_psi, d_occ, vx=vx_s, n_c=n_c_sym, stream=stream)
            b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        ms_s = statistics.median(ts)
        executed = plan.last_solve_count
        symmetric = {"ms_per_step": ms_s, "n_c": n_c_sym, "executed_solves_per_step": int(executed),
                     "executed_solves_per_s": executed / (ms_s * 1e-3),
                     "pair_equivalent_solves_per_s": w.pair_solves / (ms_s * 1e-3),
                     "applies_per_s": w.n_tgt / (ms_s * 1e-3), "speedup_vs_full": ms_per_step / ms_s,
                     "step_frac_executed": executed * w.flops_per_solve / (ms_s * 1e-3) / 1e12 / peak_dmma,
                     "E_x": float(ex_s.item()),
                     "max_rel_diff_vs_full": float(((vx_s - vx).abs().max() / vx.abs().max()).item()),
                     "what": "exx_apply_symmetric: only pairs j <= k solved; roofline credit only for executed solves"}

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        cpu_baseline, _, _ = time_oracle(w, psi.cpu(), occ.cpu(), tgt.cpu(), occ_t.cpu(), args.cpu_seconds)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, n_c, {"parallelism": f"targets sharded over {world} rank(s), orbitals replicated"}),
            "applies_per_s": world * w.n_tgt / (ms_per_step * 1e-3), "E_x": ex_val,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches_per_step * args.steps),
            "roofline": roofline, "cpu_baseline": cpu_baseline, "ace": ace, "symmetric": symmetric}
    print(json.dumps(line), flush=True)
    plan.close()
    if world > 1:
        dist.destroy_process_group()


def run_bloch(args):
    """One (k,q) pair of the complex variant on the config's grid and orbital count: phases pi/2, pi/3, pi/5 on the
    periodic axes, complex orbitals from workloads.make_complex_orbitals.  Roofline credit = executed real flops:
    per pass 2*N*n per plane product, 4 plane products on a complex axis (P and Q over two planes), 2 on a real one."""
    import math
    from paper_2501_16572_b200 import exx
    import __graft_entry__ as ge
    ge.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    w = workload_from_args(args)
    n_c = args.nc or (512 if w.N <= 200000 else 256)
    theta = tuple(t if b == wl.PERIODIC else 0.0 for t, b in zip((math.pi / 2, math.pi / 3, math.pi / 5), w.bc))
    psi = wl.make_complex_orbitals(w, dev if w.cfg >= 4 else "cpu").to(dev)
    occ = torch.from_numpy(wl.occupations(w)).to(dev)
    tgt = psi[w.tgt_start:w.tgt_start + w.n_tgt]
    plan = exx.Plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega, max_batch=max(128, n_c), device=0, theta=theta)
    plan.set_variant(args.variant)
    vx = torch.empty_like(tgt)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def step():
        return plan.apply_bloch(psi, occ, tgt, vx=vx, n_c=n_c, stream=stream)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    launches = plan.last_launch_count
    sampler = ClockSampler(0)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for e0, e1 in ev:
        flush.fill_(1)
        e0.record(stream)
        _, e_k = step()
        e1.record(stream)
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = sum(a.elapsed_time(b) for a, b in ev) / args.steps
    peak = exx.probe_fp64_peak(1, 0, 1.5)
    plan.set_profiling(True)
    flush.fill_(1)
    step()
    prof = plan.get_profile()
    plan.set_profiling(False)
    flops = sum(2 * (4 if t != 0.0 else 2) * 2.0 * w.N * n for t, n in zip(theta, (w.nx, w.ny, w.nz))) * w.pair_solves
    mp_ms = prof["mode_product"][0]
    line = {"metric": "bloch_pair_solves_per_s", "value": w.pair_solves / (ms * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128 (two f64 planes)", "data": "synthetic",
            "config": config_dict(w, n_c, {"theta": list(theta), "variant": "Bloch-periodic complex (one k-q pair)"}),
            "clocks": clocks, "gpu_launches": int(launches * args.steps), "e_k0": float(e_k[0].item()),
            "roofline": {"bound": "tensor", "kernel": "k_mode_t (real and imaginary part of V) + k_combine",
                         "achieved": flops / (mp_ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                         "frac": flops / (mp_ms * 1e-3) / 1e12 / peak,
                         "step_frac": flops / (ms * 1e-3) / 1e12 / peak, "flops_per_step": flops,
                         "class_ms_per_step": {k: v[0] for k, v in prof.items()},
                         "note": "mode_product class includes the combine kernels; executed real flops (4x a real solve on complex axes)"}}
    print(json.dumps(line), flush=True)
    plan.close()


def run_solver_sweep(args):
    """The paper's Fig. 1 (time per linear system against the batch size n_c) and Fig. 2 (batch solver, GPU against
    CPU) in shape, on the config's grid: seeded N(0,1) right-hand sides, exx_poisson_solve,
    CUDA events, median of 5 after 2 warm-ups; n_c = 1 is the non-batch limit (Eq. 8: one system per set of
    products).  The CPU column is the oracle's poisson_solve (numpy) on batches of 20 (the paper's n_c)."""
    from paper_2501_16572_b200 import exx
    import __graft_entry__ as ge
    ge.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dev = torch.device("cuda", 0)
    w = workload_from_args(args)
    n_rhs = int(max(32, min(512, (3 << 30) // (w.N * 8))))
    rhs = wl.make_rhs(w, n_rhs, dev)
    out = torch.empty_like(rhs)
    plan = exx.Plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega, max_batch=512, device=0)
    peak = exx.probe_fp64_peak(1, 0, 1.0)
    stream = torch.cuda.current_stream(dev)
    rows = []
    for n_c in (1, 2, 4, 8, 16, 20, 32, 64, 128, 256, 512):
        if n_c > n_rhs:
            break
        m = n_rhs if n_c >= 16 else max(n_c, min(n_rhs, 16 * n_c))     # fewer systems for the tiny batches
        for _ in range(2):
            plan.poisson_solve(rhs[:m], out=out[:m], n_c=n_c, stream=stream)
        ts = []
        for _ in range(5):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            plan.poisson_solve(rhs[:m], out=out[:m], n_c=n_c, stream=stream)
            b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        ms = statistics.median(ts)
        rows.append({"n_c": n_c, "systems": m, "us_per_solve": 1e3 * ms / m, "solves_per_s": m / (ms * 1e-3),
                     "frac_of_dmma_peak": m * w.flops_per_solve / (ms * 1e-3) / 1e12 / peak})
    from oracle import exx_oracle as orc   # cpu_baseline leg
    oplan = orc.make_plan(w.nx, w.ny, w.nz, w.h, w.bc, w.order, w.omega)
    c = rhs[:20].cpu().numpy()
    orc.poisson_solve(oplan, c[:2])
    t0 = time.perf_counter()
    reps = 0
    while time.perf_counter() - t0 < min(args.cpu_seconds, 10.0):
        orc.poisson_solve(oplan, c)
        reps += 1
    cpu_us = 1e6 * (time.perf_counter() - t0) / (20 * reps)
    best = min(rows, key=lambda r: r["us_per_solve"])
    print(json.dumps({"metric": "poisson_solve_sweep", "config": config_dict(w, 0), "peak_tflops": peak, "rows": rows,
                      "speedup_batch_vs_nc1": rows[0]["us_per_solve"] / best["us_per_solve"], "best_n_c": best["n_c"],
                      "cpu_baseline": {"us_per_solve": cpu_us, "cores": _oracle_threads(), "kind": "oracle",
                                       "sample": f"oracle poisson_solve, batches of 20, {reps} repetitions"},
                      "gpu_over_cpu_at_nc20": cpu_us / next(r["us_per_solve"] for r in rows if r["n_c"] == 20)}), flush=True)
    plan.close()


def main():
    args = parse_args()
    if args.solver_sweep and args.impl != "reference":
        run_solver_sweep(args)
    elif args.bloch and args.impl != "reference":
        run_bloch(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
