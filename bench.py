#!/usr/bin/env python
"""bench.py -- one JSON line for the exact-exchange hot path (BASELINE.json metric: Poisson solves/s).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--nc n_c] [--impl reference]

A "step" is one full exchange apply (all SURVEY 8(a) rows: pair density, 3+3 mode products with the
eigen-space multiply, accumulate, energy) of one BASELINE.json config over synthetic orbitals.

Default workload: BASELINE.json configs[4] (120^3 HSE bulk, 3,200 orbitals = 44 GB, 128 targets, 409,600 pair solves
per step) -- the largest single-GPU configuration, the stand-in for the paper's 6,000-electron case.  The same line
carries `roofline` (FP64 tensor pipe, measured live), `e2e` (exx_apply_host from host buffers, the orbitals streamed
in blocks), `cpu_baseline` (the oracle on a bounded sample) and, as extra objects, short measurements of configs 2-4
(`configs`) and the batch-size sweep of config 4 (`sweep_cfg4`, BASELINE.json configs[3], the paper's Fig. 1 in shape).

N > 1 (torchrun): targets are sharded across ranks, orbitals replicated; the one collective of the path (all-reduce
of the per-target energies, sharding.reduce_energy) is inside the timed region; rank 0 prints the line.
--scaling weak (default): every rank applies Vx to its own block of n_tgt targets; --scaling strong: the config's
n_tgt targets are split over the ranks.
"""
from __future__ import annotations

import argparse
import csv
import glob
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

METRIC = "poisson_pair_solves_per_s"
UNIT = "solves/s"
DEFAULT_CONFIG = 5
DEFAULT_STEPS = {1: 20, 2: 20, 3: 10, 4: 5, 5: 3}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=0, help="timed steps (0 = a per-config default that finishes in minutes)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=DEFAULT_CONFIG,
                    help="BASELINE.json config number (1-based); default 5 = configs[4], the largest single-GPU one")
    ap.add_argument("--nc", type=int, default=0, help="right-hand sides per batch (0 = workload default)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="process-group backend for --gpus N > 1.  nccl (default): one rank per GPU.  gloo: a DEBUG mode that "
                         "lets several ranks share the GPUs present (rank r uses cuda:(r mod device_count)), so the whole "
                         "multi-rank branch can be executed on a one-GPU box; its throughput is not a scaling number and "
                         "the line says so")
    ap.add_argument("--variant", type=int, default=0, help="0 = DMMA path (default), 1 = plain-kernel cross-check variant")
    ap.add_argument("--n-orb", type=int, default=0, help="override orbital count (debug; invalidates the headline)")
    ap.add_argument("--n-tgt", type=int, default=0)
    ap.add_argument("--fusion", type=int, default=-1,
                    help="exx_plan_set_fusion mask (measurement hook; -1 = library default 15: fused z pass, fused "
                         "x-backward + accumulate, half-chunk y tiles, reflection-adapted eigenbases)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the configs 2-4 / sweep_cfg4 extra objects")
    ap.add_argument("--solver-sweep", action="store_true",
                    help="bare exx_poisson_solve over n_c = 1..512 on the config's grid (the paper's Figs. 1-2 in shape)")
    ap.add_argument("--bloch", action="store_true",
                    help="measure the Bloch-periodic complex variant (SURVEY 8(f) NEXT-3) on the config's grid instead")
    ap.add_argument("--nc-sym", type=int, default=0,
                    help="batch size of the pair-symmetric apply (0 = min(n_c, 4 n_orb): larger rectangles waste more "
                         "j > k pairs inside their diagonal blocks)")
    ap.add_argument("--no-ace", action="store_true", help="skip the ACE / pair-symmetric measurements (SURVEY 8(f) NEXT-1/2)")
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="target CPU time of the oracle sample")
    args = ap.parse_args()
    if args.steps <= 0:
        args.steps = DEFAULT_STEPS.get(args.config, 5)
    return args


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
         "flops_per_solve": w.flops_per_solve,
         # one text for both arms, so that their `config` objects compare equal
         "l2": "B200 arm: flushed between timed steps (256 MiB write outside the event pair); reference arm: n/a (CPU)"}
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


def oracle_sample_workload(w: wl.Workload) -> wl.Workload:
    """The bounded sample the oracle is timed on: the config's own grid, operator and input recipe with at most 64
    (grids up to 500k points) / 16 (larger) host-generated orbitals, all of them targets.  The cost of a pair solve
    does not depend on the orbital count, so solves/s on the sample is the oracle's rate on the workload."""
    m = min(w.n_orb, 64 if w.N <= 500_000 else 16)
    return wl.scaled(w, m, m, 0)


def time_oracle(w: wl.Workload, budget_s: float, steps: int = 1, warmup: int = 0):
    """Oracle exx_apply on the bounded sample: all sample orbitals against the first n_s sample targets, n_s sized
    from a one-target calibration so that one step takes about `budget_s` seconds of CPU."""
    from oracle import exx_oracle as orc   # the one place bench.py executes oracle/ (cpu_baseline / --impl reference)
    ws = oracle_sample_workload(w)
    psi, occ, tgt, occ_t = wl.make_inputs(ws, "cpu")
    plan = orc.make_plan(ws.nx, ws.ny, ws.nz, ws.h, ws.bc, ws.order, ws.omega)
    psi_n, occ_n, tgt_n, occ_t_n = psi.numpy(), occ.numpy(), tgt.numpy(), occ_t.numpy()
    t0 = time.perf_counter()
    orc.exx_apply(plan, psi_n, occ_n, tgt_n[:1], occ_t_n[:1])
    t1 = time.perf_counter() - t0
    n_s = int(max(1, min(ws.n_tgt, budget_s / max(t1, 1e-6))))
    times = []
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        orc.exx_apply(plan, psi_n, occ_n, tgt_n[:n_s], occ_t_n[:n_s])
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
    dt = sum(times) / len(times)
    solves = ws.n_orb * n_s
    return {"value": solves / dt, "unit": UNIT, "cores": _oracle_threads(), "kind": "oracle",
            "sample": f"oracle/exx_oracle.exx_apply (numpy FP64) on the grid, operator and input recipe of {w.name} with "
                      f"{ws.n_orb} host-generated orbitals x {n_s} targets = {solves} pair solves, {dt:.2f} s per step "
                      f"(the workload itself: {w.n_orb} x {w.n_tgt} = {w.pair_solves})"}, dt, solves


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = workload_from_args(args)
    # exactly the K timed and W warm-up steps asked for; each step is a bounded sample of the workload sized so that the
    # whole run ends within a few minutes (about 150 s of oracle time in total)
    steps = max(1, args.steps)
    warmup = max(0, args.warmup)
    budget = min(args.cpu_seconds, 150.0 / (steps + warmup + 1))
    cb, dt, solves = time_oracle(w, budget, steps=steps, warmup=warmup)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": args.scaling, "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, args.nc or w.default_nc),
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

    def __init__(self, index: int, period_ms: int = 20):
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", str(period_ms)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            text, _ = self.proc.communicate(timeout=10)
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


def load_ncu_traffic():
    """Per-kernel dram bytes per launch from the committed `ncu --set full` captures: the newest
    profiles/r*_ncu_traffic.csv (columns cfg,n_c,kernel,dram_read_bytes,dram_write_bytes,...).
    {(cfg, n_c): {kernel base name: bytes}}; shapes that were not captured report null."""
    out, name = {}, None
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_ncu_traffic.csv")))
    if not files:
        return out, name
    name = os.path.basename(files[-1])
    with open(files[-1], newline="") as fh:
        for row in csv.DictReader(r for r in fh if not r.startswith("#")):
            try:
                key = (int(row["cfg"]), int(row["n_c"]))
                base = row["kernel"].split("<")[0]
                out.setdefault(key, {})[base] = float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
            except (KeyError, ValueError):
                continue
    return out, name


def hbm_peak():
    """Measured copy bandwidth (GB/s) from the driver-written MEASURED_PEAKS.json, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "of measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"


# Algorithmic HBM bytes per grid point and pair solve: SURVEY.md 8(d) counts 48 (its three-fused-pass structure: two
# round trips of the batch between the passes plus one more pass's worth for psi/tgt/vx tiles).  The five-pass structure
# this library runs moves 64 + 16/nk + 24/nj (pass 1 writes the batch, passes 2-4 read and write it, pass 5
# reads it).  The HBM leg of the step roofline uses the survey's 48; the fraction against the structure's own 64 is
# reported beside it (`frac_vs_structure_bytes`), so that "how close to the roofline" and "how close to what this design
# can reach" are both in the line.
ALG_BYTES_PER_POINT = 48.0
STRUCTURE_BYTES_PER_POINT = 64.0


def step_roofline(flops_exec_per_solve: float, N: int, peak_tflops: float, us_per_solve: float,
                  flops_dense_per_solve: float | None = None) -> dict:
    """Whole-step roofline: the slower of (executed FP64 operations / DMMA peak) and (SURVEY.md 8(d)'s algorithmic bytes /
    copy bandwidth).  `frac` = `frac_vs_survey_bytes` uses the survey's 48 B per point; `frac_vs_structure_bytes` the 64 B
    of the five-pass structure; `frac_dense_count` credits the tensor leg with the dense algorithmic operations
    4 N (nx+ny+nz) of SURVEY.md 8(d) (above 1 where the reflection-adapted bases halve the executed ones)."""
    hbm, src = hbm_peak()
    t_tensor = flops_exec_per_solve / (peak_tflops * 1e12) * 1e6
    t_hbm = ALG_BYTES_PER_POINT * N / (hbm * 1e9) * 1e6
    t_hbm_structure = STRUCTURE_BYTES_PER_POINT * N / (hbm * 1e9) * 1e6
    bound = "tensor" if t_tensor >= t_hbm else "hbm"
    out = {"bound": bound, "us_per_solve_tensor": t_tensor, "us_per_solve_hbm": t_hbm, "us_per_solve_measured": us_per_solve,
           "frac": max(t_tensor, t_hbm) / us_per_solve, "frac_vs_survey_bytes": max(t_tensor, t_hbm) / us_per_solve,
           "frac_vs_structure_bytes": max(t_tensor, t_hbm_structure) / us_per_solve,
           "us_per_solve_hbm_structure": t_hbm_structure, "hbm_peak_gbs": hbm, "hbm_peak_source": src,
           "algorithmic_bytes_per_solve": ALG_BYTES_PER_POINT * N, "algorithmic_bytes_per_point": ALG_BYTES_PER_POINT,
           "structure_bytes_per_point": STRUCTURE_BYTES_PER_POINT}
    if flops_dense_per_solve:
        t_dense = flops_dense_per_solve / (peak_tflops * 1e12) * 1e6
        out["frac_dense_count"] = max(t_dense, t_hbm) / us_per_solve
    return out


def timed_apply(step, steps: int, warmup: int, flush, stream, barrier=None):
    """`warmup` untimed steps, then exactly `steps` steps, each inside its own CUDA-event pair on `stream` with an L2
    flush (256 MiB write) before it; returns the summed milliseconds and the last step's result."""
    res = None
    for _ in range(warmup):
        res = step()
    torch.cuda.synchronize()
    if barrier:
        barrier()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for e0, e1 in ev:
        flush.fill_(1)             # evict L2 between timed steps (outside the event pair)
        e0.record(stream)
        res = step()
        e1.record(stream)
    torch.cuda.synchronize()
    if barrier:
        barrier()
    return sum(e0.elapsed_time(e1) for e0, e1 in ev), res


KERNEL_OF_PASS = {"x_forward": ("k_mode_xf_sym", "k_mode_t<X, TWO>"), "y_forward": ("k_mode_lf_sym", "k_mode_t<L>"),
                  "z": ("k_mode_zz_sym", "k_mode_zz"), "z_backward": ("k_mode_t<L, TWO>", "k_mode_t<L, TWO>"),
                  "y_backward": ("k_mode_lb_sym", "k_mode_t<L>"), "x_backward": ("k_mode_xacc_sym", "k_mode_xacc"),
                  "x_backward_orbital_side": ("k_mode_xacc_sym", "k_mode_xacc_sym")}


def instrumented(plan, step, flush, prof_steps: int, flops_step: float, peak: float, solves_step: int, dense_axis_flops):
    """Per-kernel durations from separate instrumented steps (a CUDA-event pair around every launch on the caller's
    stream; this defeats the overlap of consecutive launches, so these steps are slightly slower than the timed ones).
    Returns the mode-product class's achieved TFLOP/s, the per-class table and the per-kernel table (one kernel per pass
    of a batch, each with its executed FP64 operations / its summed launch time against the DMMA peak)."""
    plan.set_profiling(True)
    for _ in range(prof_steps):
        flush.fill_(1)
        step()
    prof = plan.get_profile()
    passes = plan.get_profile_passes()
    plan.set_profiling(False)
    mp_ms, mp_cnt = prof["mode_product"]
    all_ms = sum(v[0] for v in prof.values())
    achieved = flops_step * prof_steps / (mp_ms * 1e-3) / 1e12 if mp_ms > 0 else 0.0
    kernels = {}
    for name, (ms, cnt, fl) in passes.items():
        dense = dense_axis_flops[name[0]] * (2 if name == "z" and "z_backward" not in passes else 1)
        sym = fl < dense * (1 - 1e-9)
        tf = fl * solves_step * prof_steps / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
        kernels[name] = {"kernel": KERNEL_OF_PASS[name][0 if sym else 1], "launches_per_step": cnt // prof_steps,
                         "avg_launch_ms": ms / max(cnt, 1), "ms_per_step": ms / prof_steps,
                         "share_of_step": ms / all_ms if all_ms > 0 else None, "executed_flops_per_solve": fl,
                         "dense_flops_per_solve": dense, "achieved_tflops": tf, "frac_of_dmma_peak": tf / peak,
                         "frac_dense_count": tf / peak * dense / fl if fl > 0 else None}
    return {"achieved": achieved, "frac": achieved / peak, "avg_launch_ms": mp_ms / max(mp_cnt, 1),
            "launches": mp_cnt // prof_steps, "share_of_step": mp_ms / all_ms if all_ms > 0 else None,
            "class_ms_per_step": {k: v[0] / prof_steps for k, v in prof.items()}, "kernels": kernels}


def measure_extra(exx, cfg: int, dev, local: int, peak: float, flush, stream, n_tgt: int = 0, n_c: int = 0,
                  steps: int = 3, want_ace: bool = False, psi=None):
    """A short measurement of another BASELINE.json config (same method as the headline: L2 flush, CUDA events),
    optionally on a reduced target block (stated in the result)."""
    w0 = wl.WORKLOADS[cfg]
    w = w0 if not n_tgt or n_tgt >= w0.n_tgt else wl.scaled(w0, w0.n_orb, n_tgt, w0.tgt_start)
    n_c = n_c or w.default_nc
    if psi is None:
        psi, occ, _, _ = wl.make_inputs(w, dev)
    else:
        occ = torch.from_numpy(wl.occupations(w)).to(dev)
    tgt = psi[w.tgt_start:w.tgt_start + w.n_tgt]
    occ_t = occ[w.tgt_start:w.tgt_start + w.n_tgt]
    plan = exx.Plan.for_workload(w, max_batch=max(128, n_c), device=local)
    vx = torch.empty((w.n_tgt, w.nz, w.ny, w.nx), dtype=torch.float64, device=dev)

    def step():
        return plan.apply(psi, occ, tgt, occ_t, vx=vx, n_c=n_c, stream=stream)

    total_ms, (_, _, ex) = timed_apply(step, steps, 2, flush, stream)
    ms = total_ms / steps
    flops = w.pair_solves * plan.executed_flops_per_solve   # executed FP64 operations (<= the dense algorithmic count)
    out = {"workload": f"BASELINE.json configs[{cfg - 1}]: {w0.name}", "n_occ": w.n_orb, "n_tgt": w.n_tgt,
           "targets": "all" if w.n_tgt == w0.n_tgt else f"reduced block: {w.n_tgt} of {w0.n_tgt} targets from {w.tgt_start}",
           "n_c": n_c, "pair_solves_per_step": w.pair_solves, "steps": steps, "ms_per_step": ms,
           "value": w.pair_solves / (ms * 1e-3), "unit": UNIT, "applies_per_s": w.n_tgt / (ms * 1e-3),
           "step_frac": flops / (ms * 1e-3) / 1e12 / peak,
           "step_roofline": step_roofline(plan.executed_flops_per_solve, w.N, peak, ms * 1e3 / w.pair_solves, w.flops_per_solve),
           "executed_over_algorithmic_flops": plan.executed_flops_per_solve / w.flops_per_solve, "E_x": float(ex.item()),
           "launches_per_step": plan.last_launch_count}
    if want_ace and w.n_tgt == w.n_orb and w.tgt_start == 0:
        out.update(measure_ace_and_symmetric(plan, w, psi, occ, vx, ms, n_c, 0, peak, flush, stream, steps))
    plan.close()
    return out, psi


def measure_ace_and_symmetric(plan, w, d_psi, d_occ, vx, ms_per_step, n_c, nc_sym, peak_dmma, flush, stream, steps):
    """SURVEY 8(f) NEXT-1 (ACE tail and application on the step's own vx) and NEXT-2 (pair-symmetric apply)."""
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
           "what": "exx_ace_build(psi, W=vx) and exx_ace_apply(xi, psi): median of 5, L2 flushed, CUDA events"}
    vx_s = torch.empty_like(vx)
    n_c_sym = nc_sym or min(n_c, 4 * w.n_orb)
    for _ in range(2):
        plan.apply_symmetric(d_psi, d_occ, vx=vx_s, n_c=n_c_sym, stream=stream)
    ts = []
    for _ in range(min(steps, 5)):
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        _, _, ex_s = plan.apply_symmetric(d_psi, d_occ, vx=vx_s, n_c=n_c_sym, stream=stream)
        b.record(stream)
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    ms_s = statistics.median(ts)
    executed = plan.last_solve_count
    # executed FP64 operations of one executed solve of the pair-symmetric apply: the x-backward product runs once per
    # side of the two-sided accumulate
    flops_exec_sym = plan.executed_flops_per_symmetric_solve
    symmetric = {"ms_per_step": ms_s, "n_c": n_c_sym, "executed_solves_per_step": int(executed),
                 "executed_solves_per_s": executed / (ms_s * 1e-3),
                 "pair_equivalent_solves_per_s": w.pair_solves / (ms_s * 1e-3),
                 "applies_per_s": w.n_tgt / (ms_s * 1e-3), "speedup_vs_full": ms_per_step / ms_s,
                 "step_frac_executed": executed * flops_exec_sym / (ms_s * 1e-3) / 1e12 / peak_dmma,
                 "E_x": float(ex_s.item()),
                 "max_rel_diff_vs_full": float(((vx_s - vx).abs().max() / vx.abs().max()).item()),
                 "what": "exx_apply_symmetric: only pairs j <= k solved; roofline credit only for executed solves"}
    return {"ace": ace, "symmetric": symmetric}


def run_b200(args):
    import torch.distributed as dist
    from paper_2501_16572_b200 import exx, sharding

    t_start = time.perf_counter()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    if args.backend == "gloo":      # debug: ranks may share a GPU (NCCL refuses two ranks on one device, gloo does not)
        local = local % torch.cuda.device_count()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        if args.backend == "gloo":
            dist.init_process_group("gloo")
        else:
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
    psi, occ, _, _ = wl.make_inputs(w, gen_dev)
    d_psi, d_occ = psi.to(dev), occ.to(dev)
    del psi
    t_gen = time.perf_counter() - t_start
    # weak scaling: rank r applies Vx to n_tgt targets starting at tgt_start + r*n_tgt (wrapping);
    # strong scaling: the config's n_tgt targets are split over the ranks (sharding.shard_targets)
    if args.scaling == "strong":
        k0, k1 = sharding.shard_targets(w.n_tgt, rank, world)
        d_tgt = d_psi[w.tgt_start + k0:w.tgt_start + k1]
        d_occ_t = d_occ[w.tgt_start + k0:w.tgt_start + k1]
        n_tgt_union, k_off = w.n_tgt, k0
    elif world == 1:
        d_tgt = d_psi[w.tgt_start:w.tgt_start + w.n_tgt]
        d_occ_t = d_occ[w.tgt_start:w.tgt_start + w.n_tgt]
        n_tgt_union, k_off = w.n_tgt, 0
    else:
        idx = sharding.weak_scaling_targets(w.tgt_start, w.n_tgt, w.n_orb, rank).to(dev)
        d_tgt = d_psi[idx].contiguous()
        d_occ_t = d_occ[idx].contiguous()
        n_tgt_union, k_off = world * w.n_tgt, rank * w.n_tgt
    n_tgt_local = d_tgt.shape[0]
    solves_all_ranks = w.n_orb * n_tgt_union

    plan = exx.Plan.for_workload(w, max_batch=max(128, n_c), device=local)
    plan.set_variant(args.variant)
    if args.fusion >= 0:
        plan.set_fusion(args.fusion)
    vx = torch.empty((n_tgt_local, w.nz, w.ny, w.nx), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream(dev)

    def step_local():
        return plan.apply(d_psi, d_occ, d_tgt, d_occ_t, vx=vx, n_c=n_c, stream=stream)

    def step():
        vx_, e_k, ex = step_local()
        if world > 1:   # the path's one collective: per-target energies of the union, E_x of the union
            e_k, ex = sharding.reduce_energy(e_k, d_occ_t, k_off, n_tgt_union)
        return vx_, e_k, ex

    warmup = max(args.warmup, 3)
    period = 20 if w.pair_solves * w.flops_per_solve < 5e13 else 250
    sampler = ClockSampler(local, period) if rank == 0 else None
    total_ms, (_, e_k, ex) = timed_apply(step, args.steps, warmup, flush, stream, dist.barrier if world > 1 else None)
    launches_per_step = plan.last_launch_count
    t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms = float(t.item())
    clocks = sampler.stop() if sampler else None
    ms_per_step = total_ms / args.steps
    value = solves_all_ranks / (ms_per_step * 1e-3)
    ex_val = float(ex.item())

    # every rank has finished its collectives: tear the process group down together, rank 0 carries on alone with the
    # single-GPU instrumentation (no collective after this point)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return

    # ---- roofline of the dominant kernel class (mode products on the FP64 tensor pipe) -----------------
    peak_dmma = exx.probe_fp64_peak(1, local, 1.5)
    peak_dfma = exx.probe_fp64_peak(0, local, 0.5)
    # Roofline in EXECUTED FP64 operations: the dense algorithmic count 4 N (nx+ny+nz) per pair solve
    # unless an axis runs on the reflection-adapted basis, whose products need about half of it.  With
    # executed operations the fraction cannot exceed 1; `algorithmic_tflops` is the same time credited with the dense count.
    flops_exec = plan.executed_flops_per_solve
    flops_step = w.n_orb * n_tgt_local * flops_exec
    prof_steps = 1 if ms_per_step > 2000 else min(2, args.steps)
    dense_axis = {"x": 2.0 * w.N * w.nx, "y": 2.0 * w.N * w.ny, "z": 2.0 * w.N * w.nz}
    # (rank 0 alone from here on: the instrumented steps run the local apply, without the collective)
    inst = instrumented(plan, step_local, flush, prof_steps, flops_step, peak_dmma, w.n_orb * n_tgt_local, dense_axis)
    # the dominant kernel: the pass with the largest share of the step
    dom_pass, dom = max(inst["kernels"].items(), key=lambda kv: kv[1]["ms_per_step"]) if inst["kernels"] else (None, None)
    traffic_tab, traffic_file = load_ncu_traffic()
    traffic = None
    if dom is not None:
        traffic = traffic_tab.get((w.cfg, n_c), {}).get(dom["kernel"].split("<")[0])
    # right-hand sides of one launch of the dominant kernel: the step's pair solves over its launches (the batches are
    # nj x nk <= n_c, the last target block smaller), not n_c itself
    n_batch = (w.n_orb * n_tgt_local / dom["launches_per_step"]) if dom is not None and dom["launches_per_step"] else \
        min(n_c, w.n_orb * n_tgt_local)
    us_per_solve = ms_per_step * 1e3 / (w.n_orb * n_tgt_local)
    roofline = {"bound": "tensor",
                "kernel": (f"{dom['kernel']} ({dom_pass} pass of a batch; FP64 mma.sync -> DMMA.8x8x4, operands by TMA)"
                           if dom is not None else "mode products"),
                "achieved": dom["achieved_tflops"] if dom is not None else inst["achieved"], "peak": peak_dmma,
                "unit": "TFLOP/s", "frac": dom["frac_of_dmma_peak"] if dom is not None else inst["frac"],
                "frac_executed_count": dom["frac_of_dmma_peak"] if dom is not None else inst["frac"],
                "frac_dense_count": dom["frac_dense_count"] if dom is not None else None,
                "traffic": traffic,
                "traffic_note": (f"dram read + write bytes per launch of this kernel from the committed ncu --set full capture "
                                 f"profiles/{traffic_file}" if traffic else "no committed ncu capture for this (config, n_c)")
                                + f"; algorithmic bytes of an in-place pass over one launch's {n_batch:.1f} right-hand sides (average over "
                                  f"the step's batches) = {2 * 8 * w.N * n_batch:.4g}",
                "achieved_note": "FP64 operations this kernel EXECUTES per launch (exx_plan_get_profile_passes; the dense "
                                 "algorithmic count of its products would be higher where it runs on the reflection-adapted "
                                 "basis, DESIGN.md 6.9) / its average launch duration (CUDA events, live)",
                "peak_source": "measured live by this repo's own probe (exx_probe_fp64_peak, a register-resident DMMA issue "
                               "loop, 1.5 s): MEASURED_PEAKS.json has no FP64 entry and the profiling guide states no FP64 "
                               f"fallback; 148 SMs x 128 flop/clk x 1.965 GHz = 37.2; DFMA loop {peak_dfma:.2f} TF",
                "avg_launch_ms": dom["avg_launch_ms"] if dom is not None else inst["avg_launch_ms"],
                "launches": dom["launches_per_step"] if dom is not None else inst["launches"],
                "share_of_step": dom["share_of_step"] if dom is not None else inst["share_of_step"],
                "kernels": inst["kernels"],
                "all_mode_products": {"achieved": inst["achieved"], "frac": inst["frac"], "launches": inst["launches"],
                                      "avg_launch_ms": inst["avg_launch_ms"], "share_of_step": inst["share_of_step"]},
                "step_frac": flops_step / (ms_per_step * 1e-3) / 1e12 / peak_dmma,
                "step": step_roofline(flops_exec, w.N, peak_dmma, us_per_solve, w.flops_per_solve),
                "step_frac_dense_count": w.n_orb * n_tgt_local * w.flops_per_solve / (ms_per_step * 1e-3) / 1e12 / peak_dmma,
                "flops_per_solve_executed": flops_exec, "flops_per_solve_algorithmic": w.flops_per_solve,
                "executed_over_algorithmic_flops": flops_exec / w.flops_per_solve,
                "algorithmic_tflops_whole_step": w.n_orb * n_tgt_local * w.flops_per_solve / (ms_per_step * 1e-3) / 1e12,
                "flops_note": "achieved / frac (= frac_executed_count) / step_frac count the FP64 operations the kernels "
                              "execute (padding excluded): how busy the tensor pipe is.  frac_dense_count / "
                              "step_frac_dense_count credit the same time with SURVEY.md 8(d)'s dense algorithmic count "
                              "(2 N n per product): the reflection-adapted bases halve the executed operations, so these "
                              "exceed 1",
                "class_ms_per_step": inst["class_ms_per_step"],
                "measured": f"{prof_steps} separate instrumented step(s) (CUDA-event pair around every launch, caller's stream)"}
    if roofline["step"]["bound"] == "hbm" and dom is not None:
        # small grids (48^3): the five passes move more time through HBM than through the tensor pipe -- report the dominant
        # kernel against the copy bandwidth (algorithmic bytes of one in-place pass over a full batch), tensor numbers in "kernels"
        gbs = 2 * 8 * w.N * n_batch / (dom["avg_launch_ms"] * 1e-3) / 1e9
        roofline.update({"bound": "hbm", "achieved": gbs, "peak": roofline["step"]["hbm_peak_gbs"], "unit": "GB/s",
                         "frac": gbs / roofline["step"]["hbm_peak_gbs"],
                         "peak_source": roofline["step"]["hbm_peak_source"],
                         "achieved_note": "algorithmic bytes of one in-place pass over a full batch (2 x 8 x N x n_c) / this "
                                          "kernel's average launch duration (CUDA events, live)"})

    # ---- launch-bound steps (config 1: 64 solves in 7 launches): the same step replayed from a CUDA graph ----
    graph = None
    if world == 1 and ms_per_step < 1.0:
        try:
            side = torch.cuda.Stream()
            g = torch.cuda.CUDAGraph()
            side.wait_stream(stream)
            with torch.cuda.graph(g, stream=side):
                plan.apply(d_psi, d_occ, d_tgt, d_occ_t, vx=vx, n_c=n_c, stream=torch.cuda.current_stream())
            for _ in range(5):
                g.replay()
            torch.cuda.synchronize()
            reps = 200
            a_ev, b_ev = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_ev.record()
            for _ in range(reps):
                g.replay()
            b_ev.record()
            torch.cuda.synchronize()
            us = 1e3 * a_ev.elapsed_time(b_ev) / reps
            graph = {"us_per_step": us, "value": w.pair_solves / (us * 1e-6), "unit": UNIT, "replays": reps,
                     "what": "one exx_apply captured in a CUDA graph and replayed back to back (no L2 flush: the step is "
                             "launch bound, its data L2-resident); eager, with a flush between steps: ms_per_step"}
        except Exception as exc:   # capture is a measurement extra, never fatal
            graph = {"error": str(exc)[:200]}

    # ---- end to end through the C-ABI with host buffers (H2D + D2H inside the timed region) ------------
    e2e = None
    if not args.no_e2e and world == 1:
        e2e = measure_e2e(plan, w, d_psi, d_occ, n_c, ms_per_step)

    extra = {}
    if not args.no_ace and world == 1 and w.n_tgt == w.n_orb and w.tgt_start == 0:
        extra.update(measure_ace_and_symmetric(plan, w, d_psi, d_occ, vx, ms_per_step, n_c, args.nc_sym, peak_dmma,
                                               flush, stream, args.steps))
    plan.close()

    # ---- the other configs and the config-4 batch sweep, short runs (extra objects, not the headline) --
    if not args.no_extras and world == 1 and w.cfg == DEFAULT_CONFIG and not (args.n_orb or args.n_tgt):
        del d_psi, d_tgt, vx
        torch.cuda.empty_cache()
        configs = {}
        configs["cfg2"], _ = measure_extra(exx, 2, dev, local, peak_dmma, flush, stream, steps=10, want_ace=not args.no_ace)
        configs["cfg3"], _ = measure_extra(exx, 3, dev, local, peak_dmma, flush, stream, steps=3, want_ace=not args.no_ace)
        configs["cfg4"], psi4 = measure_extra(exx, 4, dev, local, peak_dmma, flush, stream, steps=2)   # all 256 targets
        sweep = []
        for nc in (16, 32, 64, 128, 256, 512):
            r, _ = measure_extra(exx, 4, dev, local, peak_dmma, flush, stream, n_tgt=8, n_c=nc, steps=3, psi=psi4)
            sweep.append({k: r[k] for k in ("n_c", "n_tgt", "pair_solves_per_step", "ms_per_step", "value", "step_frac")})
        del psi4
        torch.cuda.empty_cache()
        extra["configs"] = configs
        # SURVEY 8(f) NEXT-3 in the same line: the Bloch-periodic complex variant on config 2's grid (short run)
        try:
            bl = run_bloch(argparse.Namespace(config=2, nc=0, steps=5, warmup=3, variant=0, no_ace=True, n_orb=0, n_tgt=0),
                           emit=False)
            extra["bloch_cfg2"] = {"value": bl["value"], "unit": "complex pair solves/s", "ms_per_step": bl["ms_per_step"],
                                   "n_c": bl["config"]["n_c"], "theta": bl["config"]["theta"],
                                   "mode_products_frac_of_dmma_peak": bl["roofline"]["frac"],
                                   "step_frac": bl["roofline"]["step_frac"],
                                   "class_ms_per_step": bl["roofline"]["class_ms_per_step"],
                                   "what": "exx_apply_bloch, one (k,q) pair, 64 complex orbitals on 48^3; executed real flops"}
        except Exception as exc:   # an extra, never fatal for the headline
            extra["bloch_cfg2"] = {"error": str(exc)[:200]}
        extra["sweep_cfg4"] = {"what": "BASELINE.json configs[3] batch-size sweep (the paper's Fig. 1 in shape): all 1,536 "
                                       "orbitals against a reduced block of 8 targets (896..903), 3 timed steps each",
                               "unit": UNIT, "rows": sweep}

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        cpu_baseline, _, _ = time_oracle(w, args.cpu_seconds)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, n_c),
            "parallelism": f"targets sharded over {world} rank(s) ({args.scaling} scaling), orbitals replicated; one "
                           "all-reduce of the per-target energies",
            "pair_solves_all_ranks": solves_all_ranks,
            "backend": (args.backend if world > 1 else None) if args.backend == "nccl" else
                       f"gloo (DEBUG: {world} rank(s) on {torch.cuda.device_count()} GPU(s); not a scaling measurement)",
            "applies_per_s": n_tgt_union / (ms_per_step * 1e-3), "E_x": ex_val,
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches_per_step * args.steps * world),
            "roofline": roofline, "cpu_baseline": cpu_baseline,
            "vs_cpu_baseline": value / cpu_baseline["value"] if cpu_baseline else None, "cuda_graph": graph,
            "seconds": {"inputs": t_gen, "total": time.perf_counter() - t_start}}
    line.update(extra)
    print(json.dumps(line), flush=True)


def measure_e2e(plan, w, d_psi, d_occ, n_c, ms_per_step):
    """The same step through exx_apply_host: HOST buffers in, HOST results out, H2D of the orbitals (streamed in blocks,
    two resident at a time) and D2H of vx / e_k / E_x inside the timed region; wall clock around the synchronous call."""
    shape = tuple(d_psi.shape)
    pinned = True
    try:
        h_psi = torch.empty(shape, dtype=torch.float64, pin_memory=True)
    except RuntimeError:
        pinned = False
        h_psi = torch.empty(shape, dtype=torch.float64)
    chunk = max(1, (1 << 30) // (w.N * 8))
    for j0 in range(0, w.n_orb, chunk):      # the bytes the device path used, copied out in 1 GiB pieces
        h_psi[j0:j0 + chunk].copy_(d_psi[j0:j0 + chunk])
    h_occ = d_occ.cpu().contiguous()
    h_occ_t = h_occ[w.tgt_start:w.tgt_start + w.n_tgt].contiguous()
    try:
        h_vx = torch.empty((w.n_tgt, w.nz, w.ny, w.nx), dtype=torch.float64, pin_memory=pinned)
    except RuntimeError:
        h_vx = torch.empty((w.n_tgt, w.nz, w.ny, w.nx), dtype=torch.float64)
    k = int(max(2, min(5, 60e3 / max(ms_per_step, 1e-3))))
    wu = 1 if ms_per_step > 2000 else 2
    for _ in range(wu):
        plan.apply_host(h_psi, h_occ, tgt_start=w.tgt_start, n_tgt=w.n_tgt, occ_tgt=h_occ_t, vx=h_vx, n_c=n_c)
    t0 = time.perf_counter()
    for _ in range(k):
        _, _, ex_h = plan.apply_host(h_psi, h_occ, tgt_start=w.tgt_start, n_tgt=w.n_tgt, occ_tgt=h_occ_t,
                                     vx=h_vx, n_c=n_c)
    dt = (time.perf_counter() - t0) / k
    return {"value": w.pair_solves / dt, "unit": UNIT,
            "h2d_bytes_per_step": int((h_psi.numel() + w.n_tgt * w.N + h_occ.numel() + h_occ_t.numel()) * 8),
            "d2h_bytes_per_step": int(h_vx.numel() * 8 + w.n_tgt * 8 + 8), "ms_per_step": dt * 1e3,
            "steps": k, "warmup": wu,
            "api": "exx_apply_host (" + ("pinned" if pinned else "pageable: pinning failed on this box") +
                   " host buffers; orbitals uploaded in blocks while the previous block computes; synchronous; wall clock)",
            "ex": ex_h}


def run_bloch(args, emit=True):
    """One (k,q) pair of the complex variant on the config's grid and orbital count: phases pi/2, pi/3, pi/5 on the
    periodic axes, complex orbitals from workloads.make_complex_orbitals.  Roofline credit = executed real flops:
    per pass 2*N*n per plane product, 2 plane products per axis (axes with a phase run in their real form)."""
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

    sampler = ClockSampler(0)
    total_ms, (_, e_k) = timed_apply(step, args.steps, max(args.warmup, 3), flush, stream)
    launches = plan.last_launch_count
    clocks = sampler.stop()
    ms = total_ms / args.steps
    peak = exx.probe_fp64_peak(1, 0, 1.5)
    plan.set_profiling(True)
    flush.fill_(1)
    step()
    prof = plan.get_profile()
    plan.set_profiling(False)
    # an axis with a phase is held in its real form: like a real axis, one real product per plane and pass
    flops = sum(2 * 2 * 2.0 * w.N * n for n in (w.nx, w.ny, w.nz)) * w.pair_solves
    mp_ms = prof["mode_product"][0]
    line = {"metric": "bloch_pair_solves_per_s", "value": w.pair_solves / (ms * 1e-3), "unit": UNIT, "n_gpus": 1,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128 (two f64 planes)", "data": "synthetic",
            "config": config_dict(w, n_c, {"theta": list(theta), "variant": "Bloch-periodic complex (one k-q pair)"}),
            "clocks": clocks, "gpu_launches": int(launches * args.steps), "e_k0": float(e_k[0].item()),
            "roofline": {"bound": "tensor", "kernel": "k_mode_t (complex mode products)",
                         "achieved": flops / (mp_ms * 1e-3) / 1e12, "peak": peak, "unit": "TFLOP/s",
                         "frac": flops / (mp_ms * 1e-3) / 1e12 / peak,
                         "step_frac": flops / (ms * 1e-3) / 1e12 / peak, "flops_per_step": flops,
                         "class_ms_per_step": {k: v[0] for k, v in prof.items()},
                         "note": "executed real flops: 2x a dense real solve (two planes); axes with a phase run in their real form"}}
    # complex ACE tail and application on the step's own vx, targets = orbitals only
    if not args.no_ace and w.n_tgt == w.n_orb and w.tgt_start == 0:
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
        ms_build = timed(lambda: info_box.append(plan.ace_build_bloch(psi, vx, xi=xi, want_M=False, stream=stream)[2]))
        nl_build = plan.last_launch_count
        ms_apply = timed(lambda: plan.ace_apply_bloch(xi, psi, out=out, stream=stream))
        nl_apply = plan.last_launch_count
        # real flops of the embedded products: a complex Gram / expand is 4x the real one (2n x 2n over N)
        fl_build = 4 * (2.0 * n * n * w.N) + sum(4 * 2.0 * min(32, n - kb) * (kb + min(32, n - kb)) * w.N
                                                 for kb in range(0, n, 32))
        fl_apply = 4 * 4.0 * n * n * w.N
        line["ace_complex"] = {"build_ms": ms_build, "apply_ms": ms_apply, "info": int(info_box[-1].item()),
                               "build_frac_of_dmma_peak": fl_build / ms_build / 1e9 / peak,
                               "apply_frac_of_dmma_peak": fl_apply / ms_apply / 1e9 / peak,
                               "launches": [int(nl_build), int(nl_apply)],
                               "max_abs_err_ace_psi_minus_vx": float((out - vx).abs().max().item()),
                               "max_abs_vx": float(vx.abs().max().item()),
                               "what": "exx_ace_build_bloch(psi, W=vx) and exx_ace_apply_bloch(xi, psi): median of 5, L2 "
                                       "flushed, CUDA events; executed real flops (4x a real Gram / expand)"}
    plan.close()
    if emit:
        print(json.dumps(line), flush=True)
    return line


def run_solver_sweep(args):
    """The paper's Fig. 1 (time per linear system against the batch size n_c) and Fig. 2 (batch against non-batch
    solver, GPU against CPU) in shape, on the config's grid: seeded N(0,1) right-hand sides,
    exx_poisson_solve, CUDA events, median of 5 after 2 warm-ups.  `nonbatch_eq8` is the per-slice algorithm of Eq. 8
    (V1^T B_k V2 for every frontal slice, then the product with V3; exx_poisson_solve_nonbatch), one
    system at a time.  The CPU column is the oracle's poisson_solve (numpy) on batches of 20 (the paper's n_c)."""
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
    flops_exec = plan.executed_flops_per_solve
    peak = exx.probe_fp64_peak(1, 0, 1.0)
    stream = torch.cuda.current_stream(dev)

    def med(fn, reps=5):
        for _ in range(2):
            fn()
        ts = []
        for _ in range(reps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            fn()
            b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return statistics.median(ts)

    rows = []
    for n_c in (1, 2, 4, 8, 16, 20, 32, 64, 128, 256, 512):
        if n_c > n_rhs:
            break
        m = n_rhs if n_c >= 16 else max(n_c, min(n_rhs, 16 * n_c))     # fewer systems for the tiny batches
        ms = med(lambda: plan.poisson_solve(rhs[:m], out=out[:m], n_c=n_c, stream=stream))
        rows.append({"n_c": n_c, "systems": m, "us_per_solve": 1e3 * ms / m, "solves_per_s": m / (ms * 1e-3),
                     "frac_of_dmma_peak": m * flops_exec / (ms * 1e-3) / 1e12 / peak})
    nonbatch = None
    if hasattr(plan, "poisson_solve_nonbatch"):
        m = min(n_rhs, 16)
        ms = med(lambda: plan.poisson_solve_nonbatch(rhs[:m], out=out[:m], stream=stream))
        nonbatch = {"systems": m, "us_per_solve": 1e3 * ms / m, "solves_per_s": m / (ms * 1e-3),
                    "launches_per_system": plan.last_launch_count / m,
                    "what": "Eq. 8 (PAPER.md:74-78): one launch per frontal slice for V1^T B_k V2, one for the product "
                            "with V3, the multiplier, and the same back"}
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
                      "executed_over_algorithmic_flops": flops_exec / w.flops_per_solve,
                      "nonbatch_eq8": nonbatch,
                      "speedup_batch_vs_nc1": rows[0]["us_per_solve"] / best["us_per_solve"], "best_n_c": best["n_c"],
                      "speedup_batch_vs_nonbatch_eq8": nonbatch["us_per_solve"] / best["us_per_solve"] if nonbatch else None,
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
