#!/usr/bin/env python
"""bench.py -- particle-steps/s of the SPH hot path (NNPS + density + EOS + momentum + PC update) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl ours|reference]

One "step" = one predictor-corrector step of the whole hot path: fused update + cell
key -> counting sort -> cell offsets + permute -> summation density + EOS -> WCSPH acceleration, on one synthetic
workload.  Prints ONE JSON line (rank 0).

  value      device-resident throughput: inputs live in HBM, K calls of sph_pc_step(dt, 1) each bracketed by CUDA
             events on the context stream, L2 flushed (256 MiB write) between timed steps; max over ranks.
  e2e        the same metric through the C ABI with HOST (pinned) buffers: every step does sph_nnps_build(host
             arrays incl. a^n) + sph_pc_step(dt, 1) + sph_sync_state(host, incl. a^{n+1}); copies inside the timing.
  roofline   the dominant kernel (a pair loop: k_density searches + sums eq.3, k_accel_list replays its hit masks
             for eq.8-9): algorithmic flops per launch / its mean launch duration from CUDA event pairs recorded
             around every launch (sph_set_profiling) during a second pass of the same K steps.  bound = "alu"
             (plain FP32 pipes); peak = the FMA rate sph_fp32_probe measures in this run.
  cpu_baseline  the fp64 oracle (oracle/, as it stands, OpenMP over destinations) on this box's host cores.

N > 1: the path does not shard (north_star: one GPU) -> N independent replicas (seed + rank), no data-path
collective; value = particles of all ranks x K / max-over-ranks time ("scaling": "weak").
--impl reference times the oracle (the tier's reference arm) on a bounded sample of the same workload.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "particle_steps_per_sec"
UNIT = "particle-steps/s"
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965                 # B200_PROFILING.md "Nominal figures"
ALU_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_GHZ / 1e3      # 74.4 TFLOP/s if every issue slot were an FFMA


# ---------------------------------------------------------------------------------------------------------
# workloads (BASELINE.json configs)
# ---------------------------------------------------------------------------------------------------------
def make_workload(name: str, rank: int = 0, small: bool = False):
    from paper_1909_04504_b200 import workloads as W
    if name == "C1":
        return W.taylor_green_2d(seed=0 + 100 * rank)
    if name == "C2":
        return W.dam_break_2d()
    if name == "C3":
        return W.periodic_box_3d((64, 64, 64) if small else (128, 128, 128), seed=1 + 100 * rank, dx=1.0 / 128)
    if name == "C4":
        return W.dam_break_3d(dx=0.01 if small else 0.005)
    if name == "C5":
        return W.gaussian_mixture_3d(N=(1 << 20) if small else (1 << 24), seed=2 + 100 * rank)
    raise SystemExit(f"unknown workload {name}")


# Algorithmic flops per unit (FMA = 2, rsqrt/rcp = 1, compares/selects = 0).
def flops_per_test(dim: int, variable_h: bool) -> int:
    return (8 if dim == 3 else 5) + (3 if variable_h else 0)


def flops_per_pair(kind: str, kernel: str, dim: int, variable_h: bool, arho: bool) -> int:
    geom = 11 if dim == 3 else 8                     # d, r2, rsqrt, r, q
    varh = (6 if dim == 3 else 5) if variable_h else 0
    f = {"cubic": 5, "quintic": 16, "wendland_c2": 7}[kernel]
    df = {"cubic": 3, "quintic": 14, "wendland_c2": 6}[kernel]
    if kind == "density":
        return geom + varh + f + 3
    body = (30 if dim == 3 else 25)                  # grad scale, v_ij, v.r, Pi_ij, pressure terms, accumulate
    return geom + varh + df + body + (3 if arho else 0)


# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark(self):
        return time.time()

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows[-3:]]
        sm, smax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except Exception:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def ncu_traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload`, from the committed
    `ncu --set full` capture summarised in profiles/r1_dram_traffic.csv (kernel,workload,read_bytes,write_bytes),
    or None when no capture of that kernel/workload is committed."""
    path = os.path.join(ROOT, "profiles", "r1_dram_traffic.csv")
    try:
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and f[0] == kernel and f[1] == workload:
                return float(f[2]) + float(f[3])
    except OSError:
        pass
    return None


def aggregate(elapsed_ms: float, units: float, world: int):
    """max-over-ranks time and summed units (replicas): returns (ms, total_units).  gloo/nccl all_reduce."""
    if world <= 1:
        return elapsed_ms, units
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=dev)
    u = torch.tensor([units], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


# ---------------------------------------------------------------------------------------------------------
# reference arm: the oracle on host cores
# ---------------------------------------------------------------------------------------------------------
def oracle_steps(wl, steps: int, warmup: int, budget_s: float = None):
    """Times `steps` oracle PC steps (after the a^0 evaluation and `warmup` steps); with budget_s it stops after
    the first step that ends past the budget.  Returns (seconds, pairs, threads, steps done)."""
    from oracle import sph_oracle as O
    st = O.State(wl)
    O.evaluate(wl, st, wl.density_mode)
    move = "no position update" not in wl.note
    for _ in range(warmup):
        O.pc_step(wl, st, wl.dt, wl.density_mode, move=move)
    t0 = time.perf_counter()
    pairs = 0
    done = 0
    for _ in range(steps):
        pairs += O.pc_step(wl, st, wl.dt, wl.density_mode, move=move)
        done += 1
        if budget_s is not None and time.perf_counter() - t0 > budget_s:
            break
    return time.perf_counter() - t0, pairs, O.num_threads(), done


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_workload(args.workload, 0, small=True)
    sec, pairs, cores, _ = oracle_steps(wl, args.steps, args.warmup)
    val = wl.n_total * args.steps / sec
    sample = f"{wl.name}: {wl.n_total} particles per step (same spacing, h, kernel and parameters as the full workload)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(args.workload), "sample": sample, "density_mode": wl.density_mode},
            "pair_interactions_per_sec": pairs / sec,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


def workload_label(name: str) -> str:
    return {"C1": "C1: 2-D periodic Taylor-Green, 4,096 particles, cubic spline h=1.3dx (BASELINE configs[0])",
            "C2": "C2: 2-D dam break, 20,000 fluid + 3,618 solid particles, quintic h=1.0dx (BASELINE configs[1])",
            "C3": "C3: 3-D periodic unit cube, 128^3 jittered lattice = 2,097,152 particles (BASELINE configs[2] prints 1,048,576 for 128^3; DESIGN.md R21), Wendland-C2 h=1.2dx, density+momentum+PC update",
            "C4": "C4: 3-D dam break, 3,456,000 fluid + 765,468 solid particles, cubic h=1.3dx (BASELINE configs[3])",
            "C5": "C5: 3-D Gaussian mixture, 16,777,216 particles, variable h, Wendland-C2 (BASELINE configs[4])"}[name]


# ---------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_1909_04504_b200 import binding

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SPH path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()

    wl = make_workload(args.workload, rank)
    mode = wl.density_mode
    move = "no position update" not in wl.note
    N = wl.n_total
    fixed = [a.fixed for a in wl.arrays]
    stream = torch.cuda.Stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    K, Wm = args.steps, args.warmup

    with torch.cuda.stream(stream):
        ctx = binding.SphContext.from_workload(wl, stream=stream, move=move)
        dev = binding.device_arrays(wl)
        fp32_peak = None
        if rank == 0:
            fp32_peak = {"ffma": ctx.fp32_probe(False, 8192)[0], "ffma2": ctx.fp32_probe(True, 8192)[0]}
        ctx.nnps_build(dev, fixed)
        ctx.pc_step(wl.dt, 1, mode)                       # a^0 + first step
        for _ in range(max(Wm - 1, 0)):
            ctx.pc_step(wl.dt, 1, mode)
        ctx.synchronize()

        def timed_pass(profile: bool):
            ctx.set_profiling(profile)
            l0 = ctx.get_stats().kernel_launches
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
            barrier(); torch.cuda.synchronize()
            for a, b in ev:
                flush.zero_()                             # L2 flush between timed steps (on the same stream)
                a.record(stream)
                ctx.pc_step(wl.dt, 1, mode)
                b.record(stream)
            torch.cuda.synchronize(); barrier()
            ms = sum(a.elapsed_time(b) for a, b in ev)
            return ms, ctx.get_stats().kernel_launches - l0

        sampler = ClockSampler(local_rank) if rank == 0 else None
        t_mark0 = time.time()
        ms_total, launches = timed_pass(False)
        t_mark1 = time.time()
        clocks = sampler.stop(t_mark0, t_mark1) if sampler else None

        # back-to-back variant: one call, K steps, no flush, no host involvement inside
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); ctx.pc_step(wl.dt, K, mode); b.record(stream); torch.cuda.synchronize()
        ms_b2b = a.elapsed_time(b)

        # second pass of the same K steps with an event pair around every launch -> per-kernel durations
        _, _ = timed_pass(True)
        prof = ctx.get_profile()
        ctx.set_profiling(False)
        stats = ctx.get_stats()                           # pair / candidate counts of the LAST evaluation
        ctx.synchronize()

        # ---- e2e through the C ABI with host buffers
        host = binding.pinned_arrays(wl)
        dim = wl.dim
        acc_keys = ("ax", "ay", "az", "arho") if dim == 3 else ("ax", "ay", "arho")
        out_keys = tuple(k for k in ("x", "y", "z", "u", "v", "w", "rho", "p") if dim == 3 or k not in ("z", "w")) + acc_keys
        for hA in host:
            n = hA["x"].shape[0]
            for k in acc_keys + ("p",):
                hA[k] = torch.zeros(n, dtype=torch.float32).pin_memory()
        in_keys = [k for k in host[0].keys() if k != "p" and not (dim == 2 and k in ("z", "w", "az"))]
        Ke = max(1, min(K, args.e2e_steps))

        def e2e_step():
            ctx.nnps_build([{k: hA[k] for k in in_keys} for hA in host], fixed)
            ctx.pc_step(wl.dt, 1, mode)
            for ai, hA in enumerate(host):
                ctx.sync_state(ai, host=True, out={k: hA[k] for k in out_keys})
        # first call has no a^n on the host yet (zeros would be wrong): evaluate once through the device path
        ctx.nnps_build([{k: hA[k] for k in in_keys if k not in acc_keys} for hA in host], fixed)
        ctx.pc_step(wl.dt, 1, mode)
        for ai, hA in enumerate(host):
            ctx.sync_state(ai, host=True, out={k: hA[k] for k in out_keys})
        for _ in range(2):
            e2e_step()
        barrier(); torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        a.record(stream)
        for _ in range(Ke):
            e2e_step()
        b.record(stream); torch.cuda.synchronize()
        e2e_wall_ms = 1e3 * (time.perf_counter() - t0)
        e2e_ms = max(a.elapsed_time(b), e2e_wall_ms)
        barrier()
        h2d = sum(hA[k].numel() * 4 for hA in host for k in in_keys)
        d2h = sum(hA[k].numel() * 4 for hA in host for k in out_keys)

    ms_max, units = aggregate(ms_total, float(N) * K, world)
    e2e_max, e2e_units = aggregate(e2e_ms, float(N) * Ke, world)
    ms_b2b_max, _ = aggregate(ms_b2b, 0.0, world)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    value = units / (ms_max * 1e-3)
    pairs_per_step = stats.pairs_density + stats.pairs_accel
    variable_h = bool(stats.variable_h)
    step_kernel_ms = sum(v["ms"] for k, v in prof.items() if not k.startswith("_"))
    kernels = {k: {"launches": v["launches"], "ms_per_launch": v["ms"] / v["launches"], "share": v["ms"] / step_kernel_ms}
               for k, v in prof.items() if not k.startswith("_")}
    cont = mode == "continuity"
    # ---- ALU roofline of the pair kernels (DESIGN.md "Rooflines" / "Algorithmic work"):
    # algorithmic flops of one launch = [searching passes only] the paper's own candidate set, the 3^d cells of
    # size >= the support radius around each destination (L158), x flops per predicate test, + the true pairs x
    # flops per pair.  The candidates the kernel REALLY tests (stats.candidates_*) are reported beside it, not used.
    c_test = flops_per_test(wl.dim, variable_h)
    coarse_cells = 1
    for k in range(wl.dim):
        coarse_cells *= max(1, stats.n_cells[k] // (stats.xsub if k == 0 else 1))
    ref_candidates = (3 ** wl.dim) * float(N) * float(N) / coarse_cells          # uniform-occupancy figure
    alu = {}
    if "k_density" in prof:
        nl_ = prof["k_density"]["launches"] / K
        fl = (ref_candidates * c_test + stats.pairs_density * flops_per_pair("density", wl.kernel, wl.dim, variable_h, False)) / max(nl_, 1)
        alu["k_density"] = {"flops": fl, "searches": True}
    for kname, searches in (("k_accel", True), ("k_accel_list", False)):
        if kname in prof:
            nl_ = prof[kname]["launches"] / K
            fl = ((ref_candidates * c_test if searches else 0.0)
                  + stats.pairs_accel * flops_per_pair("accel", wl.kernel, wl.dim, variable_h, cont)) / max(nl_, 1)
            alu[kname] = {"flops": fl, "searches": searches}
    peak_tf, peak_src = ALU_PEAK_TFLOPS, "derived: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz"
    if fp32_peak:
        peak_tf = max(fp32_peak.values())
        peak_src = ("measured in this run by sph_fp32_probe (dependent-free FMA streams, 8 blocks x 256 threads per SM): "
                    f"FFMA {fp32_peak['ffma']:.1f}, FFMA2 {fp32_peak['ffma2']:.1f} TFLOP/s; nominal {ALU_PEAK_TFLOPS:.1f}")
    for kname, v in alu.items():
        dur = prof[kname]["ms"] / prof[kname]["launches"]
        v["achieved_tflops"] = v["flops"] / (dur * 1e-3) / 1e12
        v["frac"] = v["achieved_tflops"] / peak_tf
        kernels[kname].update({"algorithmic_flops_per_launch": v["flops"], "achieved_tflops": v["achieved_tflops"],
                               "alu_frac": v["frac"]})
    dom = max(alu, key=lambda k: prof[k]["ms"]) if alu else max((k for k in prof if not k.startswith("_")), key=lambda k: prof[k]["ms"])
    dur_ms = prof[dom]["ms"] / prof[dom]["launches"]
    roofline = {"kernel": dom, "bound": "alu", "achieved": alu[dom]["achieved_tflops"], "peak": peak_tf, "unit": "TFLOP/s",
                "frac": alu[dom]["frac"], "traffic": ncu_traffic(dom, args.workload),
                "peak_source": peak_src,
                "algorithmic_flops_per_launch": alu[dom]["flops"],
                "counts": (f"{'3^d-cell candidates of L158 x ' + str(c_test) + ' flop + ' if alu[dom]['searches'] else ''}"
                           f"true pairs x flops per pair (DESIGN.md Algorithmic work); the kernel really tested "
                           f"{stats.candidates_density if dom == 'k_density' else stats.candidates_accel} candidates"),
                "ms_per_launch": dur_ms,
                "share_of_step_kernel_time": prof[dom]["ms"] / step_kernel_ms,
                "timing": "CUDA event pair around every launch in a second pass of the same K steps"}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        hbm_peak, hbm_src = float(peaks["hbm_gbs"]), "measured"
    except Exception:
        hbm_peak, hbm_src = 6650.0, "fallback"
    # HBM-bound streaming kernels: algorithmic bytes per particle
    bytes_pp = {"k_update": 16 + 4 + 16 + 16 + 16 + 16 + 8 + 4 + 4, "k_scatter": 4 + 4 + 4 + 2 * (16 + 16 + 8 + 4) + 4}
    hbm = {}
    for k, bpp in bytes_pp.items():
        if k in kernels:
            gbs = bpp * N / (kernels[k]["ms_per_launch"] * 1e-3) / 1e9
            hbm[k] = {"bytes_per_particle": bpp, "achieved_gbs": gbs, "peak_gbs": hbm_peak, "frac": gbs / hbm_peak, "peak_source": hbm_src}

    cpu = None
    if not args.no_cpu_baseline:
        wl_small = make_workload(args.workload, 0, small=True)
        sec, _, cores, done = oracle_steps(wl_small, args.cpu_steps, 0, budget_s=args.cpu_seconds)
        cpu = {"value": wl_small.n_total * done / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{wl_small.name}: {done} oracle PC steps of {wl_small.n_total} particles "
                         f"(same spacing, h, kernel, parameters) after the a^0 evaluation; {sec:.1f} s"}

    # BASELINE.json configs[1] (C2, the 2-D dam break run for its 1,000 steps) beside the headline workload: it is
    # launch-latency bound at 23,618 particles, so it is reported, not used for the roofline
    also = None
    if args.workload == "C3" and not args.no_also:
        wl2 = make_workload("C2", 0)
        with torch.cuda.stream(stream):
            c2 = binding.SphContext.from_workload(wl2, stream=stream)
            c2.nnps_build(binding.device_arrays(wl2), [a.fixed for a in wl2.arrays])
            c2.pc_step(wl2.dt, 20, wl2.density_mode)                     # a^0 + warm-up steps
            c2.synchronize()
            a2, b2 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a2.record(stream); c2.pc_step(wl2.dt, wl2.n_steps, wl2.density_mode); b2.record(stream)
            torch.cuda.synchronize()
            c2.synchronize()                                             # raises on out-of-domain / non-finite (no fallback)
            ms2 = a2.elapsed_time(b2)
            s2 = c2.get_stats()
            c2.close()
        also = {"workload": workload_label("C2"), "steps": wl2.n_steps, "ms_total": ms2, "us_per_step": 1e3 * ms2 / wl2.n_steps,
                "value": wl2.n_total * wl2.n_steps / (ms2 * 1e-3), "unit": UNIT,
                "pair_interactions_per_sec": (s2.pairs_density + s2.pairs_accel) * wl2.n_steps / (ms2 * 1e-3),
                "note": "one sph_pc_step(dt, 1000) call, continuity mode, device-resident, CUDA events; launch-latency bound"}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": workload_label(args.workload), "particles_per_gpu": N, "density_mode": mode,
                       "kernel": wl.kernel, "dim": wl.dim, "grid_cells": list(stats.n_cells),
                       "l2": "flushed between timed steps (256 MiB write); events bracket each sph_pc_step(dt,1)",
                       "parallelism": "replicas" if world > 1 else "single GPU"},
            "pair_interactions_per_sec": pairs_per_step * world * K / (ms_max * 1e-3),
            "pairs_per_step": pairs_per_step, "candidate_tests_per_step": stats.candidates,
            "back_to_back": {"value": units / (ms_b2b_max * 1e-3), "ms_per_step": ms_b2b_max / K,
                             "note": "one sph_pc_step(dt,K) call, no L2 flush"},
            "e2e": {"value": e2e_units / (e2e_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "steps": Ke, "what": "sph_nnps_build(host pinned arrays + a^n) + sph_pc_step(dt,1) + sph_sync_state(host) per step"},
            "gpu_launches": int(launches),
            "roofline": roofline, "kernels": kernels, "hbm_kernels": hbm,
            "cpu_baseline": cpu, "clocks": clocks, "configs1_dam_break_2d": also}
    print(json.dumps(line), flush=True)
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--cpu-steps", type=int, default=1000)
    ap.add_argument("--cpu-seconds", type=float, default=20.0, help="time budget of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the C2 (BASELINE configs[1]) side measurement")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
