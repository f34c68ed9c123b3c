#!/usr/bin/env python
"""bench.py -- particle-steps/s of the SPH hot path (NNPS + density + EOS + momentum + PC update) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5] [--impl ours|reference]

One "step" = one predictor-corrector step of the whole hot path: fused update + cell
key -> counting sort -> cell offsets + permute -> neighbour search (tensor-core filter -> mask records) ->
summation density + EOS -> WCSPH acceleration, on one synthetic workload.  Prints ONE
JSON line (rank 0).  The headline workload is the largest single-GPU configuration of BASELINE.json (C5); the other
four configurations are measured the same way in the same run and reported under "configs".

  value      device-resident throughput: inputs live in HBM, K calls of sph_pc_step(dt, 1) each bracketed by CUDA
             events on the context stream, L2 flushed (256 MiB write) between timed steps; three such passes, the
             median pass is reported; max over ranks.
  e2e        the same metric through the C ABI with HOST (pinned) buffers: every step does sph_nnps_build(host
             arrays incl. a^n) + sph_pc_step(dt, 1) + sph_sync_state(host, incl. a^{n+1}); copies inside the timing.
  roofline   the dominant kernel of the step: algorithmic flops per launch / its mean launch duration from CUDA
             event pairs recorded around every launch (sph_set_profiling) during an extra pass of the same K steps.
             bound = "alu" (plain FP32 pipes); peak = the FMA rate sph_fp32_probe measures
             in this run.  Work units: the search is charged the candidate set of the
             PAPER's own cell-list search on the current state (sph_stencil_candidates: 3^d cells >= k h_max, L158)
             x flops per predicate; a pair pass its true pairs x flops per pair.
  cpu_baseline  the fp64 oracle (oracle/, as it stands, OpenMP over destinations) on this box's host cores, all
             threads and one thread, on a bounded sample of the same workload.

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
L2_BYTES = 126e6
ALL = ("C1", "C2", "C3", "C4", "C5")


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
        return W.gaussian_mixture_3d(N=(1 << 18) if small else (1 << 24), seed=2 + 100 * rank)
    raise SystemExit(f"unknown workload {name}")


def workload_label(name: str) -> str:
    return {"C1": "C1: 2-D periodic Taylor-Green, 4,096 particles, cubic spline h=1.3dx (BASELINE configs[0])",
            "C2": "C2: 2-D dam break, 20,000 fluid + 3,618 solid particles, quintic h=1.0dx, continuity mode (BASELINE configs[1])",
            "C3": "C3: 3-D periodic unit cube, 128^3 jittered lattice = 2,097,152 particles (BASELINE configs[2] prints 1,048,576 for 128^3; DESIGN.md R21), Wendland-C2 h=1.2dx, density+momentum+PC update",
            "C4": "C4: 3-D dam break, 3,456,000 fluid + 765,468 solid particles, cubic h=1.3dx, continuity mode (BASELINE configs[3])",
            "C5": "C5: 3-D Gaussian mixture, 16,777,216 particles, variable h (ratio 4), Wendland-C2, density+momentum, no position update (BASELINE configs[4], the largest single-GPU configuration)"}[name]


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


# Algorithmic bytes per particle of the streaming kernels, per launch variant (DESIGN.md "NNPS" / "Algorithmic work")
def hbm_bytes_per_particle(kernel: str, cont: bool, move: bool) -> int:
    if kernel == "k_update":          # eq.14 + eq.12 + eq.13 + key: posh R(+W when moving), velm R+W, acc R, meta R, key W, rank W
        return 16 + (16 if move else 0) + 32 + 16 + 4 + 4 + 4 + (16 if cont else 0)      # continuity: rp R+W
    if kernel == "k_update_kick":     # eq.14 only: velm R+W, acc R, meta R
        return 32 + 16 + 4 + (16 if cont else 0)
    if kernel == "k_scatter":         # key, rank, cell_start R; posh, velm, rp, meta R+W; cell W
        return 12 + 2 * (16 + 16 + 8 + 4) + 4
    raise KeyError(kernel)


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
    """(bytes, source): dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload` from the
    committed `ncu --set full` capture summarised in profiles/r2_dram_traffic.csv (kernel,workload,read_bytes,
    write_bytes,capture); not measured in this run (no number of a bench run is taken under a profiler)."""
    path = os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")
    try:
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 4 and f[0] == kernel and f[1] == workload:
                return float(f[2]) + float(f[3]), f"profiles/r2_dram_traffic.csv ({f[4] if len(f) > 4 else 'ncu --set full capture'}); not measured in this run"
    except OSError:
        pass
    return None, "no committed ncu capture of this kernel on this workload"


def ncu_limiter(kernel: str, workload: str):
    """What the committed ncu capture shows to hold the kernel (columns 6-7 of profiles/r2_dram_traffic.csv:
    l1tex__data_pipe_lsu_wavefronts and smsp__issue_active, % of peak); not measured in this run."""
    try:
        for line in open(os.path.join(ROOT, "profiles", "r2_dram_traffic.csv")):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 7 and f[0] == kernel and f[1] == workload:
                return {"l1_lsu_data_pipe_pct_of_peak": float(f[5]), "issue_slots_pct_of_peak": float(f[6]), "source": f[4] + "; not measured in this run",
                        "note": "the replaying pair kernels are held by the L1 LSU data pipe (one cycle per 128-byte line a gather touches) "
                                "with the issue slots close behind; the search by issue / the ALU pipe (DESIGN.md 'What bounds them')"}
    except (OSError, ValueError):
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
# reference arm / cpu_baseline: the oracle on host cores
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


def oracle_single_core(wl, n_dest: int = 2048):
    """One evaluation (density + momentum, or momentum + continuity) of the oracle on ONE thread for a seeded
    subset of destination particles against all sources, extrapolated to particle-steps/s of one core."""
    from oracle import sph_oracle as O
    nthr = O.num_threads()
    O.set_num_threads(1)
    try:
        st = O.State(wl)
        for A in st.arrays:
            A["p"] = O.eos(wl, A["rho"])
        na = len(wl.arrays)
        t_total, n_total = 0.0, 0
        for d in range(na):
            n = wl.arrays[d].n
            if n == 0:
                continue
            sub = np.sort(np.random.default_rng(7 + d).choice(n, size=min(n_dest, n), replace=False))
            t0 = time.perf_counter()
            if wl.density_mode == "summation":
                O.density(wl, st, d, wl.density_sources[d], pred32=False, subset=sub)
            srcs = wl.accel_sources[d] if not wl.arrays[d].fixed else (wl.arho_sources[d] if wl.density_mode == "continuity" else [])
            if srcs:
                O.accel(wl, st, d, srcs, pred32=False, subset=sub)
            t_total += (time.perf_counter() - t0) * (n / len(sub))
            n_total += n
        return {"value": n_total / t_total if t_total > 0 else None, "unit": UNIT, "cores": 1,
                "sample": f"one evaluation of {min(n_dest, wl.arrays[0].n)} seeded destination particles per array against all "
                          f"sources of {wl.name}, extrapolated to all particles"}
    finally:
        O.set_num_threads(nthr)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_workload(args.workload, 0, small=True)
    sec, pairs, cores, done = oracle_steps(wl, args.steps, args.warmup)
    val = wl.n_total * done / sec
    sample = f"{wl.name}: {wl.n_total} particles per step (same spacing law, h, kernel and parameters as the full workload)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * sec / max(done, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_label(args.workload), "sample": sample, "density_mode": wl.density_mode},
            "pair_interactions_per_sec": pairs / sec,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ---------------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------------
def measure(name, rank, world, K, Wm, passes, e2e_steps, stream, flush, barrier, fp32_peak, hbm_peak, overrides):
    """Measures one configuration on this rank's GPU.  Returns a dict of per-rank results (aggregated by the caller)."""
    import torch
    from paper_1909_04504_b200 import binding
    wl = make_workload(name, rank)
    mode = wl.density_mode
    cont = mode == "continuity"
    move = "no position update" not in wl.note
    N = wl.n_total
    fixed = [a.fixed for a in wl.arrays]
    with torch.cuda.stream(stream):
        ctx = binding.SphContext.from_workload(wl, stream=stream, move=move, **overrides)
        dev = binding.device_arrays(wl)
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
            return sum(a.elapsed_time(b) for a, b in ev), ctx.get_stats().kernel_launches - l0

        t0 = time.time()
        runs = [timed_pass(False) for _ in range(passes)]
        t1 = time.time()
        ms_passes = sorted(r[0] for r in runs)
        ms_total, launches = ms_passes[len(ms_passes) // 2], runs[0][1]

        # back-to-back variant: one call, K' steps, no flush, no host involvement inside (captured step graph)
        Kb = max(K, 20)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); ctx.pc_step(wl.dt, Kb, mode); b.record(stream); torch.cuda.synchronize()
        ms_b2b = a.elapsed_time(b) / Kb

        # one more pass of the same K steps with an event pair around every launch -> per-kernel durations
        timed_pass(True)
        prof = ctx.get_profile()
        ctx.set_profiling(False)
        stats = ctx.get_stats()                           # pair / candidate counts of the LAST evaluation
        stencil = ctx.stencil_candidates()                # candidate set of the paper's cell-list search on this state
        ctx.synchronize()

        # ---- e2e through the C ABI with host buffers
        e2e = None
        if e2e_steps > 0:
            host = binding.pinned_arrays(wl)
            dim = wl.dim
            acc_keys = ("ax", "ay", "az", "arho") if dim == 3 else ("ax", "ay", "arho")
            out_keys = tuple(k for k in ("x", "y", "z", "u", "v", "w", "rho", "p") if dim == 3 or k not in ("z", "w")) + acc_keys
            for hA in host:
                n = hA["x"].shape[0]
                for k in acc_keys + ("p",):
                    hA[k] = torch.zeros(n, dtype=torch.float32).pin_memory()
            in_keys = [k for k in host[0].keys() if k != "p" and not (dim == 2 and k in ("z", "w", "az"))]

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
            e2e_step()
            barrier(); torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            tw = time.perf_counter()
            a.record(stream)
            for _ in range(e2e_steps):
                e2e_step()
            b.record(stream); torch.cuda.synchronize()
            e2e_ms = max(a.elapsed_time(b), 1e3 * (time.perf_counter() - tw))
            barrier()
            e2e = {"ms": e2e_ms, "steps": e2e_steps,
                   "h2d": sum(hA[k].numel() * 4 for hA in host for k in in_keys),
                   "d2h": sum(hA[k].numel() * 4 for hA in host for k in out_keys)}
            del host
        ctx.close()
        del dev
    torch.cuda.empty_cache()
    return {"wl": wl, "N": N, "mode": mode, "cont": cont, "move": move, "ms_total": ms_total, "ms_passes": ms_passes,
            "launches": int(launches), "ms_b2b": ms_b2b, "prof": prof, "stats": stats, "stencil": stencil, "e2e": e2e,
            "t_timed": (t0, t1)}


def report(name, r, K, world, ms_max, units, e2e_agg, fp32_peak, hbm_peak, hbm_src):
    """Turns the measurements of one configuration into the reported numbers (rank 0)."""
    wl, stats, prof, N, cont = r["wl"], r["stats"], r["prof"], r["N"], r["cont"]
    variable_h = bool(stats.variable_h)
    kprof = {k: v for k, v in prof.items() if not k.startswith("_")}
    step_ms = sum(v["ms"] for v in kprof.values())
    kernels = {k: {"launches": v["launches"], "ms_per_launch": v["ms"] / v["launches"], "share": v["ms"] / step_ms} for k, v in kprof.items()}
    c_test = flops_per_test(wl.dim, variable_h)
    pair_d = flops_per_pair("density", wl.kernel, wl.dim, variable_h, False)
    pair_a = flops_per_pair("accel", wl.kernel, wl.dim, variable_h, cont)
    # algorithmic flops per launch: a searching launch is charged the candidate set of
    # the paper's cell-list search (3^d cells >= k h_max) -- or, where the level grids of this library stream FEWER
    # candidates than that (variable h), what it really streams: the fraction never credits work that was avoided
    search_units = min(r["stencil"], stats.candidates_search) if stats.candidates_search > 0 else r["stencil"]
    work = {"k_search": search_units * c_test,
            "k_density_list": stats.pairs_density * pair_d, "k_accel_list": stats.pairs_accel * pair_a,
            "k_density": r["stencil"] * c_test + stats.pairs_density * pair_d,
            "k_accel": r["stencil"] * c_test + stats.pairs_accel * pair_a}
    peak_tf = max(fp32_peak.values()) if fp32_peak else ALU_PEAK_TFLOPS
    peak_src = (f"measured in this run by sph_fp32_probe (dependent-free FMA streams, 8 blocks x 256 threads per SM): FFMA "
                f"{fp32_peak['ffma']:.1f}, FFMA2 {fp32_peak['ffma2']:.1f} TFLOP/s; nominal {ALU_PEAK_TFLOPS:.1f}") if fp32_peak else \
               "derived: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz"
    alu = {}
    for kname, fl in work.items():
        if kname in kprof:
            per_launch = fl / max(kprof[kname]["launches"] / K, 1)
            dur = kprof[kname]["ms"] / kprof[kname]["launches"]
            tf = per_launch / (dur * 1e-3) / 1e12
            alu[kname] = {"flops": per_launch, "tflops": tf, "frac": tf / peak_tf}
            kernels[kname].update({"algorithmic_flops_per_launch": per_launch, "achieved_tflops": tf, "alu_frac": tf / peak_tf})
    roofline = None
    if alu:
        dom = max(alu, key=lambda k: kprof[k]["ms"])
        traffic, tsrc = ncu_traffic(dom, name)
        tot_fl = sum(alu[k]["flops"] * kprof[k]["launches"] / K for k in alu)
        tot_ms = sum(kprof[k]["ms"] / K for k in alu)
        roofline = {"kernel": dom, "bound": "alu", "achieved": alu[dom]["tflops"], "peak": peak_tf, "unit": "TFLOP/s",
                    "frac": alu[dom]["frac"], "traffic": traffic, "traffic_source": tsrc, "peak_source": peak_src,
                    "algorithmic_flops_per_launch": alu[dom]["flops"], "ncu_limiter": ncu_limiter(dom, name),
                    "counts": "k_search: min(candidates of the paper's cell-list search (sph_stencil_candidates on this state: "
                              f"{r['stencil']} = {r['stencil'] / max(N, 1):.0f} per particle), candidates streamed) x {c_test} flop; pair passes: true pairs x "
                              f"{pair_d} (density) / {pair_a} (momentum) flop; this library streamed {stats.candidates} candidates "
                              f"({stats.candidates / max(N, 1):.0f} per particle) through its filter",
                    "ms_per_launch": kprof[dom]["ms"] / kprof[dom]["launches"],
                    "share_of_step_kernel_time": kprof[dom]["ms"] / step_ms,
                    "pair_path": {"kernels": sorted(alu), "achieved": tot_fl / (tot_ms * 1e-3) / 1e12, "frac": tot_fl / (tot_ms * 1e-3) / 1e12 / peak_tf,
                                  "share_of_step_kernel_time": tot_ms * K / step_ms,
                                  "vs_paper_search": (r["stencil"] * c_test * (2 if "k_density_list" in alu or "k_density" in alu else 1)
                                                      + stats.pairs_density * pair_d + stats.pairs_accel * pair_a) / (tot_ms * 1e-3) / 1e12 / peak_tf,
                                  "vs_paper_search_note": "the same time against the work of the paper's scheme: one 3^d-cell search per pair pass"},
                    "timing": "CUDA event pair around every launch in an extra pass of the same K steps"}
    state_bytes = N * (16 + 16 + 8 + 4 + 4 + 16)
    hbm = {}
    for k in ("k_update", "k_update_kick", "k_scatter"):
        if k in kernels:
            bpp = hbm_bytes_per_particle(k, cont, r["move"])
            gbs = bpp * N / (kernels[k]["ms_per_launch"] * 1e-3) / 1e9
            hbm[k] = {"bytes_per_particle": bpp, "achieved_gbs": gbs, "peak_gbs": hbm_peak, "frac": gbs / hbm_peak, "peak_source": hbm_src,
                      "l2_resident": bool(state_bytes < L2_BYTES)}
    if "k_scan" in kernels:
        # tables of >= 1024 tiles are scanned by three launches (tile sums, their scan, the pass that applies them: the
        # table is read twice); the algorithmic bytes stay 12 per key (counts read, offsets written, counts cleared)
        parts = [k for k in ("k_scan_reduce", "k_scan_tiles", "k_scan") if k in kernels]
        scan_ms = sum(kernels[k]["ms_per_launch"] for k in parts)
        gbs = 12.0 * stats.n_keys / (scan_ms * 1e-3) / 1e9
        hbm["k_scan"] = {"bytes_per_key": 12, "keys": int(stats.n_keys), "achieved_gbs": gbs, "peak_gbs": hbm_peak, "frac": gbs / hbm_peak,
                         "peak_source": hbm_src, "l2_resident": bool(12.0 * stats.n_keys < L2_BYTES), "launches": parts, "ms": scan_ms}
    pairs_per_step = stats.pairs_density + stats.pairs_accel
    out = {"workload": workload_label(name), "particles_per_gpu": N, "density_mode": r["mode"], "kernel": wl.kernel, "dim": wl.dim,
           "value": units / (ms_max * 1e-3), "unit": UNIT, "ms_per_step": ms_max / K,
           "ms_per_step_passes": [m / K for m in r["ms_passes"]],
           "pair_interactions_per_sec": pairs_per_step * world * K / (ms_max * 1e-3), "pairs_per_step": int(pairs_per_step),
           "candidates_streamed_per_step": int(stats.candidates), "stencil_candidates_per_step": int(r["stencil"]),
           "grid": {"levels": int(stats.n_levels), "coarsest_cells": list(stats.n_cells), "xsub": int(stats.xsub), "keys": int(stats.n_keys)},
           "records": {"replayed": bool(stats.used_rows), "rows_used": int(stats.nlist_rows_used), "rows_capacity": int(stats.nlist_rows_capacity),
                       "fallback_warps": int(stats.nlist_fallback_warps)},
           "back_to_back": {"ms_per_step": r["ms_b2b"], "value": N * world / (r["ms_b2b"] * 1e-3),
                            "note": "one sph_pc_step(dt, >= 20) call: no L2 flush, captured two-step CUDA graph"},
           "gpu_launches": r["launches"], "roofline": roofline, "kernels": kernels, "hbm_kernels": hbm}
    if e2e_agg is not None:
        e_ms, e_units = e2e_agg
        out["e2e"] = {"value": e_units / (e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": r["e2e"]["h2d"], "d2h_bytes_per_step": r["e2e"]["d2h"],
                      "steps": r["e2e"]["steps"], "ms_per_step": e_ms / r["e2e"]["steps"],
                      "pcie_gbs": (r["e2e"]["h2d"] + r["e2e"]["d2h"]) * r["e2e"]["steps"] / (e_ms * 1e-3) / 1e9,
                      "what": "sph_nnps_build(host pinned arrays + a^n) + sph_pc_step(dt,1) + sph_sync_state(host) per step"}
    return out


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

    stream = torch.cuda.Stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    K, Wm = args.steps, args.warmup
    overrides = {k: v for k, v in (("xsub", args.xsub), ("levels", args.levels), ("nlist_slots", args.nlist_slots)) if v}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        hbm_peak, hbm_src = float(peaks["hbm_gbs"]), "measured (MEASURED_PEAKS.json, torch copy)"
    except Exception:
        hbm_peak, hbm_src = 6650.0, "fallback (B200_PROFILING.md)"

    fp32_peak = None
    with torch.cuda.stream(stream):
        from paper_1909_04504_b200 import workloads as W
        tiny = W.taylor_green_2d()
        pctx = binding.SphContext.from_workload(tiny, stream=stream)
        fp32_peak = {"ffma": pctx.fp32_probe(False, 8192)[0], "ffma2": pctx.fp32_probe(True, 8192)[0]}
        pctx.close()

    names = [args.workload] + ([n for n in ALL if n != args.workload] if not args.no_configs else [])
    results, sampler, clocks = {}, None, None
    for idx, name in enumerate(names):
        head = idx == 0
        if head and rank == 0:
            sampler = ClockSampler(local_rank)
        r = measure(name, rank, world, K if head else min(K, args.config_steps), Wm, args.passes if head else 3,
                    args.e2e_steps if head else min(args.e2e_steps, 2), stream, flush, barrier, fp32_peak, hbm_peak, overrides)
        r["K"] = K if head else min(K, args.config_steps)
        if head and sampler:
            clocks = sampler.stop(*r["t_timed"])
        ms_max, units = aggregate(r["ms_total"], float(r["N"]) * r["K"], world)
        e2e_agg = aggregate(r["e2e"]["ms"], float(r["N"]) * r["e2e"]["steps"], world) if r["e2e"] else None
        if rank == 0:
            results[name] = report(name, r, r["K"], world, ms_max, units, e2e_agg, fp32_peak, hbm_peak, hbm_src)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    head = results[args.workload]
    cpu = None
    if not args.no_cpu_baseline:
        from oracle import sph_oracle as O
        wl_small = make_workload(args.workload, 0, small=True)
        sec, _, cores, done = oracle_steps(wl_small, args.cpu_steps, 0, budget_s=args.cpu_seconds)
        cpu = {"value": wl_small.n_total * done / sec, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{wl_small.name}: {done} oracle PC steps of {wl_small.n_total} particles (same spacing law, h, kernel, "
                         f"parameters) after the a^0 evaluation; {sec:.1f} s",
               "single_core": oracle_single_core(wl_small)}

    line = {"metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": head["workload"], "particles_per_gpu": head["particles_per_gpu"], "density_mode": head["density_mode"],
                       "kernel": head["kernel"], "dim": head["dim"], "grid": head["grid"], "passes": args.passes,
                       "l2": "flushed between timed steps (256 MiB write); events bracket each sph_pc_step(dt,1); median of the passes",
                       "parallelism": "replicas" if world > 1 else "single GPU"},
            "pair_interactions_per_sec": head["pair_interactions_per_sec"], "pairs_per_step": head["pairs_per_step"],
            "candidates_streamed_per_step": head["candidates_streamed_per_step"],
            "stencil_candidates_per_step": head["stencil_candidates_per_step"],
            "ms_per_step_passes": head["ms_per_step_passes"], "records": head["records"], "back_to_back": head["back_to_back"],
            "e2e": head.get("e2e"), "gpu_launches": head["gpu_launches"],
            "roofline": head["roofline"], "kernels": head["kernels"], "hbm_kernels": head["hbm_kernels"],
            "cpu_baseline": cpu, "clocks": clocks,
            "configs": {n: results[n] for n in names if n != args.workload}}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=list(ALL))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--passes", type=int, default=3, help="timed passes of K steps; the median is reported")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--config-steps", type=int, default=20, help="steps per pass of the non-headline configurations")
    ap.add_argument("--cpu-steps", type=int, default=1000)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="time budget of the cpu_baseline sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="measure the headline workload only")
    ap.add_argument("--xsub", type=int, default=0, help="tuning: sph_params.xsub (0 = default)")
    ap.add_argument("--levels", type=int, default=0, help="tuning: sph_params.levels (0 = default)")
    ap.add_argument("--nlist-slots", type=int, default=0, help="tuning: sph_params.nlist_slots (0 = default, < 0: no record pool)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    args.passes = max(args.passes, 3) if args.impl == "ours" else args.passes
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
