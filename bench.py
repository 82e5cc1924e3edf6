#!/usr/bin/env python
"""bench.py -- the driver's measurement contract for the NanoBTE hot path.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload finfet|cube|nongray_square|gray_square|triangles]
                    [--mode plain|synthetic] [--impl reference] [--no-cpu-baseline]

A "step" is one pass of the whole hot path over one batch of synthetic input: transport sweep (a2-a5), closures +
moments + temperature update (a3, a6, a8) and, in synthetic mode, the CG diffusion correction (a7).  The default
workload is BASELINE.json configs[3] (FinFET-like masked grid, 844 M cell.band.direction updates per sweep, the
"largest structured config" the north_star's roofline bar is set on), in the mode that config names (synthetic).
Prints ONE JSON line (rank 0).  Multi-GPU: the path is single-GPU by the north_star, so --gpus N runs N independent
replicas (one per rank under torchrun), no data-path collective; value is the whole-job aggregate.

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-band-direction updates/s through one source iteration (sweep + closures + moments [+ CG]), fp64"
UNIT = "updates/s"
SMI_QUERY = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="finfet")
    ap.add_argument("--mode", default=None, help="plain | synthetic (default: the config's own)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-convergence", action="store_true", help="skip the time-to-convergence run")
    ap.add_argument("--cpu-sample-bands", type=int, default=0, help="bands in the oracle's sample (0 = auto)")
    ap.add_argument("--shard", default="replicas", choices=["replicas", "bands"],
                    help="N > 1: independent replicas (default; the north_star keeps the path on one GPU) or ONE problem with the band "
                         "table split over the ranks and one all-reduce per iteration (PAPER.md:115-121; strong scaling)")
    ap.add_argument("--sweep-G", type=int, default=0)
    ap.add_argument("--sweep-threads", type=int, default=0)
    ap.add_argument("--sweep-variant", type=int, default=0)
    return ap.parse_args()


def make_problem(name):
    from paper_2607_03226_b200 import workloads as wl
    return wl.CONFIGS[name]()


def workload_config(pr, mode, extra=None):
    from paper_2607_03226_b200 import workloads as wl
    m = pr["mesh"]
    grid = f"{m['nx']}x{m['ny']}x{m['nz']}" if pr["kind"] == "structured" else f"{m['n_cells']} triangles"
    cfg = {"workload": pr["name"], "grid": grid, "active_cells": wl.n_active(pr), "bands": len(pr["bands"]["C"]),
           "directions": len(pr["quad"]["w"]), "updates_per_sweep": wl.n_updates(pr), "mode": mode,
           "l2_policy": "inputs larger than L2 (e array >> 126 MB); no flush needed" if wl.n_updates(pr) * 8 > 4 * 126e6
           else "e array fits L2: numbers are L2-resident, no roofline claim"}
    if extra:
        cfg.update(extra)
    return cfg


# ---------------------------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi polled every 100 ms during the timed region (B200_PROFILING.md 'clocks' line)."""

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={SMI_QUERY}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in open(self.path):
            f = [x.strip() for x in line.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[5 + k].lower().startswith("active"):
                    reasons.add(nm)
        try:
            os.unlink(self.path)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # samples under load = the upper half (the sampler also sees the idle edges of the region)
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy_)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline / --impl reference)
# ---------------------------------------------------------------------------------------------------------------------
def oracle_sample_problem(pr, n_bands):
    """Same mesh, quadrature, tags and source; the first n_bands bands of the table, each with the source share it has
    in the full table.  (band, direction) systems are independent, so the cost per update is the workload's own."""
    B = len(pr["bands"]["C"])
    n_bands = max(1, min(B, n_bands))
    sub = dict(pr)
    sub["bands"] = {k: np.ascontiguousarray(v[:n_bands]) for k, v in pr["bands"].items()}
    C = np.asarray(pr["bands"]["C"], dtype=np.float64)
    return sub, n_bands, C[:n_bands] / C.sum()


def auto_sample_bands(pr, target_updates=1.0e8):
    from paper_2607_03226_b200 import workloads as wl
    per_band = wl.n_active(pr) * len(pr["quad"]["w"])
    return int(max(1, min(len(pr["bands"]["C"]), round(target_updates / per_band))))


def run_oracle(pr, mode, steps, warmup, n_bands, threads):
    """Times the oracle PER PHASE on a band sample of the workload and extrapolates to the full band table:

        t_step(full) = (t_sweep + t_moments) * B / n_bands + t_cg

    The sweep (O2/O3) and the moment pass (O4) cost the same per (cell, band, direction) update whatever the band, so
    they scale with the band count; the diffusion correction (O6, CG on the full mesh) does not depend on the band
    count at all, so it is taken as measured (a sample that divides the fixed CG cost by the sample's updates
    understates the CPU rate).  Returns a dict."""
    from oracle.ref import RefSolver
    from paper_2607_03226_b200 import workloads as wl
    sub, nb, share = oracle_sample_problem(pr, n_bands)
    B = len(pr["bands"]["C"])
    r = RefSolver(sub, threads=threads, share=share)
    threads = r.threads
    synthetic = mode == "synthetic"
    t = {"sweep": 0.0, "moments": 0.0, "cg": 0.0}
    cg_iters = []
    for k in range(warmup + steps):
        t0 = time.perf_counter()
        r.sweep()
        t1 = time.perf_counter()
        r.update_temperature()
        t2 = time.perf_counter()
        if synthetic:
            it, _ = r.diffusion_correct()
        t3 = time.perf_counter()
        if k >= warmup:
            t["sweep"] += t1 - t0
            t["moments"] += t2 - t1
            t["cg"] += t3 - t2
            if synthetic:
                cg_iters.append(it)
    r.close()
    for k in t:
        t[k] /= max(1, steps)
    scale = B / nb
    t_full = (t["sweep"] + t["moments"]) * scale + t["cg"]
    upd_full = wl.n_updates(pr)
    return {"value": upd_full / t_full, "s_per_step_full": t_full, "cores": threads,
            "sweep_updates_per_s": wl.n_updates(sub) / t["sweep"],
            "phases_s_sample": dict(t), "phases_s_full": {"sweep": t["sweep"] * scale, "moments": t["moments"] * scale, "cg": t["cg"]},
            "cg_iters_per_step": float(np.mean(cg_iters)) if cg_iters else 0.0,
            "sample": (f"{pr['name']}: same mesh/quadrature/walls/source, first {nb} of {B} bands ({wl.n_updates(sub)} updates per "
                       f"sample step), {steps} timed steps after {warmup} warm-up, mode {mode}; sweep and moments timed separately "
                       f"and scaled by {B}/{nb}, CG (full mesh, band independent) as measured")}


# ---------------------------------------------------------------------------------------------------------------------
def bench_band_shards(args, pr, mode, rank, world, local, dist, skw):
    """--shard bands: ONE problem, the band table split over the ranks (paper_2607_03226_b200/sharded.py), one NCCL all-reduce
    of the update tensor per source iteration.  Strong scaling: value = updates of the whole problem / time."""
    import torch
    from paper_2607_03226_b200 import replicas, sharded
    from paper_2607_03226_b200 import workloads as wl
    s = sharded.ShardedSolver(pr, rank, world, dist=dist, **skw)
    upd = wl.n_updates(pr)
    for _ in range(args.warmup):
        s.step(mode)
    replicas.barrier(dist, torch.cuda.synchronize)
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ else local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = s.local.launches
    sampler.start()
    e0.record()
    cg = [s.step(mode)[1] for _ in range(args.steps)]
    e1.record()
    replicas.barrier(dist, torch.cuda.synchronize)
    clocks = sampler.stop()
    ms = replicas.max_over_ranks(e0.elapsed_time(e1), dist, "cuda") / args.steps
    n_len = 5 * s.local.n_active + s.local.n_bf
    out = {"metric": METRIC, "value": upd / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_config(pr, mode, {"parallelism": f"band shards x{world}, one all-reduce of {n_len} doubles per iteration",
                                                "bands_of_rank0": len(s.bands)}),
           "cg_iters_per_step": float(np.mean(cg)) if cg else 0.0, "gpu_launches": int(s.local.launches - l0), "clocks": clocks,
           "e2e": {"value": upd / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 16,
                   "note": "band-shard arm: device-resident state, one 16-byte read per step (max|dT|, CG count)"}}
    s.close()
    if rank == 0:
        print(json.dumps(out))
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    from paper_2607_03226_b200 import replicas
    rank, world, local = replicas.env_rank()
    pr = make_problem(args.workload)
    mode = args.mode or pr["mode"]

    if args.impl == "reference":
        if rank != 0:
            return 0
        nb = args.cpu_sample_bands or auto_sample_bands(pr, 6.0e7)
        steps, warmup = max(1, min(args.steps, 3)), max(1, min(args.warmup, 1))
        cores = len(os.sched_getaffinity(0))
        o = run_oracle(pr, mode, steps, warmup, nb, cores)
        val = o["value"]
        out = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
               "warmup": warmup, "ms_per_step": o["s_per_step_full"] * 1e3, "higher_is_better": True, "scaling": "weak",
               "vs_baseline": None, "dtype": "f64", "data": "synthetic",
               "config": workload_config(pr, mode, {"note": "CPU oracle; per-phase timing on a band sample, extrapolated to the full "
                                                            "band table (ms_per_step is that extrapolation)"}),
               "cpu_baseline": {"value": val, "unit": UNIT, "cores": o["cores"], "kind": "oracle", "sample": o["sample"],
                                "phases_s_full": o["phases_s_full"], "cg_iters_per_step": o["cg_iters_per_step"]},
               "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
               "gpu_launches": 0}
        print(json.dumps(out))
        return 0

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: libnanobte has no CPU fallback")
    torch.cuda.set_device(local)
    dist = replicas.init("nccl", torch.device("cuda", local))
    from paper_2607_03226_b200 import build as nb_build
    from paper_2607_03226_b200 import workloads as wl
    if rank == 0:
        nb_build.build()
    if dist:
        dist.barrier()
    from paper_2607_03226_b200.binding import Solver

    skw = dict(sweep_G=args.sweep_G, sweep_threads=args.sweep_threads, sweep_variant=args.sweep_variant)
    if args.shard == "bands":
        return bench_band_shards(args, pr, mode, rank, world, local, dist, skw)
    t_c0 = time.perf_counter()
    g = Solver(pr, **skw)
    g.set_keep_e(False)  # the sweeps of an iteration leave eps where solve() leaves it (on chip where the kernel can)
    torch.cuda.synchronize()
    create_s = time.perf_counter() - t_c0
    upd = wl.n_updates(pr)
    synthetic = mode == "synthetic"

    def step(s, ev=None, cg=None):
        """One source iteration through the C ABI: sweep (a2-a5), closures + moments + update (a3, a6, a8), CG (a7)."""
        if ev is not None:
            ev[0].record()
        s.sweep()
        if ev is not None:
            ev[1].record()
        if synthetic:
            s.update_temperature(sync=False)
            if ev is not None:
                ev[2].record()
            it, _ = s.diffusion_correct()
            if cg is not None:
                cg.append(it)
        else:
            s.update_temperature(sync=True)
            if ev is not None:
                ev[2].record()
        if ev is not None:
            ev[3].record()

    def barrier():
        replicas.barrier(dist, torch.cuda.synchronize)

    # ---- device-resident arm: outer iterations W+1 .. W+K of the solve from T_ref ------------------------------------
    for _ in range(args.warmup):
        step(g)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(args.steps)]
    sampler = ClockSampler(torch.cuda.current_device() if "CUDA_VISIBLE_DEVICES" not in os.environ else local)
    l0 = g.launches
    cg_dev = []
    barrier()
    sampler.start()
    for k in range(args.steps):
        step(g, evs[k], cg_dev)
    barrier()
    clocks = sampler.stop()
    launches = g.launches - l0
    total_ms = evs[0][0].elapsed_time(evs[-1][3])
    sweep_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    update_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    cg_ms = float(np.mean([e[2].elapsed_time(e[3]) for e in evs])) if synthetic else 0.0
    total_ms = replicas.max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / args.steps
    value = replicas.whole_job_rate(upd, world, ms_per_step * 1e-3)
    info = dict(g.info)
    g.close()

    # ---- end-to-end arm: the SAME outer iterations (fresh solver, same warm-up), host buffers through the C ABI, the
    # host<->device copies of every step inside the timed region ----------------------------------------------------------
    g = Solver(pr, **skw)
    g.set_keep_e(False)
    T_host = torch.empty(g.n_cells, dtype=torch.float64).pin_memory()
    T_host.copy_(torch.as_tensor(g.get_T(0)))
    T_np = T_host.numpy()
    cg_e2e = []

    def e2e_step(cg=None):
        g.set_T(T_np)                       # H2D: n_cells doubles from pinned host memory
        step(g, None, cg)                   # D2H inside: max|dT| (+ CG iterations)
        g.get_T(0, out=T_np)                # D2H: n_cells doubles, straight into the pinned buffer

    for _ in range(args.warmup):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step(cg_e2e)
    barrier()
    e2e_s = (time.perf_counter() - t0) / args.steps
    e2e_s = replicas.max_over_ranks(e2e_s, dist, "cuda")
    e2e = {"value": replicas.whole_job_rate(upd, world, e2e_s), "unit": UNIT, "h2d_bytes_per_step": int(g.n_cells * 8),
           "d2h_bytes_per_step": int(g.n_cells * 8 + 16), "ms_per_step": e2e_s * 1e3,
           "cg_iters_per_step": float(np.mean(cg_e2e)) if cg_e2e else 0.0,
           "note": "same outer iterations as the device arm (fresh solver, same warm-up); timed with the host clock around "
                   "barrier + synchronize"}
    g.close()

    # ---- roofline of the dominant kernel (the sweep): 8 algorithmic bytes per update (the eps store of the sweep;
    # DESIGN.md section 6).  The tile-dataflow kernel also does the moments (SURVEY: 8 B/update more, the eps load) and moves
    # neither through HBM, so for it the HBM figure is an equivalent rate, not traffic: the measured DRAM bytes are in
    # "traffic", and what bounds the kernel itself is in "on_chip" (fp64 pipe and shared-memory crossbar).
    peak, peak_src = measured_peaks()
    alg_bytes = 8.0 * upd
    achieved = alg_bytes / (sweep_ms * 1e-3) / 1e9
    brick = pr["kind"] == "structured" and info.get("sweep_variant") == 5
    kernel = (("sweep_brick_kernel" if brick else "sweep_structured_kernel") if pr["kind"] == "structured" else
              ("sweep_unstructured_staged_kernel" if info.get("sweep_rmax", 0) == 0 else "sweep_unstructured_kernel"))
    roofline = {"bound": "hbm", "kernel": kernel,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / 8000.0,
                "algorithmic_bytes_per_launch": alg_bytes, "launch_ms": sweep_ms}
    if brick:
        # fp64 operations per update: 4 (substitution) + 3 (band sums of the moments) + 5/B per direction weight ~ 7.2;
        # peak = 64 DFMA/clk/SM x SMs x clock (B300_MICROARCH.md unit counts; 58/clk measured with a DFMA-only kernel)
        sm_clock = (clocks.get("sm_mhz") or 1965.0) * 1e6
        ops = (7.0 + 5.0 / max(1, len(pr["bands"]["C"]))) * upd
        alu_peak = 64.0 * 148 * sm_clock
        # shared-memory bytes per update: STS 8 + LDS 8 (u-upwind) + 8 (theta: a broadcast still returns 8 B per lane) + LDS 8
        # (moments) + ~3 (band coefficients, 16 B per 6 values) = 35; ncu counts 48 B/update (rows of a 7-row tile padded to 8, conflicts)
        smem_bytes = 35.0 * upd
        roofline["fused"] = {"note": "sweep + moments in one kernel: nothing of eps goes to HBM unless asked for",
                             "algorithmic_bytes_sweep_plus_moments": 16.0 * upd,
                             "equivalent_GBs_sweep_plus_moments": 16.0 * upd / (sweep_ms * 1e-3) / 1e9}
        roofline["on_chip"] = {"alu": {"bound": "alu", "achieved": ops / (sweep_ms * 1e-3) / 1e12, "peak": alu_peak / 1e12,
                                       "unit": "T fp64 op/s", "frac": ops / (sweep_ms * 1e-3) / alu_peak},
                               "smem": {"achieved": smem_bytes / (sweep_ms * 1e-3) / 1e12, "peak": 128.0 * 148 * sm_clock / 1e12,
                                        "unit": "TB/s", "frac": smem_bytes / (sweep_ms * 1e-3) / (128.0 * 148 * sm_clock)}}
    else:
        roofline["moments_pass"] = {"achieved": alg_bytes / (update_ms * 1e-3) / 1e9, "launch_ms": update_ms,
                                    "note": "closures + moments + update; 8 B/update read"}
    tr = os.path.join(ROOT, "profiles", "traffic.json")  # copied from ncu --set full captures; each entry names its capture
    if os.path.exists(tr):
        try:
            ent = json.load(open(tr)).get(pr["name"], {})
            roofline["traffic"] = ent.get("sweep_dram_bytes_per_launch")
            roofline["traffic_source"] = {k: ent.get(k) for k in ("capture", "commit", "kernel") if k in ent}
        except Exception:
            pass

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": workload_config(pr, mode, {"parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                                                "sweep": {k: info[k] for k in ("sweep_G", "sweep_threads", "sweep_rmax", "n_tasks", "n_planes",
                                                                               "sweep_smem_bytes", "pencil_axis")},
                                                "cg": {k: info[k] for k in ("cg_multigrid", "cg_mg_levels", "cg_fused", "cg_cells_per_thread",
                                                                            "cg_ctas", "cg_face_uniform", "cg_recycle")},
                                                "device_bytes": info["device_bytes"]}),
           "sweep_updates_per_s": world * upd / (sweep_ms * 1e-3), "s_per_iteration": ms_per_step * 1e-3,
           "breakdown_ms": {"sweep": sweep_ms, "closures_moments_update": update_ms, "cg": cg_ms},
           "cg_iters_per_step": float(np.mean(cg_dev)) if cg_dev else 0.0,
           "create_s": create_s, "roofline": roofline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}
    # ---- time to convergence (north_star: reported beside the per-iteration numbers): a fresh solver, solve() to the
    # workload's own tolerance, wall clock around the call (one 16-byte D2H per iteration is part of it)
    if not args.no_convergence:
        g2 = Solver(pr, **skw)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        res = g2.solve(pr["tol"], pr["max_iter"], mode)
        torch.cuda.synchronize()
        out["time_to_convergence"] = {"seconds": time.perf_counter() - t0, "iterations": res["iters"],
                                      "converged": res["converged"], "tol_K": pr["tol"], "last_dT_K": res["last_dT"],
                                      "cg_iters_total": int(g2.get_history()[1].sum())}
        g2.close()
        if pr["mode"] == "synthetic" or any(t[0] == 0 for t in pr["mesh"]["tags"]):
            # the same solve started from the Fourier field (nanobte_init_fourier), the guess inside the clock
            g3 = Solver(pr, **skw)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            cg0 = g3.init_fourier()
            res = g3.solve(pr["tol"], pr["max_iter"], mode)
            torch.cuda.synchronize()
            out["time_to_convergence"]["fourier_start"] = {"seconds": time.perf_counter() - t0, "iterations": res["iters"],
                                                           "converged": res["converged"], "guess_cg_iters": cg0,
                                                           "cg_iters_total": int(g3.get_history()[1].sum())}
            g3.close()
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # the oracle as it stands on this box's host cores: all cores and one core, per phase
        cores = len(os.sched_getaffinity(0))
        nb = args.cpu_sample_bands or auto_sample_bands(pr)
        oN = run_oracle(pr, mode, 2, 1, nb, cores)
        o1 = run_oracle(pr, mode, 1, 0, 1 if wl.n_updates(pr) > 1e7 else nb, 1)
        out["cpu_baseline"] = {"value": oN["value"], "unit": UNIT, "cores": oN["cores"], "kind": "oracle", "sample": oN["sample"],
                               "s_per_step_full": oN["s_per_step_full"], "phases_s_full": oN["phases_s_full"],
                               "sweep_updates_per_s": oN["sweep_updates_per_s"], "cg_iters_per_step": oN["cg_iters_per_step"],
                               "one_thread": {k: o1[k] for k in ("value", "cores", "s_per_step_full", "phases_s_full",
                                                                  "sweep_updates_per_s", "sample")}}
        if "time_to_convergence" in out:
            out["cpu_baseline"]["time_to_convergence_extrapolated_s"] = oN["s_per_step_full"] * out["time_to_convergence"]["iterations"]
    if rank == 0:
        print(json.dumps(out))
    if dist:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
