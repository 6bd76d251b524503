#!/usr/bin/env python
"""bench.py -- SPH particle-updates/s per full leapfrog step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cube256|cube128|sod|disc|...] [--impl reference]

A "step" is one pass of the whole hot path: predictor, Morton keys, onesweep sort,
permute, Karras tree, AABB/hmax, traversal -> neighbour cache, h/density Newton iteration, forces + CFL dt,
corrector. Default workload: BASELINE.json configs[2], the 256^3 uniform periodic cube the metric's target is
quoted on (16.8 M particles, ~13 GB resident: far larger than L2, so no L2 flush is needed between steps).
Multi-GPU: replicas only (the path has no exchange step in scope) -- every rank runs the same
workload with a different seed; value = particles stepped by all ranks / max-over-ranks time.
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

METRIC = "sph_particle_updates_per_sec_per_full_step"
UNIT = "particle-updates/s"

# Algorithmic work per unit, stated in DESIGN.md "Rooflines": FP64 flop per neighbour pair (fma = 2, div = sqrt = 1)
FLOP_PER_PAIR_DENSITY_GATHER = 11     # separation, d^2, sqrt (once per pair per density solve)
FLOP_PER_PAIR_DENSITY_SWEEP = 16      # q, f, f', two accumulations (per pair per Newton sweep)
FLOP_PER_PAIR_FORCE = 93              # Eq. 3-6, 8-10 per pair
FLOP_PER_PAIR_TEST = 13               # exact object-object test per found pair (single pass)

KERNEL_NAMES = ("M4", "M5", "M6", "Wendland C2", "Wendland C4", "Wendland C6")   # FLOP_PER_PAIR_* below are the M4 counts
# dram__bytes_read.sum + dram__bytes_write.sum per launch, copied from the committed ncu --set full capture of this
# workload: NOT measured by this run (bench.py never runs under a profiler); only quoted when bench runs that workload
NCU_TRAFFIC_SOURCE = "profiles/r2_ncu_all.md"
NCU_TRAFFIC_BYTES_CUBE256 = {"forces": 6.54e9, "traverse": 4.71e9, "density": 5.10e9}   # profiles/r2_ncu_all.md rows 24, 19, 21


def reduce_over_ranks(ms_local: float, n_local: float, world: int, device):
    """Whole-job aggregate: max over ranks of the device time, sum over ranks of the particles stepped."""
    import torch
    import torch.distributed as dist
    tmax = torch.tensor([ms_local], dtype=torch.float64, device=device)
    ntot = torch.tensor([float(n_local)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(ntot, op=dist.ReduceOp.SUM)
    return float(tmax.item()), float(ntot.item())


def make_workload(name: str, seed_offset: int = 0):
    from paper_2503_09713_b200 import workloads as W
    seed = W.DEFAULT_SEED + seed_offset
    if name.startswith("cube"):
        n = int(name[4:])
        return W.cube(n, jitter=0.1, seed=seed, steps=5, name=f"C2-recipe uniform periodic cube {n}^3")
    if name == "sod":
        return W.config(1)
    if name.startswith("sedov"):   # the paper's timing set-up: both CFL numbers 1e-3
        return W.sedov(int(name[5:] or 256), cfl=1e-3, name=f"Sedov-Taylor blast, HCP lattice, n_side {name[5:] or 256}")
    if name.startswith("disc"):
        n = int(name[4:] or 10_000_000)
        return W.disc(n, seed=seed)
    if name == "c0":
        return W.config(0)
    raise SystemExit(f"unknown workload {name}")


class ClockSampler(threading.Thread):
    """Samples SM clock, power and throttle reasons during the timed region (B200_PROFILING.md recipe) through NVML
    every 20 ms (nvidia-smi itself takes longer to start than a whole step lasts)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag, self.max_mhz = index, [], False, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            h = nv.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            while not self.stop_flag:
                self.rows.append((float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)),
                                  nv.nvmlDeviceGetPowerUsage(h) / 1000.0,
                                  int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(h))))
                time.sleep(0.02)
        except Exception as e:          # no NVML: report that instead of a clock
            self.err = repr(e)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable: " + getattr(self, "err", "no samples")]}
        bits = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4,
                "hw_power_brake_slowdown": 0x80}
        seen = 0
        for r in self.rows:
            seen |= r[2]
        return {"sm_mhz": float(np.median([r[0] for r in self.rows])), "sm_max_mhz": self.max_mhz,
                "power_w_max": max(r[1] for r in self.rows), "samples": len(self.rows),
                "reasons": [k for k, b in bits.items() if seen & b]}


def host_cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_c0_rate():
    """BASELINE config 0 in full on the oracle: one tree build + density iteration + force evaluation of 16^3 particles."""
    import oracle as O
    from paper_2503_09713_b200 import workloads as W
    w = W.config(0)
    t0 = time.perf_counter()
    O.State(w, "grid")
    dt = time.perf_counter() - t0
    return w.n / dt, dt


def oracle_step_rate(n_side: int, steps: int, warmup: int):
    """Time the oracle (as it stands, 1 thread) on the C2 recipe at n_side^3 particles."""
    import oracle as O
    from paper_2503_09713_b200 import workloads as W
    w = W.cube(n_side, jitter=0.1, steps=steps)
    t_init = time.perf_counter()
    s = O.State(w, "grid")
    t_init = time.perf_counter() - t_init
    for _ in range(warmup):
        s.step()
    t0 = time.perf_counter()
    for _ in range(steps):
        s.step()
    dt = time.perf_counter() - t0
    return w.n * steps / dt, dt / steps, w.n, t_init


def run_reference(args):
    """--impl reference: the oracle on the host cores (reference arm for this tier)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_side = args.ref_side
    rate, s_per_step, n, _ = oracle_step_rate(n_side, args.steps, args.warmup)
    sample = f"C2 recipe at {n_side}^3 = {n} particles (bounded sample of the 256^3 workload), {args.steps} full oracle steps"
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": s_per_step * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload} (oracle sample {n_side}^3)", "n_particles": n, "l2": "n/a (CPU)"},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                             "host_cpu": host_cpu_model()},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def run_sweep(args):
    """BASELINE config 4: the C2 recipe at 64^3 ... 512^3 on one GPU; one JSON line per size with per-kernel times."""
    import torch
    from paper_2503_09713_b200 import binding as B, workloads as W
    torch.cuda.set_device(0)
    for n_side in (64, 128, 256, 384, 512):
        w = W.cube(n_side, jitter=0.1, steps=args.steps)
        try:
            sim = B.Sim.from_workload(w)
        except B.SphError as e:
            print(json.dumps({"sweep_n_side": n_side, "n_particles": w.n, "error": str(e)}))
            break
        n = w.n
        del w
        for _ in range(max(args.warmup, 1)):
            sim.step_leapfrog()
        torch.cuda.synchronize()
        sim.reset_timers()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            sim.step_leapfrog()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        st = sim.stats()
        print(json.dumps({"sweep_n_side": n_side, "n_particles": n, "ms_per_step": ms, "value": n / (ms * 1e-3), "unit": UNIT,
                          "ms_per_kernel": {k[3:]: st[k] / args.steps for k in st if k.startswith("ms_") and k != "ms_total"
                                            and st[k] > 0},
                          "neighbours_mean": st["nbr_mean"], "bytes_allocated": st["bytes_allocated"]}), flush=True)
        sim.close()
        del sim
        torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cube256")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--ref-side", type=int, default=40, help="lattice side of the oracle's bounded sample (--impl reference)")
    ap.add_argument("--cpu-side", type=int, default=64, help="lattice side of the cpu_baseline leg (64 = the smallest point of BASELINE config 4)")
    ap.add_argument("--group-max", type=int, default=0,
                    help="particles per leaf group / bucket, 1..32 (0 = the default 32): the particles-per-leaf sweep of PAPER.md:382")
    ap.add_argument("--leaf-reduction", type=int, default=0,
                    help="0 = off (group_max rule); k >= 1: leaf groups from the paper's Alg. 1 with n_red = k - 1 passes (PAPER.md:911-963)")
    ap.add_argument("--morton-bits", type=int, default=0, help="21 (default) or 10: the paper's 30-bit Morton codes (PAPER.md:582, 378)")
    ap.add_argument("--sph-kernel", type=int, default=0, help="0 M4 (default, the BASELINE configs), 1 M5, 2 M6, 3/4/5 Wendland C2/C4/C6")
    ap.add_argument("--hfact", type=float, default=0.0, help="h_fact (default 1.2; the paper uses 1.0 with M6, PAPER.md:208)")
    ap.add_argument("--sweep", action="store_true", help="BASELINE config 4: sizes 64^3..512^3, one line each")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)

    import torch
    import torch.distributed as dist
    from paper_2503_09713_b200 import binding as B, build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if not os.path.exists(B.LIB_PATH):
        if rank == 0:
            build.build()
        if world > 1:
            dist.barrier()

    w = make_workload(args.workload, seed_offset=rank)
    if args.sph_kernel or args.hfact:      # other kernels: the same particles, h0 rescaled to the chosen h_fact
        hf = args.hfact or w.hfact
        w.h0 = w.h0 * (hf / w.hfact)
        w.kernel, w.hfact = args.sph_kernel, hf
    n = w.n
    sim = B.Sim.from_workload(w, params=B.params_for(w, group_max=args.group_max, morton_bits=args.morton_bits, leaf_reduction=args.leaf_reduction))   # inputs resident in HBM; includes the white step
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        sim.step_leapfrog()
    barrier()
    sim.reset_timers()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        sim.step_leapfrog()
    e1.record(stream)
    barrier()
    sampler.stop_flag = True
    ms = e0.elapsed_time(e1)
    st = sim.stats()
    ms_all, n_all = reduce_over_ranks(ms, n, world, "cuda")
    value = n_all * args.steps / (ms_all * 1e-3)

    # ---- end-to-end through the C ABI with HOST buffers: upload state, step, download results, every step
    e2e = None
    if not args.no_e2e:
        host = sim.get_fields(("pos", "vel", "u", "h", "acc", "dudt"), host=True)
        out = {k: torch.empty_like(v).pin_memory() for k, v in
               sim.get_fields(("pos", "vel", "u", "h", "rho", "acc", "dudt"), host=True).items()}
        h2d = sum(v.numel() * 8 for v in host.values())
        d2h = sum(v.numel() * 8 for v in out.values())
        k_e2e = max(2, min(args.steps, 3))
        for it in range(1 + k_e2e):
            if it == 1:
                barrier()
                t0 = time.perf_counter()
            sim.set_fields(**host)
            sim.step_leapfrog()
            res = sim.get_fields(tuple(out.keys()), host=True, out=out)
            host = {k: res[k] for k in host}     # the downloaded state is the next step's input (no host-side copy)
        barrier()
        t_e2e = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t_e2e, op=dist.ReduceOp.MAX)
        e2e = {"value": n_all * k_e2e / float(t_e2e.item()), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": k_e2e}

    if rank == 0:
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        hbm_src = "measured (MEASURED_PEAKS.json)" if "hbm_gbs" in peaks else "fallback (B200_PROFILING.md)"
        fp64_peak = B.measure_fp64_peak()      # TFLOP/s, DFMA microbenchmark run now on this GPU
        K = args.steps
        pairs = st["n_neighbours"]             # pairs in the cache of the last step (self included)
        # Newton sweeps + the closing pass at the converged h, counted on the device by k_density: mean per particle
        sweeps = st["density_sweeps"] / n if st.get("density_sweeps", 0) > 0 else max(st["h_iter_max"], 1) + 1
        per_stage = {k[3:]: st[k] / K for k in st if k.startswith("ms_") and k != "ms_total"}
        flops = {"density": pairs * (FLOP_PER_PAIR_DENSITY_GATHER + FLOP_PER_PAIR_DENSITY_SWEEP * sweeps),
                 "forces": pairs * FLOP_PER_PAIR_FORCE,
                 "traverse": pairs * FLOP_PER_PAIR_TEST}
        bytes_ = {"keys": 36 * n, "sort": (8 + 24 * st.get("sort_passes", 8)) * n, "permute": 220 * n, "tree": 60 * n, "aabb": 148 * n,
                  "scan": 12 * n, "leapfrog": 272 * n}
        kernels = {}
        per_stage = {k: v for k, v in per_stage.items() if v > 0.0}
        fp32_peak = 148 * 128 * 2 * 1.965e9 * 1e-12     # nominal: 148 SMs x 128 FP32 lanes x 2 x 1.965 GHz
        for k, v in per_stage.items():
            if k == "traverse":     # the pair test runs in packed fp32 (fp64 only for the rare uncertain buckets)
                ach = flops[k] / (v * 1e-3) * 1e-12
                kernels[k] = {"ms": v, "bound": "alu", "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s (fp32, nominal peak)", "frac": ach / fp32_peak}
            elif k in flops:
                ach = flops[k] / (v * 1e-3) * 1e-12
                kernels[k] = {"ms": v, "bound": "alu", "achieved": ach, "peak": fp64_peak, "unit": "TFLOP/s (fp64)", "frac": ach / fp64_peak}
            else:
                ach = bytes_[k] / (v * 1e-3) * 1e-9 if v > 0 else 0.0
                kernels[k] = {"ms": v, "bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak}
        dom = max(per_stage, key=per_stage.get)
        roofline = dict(kernels[dom])
        traffic = NCU_TRAFFIC_BYTES_CUBE256.get(dom) if (args.workload == "cube256" and not args.sph_kernel and not args.hfact
                                                          and args.group_max in (0, 32)) else None
        roofline.update({"kernel": dom, "traffic": traffic, "traffic_unit": "bytes per launch (ncu dram read+write)",
                         "traffic_source": f"{NCU_TRAFFIC_SOURCE} (committed ncu capture of this kernel), not measured by this run" if traffic else None,
                         "peak_note": "hbm peak is the measured copy bandwidth of MEASURED_PEAKS.json, so an hbm frac can read slightly above 1 (nominal 7.7 TB/s)",
                         "peak_source": "sph_measure_fp64_peak DFMA microbenchmark, this run" if dom in flops else hbm_src,
                         "share_of_step": per_stage[dom] / sum(per_stage.values())})
        cpu = None
        if not args.no_cpu_baseline:
            # BASELINE configs on the oracle: config 0 in full (one evaluation of 16^3 particles) and the 64^3 point
            # of config 4 (the C2 recipe), one full leapfrog step after its white step: ~45 s of CPU work in all
            c0_rate, c0_s = oracle_c0_rate()
            rate, s_per_step, n_s, t_init = oracle_step_rate(args.cpu_side, 1, 0)
            cpu = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "host_cpu": host_cpu_model(),
                   "sample": f"BASELINE config 4 point {args.cpu_side}^3 = {n_s} particles (the C2 recipe), 1 full oracle leapfrog step "
                             f"({s_per_step:.1f} s) after its white step ({t_init:.1f} s)",
                   "config0": {"value": c0_rate, "unit": "particles/s per evaluation (build + density + forces)",
                               "seconds": c0_s, "sample": "BASELINE config 0 in full: 16^3 particles, one evaluation"}}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_all / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "n_particles": n, "neighbours_mean": st["nbr_mean"], "kernel": KERNEL_NAMES[args.sph_kernel], "group_max": args.group_max or 32, "morton_bits": args.morton_bits or 21, "leaf_reduction": args.leaf_reduction, "n_groups": st["n_groups"],
                           "density_sweeps_mean": sweeps, "cache_pairs": pairs, "cache_pairs_inner": st.get("n_inner", 0),
                           "hfact": w.hfact, "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": "inputs (~0.8 kB/particle resident) larger than the 126 MB L2; no flush",
                           "restarts_last_step": st["restarts"], "h_iter_max": st["h_iter_max"]},
                "clocks": sampler.summary(), "e2e": e2e, "gpu_launches": int(st["kernel_launches"]),
                "roofline": roofline, "kernels": kernels, "cpu_baseline": cpu,
                "context": {"paper_a100_particles_per_s": 12e6, "fp64_peak_tflops_measured": fp64_peak,
                            "hbm_peak_gbs": hbm_peak, "bytes_allocated": st["bytes_allocated"]}}
        print(json.dumps(line))
    sim.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
