#!/usr/bin/env python
"""bench.py -- whole-path throughput of the PM force evaluation (BASELINE.json metric).

    python bench.py --gpus 1 --steps K --warmup W            # our arm (libpmforce.so on the GPU)
    python bench.py --impl reference --steps K --warmup W    # the fp64 oracle on the host cores
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N   # N independent replicas

A "step" is one complete force evaluation A(X): bin, assign, R2C FFT, Fourier-space kernel, three C2R FFTs,
gather (include/pmforce.h: pm_force).  The N = 1 workload is the north_star target ("headline" in
pm_inputs.CONFIGS): N = 512^3 particles, 512^3 mesh, CIC, 4th-order gradient kernel, deconvolved, fp32; a
seeded lattice with rms 1-cell Gaussian displacement.  One JSON line on stdout.
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

METRIC = "pm_force_particles_per_s"
UNIT = "particles/s"


# ---------------------------------------------------------------------------------------------------------
def algorithmic_bytes(n: int, g: int) -> dict:
    """SURVEY 8(d) / DESIGN.md "Algorithmic bytes": what the method itself must move (fp32), per stage."""
    return {
        "bin": 12 * n + 16 * n,            # the build's own step: one read of the positions + the records written
                                           # (single-pass bucketed sort; its zero-fill of the mesh is not counted)
        "assign": 12 * n + 4 * g,          # positions in, mesh written once
        "fft_fwd": 8 * g,                  # floor: one read + one write
        "kspace": 4 * g + 12 * g,
        "fft_inv": 24 * g,
        "interp": 12 * n + 12 * g + 12 * n,  # positions + 3 meshes in, forces out
    }


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_sample_run(cfg_name: str, n_p: int):
    """One oracle force evaluation of the same configuration at reduced size; returns (seconds, particles)."""
    from oracle import pm_oracle as po
    from pm_inputs import generators as gen

    pos, c = gen.make_config_positions(cfg_name, n_p=n_p)
    t0 = time.perf_counter()
    po.force(pos, c["m"], c["box"], worder=c["worder"], interlace=c["interlace"], grad_order=c["grad_order"],
             lap_order=c["lap_order"], deconv_pow=c["deconv_pow"])
    return time.perf_counter() - t0, pos.shape[0]


def replica_seed(seed: int, rank: int) -> int:
    """Seed of rank's independent replica (replicas only, no data-path collective)."""
    return int(seed) + 100 * int(rank)


def max_over_ranks(values, world: int, device="cpu"):
    """Element-wise MAX of per-rank timings over all ranks (the only collective of the bench)."""
    import torch
    import torch.distributed as dist

    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def whole_job_rate(world: int, units_per_rank: int, steps: int, ms_total: float) -> float:
    """Units all ranks processed / the slowest rank's time (weak scaling: per-rank work is fixed)."""
    return world * units_per_rank * steps / (ms_total * 1e-3)


def host_threads() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


# ---------------------------------------------------------------------------------------------------------
def run_reference(args) -> int:
    """The oracle as it stands, on the host cores, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n_p = args.ref_np
    times, npart = [], 0
    for i in range(args.warmup + args.steps):
        dt, npart = oracle_sample_run(args.config, n_p)
        if i >= args.warmup:
            times.append(dt)
    total = float(np.sum(times))
    value = npart * len(times) / total
    from pm_inputs import generators as gen
    c = gen.CONFIGS[args.config]
    sample = (f"{args.config} at n_p={n_p} (N={npart}, mesh {int(round(n_p * c['m'] / c['n_p']))}^3), same kernels "
              f"and cell size; NumPy oracle, fp64")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 0, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.config} (oracle sample)", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_ours(args) -> int:
    import torch
    import torch.distributed as dist

    import paper_2510_05206_b200 as pm
    from pm_inputs import generators as gen

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback for the force path")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    # ---- workload: one independent replica per rank (replicas only, no collective) ----------
    c = dict(gen.CONFIGS[args.config])
    if args.n_p:
        pos_np, c = gen.make_config_positions(args.config, n_p=args.n_p)
    else:
        c["seed"] = replica_seed(c["seed"], rank)
        if c.get("clustered"):
            pos_np = gen.clustered_halos(c["n_p"] ** 3, c["m"], c["box"], c["seed"],
                                         lattice_shape=(c["n_p"], c["n_p"], c["n_p"] // 2), rms_cells=c["rms"])
        else:
            pos_np = gen.lattice_displaced(c["n_p"], c["m"], c["box"], c["rms"], c["seed"])
    n = pos_np.shape[0]
    g = c["m"] ** 3
    params = pm.PMParams(m=c["m"], box=c["box"], max_particles=n, worder=c.get("worder", 2),
                         interlace=c.get("interlace", 0), deconv_pow=c.get("deconv_pow", 2),
                         grad_order=c.get("grad_order", 0), lap_order=c.get("lap_order", 0),
                         method=1 if c.get("nufft") else 0, nufft_sigma=c.get("sigma", 2.0),
                         nufft_eps=c.get("eps", 1e-6))
    ctx = pm.pm_create(params)
    pos_host = torch.from_numpy(pos_np).pin_memory()
    force_host = torch.empty(n, 3, dtype=torch.float32).pin_memory()
    pos = pos_host.cuda()
    force = torch.empty(n, 3, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing ---------------------------------------------------------------------------
    pm.pm_set_profiling(ctx, True)
    for _ in range(args.warmup):
        pm.pm_force(ctx, pos, force)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stage_acc = {k: 0.0 for k in pm.STAGE_NAMES}
    launches = 0
    barrier()
    e0.record()
    for _ in range(args.steps):
        pm.pm_force(ctx, pos, force)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    # per-stage durations: a separate profiled pass (pm_get_stage_ms synchronises, so not inside the timed loop)
    for _ in range(args.steps):
        pm.pm_force(ctx, pos, force)
        ms, nl = pm.pm_get_stage_ms(ctx)
        launches = nl
        for k in stage_acc:
            stage_acc[k] += ms[k] / args.steps
    clocks = sampler.stop()

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region) -------------------
    pm.pm_set_profiling(ctx, False)
    pm.pm_force_host(ctx, pos_host, force_host)  # warm-up (allocates the staging buffers)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(args.steps, 5))
    for _ in range(e2e_steps):
        pm.pm_force_host(ctx, pos_host, force_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    checksum = float(force_host[:: max(1, n // 1000)].double().abs().sum())

    ms_total, e2e_ms = max_over_ranks([ms_total, e2e_s * 1e3], world, device="cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    value = whole_job_rate(world, n, args.steps, ms_total)
    e2e_value = whole_job_rate(world, n, e2e_steps, e2e_ms)

    # ---- roofline of the dominant hand-written kernel -----------------------------------------------------
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        peak = float(json.load(open(peaks_path))["hbm_gbs"])
        peak_src = "MEASURED_PEAKS.json hbm_gbs (burst copy)"
    else:
        peak, peak_src = 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"
    ab = algorithmic_bytes(n, g)
    stages = {}
    for k in ("bin", "assign", "fft_fwd", "kspace", "fft_inv", "interp"):
        if stage_acc[k] > 0:
            gbs = ab[k] / (stage_acc[k] * 1e-3) / 1e9
            stages[k] = {"ms": round(stage_acc[k], 4), "alg_GB": round(ab[k] / 1e9, 4), "GBps": round(gbs, 1),
                         "frac": round(gbs / peak, 4)}
    # the dominant hand-written KERNEL: stages that are one kernel launch each (assign = k_scatter_warp / k_scatter,
    # kspace = k_xfft_kspace / k_kspace_fwd, interp = k_gather); "bin" is six launches and is listed in `stages`
    own = {k: v for k, v in stages.items() if k in ("assign", "kspace", "interp")}
    dom = max(own, key=lambda k: own[k]["ms"])
    traffic = None
    tp = os.path.join(ROOT, "profiles", "dram_traffic.json")  # written from an ncu --set full capture
    if os.path.exists(tp):
        traffic = json.load(open(tp)).get(args.config, {}).get(dom)
    kernel_names = {"assign": "k_scatter_warp / k_scatter", "kspace": "k_xfft_kspace (x-FFTs + k-space) or k_kspace_fwd",
                    "interp": "k_gather"}
    roofline = {"bound": "hbm", "kernel": kernel_names[dom], "stage": dom, "achieved": stages[dom]["GBps"],
                "peak": peak, "unit": "GB/s", "frac": stages[dom]["frac"], "traffic": traffic,
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                "peak_source": peak_src}

    # ---- oracle timed beside it (bounded sample) ----------------------------------------------------------
    cpu = None
    if not args.no_cpu_baseline and not c.get("nufft"):
        dt, npart = oracle_sample_run(args.config, args.ref_np)
        cpu = {"value": npart / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{args.config} at n_p={args.ref_np} (N={npart}), one evaluation, {dt:.1f} s; "
                         f"NumPy fp64, single-threaded ({host_threads()} host threads available)"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.config}: N={c['n_p']}^3 particles, mesh {c['m']}^3, box {c['box']}, "
                               f"worder={c.get('worder', 2)}, grad_order={c.get('grad_order', 0)}, "
                               f"deconv_pow={c.get('deconv_pow', 2)}, interlace={c.get('interlace', 0)}"
                               + (", NUFFT" if c.get("nufft") else ""),
                   "particles": n, "mesh_cells": g, "replicas": world,
                   "l2_policy": "inputs larger than L2 (positions 1.6 GB, meshes 0.5 GB each); no flush",
                   "paper_context": "A100 40GB, JAX: 0.2 s/step at this setting (PAPER.md:552) = 6.7e8 particles/s"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 12 * n, "d2h_bytes_per_step": 12 * n,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps, "checksum": checksum},
        "gpu_launches": launches * args.steps,
        "roofline": roofline,
        "stages": stages,
        "cpu_baseline": cpu,
    }
    print(json.dumps(line))
    pm.pm_destroy(ctx)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main(argv=None) -> int:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--config", default="headline", help="name in pm_inputs.CONFIGS")
    ap.add_argument("--n-p", dest="n_p", type=int, default=0, help="reduced particles per dim (tests only)")
    ap.add_argument("--ref-np", dest="ref_np", type=int, default=0,
                    help="oracle sample size, particles per dim (default 192 beside our arm, 128 per reference step)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args(argv)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3  # timing rule: at least 3 warm-up steps
    if not args.ref_np:
        args.ref_np = 128 if args.impl == "reference" else 192
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    raise SystemExit(main())
