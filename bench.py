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
NOMINAL_HBM_GBS = 8000.0  # north_star: "B200's ~8 TB/s peak"


def algorithmic_bytes(n: int, g: int, grad_real: bool = False) -> dict:
    """SURVEY 8(d) / DESIGN.md "Algorithmic bytes": what the method itself must move (fp32), per stage."""
    ab = {
        "bin": 12 * n + 16 * n,            # the build's own step: one read of the positions + the records written
                                           # (single-pass bucketed sort; its zero-fill of the mesh is not counted)
        "assign": 12 * n + 4 * g,          # positions in, mesh written once
        "fft_fwd": 8 * g,                  # floor: one read + one write
        "kspace": 4 * g + 12 * g,
        "fft_inv": 24 * g,
        "interp": 12 * n + 12 * g + 12 * n,  # positions + 3 meshes in, forces out
        # reverse mode (SURVEY 8(d) "force-VJP extra")
        "vjp_scatter": 24 * n + 12 * g,    # positions + cotangents in, 3 meshes out
        "vjp_kspace": 24 * g + 16 * g + 8 * g,  # 3 R2C floors, transposed kernel 12G in + 4G out, 1 C2R floor
        "vjp_gather": 36 * n + 16 * g,     # positions, cotangents, position cotangents out; 4 meshes in
        # DKD elementwise pass: X, V read, X written
        "step": 36 * n,
    }
    if grad_real:  # PM_FLAG_GRAD_REAL: potential only through Fourier space, stencil in real space
        ab.update(kspace=4 * g + 4 * g, fft_inv=8 * g, gradient=4 * g + 12 * g)  # (the VJP stays in Fourier space)
    return ab


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


def oracle_sample_run(cfg_name: str, n_p: int, fft_workers: int = 1):
    """One oracle force evaluation of the same configuration at reduced size; returns (seconds, particles).
    fft_workers != 1 runs the oracle's FFT library step on that many host threads (-1: all); its scatter / gather
    loops are single-threaded NumPy by construction."""
    from oracle import pm_oracle as po
    from pm_inputs import generators as gen

    pos, c = gen.make_config_positions(cfg_name, n_p=n_p)
    old = po.FFT_WORKERS
    po.FFT_WORKERS = fft_workers
    try:
        t0 = time.perf_counter()
        po.force(pos, c["m"], c["box"], worder=c["worder"], interlace=c["interlace"], grad_order=c["grad_order"],
                 lap_order=c["lap_order"], deconv_pow=c["deconv_pow"])
        return time.perf_counter() - t0, pos.shape[0]
    finally:
        po.FFT_WORKERS = old


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


def csrc_fingerprint() -> str:
    """Hash of the kernel sources: an ncu traffic figure is only quoted for the library it was measured on."""
    import hashlib

    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2510_05206_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def load_peak():
    peaks_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(peaks_path):
        return float(json.load(open(peaks_path))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (burst copy)"
    return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


def make_positions(gen, name, rank, n_p=0):
    c = dict(gen.CONFIGS[name])
    if n_p:
        return gen.make_config_positions(name, n_p=n_p)
    c["seed"] = replica_seed(c["seed"], rank)
    if c.get("clustered"):
        pos = gen.clustered_halos(c["n_p"] ** 3, c["m"], c["box"], c["seed"],
                                  lattice_shape=(c["n_p"], c["n_p"], c["n_p"] // 2), rms_cells=c["rms"])
    else:
        pos = gen.lattice_displaced(c["n_p"], c["m"], c["box"], c["rms"], c["seed"])
    return pos, c


def params_for(pm, c, n, flags=0):
    return pm.PMParams(m=c["m"], box=c["box"], max_particles=n, worder=c.get("worder", 2),
                       interlace=c.get("interlace", 0), deconv_pow=c.get("deconv_pow", 2),
                       grad_order=c.get("grad_order", 0), lap_order=c.get("lap_order", 0),
                       method=1 if c.get("nufft") else 0, nufft_sigma=c.get("sigma", 2.0),
                       nufft_eps=c.get("eps", 1e-6), nufft_width=c.get("width", 0), flags=flags)


def stage_table(stage_ms, ab, peak, names):
    out = {}
    for k in names:
        if stage_ms.get(k, 0.0) > 0 and k in ab:
            gbs = ab[k] / (stage_ms[k] * 1e-3) / 1e9
            out[k] = {"ms": round(stage_ms[k], 4), "alg_GB": round(ab[k] / 1e9, 4), "GBps": round(gbs, 1),
                      "frac": round(gbs / peak, 4), "frac_nominal_8TBps": round(gbs / NOMINAL_HBM_GBS, 4)}
        elif stage_ms.get(k, 0.0) > 0:
            out[k] = {"ms": round(stage_ms[k], 4)}
    return out


FORCE_STAGES = ("bin", "assign", "fft_fwd", "kspace", "fft_inv", "gradient", "interp")
VJP_STAGES = FORCE_STAGES[:-1] + ("vjp_scatter", "vjp_kspace", "vjp_gather")


def time_call(torch, fn, steps, warmup, barrier=None):
    """ms per call: `steps` calls between two CUDA events on the current stream (the stream the library launches on)."""
    for _ in range(warmup):
        fn()
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        fn()
    e1.record()
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    return e0.elapsed_time(e1) / steps


def profile_stages(pm, ctx, fn, steps):
    """Per-stage CUDA-event durations from a separate pass (events are only recorded here, never in a timed loop)."""
    pm.pm_set_profiling(ctx, True)
    acc = {k: 0.0 for k in pm.STAGE_NAMES}
    launches = 0
    for _ in range(steps):
        fn()
        ms, launches = pm.pm_get_stage_ms(ctx)
        for k in acc:
            acc[k] += ms[k] / steps
    pm.pm_set_profiling(ctx, False)
    return acc, launches


def run_config(torch, pm, gen, name, rank, local, peak, steps, warmup, with_vjp, flags=0, n_p=0, pos_c=None):
    """Force (and VJP) throughput and stage times of one named configuration; its own clock sample."""
    pos_np, c = pos_c if pos_c is not None else make_positions(gen, name, rank, n_p)
    n = pos_np.shape[0]
    ctx = pm.pm_create(params_for(pm, c, n, flags))
    g = ctx.G  # mesh the FFTs and the scatter / gather run on (NUFFT: the fine grid)
    pos = torch.from_numpy(pos_np).cuda()
    out = torch.empty(n, 3, device="cuda")
    sampler = ClockSampler(local)
    sampler.start()
    ms = time_call(torch, lambda: pm.pm_force(ctx, pos, out), steps, warmup)
    st, launches = profile_stages(pm, ctx, lambda: pm.pm_force(ctx, pos, out), max(2, steps // 2))
    ab = algorithmic_bytes(n, g, bool(flags & pm.FLAG_GRAD_REAL))
    res = {"workload": f"{name}: N={c['n_p']}^3, mesh {c['m']}^3" + (", NUFFT fine grid %d^3 w=%d" % (ctx.mg, ctx.nufft_width) if c.get("nufft") else ""),
           "particles": n, "ms_per_step": round(ms, 4), "particles_per_s": n / (ms * 1e-3), "launches_per_step": launches,
           "stages": stage_table(st, ab, peak, FORCE_STAGES)}
    if c.get("nufft"):  # spreading / interpolation against the measured shared-memory ceilings, not HBM
        w3 = ctx.nufft_width ** 3
        atom, lds = pm.pm_smem_peak(ctx, 1), pm.pm_smem_peak(ctx, 0)
        res["smem_ceiling"] = {"atomics_per_s": atom, "loads_per_s": lds, "how": "pm_smem_peak: conflict-free micro-kernel"}
        for k, ops, ceil in (("assign", w3 * n, atom), ("interp", 3 * w3 * n, lds)):
            if k in res["stages"]:
                res["stages"][k].update(bound="smem", lane_ops_per_s=ops / (st[k] * 1e-3), frac_smem=round(ops / (st[k] * 1e-3) / ceil, 4))
    if with_vjp:
        lam = torch.from_numpy(gen.gaussian_cotangent(n, c.get("cot_seed", 2000))).cuda()
        ms_v = time_call(torch, lambda: pm.pm_force_vjp(ctx, pos, lam, out), max(2, steps // 2), 2)
        stv, _ = profile_stages(pm, ctx, lambda: pm.pm_force_vjp(ctx, pos, lam, out), 2)
        res["vjp"] = {"ms_per_call": round(ms_v, 4), "stages": stage_table(stv, ab, peak, VJP_STAGES)}
        del lam
    res["clocks"] = sampler.stop()
    pm.pm_destroy(ctx)
    del pos, out
    torch.cuda.empty_cache()
    return res


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
    peak, peak_src = load_peak()

    # ---- workload: one independent replica per rank (replicas only, no collective) ----------
    pos_np, c = make_positions(gen, args.config, rank, args.n_p)
    n = pos_np.shape[0]
    g = c["m"] ** 3
    ctx = pm.pm_create(params_for(pm, c, n))
    pos_host = torch.from_numpy(pos_np).pin_memory()
    force_host = torch.empty(n, 3, dtype=torch.float32).pin_memory()
    pos = pos_host.cuda()
    force = torch.empty(n, 3, device="cuda")

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing (no events inside the library during the timed loop) ------------------------
    pm.pm_set_profiling(ctx, False)
    for _ in range(args.warmup):
        pm.pm_force(ctx, pos, force)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ms_total = time_call(torch, lambda: pm.pm_force(ctx, pos, force), args.steps, 0, barrier) * args.steps
    stage_acc, launches = profile_stages(pm, ctx, lambda: pm.pm_force(ctx, pos, force), args.steps)
    clocks = sampler.stop()

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region) -------------------
    pm.pm_force_host(ctx, pos_host, force_host)  # warm-up (allocates the staging buffers)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(args.steps, 5))
    for _ in range(e2e_steps):
        pm.pm_force_host(ctx, pos_host, force_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    checksum = float(force_host[:: max(1, n // 1000)].double().abs().sum())

    # The same with TWO evaluations in flight (two ctx, two streams, pm_force_host_async): one evaluation cannot overlap
    # its own copies -- every force depends on every position -- but the device-to-host copy of one overlaps the
    # host-to-device copy of the next, so both directions of the host link stay busy.  Every step still copies its own
    # inputs in and its own result out inside the timed region.
    nl = max(2, args.e2e_lanes)
    pipe_ms, pipe_steps, pipe_err = None, nl * max(3, e2e_steps), 0.0
    if not args.no_pipeline:
        lanes = [(ctx, force_host, torch.cuda.Stream())]
        for _ in range(nl - 1):
            lanes.append((pm.pm_create(params_for(pm, c, n)), torch.empty(n, 3, dtype=torch.float32).pin_memory(),
                          torch.cuda.Stream()))
        for cx, fh, s_ in lanes:  # warm-up: staging buffers of the extra ctx, plans, first-launch costs
            with torch.cuda.stream(s_):
                pm.pm_force_host_async(cx, pos_host, fh)
        barrier()
        t0 = time.perf_counter()
        for i in range(pipe_steps):
            cx, fh, s_ = lanes[i % nl]
            with torch.cuda.stream(s_):
                pm.pm_force_host_async(cx, pos_host, fh)
        torch.cuda.synchronize()
        pipe_ms = (time.perf_counter() - t0) * 1e3
        stride = max(1, n // 1000)
        pipe_err = max(float((fh[::stride] - force_host[::stride]).abs().max()) for _, fh, _ in lanes[1:])
        for cx, _, _ in lanes[1:]:
            pm.pm_destroy(cx)
        del lanes

    ms_total, e2e_ms = max_over_ranks([ms_total, e2e_s * 1e3], world, device="cuda")
    if pipe_ms is not None:
        (pipe_ms,) = max_over_ranks([pipe_ms], world, device="cuda")

    # ---- beside the headline (rank 0 of a single-GPU run only; every block is a measurement of this run) ------
    extras = {}
    if rank == 0 and world == 1 and not args.headline_only and not c.get("nufft"):
        lam = torch.from_numpy(gen.gaussian_cotangent(n, 2005)).cuda()
        xbar = torch.empty(n, 3, device="cuda")
        ab = algorithmic_bytes(n, g)
        # reverse mode on the same workload
        ms_v = time_call(torch, lambda: pm.pm_force_vjp(ctx, pos, lam, xbar), 5, 2)
        stv, _ = profile_stages(pm, ctx, lambda: pm.pm_force_vjp(ctx, pos, lam, xbar), 3)
        extras["vjp"] = {"call": "pm_force_vjp (forward meshes recomputed)", "ms_per_call": round(ms_v, 4),
                         "stages": stage_table(stv, ab, peak, VJP_STAGES)}
        pm.pm_bin(ctx, pos)
        pm.pm_force(ctx, pos, force)
        ms_r = time_call(torch, lambda: pm.pm_force_vjp(ctx, pos, lam, xbar), 5, 2)
        extras["vjp"]["ms_per_call_reusing_pinned_force_meshes"] = round(ms_r, 4)
        # one DKD step and one backward-in-time adjoint step on copies of the state
        X, V = pos.clone(), (torch.randn(n, 3, device="cuda") * (0.3 * c["box"] / c["m"]))
        Xs, Vs = lam.clone(), xbar.normal_()
        coef = (0.5, 0.5, 0.97, 0.2)
        ms_s = time_call(torch, lambda: pm.pm_dkd_step(ctx, X, V, *coef), 5, 2)
        ms_a = time_call(torch, lambda: pm.pm_dkd_step_adjoint(ctx, X, V, Xs, Vs, *coef), 3, 1)
        extras["dkd"] = {"step_ms": round(ms_s, 4), "adjoint_step_ms": round(ms_a, 4),
                         "note": "Eq. 2.14 / Table 3 at the headline size; kick, second drift and the alpha*, beta* "
                                 "reductions ride on the gather; the adjoint step shares one set of force meshes "
                                 "between the primal kick-back and the VJP"}
        del X, V, Xs, Vs, lam, xbar
        pm.pm_destroy(ctx)
        ctx = None
        del pos, force
        torch.cuda.empty_cache()
        # the one-C2R variant (PM_FLAG_GRAD_REAL) on the same workload
        extras["variants"] = {"grad_real": run_config(torch, pm, gen, args.config, rank, local, peak, args.steps,
                                                      args.warmup, True, flags=pm.FLAG_GRAD_REAL, n_p=args.n_p,
                                                      pos_c=(pos_np, c))}
        if not args.no_other_configs and not args.n_p:
            oc = {}
            for name, vjp in (("cfg2", False), ("cfg4", True), ("cfg3", True), ("cfg3_paper", True)):
                oc[name] = run_config(torch, pm, gen, name, rank, local, peak, 5, 3, vjp)
            extras["other_configs"] = oc
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    value = whole_job_rate(world, n, args.steps, ms_total)
    e2e_value = whole_job_rate(world, n, e2e_steps, e2e_ms)
    seq = {"value": e2e_value, "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps,
           "call": "pm_force_host, one blocking evaluation after the other"}
    e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 12 * n, "d2h_bytes_per_step": 12 * n,
           "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps, "checksum": checksum, "mode": seq["call"]}
    if pipe_ms is not None:  # the headline end-to-end number: both directions of the host link busy
        e2e.update(value=whole_job_rate(world, n, pipe_steps, pipe_ms), ms_per_step=pipe_ms / pipe_steps,
                   steps=pipe_steps, sequential=seq, max_abs_diff_between_lanes=pipe_err,
                   lanes=nl,
                   mode=f"pm_force_host_async, {nl} evaluations in flight ({nl} ctx on {nl} streams): the D2H copy of "
                        "one overlaps the H2D copy of the next; every step copies its inputs in and its result out")

    # ---- roofline of the dominant hand-written kernel -----------------------------------------------------
    ab = algorithmic_bytes(n, g)
    stages = stage_table(stage_acc, ab, peak, FORCE_STAGES)
    # the dominant hand-written KERNEL: stages that are one kernel launch each (assign = k_scatter_warp / k_scatter,
    # kspace = k_xfft_kspace / k_kspace_fwd, interp = k_gather); "bin" is six launches and is listed in `stages`
    own = {k: v for k, v in stages.items() if k in ("assign", "kspace", "interp")}
    dom = max(own, key=lambda k: own[k]["ms"])
    traffic, traffic_src = None, "none: no ncu capture of this configuration"
    tp = os.path.join(ROOT, "profiles", "dram_traffic_r2.json")  # written from an ncu --set full capture
    if os.path.exists(tp):
        tj = json.load(open(tp))
        if tj.get("csrc_fingerprint") == csrc_fingerprint():
            traffic = tj.get(args.config, {}).get(dom)
            traffic_src = tj.get("source", "")
        else:
            traffic_src = "stale: the kernels changed since the ncu capture in profiles/ (" + tj.get("source", "") + ")"
    kernel_names = {"assign": "k_scatter_warp / k_scatter", "kspace": "k_xfft_kspace (x-FFTs + k-space) or k_kspace_fwd",
                    "interp": "k_gather"}
    roofline = {"bound": "hbm", "kernel": kernel_names[dom], "stage": dom, "achieved": stages[dom]["GBps"],
                "peak": peak, "unit": "GB/s", "frac": stages[dom]["frac"],
                "frac_nominal_8TBps": stages[dom]["frac_nominal_8TBps"], "traffic": traffic,
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum)",
                "traffic_source": traffic_src, "peak_source": peak_src}

    # ---- oracle timed beside it (bounded samples; one core, and its FFT step on all cores) --------------------
    cpu = None
    if not args.no_cpu_baseline and not c.get("nufft"):
        dt, npart = oracle_sample_run(args.config, args.ref_np)
        dta, _ = oracle_sample_run(args.config, args.ref_np, fft_workers=-1)
        cpu = {"value": npart / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": f"{args.config} at n_p={args.ref_np} (N={npart}), one evaluation, {dt:.1f} s; NumPy fp64, "
                         f"single-threaded as it stands",
               "all_cores": {"value": npart / dta, "cores": host_threads(), "seconds": round(dta, 2),
                             "note": "same evaluation with the FFT library step on all host threads "
                                     "(scipy.fft workers); the oracle's scatter / gather loops are single-threaded "
                                     "NumPy by construction"}}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": f"{args.config}: N={c['n_p']}^3 particles, mesh {c['m']}^3, box {c['box']}, "
                               f"worder={c.get('worder', 2)}, grad_order={c.get('grad_order', 0)}, "
                               f"deconv_pow={c.get('deconv_pow', 2)}, interlace={c.get('interlace', 0)}"
                               + (", NUFFT" if c.get("nufft") else "") + "; reference path (three inverse FFTs)",
                   "particles": n, "mesh_cells": g, "replicas": world,
                   "l2_policy": "inputs larger than L2 (positions 1.6 GB, meshes 0.5 GB each); no flush",
                   "paper_context": "A100 40GB, JAX: 0.2 s/step at this setting (PAPER.md:552) = 6.7e8 particles/s"},
        "clocks": clocks,
        "e2e": e2e,
        "gpu_launches": launches * args.steps,
        "roofline": roofline,
        "stages": stages,
        "cpu_baseline": cpu,
    }
    line.update(extras)
    print(json.dumps(line))
    if ctx is not None:
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
    ap.add_argument("--e2e-lanes", dest="e2e_lanes", type=int, default=3,
                    help="evaluations in flight in the pipelined end-to-end measurement (one ctx and stream each)")
    ap.add_argument("--no-pipeline", dest="no_pipeline", action="store_true",
                    help="skip the two-evaluations-in-flight end-to-end measurement (second ctx)")
    ap.add_argument("--config", default="headline", help="name in pm_inputs.CONFIGS")
    ap.add_argument("--n-p", dest="n_p", type=int, default=0, help="reduced particles per dim (tests only)")
    ap.add_argument("--ref-np", dest="ref_np", type=int, default=0,
                    help="oracle sample size, particles per dim (default 192 beside our arm, 128 per reference step)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--headline-only", action="store_true", help="skip the VJP / DKD / variant / other-config blocks")
    ap.add_argument("--no-other-configs", action="store_true", help="skip cfg2 / cfg4 / cfg3 beside the headline")
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
