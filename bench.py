#!/usr/bin/env python
"""bench.py -- RAAR frame-iterations/s of the SHARP projection loop (arXiv 1602.01448) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2|3|4|5|1] [--impl ours|reference]

A "step" is one pass of the whole hot path over one synthetic scan: z0 = Q psi0
(split), `iters` RAAR iterations (fused FFT / magnitude projection / IFFT / frame combine + gather overlap with
the object-space combine [+ Eq. 10 probe refinement on the blind configs]) and the three error norms.  The
metric is frame-iterations/s = ranks * K_frames * iters * steps / time.

  value      inputs resident in HBM when the timed region starts; CUDA events on the library's stream
  e2e        the same metric through sharp_reconstruct_host: HOST (pinned) intensities and probe in, HOST object,
             probe and residuals out, copies inside the timed region
  roofline   the fused per-frame kernel: algorithmic bytes (20 B per frame pixel) / its average
             launch duration, measured with CUDA events around each of its launches in a second pass over the
             same steps, against MEASURED_PEAKS.json's HBM copy bandwidth
  cpu_baseline / --impl reference   the CPU oracle (oracle/, double precision, OpenMP over the host cores) as it
             stands, on a bounded sub-raster sample of the same recipe

  secondary  the default run (config 2, m = 128) also measures config 4 (m = 256, full size) the same way and
             reports it under `secondary` (BASELINE.json's metric names both sizes); --no-secondary skips it

N > 1 (torchrun): every rank reconstructs its own scan (same recipe, seed + 1000 rank), no data-path collective:
weak scaling.  Timing is the max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "RAAR frame-iterations/s"
UNIT = "frame-iterations/s"
BYTES_PER_PX_FRAME_KERNEL = 20          # read c (8) + read a (4) + write c' (8): SURVEY.md 8(d) "M20"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2,
                    help="BASELINE.json configs[n-1]; 2 = medium raster (default); 6 = the paper's Fig. 3 shape (periodic)")
    ap.add_argument("--iters", type=int, default=0, help="RAAR iterations per step (0 = the config's own count)")
    ap.add_argument("--grid", type=int, default=0, help="reduce the raster to grid x grid (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the config-4 (m = 256) block of the default run")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: ONE scan, its frames partitioned over the ranks by region, object numerator all-reduced "
                         "every iteration (sharp_set_sharded; strong scaling) instead of one independent scan per rank")
    return ap.parse_args()


def workload(args, rank=0):
    import synth
    cfg = synth.config(args.config)
    if args.grid:
        cfg = synth.reduced(cfg, args.grid)
    if rank:
        import dataclasses
        cfg = dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)
    iters = args.iters or cfg.iters
    return cfg, iters


def workload_name(cfg, iters):
    return (f"{cfg.name}: {cfg.K} frames {cfg.m}x{cfg.m} c64, object {cfg.shape[0]}x{cfg.shape[1]}, "
            f"beta {cfg.beta}, {iters} RAAR iterations/step, probe "
            + (f"refined every {cfg.refine_every}" if cfg.refine_every else "fixed")
            + (", periodic boundary" if cfg.periodic else ""))


# ---- the CPU oracle, timed as it stands (cpu_baseline and --impl reference) ---------------------------------------
def oracle_sample(args):
    """A sub-raster of the same recipe that the oracle advances in a few seconds per step."""
    import synth
    cfg = synth.config(args.config)
    g = {64: 10, 128: 12, 256: 6, 512: 9}[cfg.m]          # frames: 100 / 144 / 36 / 9
    if cfg.periodic:
        g = 16                                              # the torus must stay larger than the frame: 160 x 160
    scfg = synth.reduced(cfg, min(g, cfg.grid))
    its = 2 if cfg.m <= 128 else 1
    return scfg, its


def time_oracle(args, steps, warmup):
    import synth
    from oracle import sharp_oracle as orc
    orc.build()
    scfg, its = oracle_sample(args)
    pos, shape, I, w0, obj, wt = synth.make(scfg)
    o = orc.Oracle(scfg.m, pos, shape, I, w0, refine_every=scfg.refine_every)
    for _ in range(warmup):
        o.iterate(its, scfg.beta)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.iterate(its, scfg.beta)
    dt = time.perf_counter() - t0
    eps = o.errors()
    return dict(value=scfg.K * its * steps / dt, unit=UNIT, cores=orc.n_threads(), kind="oracle",
                sample=f"{scfg.K} frames {scfg.m}x{scfg.m} ({scfg.name}, same recipe), {its} RAAR iteration(s)/step, "
                       f"{steps} timed steps after {warmup} warm-up, C double precision + OpenMP",
                seconds=dt, ms_per_step=1e3 * dt / steps, eps=[float(e) for e in eps]), scfg, its


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg, iters = workload(args)
    base, scfg, its = time_oracle(args, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": base["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": base["ms_per_step"], "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg, iters), "timed_sample": base["sample"]},
        "cpu_baseline": {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": base["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ---- clocks during the timed region -------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.FIELDS}",
                                       "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 8:
                continue
            try:
                sm.append(float(parts[0])); smax.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for nm, v in zip(names, parts[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        # "under load": samples drawing more than half of the peak power seen
        pmax = max(power)
        load = [s for s, pw in zip(sm, power) if pw >= 0.5 * pmax] or sm
        return {"sm_mhz": statistics.median(load), "sm_max_mhz": max(smax), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": pmax}


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, torch copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def max_over_ranks(x, dist, device):
    """MAX of a scalar over all ranks (identity when not distributed)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, K, iters, steps, ms):
    """whole-job frame-iterations/s: every rank advanced K frames by iters*steps iterations in `ms` (max over ranks)."""
    return world * K * iters * steps / (ms * 1e-3)


# ---- our arm ----------------------------------------------------------------------------------------------------
def spans_per_step(cfg, iters):
    """kernel launches the library brackets with events in one step (sharp_profile caps the record at 8192)."""
    per_it = 2 + (2 if cfg.refine_every else 0)      # frame + overlap (+ Eq. 10 partial sums + final)
    return per_it * iters + 8


def measure(args, config_number, steps, warmup, rank, world, dev, dist, want_e2e, sample_clocks):
    """One workload (BASELINE.json configs[config_number-1]) on this rank: device-resident throughput, per-kernel
    durations and the roofline of the fused frame kernel, and the host-buffer end-to-end number."""
    import dataclasses
    import torch
    import paper_1602_01448_b200 as sharp
    import synth

    cfg = synth.config(config_number)
    if args.grid:
        cfg = synth.reduced(cfg, args.grid)
    sharded = bool(args.sharded) and dist is not None
    if rank and not sharded:
        cfg = dataclasses.replace(cfg, seed=cfg.seed + 1000 * rank)
    iters = args.iters or cfg.iters
    pos, shape, I, w0, obj, wt = synth.make(cfg)
    K_total = cfg.K
    if sharded:                                  # this rank's region of the one scan
        from paper_1602_01448_b200.sharding import partition_by_region
        mine = partition_by_region(pos, world)[rank]
        pos, I = pos[mine], np.ascontiguousarray(I[mine])
    K, m = len(pos), cfg.m
    I_host = torch.from_numpy(np.ascontiguousarray(I)).pin_memory()
    w_host = torch.from_numpy(np.ascontiguousarray(w0)).pin_memory()
    rec = sharp.Reconstruction(m, pos, shape, device=dev, periodic=bool(cfg.periodic))
    if sharded:
        rec.set_sharded(lambda t: dist.all_reduce(t), K_total)
    rec.set_probe_refine(cfg.refine_every)
    I_dev = I_host.to(dev)
    rec.set_intensities(I_dev)
    w_dev = w_host.to(dev)
    rec.set_probe(w_dev)

    def step():
        if cfg.refine_every:                 # the blind loop replaces the probe: every step restarts from w0
            rec.set_probe(w_dev)
        rec.set_object(None)                 # a1: z0 = Q psi0, flat start
        rec.iterate(iters, cfg.beta)         # a2-a6 (+ a7 on blind configs)
        return rec.errors()                  # a8 (synchronises)

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(max(warmup, 3)):
        eps = step()

    # ---- timed region: device-resident ------------------------------------------------------------------------
    sampler = ClockSampler(dev.index) if sample_clocks else None
    barrier()
    l0 = rec.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        eps = step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = rec.launch_count() - l0
    clocks = sampler.stop() if sampler else None
    ms = max_over_ranks(ms, dist, dev)
    value = job_value(1 if sharded else world, K_total, iters, steps, ms)

    # ---- second pass over the same steps with events around every launch: per-kernel durations -----------------
    rec.profile(True)
    nprof = max(1, min(steps, 8192 // spans_per_step(cfg, iters)))
    for _ in range(nprof):
        step()
    prof = rec.profile_read()
    rec.profile(False)
    f_ms, f_n = prof["frame"]
    peak, peak_src = measured_peak()
    alg_bytes = BYTES_PER_PX_FRAME_KERNEL * K * m * m
    achieved = alg_bytes / (f_ms / f_n * 1e-3) / 1e9 if f_n else None
    tot_ms = sum(v[0] for v in prof.values())
    roofline = {
        "kernel": ("k_frame_r" if m <= 128 else "k_frame_s") + "<FRAME_ITER> (fused split-add / FFT2 / magnitude "
                  "projection / IFFT2 / frame combine)",
        "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": (achieved / peak) if achieved else None, "traffic": None,
        "frac_of_nominal_8TBs": (achieved / 8000.0) if achieved else None,
        "peak_source": peak_src, "algorithmic_bytes_per_launch": alg_bytes,
        "avg_launch_ms": f_ms / f_n if f_n else None, "launches_timed": f_n,
        "share_of_kernel_time": {k: (v[0] / tot_ms if tot_ms else None) for k, v in prof.items()},
        "avg_ms": {k: (v[0] / v[1] if v[1] else None) for k, v in prof.items()},
    }
    traffic_file = os.path.join(ROOT, "profiles", f"traffic_cfg{config_number}.json")
    if os.path.exists(traffic_file) and not args.grid:
        # DRAM bytes per launch of the frame kernel, read off this round's committed `ncu --set full` capture of the
        # same kernel at this config (profiles/r02_summary.md names the command); null when there is no capture
        try:
            with open(traffic_file) as f:
                t = json.load(f)
            # the capture may hold fewer frames per launch than this workload (config 4 is captured on a 40 x 40
            # sub-raster): DRAM bytes per frame x the frames of this launch
            roofline["traffic"] = int(t["frame_kernel_dram_bytes_per_frame"] * K)
            roofline["traffic_source"] = t.get("source") + f"; {t['frames_per_launch_in_capture']} frames per launch in the capture, scaled to {K}"
        except Exception:
            pass

    # ---- end to end: host buffers in, host buffers out ---------------------------------------------------------
    e2e = None
    if want_e2e:
        n_e2e = max(1, min(steps, 5))
        rec.reconstruct_host(I_host, w_host, iters, cfg.beta)      # warm-up (allocates the pinned outputs)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            psi, w, eps_h = rec.reconstruct_host(I_host, w_host, iters, cfg.beta)   # synchronous
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dt, dist, dev)
        e2e = {"value": (1 if sharded else world) * K_total * iters * n_e2e / dt, "unit": UNIT,
               "h2d_bytes_per_step": int(I_host.numel() * 4 + w_host.numel() * 8),
               "d2h_bytes_per_step": int(shape[0] * shape[1] * 8 + m * m * 8 + 12),
               "steps": n_e2e, "ms_per_step": 1e3 * dt / n_e2e,
               "api": "sharp_reconstruct_host (pinned host intensities + probe in; object, probe, residuals out)"}
    eps0 = None
    if hasattr(rec, "eps0"):
        try:
            eps0 = float(rec.eps0(obj, wt))  # Eq. 14: error against the known synthetic object and its illumination
        except Exception:
            eps0 = None
    rec.close()
    del rec, I_dev
    torch.cuda.empty_cache()
    return {
        "value": value, "ms": ms, "steps": steps, "iters": iters, "eps": [float(x) for x in eps], "eps0": eps0,
        "launches": int(launches), "clocks": clocks, "roofline": roofline, "e2e": e2e,
        "workload": workload_name(cfg, iters), "K": K, "m": m, "sharded": sharded,
        "l2": "inputs larger than L2 (frame state 2x%.0f MB + amplitudes %.0f MB per iteration vs 126 MB L2)"
              % (K * m * m * 8 / 1e6, K * m * m * 4 / 1e6),
    }


def run_ours(args):
    import torch
    import paper_1602_01448_b200 as sharp

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the library has no CPU path (use --impl reference for the oracle)")
    sharp.load_library()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1 or (args.sharded and "RANK" in os.environ):
        # (a one-rank group under torchrun --nproc-per-node 1 --sharded runs the sharded path through a real NCCL
        # all-reduce: the only multi-GPU plumbing a one-GPU box can exercise)
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    warm = max(args.warmup, 3)
    main_ = measure(args, args.config, args.steps, warm, rank, world, dev, dist, not args.no_e2e, rank == 0)
    # BASELINE.json's metric names m = 128 AND m = 256: the second headline size (config 4, full size) rides on the
    # same line as `secondary` whenever the default workload (config 2) is benched
    second = None
    if args.config == 2 and not args.grid and not args.no_secondary:
        second = measure(args, 4, max(1, min(args.steps, 3)), 3, rank, world, dev, dist, not args.no_e2e, rank == 0)

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        base, _, _ = time_oracle(args, steps=3, warmup=1)
        cpu = {k: base[k] for k in ("value", "unit", "cores", "kind", "sample")}

    def block(r, config_number):
        return {
            "config": {"workload": r["workload"], "config_number": config_number, "l2": r["l2"],
                       "parallelism": ("one scan sharded by region over the GPUs, object numerator all-reduced every iteration"
                                       if r["sharded"] else "independent scan per GPU, no collective") if world > 1 else "single GPU",
                       "step": "set_object(flat) + iterate(iters, beta) + errors()"},
            "value": r["value"], "unit": UNIT, "steps": r["steps"], "ms_per_step": r["ms"] / r["steps"],
            "ms_per_iteration": r["ms"] / r["steps"] / r["iters"], "eps": r["eps"], "eps0": r["eps0"],
            "gpu_launches": r["launches"], "clocks": r["clocks"], "roofline": r["roofline"], "e2e": r["e2e"],
        }

    m1 = block(main_, args.config)
    line = {
        "metric": METRIC, "value": m1["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": warm, "ms_per_step": m1["ms_per_step"], "higher_is_better": True,
        "scaling": "strong" if main_["sharded"] else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": m1["config"],
        "ms_per_iteration": m1["ms_per_iteration"], "eps": m1["eps"], "eps0": m1["eps0"],
        "gpu_launches": m1["gpu_launches"] + (second["launches"] if second else 0),
        "clocks": m1["clocks"], "roofline": m1["roofline"], "e2e": m1["e2e"], "cpu_baseline": cpu,
        "secondary": block(second, 4) if second else None,
    }
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    return 0


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    # stdout carries the JSON line and nothing else: libraries that write banners to file descriptor 1 (NCCL prints its
    # version there when NCCL_DEBUG=VERSION) are sent to stderr for the duration of the run
    sys.stdout.flush()
    saved = os.dup(1)
    os.dup2(2, 1)
    real_stdout = os.fdopen(saved, "w")
    py_stdout, sys.stdout = sys.stdout, real_stdout
    try:
        return run_ours(args)
    finally:
        real_stdout.flush()
        sys.stdout = py_stdout


if __name__ == "__main__":
    sys.exit(main())
