#!/usr/bin/env python
"""bench.py -- one JSON line for the w-stacking hot path on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path (rick_bin -> rick_grid (zero + grid) -> rick_fft_planes ->
rick_wcorrect_accumulate) over one batch of seeded synthetic visibilities already resident in HBM.
Workload at N=1: BASELINE.json configs[1] ("10M": 1e7 visibilities, 2048^2 x 32 planes, complex64 mesh).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 10M] [--impl reference]

N > 1 (torchrun): the path does not shard ("replicas only"): every rank images its own copy
of the workload on its own GPU, no data-path collective; value = visibilities of all ranks / max time.
--impl reference times the CPU oracle (oracle/) on the host cores, rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gridded_visibilities_per_sec"
UNIT = "visibilities/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


def _traffic(kernel: str, workload: str = "10M"):
    """dram bytes per launch of `kernel` from the committed ncu --set full summary (captured on the
    workload the file names), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            d = json.load(f)
            return d.get(kernel) if d.get("_workload", "10M") == workload else None
    except Exception:
        return None


def max_over_ranks(x: float, dist, device) -> float:
    """Replicas-only multi-GPU accounting: a timed quantity of the job is the slowest
    rank's; there is no data-path collective, this all-reduce of one scalar is the only exchange."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(per_rank_units: int, world: int, ms_per_step: float) -> float:
    """Whole-job throughput: every rank images its own replica of the workload (weak scaling)."""
    return world * per_rank_units / (ms_per_step * 1e-3)


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.02):
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._loop, daemon=True)
            self._thread.start()

    def stop(self):
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML unavailable or region too short"}
        return {"sm_mhz": statistics.median(self.samples), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def _oracle_sample(cfg, vis_host, pa, sample_M: int):
    """Time the oracle, as it stands, on the first `sample_M` visibilities with the full plan (all Nw planes
    are gridded, transformed and w-corrected).  Returns (seconds per stage, n_kept of the sample, threads)."""
    from oracle import rick_oracle as O
    u, v, w, vv, wt = (a[:sample_M] for a in vis_host)
    t0 = time.perf_counter()
    _, n_kept, st = O.image(O.Plan(**pa), u, v, w, vv, wt, return_timing=True)
    total = time.perf_counter() - t0
    return st, n_kept, total, O.threads()


def cpu_baseline(cfg, vis_host, pa, M: int):
    """The oracle timed on a bounded sample; the whole-workload time is per-visibility stages scaled by
    M / M_sample plus the per-plane stages (FFT, w-correction), which do not depend on M."""
    sample_M = min(M, 1_000_000)
    st, n_kept_s, total, threads = _oracle_sample(cfg, vis_host, pa, sample_M)
    scale = M / sample_M
    est = (st["keys"] + st["grid"]) * scale + st["fft"] + st["wcorrect"]
    return {
        "value": M / est, "unit": UNIT, "cores": threads, "kind": "oracle",
        "sample": (f"first {sample_M} of {M} visibilities through the full plan ({pa['N']}^2 x {pa['Nw']} planes): "
                   f"keys+grid {st['keys'] + st['grid']:.2f} s scaled x{scale:.1f}, fft {st['fft']:.2f} s and "
                   f"w-correct {st['wcorrect']:.2f} s taken as measured; sample wall {total:.2f} s"),
        "stage_seconds_sample": {k: round(float(x), 4) for k, x in st.items()},
        "est_seconds_full": est,
    }


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np  # noqa: F401
    from paper_2411_07321_b200 import workloads as W
    cfg = W.CONFIGS[args.config]
    sample_M = min(cfg.M, args.ref_sample)
    scfg = W.scaled(cfg, sample_M)
    vis = W.generate(scfg, device="cpu")
    pa = W.plan_args(scfg, vis)
    pa = dict(pa, kernel=args.kernel, beta=2.34 * cfg.support if args.kernel == "kb" else 0.0)
    host = vis.numpy()
    times = []
    last = None
    for i in range(args.warmup + args.steps):
        st, n_kept, total, threads = _oracle_sample(scfg, host, pa, sample_M)
        if i >= args.warmup:
            times.append(total)
        last = (st, n_kept, threads)
    sec = sum(times) / len(times)
    value = sample_M / sec
    st, n_kept, threads = last
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.config, "N": pa["N"], "Nw": pa["Nw"], "support": pa["support"],
                   "sample": f"each step images the first {sample_M} visibilities of the workload with the full plan"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle",
                         "sample": f"first {sample_M} of {cfg.M} visibilities, all {pa['Nw']} planes, per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="10M")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-sample", type=int, default=1_000_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fusion", action="store_true", help="2-D cuFFT + separate w-correction kernel")
    ap.add_argument("--fusion", type=int, default=2, choices=[1, 2],
                    help="rick_plan_set_fusion mode where the plan supports it: 1 fused column transform, 2 + row occupancy")
    ap.add_argument("--kernel", default="gauss", choices=["gauss", "kb"],
                    help="gridding kernel: the Gaussian of BASELINE.json (default) or the paper's Kaiser-Bessel (beta = 2.34 S)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--e2e-chunks", type=int, default=4,
                    help="time slices of rick_image_from_host_chunked in the e2e region (1: one copy, then compute)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    if args.impl == "reference":
        run_reference(args)
        return

    import torch
    from paper_2411_07321_b200 import binding as B
    from paper_2411_07321_b200 import workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path is the only implementation")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    cfg = W.CONFIGS[args.config]
    vis = W.generate(cfg, device=dev)
    pa = W.plan_args(cfg, vis)
    M = vis.M
    im = B.Imager(dtype=cfg.dtype, M_max=M, fused=0 if args.no_fusion else args.fusion, kernel=args.kernel, beta=2.34 * cfg.support, **pa)
    cell = 16 if cfg.dtype == "c128" else 8
    mesh_bytes = cfg.Nw * cfg.N * cfg.N * cell

    def step():
        im.run(vis.u, vis.v, vis.w, vis.vis, vis.weight)

    for _ in range(args.warmup):
        step()
    torch.cuda.synchronize()
    n_kept = int(im.n_kept.item())
    if dist is not None:
        dist.barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = im.launches()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStart()      # `ncu --profile-from-start off` sees the timed region only
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    torch.cuda.cudart().cudaProfilerStop()
    launches = im.launches() - l0
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, dist, dev)
    if dist is not None:
        dist.barrier()
    ms_per_step = ms / args.steps
    value = job_value(M, world, ms_per_step)

    # per-stage CUDA-event times (events recorded by the library on the launch stream), same workload
    per = {k: [] for k in B.RICK_T_NAMES}
    for _ in range(max(5, min(args.steps, 20))):
        step()
        tm = im.timings()
        for k in per:
            per[k].append(tm[k])
    stage_ms = {k: statistics.median(v) for k, v in per.items()}
    peak, peak_src = _peaks()
    _, n_pass, _ = B.rick_plan_sort_layout(im.plan)
    # fusion mode 2 clears / transforms / reads only the mesh rows some footprint touches: those are the bytes
    # the path needs; the dense-mesh figure of SURVEY.md section 8(d) is kept beside it for zero+grid
    rows_total = cfg.Nw * cfg.N
    rows_defined = B.rick_plan_rows_defined(im.plan) if im.fused == 2 else rows_total
    live_bytes = mesh_bytes * rows_defined // rows_total
    alg = {   # algorithmic bytes per launch
        "keygen": (24 + 4 + 32) * M,                 # SoA in, sort key + 32-B staging record out
        # sort: first pass 4 r + 8 w, middle passes 8 r + 8 w, last pass 8 r and, fused into it, the gather
        # (one 32-B record in, sorted SoA 24 B + gridder records 24 B out per kept visibility)
        "sort": ((12 if n_pass > 1 else 4) + 16 * max(n_pass - 2, 0) + (8 if n_pass > 1 else 0)) * M + (32 + 48) * n_kept,
        "gather": 0,                                 # rides in the last sort pass (rick_bin without perm_out)
        "zero": live_bytes,
        "grid": 24 * n_kept,
        "fft": (2 if im.fused else 4) * live_bytes,      # fused: row transforms only (one read + write)
        "wcorrect": live_bytes + cfg.N * cfg.N * 8,      # fused: column transforms + screen + sum, one read
    }
    stages = {}
    for k, b in alg.items():
        if k == "gather":
            continue
        t = stage_ms[k]
        stages[k] = {"ms": round(t, 4), "alg_bytes": b, "gbs": (b / (t * 1e-3) / 1e9) if t > 0 else None,
                     "frac": (b / (t * 1e-3) / 1e9 / peak) if t > 0 else None}
    zg = stage_ms["zero"] + stage_ms["grid"]
    stages["zero+grid"] = {"ms": round(zg, 4), "alg_bytes": alg["zero"] + alg["grid"],
                           "gbs": (alg["zero"] + alg["grid"]) / (zg * 1e-3) / 1e9,
                           "frac": (alg["zero"] + alg["grid"]) / (zg * 1e-3) / 1e9 / peak,
                           "vis_per_s": n_kept / (zg * 1e-3),
                           "frac_dense_mesh_definition": (mesh_bytes + alg["grid"]) / (zg * 1e-3) / 1e9 / peak}
    # the dominant kernel = the library kernel with the largest total time in a step; its roofline numbers
    # are per launch (sort: n_pass launches of k_onesweep, the average pass)
    kernels = {"grid": ("k_grid_rec" if cfg.dtype == "c64" else "k_grid_runs", 1),
               "wcorrect": ("k_colfft_wcorrect" if im.fused else "k_wcorrect", 1), "keygen": ("k_keygen", 1),
               "sort": ("k_onesweep", n_pass)}
    dom = max(kernels, key=lambda k: stage_ms[k])
    kname, n_launch = kernels[dom]
    launch_ms = stage_ms[dom] / n_launch
    launch_bytes = alg[dom] / n_launch
    achieved = launch_bytes / (launch_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": kname, "stage": dom, "launches_per_step": n_launch,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": _traffic(kname, args.config), "peak_source": peak_src,
                "launch_ms": launch_ms, "alg_bytes_per_launch": launch_bytes}
    if kname == "k_colfft_wcorrect":
        # the fused column transform is bound by fp32 instruction issue, not by HBM (profiles/): report it against
        # the fp32 ALU peak DESIGN.md section 5 derives (148 SMs x 128 lanes x 2 flop x 1.965 GHz), with the
        # 5 N log2 N flop of every column transform; the HBM view stays beside it
        import math
        flops = 5.0 * cfg.N * math.log2(cfg.N) * cfg.N * cfg.Nw
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
        roofline = {"bound": "alu", "kernel": kname, "stage": dom, "launches_per_step": n_launch,
                    "achieved": flops / (launch_ms * 1e-3) / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
                    "frac": flops / (launch_ms * 1e-3) / 1e12 / alu_peak,
                    "traffic": _traffic(kname + ("_mode2" if im.fused == 2 else ""), args.config),
                    "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 (FMA) x 1.965 GHz (DESIGN.md section 5)",
                    "launch_ms": launch_ms, "alg_flops_per_launch": flops,
                    "hbm": {"achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                            "alg_bytes_per_launch": launch_bytes}}

    # end to end through rick_image_from_host: pinned host inputs -> host image, copies inside the region
    host = [x.cpu() for x in (vis.u, vis.v, vis.w, vis.vis, vis.weight)]
    e2e = None
    if args.e2e_steps > 0:
        host = [x.pin_memory() for x in host]
        out = torch.empty((cfg.N, cfg.N), dtype=torch.float64).pin_memory()
        def timed_from_host(chunks):
            im.run_from_host(*host, out, chunks=chunks)
            torch.cuda.synchronize()
            if dist is not None:
                dist.barrier()
            t0 = time.perf_counter()
            for _ in range(args.e2e_steps):
                im.run_from_host(*host, out, chunks=chunks)
            torch.cuda.synchronize()
            return max_over_ranks((time.perf_counter() - t0) / args.e2e_steps, dist, dev)

        e2e_s = timed_from_host(args.e2e_chunks)
        e2e = {"value": world * M / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 24 * M,
               "d2h_bytes_per_step": cfg.N * cfg.N * 8, "ms_per_step": e2e_s * 1e3, "steps": args.e2e_steps,
               "chunks": args.e2e_chunks,
               "call": "rick_image_from_host_chunked" if args.e2e_chunks > 1 else "rick_image_from_host"}
        if args.e2e_chunks > 1:
            e2e["ms_per_step_one_chunk"] = timed_from_host(1) * 1e3

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if cfg.dtype == "c64" else "f64", "data": "synthetic",
        "config": {"workload": args.config, "M": M, "M_kept": n_kept, "sort_passes": n_pass, "N": cfg.N, "Nw": cfg.Nw,
                   "support": cfg.support, "sigma": cfg.sigma, "gridding_kernel": args.kernel, "mesh": cfg.dtype, "fusion_mode": int(im.fused), "mesh_rows_defined": rows_defined, "mesh_rows": rows_total,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": "inputs (240 MB) and mesh (1.07 GB) exceed the 126 MB L2; no explicit flush"
                   if args.config == "10M" else "inputs and mesh exceed L2; no explicit flush"},
        "image_seconds": ms_per_step * 1e-3,
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roofline, "stages": stages,
    }
    if world == 1 and not args.no_cpu_baseline:
        opa = dict(pa, kernel=args.kernel, beta=2.34 * cfg.support if args.kernel == "kb" else 0.0)
        line["cpu_baseline"] = cpu_baseline(cfg, [h.numpy() for h in host], opa, M)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
