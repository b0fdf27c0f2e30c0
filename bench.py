#!/usr/bin/env python
"""bench.py -- one JSON line for the w-stacking hot path on B200 (contract: see DESIGN.md "Measurement").

A step = one pass of the whole hot path (rick_bin -> rick_grid (zero + grid) -> rick_fft_planes ->
rick_wcorrect_accumulate) over one batch of seeded synthetic visibilities already resident in HBM.
Workload at N=1: BASELINE.json configs[4] ("hotspot": 1e9 visibilities, 16384^2 x 16 planes, complex64 mesh,
support 9), the largest configuration that fits one GPU; the other four by --config.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config hotspot] [--impl reference]

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


def _traffic(kernel: str, workload: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full
    summary captured on `workload` (profiles/traffic.json: {workload: {kernel: bytes}}), or None when there is
    no capture of this kernel on this workload."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f).get(workload, {}).get(kernel)
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


def _one_plane(pa, vis_host, sample_M: int):
    """The bounded oracle sample: the first `sample_M` visibilities imaged through ONE w-plane of the
    configuration's mesh (same N, support, sigma, dl; the plan's whole w range mapped to a single plane), by
    the oracle's own whole-path call as it stands.  Its per-visibility stages (keys, gridding) scale with M,
    its per-plane stages (FFT, w-correction) with the plane count.
    -> (stage seconds, n_kept, wall s, threads, the oracle's image of the sample)"""
    from oracle import rick_oracle as O
    u, v, w, vv, wt = (a[:sample_M] for a in vis_host)
    pa1 = dict(pa, Nw=1)
    t0 = time.perf_counter()
    img, n_kept, st = O.image(O.Plan(**pa1), u, v, w, vv, wt, return_timing=True)
    total = time.perf_counter() - t0
    return st, n_kept, total, O.threads(), img


def _sample_parity(pa, vis_host, sample_M: int, oracle_img, oracle_kept: int, gpu_image, dtype: str):
    """Parity record of the bench line: the CUDA path, configured as the timed run (fusion mode, rick_bin mode,
    gridding kernel), images the oracle's bounded sample (one w-plane of the configuration's mesh) and is compared
    with the oracle image through the two gates of DESIGN.md "Parity gate".  (The whole workload against the whole
    oracle image is tests/test_gpu_full_configs.py: minutes of oracle time.)"""
    import numpy as np
    from oracle import rick_oracle as O
    img, kept = gpu_image(dict(pa, Nw=1), [a[:sample_M] for a in vis_host])
    N = pa["N"]
    t = O.taper(N, pa["support"], pa["sigma"], pa.get("kernel", "gauss"), pa.get("beta", 0.0))
    tt = t / t[N // 2]
    inner = slice(N // 4, 3 * N // 4)
    peak = float(np.abs(oracle_img[inner, inner]).max())
    a = b = 0.0
    for q0 in range(0, N, 512):                       # row blocks keep the temporaries small
        tw = np.outer(tt[q0:q0 + 512], tt)
        d = np.abs(img[q0:q0 + 512] - oracle_img[q0:q0 + 512])
        b = max(b, float((d * tw).max()))
        m = tw >= 1e-2
        if m.any():
            a = max(a, float(d[m].max()))
    tol = 1e-10 if dtype == "c128" else 1e-5
    return {"against": "oracle", "sample": f"first {sample_M} visibilities through one {N}^2 plane (the cpu_baseline sample)",
            "gate_a": a / peak, "gate_b": b / peak, "tol": tol, "n_kept_equal": bool(kept == oracle_kept),
            "ok": bool(kept == oracle_kept and a <= tol * peak and b <= tol * peak)}


def cpu_baseline(cfg, vis_host, pa, M: int, n_kept: int, sample_M: int = 1_000_000, gpu_image=None):
    """The oracle timed on a bounded sample (see _one_plane); the whole-workload time is estimated as
    per-visibility stages x M / M_sample + per-plane stages x Nw.  Same numerator as the GPU line (kept
    visibilities)."""
    sample_M = min(M, sample_M)
    st, n_kept_s, total, threads, oracle_img = _one_plane(pa, vis_host, sample_M)
    scale = M / sample_M
    est = (st["keys"] + st["grid"]) * scale + (st["fft"] + st["wcorrect"]) * pa["Nw"]
    parity = _sample_parity(pa, vis_host, sample_M, oracle_img, n_kept_s, gpu_image, cfg.dtype) if gpu_image else None
    return parity, {
        "value": n_kept / est, "unit": UNIT, "cores": threads, "kind": "oracle",
        "sample": (f"first {sample_M} of {M} visibilities through one of the {pa['Nw']} planes of the {pa['N']}^2 mesh: "
                   f"keys+grid {st['keys'] + st['grid']:.2f} s scaled x{scale:.1f}, fft {st['fft']:.2f} s and "
                   f"w-correct {st['wcorrect']:.2f} s per plane scaled x{pa['Nw']}; sample wall {total:.2f} s"),
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
        st, n_kept, total, threads, _ = _one_plane(pa, host, sample_M)
        if i >= args.warmup:
            times.append(total)
        last = (st, n_kept, threads)
    sec = sum(times) / len(times)
    st, n_kept, threads = last
    value = n_kept / sec
    sample = (f"each step images the first {sample_M} visibilities of the workload ({n_kept} kept) through ONE w-plane "
              f"of the {pa['N']}^2 mesh (the oracle's per-plane FFT and w-correction cost {st['fft'] + st['wcorrect']:.1f} s "
              f"per plane at this size; all {pa['Nw']} planes per step would not end within minutes)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.config, "N": pa["N"], "Nw": pa["Nw"], "support": pa["support"], "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="hotspot", choices=["tiny", "10M", "100M", "500M", "hotspot"],
                    help="BASELINE.json workload; default: the largest single-GPU configuration")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--ref-sample", type=int, default=200_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fusion", action="store_true", help="2-D cuFFT + separate w-correction kernel")
    ap.add_argument("--fusion", type=int, default=2, choices=[1, 2],
                    help="rick_plan_set_fusion mode: 1 fused column transform, 2 + row occupancy")
    ap.add_argument("--kernel", default="gauss", choices=["gauss", "kb"],
                    help="gridding kernel: the Gaussian of BASELINE.json (default) or the paper's Kaiser-Bessel (beta = 2.34 S)")
    ap.add_argument("--M", type=int, default=0, help="profiling subset: only the first M visibilities of the workload")
    ap.add_argument("--Nw", type=int, default=0, help="profiling subset: this many w-planes instead of the workload's")
    ap.add_argument("--sorted-outputs", action="store_true",
                    help="fp32 mesh: ask rick_bin for the sorted SoA copies (the gather runs in the last sort pass and the "
                         "gridder streams its records) instead of the default indirect mode")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--e2e-chunks", type=int, default=8,
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
    if args.M or args.Nw:       # a subset for profiler captures (ncu saves and restores what a kernel writes); not a bench line
        cfg = W.scaled(cfg, args.M or cfg.M, Nw=args.Nw or cfg.Nw)
    vis = W.generate(cfg, device=dev)
    pa = W.plan_args(cfg, vis)
    M = vis.M
    fma_tflops, add_tinst, fma2_tflops = B.rick_measure_fp32_rate()
    rand_grec = B.rick_measure_random_read_rate()        # before the big buffers exist: it borrows 2 GB
    im = B.Imager(dtype=cfg.dtype, M_max=M, fused=0 if args.no_fusion else args.fusion, kernel=args.kernel, beta=2.34 * cfg.support,
                  sorted_outputs=True if (args.sorted_outputs or cfg.dtype == "c128") else None, **pa)
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
    value = job_value(n_kept, world, ms_per_step)            # gridded (kept) visibilities per second, SURVEY 8(d)

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
    # where the long-row kernel runs, clearing and the row transform's reads are by segment of a row (rows.cu)
    seg_bytes = B.rick_plan_cells_defined(im.plan) * cell if im.fused == 2 else mesh_bytes
    one_sweep = bool(im.fused) and cfg.dtype == "c64" and cfg.N <= 2048      # colfft.cu; else the split engine (colsplit.cu)
    split = bool(im.fused) and not one_sweep
    if not im.fused:
        fft_rows_b, col_a_b, fft_b, wc_b = 0, 0, 4 * mesh_bytes, mesh_bytes + cfg.N * cfg.N * 8
    elif one_sweep:
        fft_rows_b = 2 * live_bytes          # mode 2: own row kernel on the defined rows; mode 1: live = mesh
        col_a_b, fft_b, wc_b = 0, fft_rows_b, live_bytes + cfg.N * cfg.N * 8
    else:
        own_rows = im.fused == 2 and cfg.N >= 4096 and not (cfg.dtype == "c128" and cfg.N > 8192)   # rowbig.cu
        fft_rows_b = seg_bytes + live_bytes if own_rows else 2 * mesh_bytes      # reads the defined segments, writes the defined rows; else batched library transforms of every row
        col_a_b = live_bytes + mesh_bytes    # sweep A reads the defined rows, writes every row
        fft_b, wc_b = fft_rows_b + col_a_b, mesh_bytes + cfg.N * cfg.N * 8
    indirect = not im.sorted_outputs    # fp32 mesh: rick_bin gathers nothing; the gridder fetches 32-B records by index
    alg = {   # algorithmic bytes per stage
        "keygen": (24 + 4 + 32) * M,                 # SoA in, sort key + 32-B staging record out
        # sort: first pass 4 r + 8 w, middle passes 8 r + 8 w, last pass 8 r and, fused into it, the gather
        # (one 32-B record in, sorted SoA 24 B + gridder records 24 B out per kept visibility)
        # (indirect: every pass after the first is 8 r + 8 w and nothing is gathered; the gridder reads 4 B of index
        # and one 32-B record per kept visibility)
        "sort": ((12 + 16 * (n_pass - 1)) * M if indirect else
                 ((12 if n_pass > 1 else 4) + 16 * max(n_pass - 2, 0) + (8 if n_pass > 1 else 0)) * M + (32 + 48) * n_kept),
        "zero": seg_bytes if im.fused == 2 else mesh_bytes,
        "grid": (4 + 32) * n_kept if indirect else 24 * n_kept,
        "fft": fft_b, "fft_rows": fft_rows_b, "fft_col_a": col_a_b,
        "wcorrect": wc_b,
    }
    stages = {}
    for k, b in alg.items():
        t = stage_ms[k]
        if b == 0 or t <= 0:
            continue
        stages[k] = {"ms": round(t, 4), "alg_bytes": b, "gbs": b / (t * 1e-3) / 1e9, "frac": b / (t * 1e-3) / 1e9 / peak}
    zg = stage_ms["zero"] + stage_ms["grid"]
    stages["zero+grid"] = {"ms": round(zg, 4), "alg_bytes": alg["zero"] + alg["grid"],
                           "gbs": (alg["zero"] + alg["grid"]) / (zg * 1e-3) / 1e9,
                           "frac": (alg["zero"] + alg["grid"]) / (zg * 1e-3) / 1e9 / peak,
                           "vis_per_s": n_kept / (zg * 1e-3),
                           "frac_dense_mesh_definition": (mesh_bytes + alg["grid"]) / (zg * 1e-3) / 1e9 / peak}
    binzg = stage_ms["bin"] + zg
    stages["bin+zero+grid"] = {"ms": round(binzg, 4), "vis_per_s": n_kept / (binzg * 1e-3)}
    # the dominant kernel = the library kernel with the largest total time in a step; its roofline numbers
    # are per launch (sort: n_pass launches of k_onesweep, the average pass), against the measured HBM copy rate
    kernels = {"grid": ("k_grid_rec" if cfg.dtype == "c64" else "k_grid_runs", 1), "keygen": ("k_keygen", 1),
               "sort": ("k_onesweep", n_pass),
               "wcorrect": ("k_col_b" if split else ("k_colfft_wcorrect" if one_sweep else "k_wcorrect"), 1)}
    if split:
        kernels["fft_col_a"] = ("k_col_a", 1)
        if own_rows:
            kernels["fft_rows"] = ("k_row_big", 1)
    elif one_sweep and im.fused == 2:
        kernels["fft_rows"] = ("k_rowfft", 1)
    dom = max(kernels, key=lambda k: stage_ms[k])
    kname, n_launch = kernels[dom]
    launch_ms = stage_ms[dom] / n_launch
    launch_bytes = alg[dom] / n_launch
    achieved = launch_bytes / (launch_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": kname, "stage": dom, "launches_per_step": n_launch,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": _traffic(kname, args.config), "peak_source": peak_src,
                "launch_ms": launch_ms, "alg_bytes_per_launch": launch_bytes,
                "share_of_step": stage_ms[dom] / ms_per_step}
    # instruction-issue view of the transform kernels against the fp32 rates measured in this run
    # (rick_measure_fp32_rate: a register-resident FMA / ADD chain on every SM), 5 L log2 L flop per L-point transform
    import math
    alu = {"fp32_fma_tflops_measured": fma_tflops, "fp32_add_tinst_measured": add_tinst,
           "fp32x2_fma_tflops_measured": fma2_tflops}
    if cfg.dtype == "c64" and im.fused:
        n_el = cfg.N * cfg.N * cfg.Nw
        if one_sweep:
            alu["k_colfft_wcorrect_tflops"] = 5.0 * math.log2(cfg.N) * n_el / (stage_ms["wcorrect"] * 1e-3) / 1e12
        else:
            n2 = 1 << ((int(math.log2(cfg.N)) + 1) // 2)
            alu["k_col_a_tflops"] = 5.0 * math.log2(cfg.N // n2) * n_el / (stage_ms["fft_col_a"] * 1e-3) / 1e12
            alu["k_col_b_tflops"] = 5.0 * math.log2(n2) * n_el / (stage_ms["wcorrect"] * 1e-3) / 1e12
    roofline["alu_view"] = alu
    # the gather (in the last sort pass, or, in indirect mode, inside the gridder) is bound by the GPU's random-access
    # rate, measured in this run (rick_measure_random_read_rate: random 32-byte records of a 2 GB array)
    roofline["random_access_view"] = {
        "measured_grecords_per_s": rand_grec,
        "gathered_records": n_kept,
        "floor_ms": n_kept / (rand_grec * 1e9) * 1e3 if rand_grec > 0 else None,
        "where": "k_grid_rec (indirect mode)" if indirect else "last k_onesweep pass (fused gather)",
        "grid_stage_grecords_per_s": n_kept / (stage_ms["grid"] * 1e-3) / 1e9 if indirect else None,
        "frac": (n_kept / (stage_ms["grid"] * 1e-3) / 1e9 / rand_grec) if (indirect and rand_grec > 0) else None}

    # end to end through rick_image_from_host(_chunked): pinned host inputs -> host image, copies inside the region
    host = [torch.empty(x.shape, dtype=x.dtype, pin_memory=args.e2e_steps > 0) for x in (vis.u, vis.v, vis.w, vis.vis, vis.weight)]
    for h, x in zip(host, (vis.u, vis.v, vis.w, vis.vis, vis.weight)):
        h.copy_(x)
    torch.cuda.synchronize()
    del vis                      # the device-resident inputs make room for the staging buffers of the host entry
    torch.cuda.empty_cache()
    e2e = None
    if args.e2e_steps > 0:
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
        e2e = {"value": world * n_kept / e2e_s, "unit": UNIT, "h2d_bytes_per_step": 24 * M,
               "d2h_bytes_per_step": cfg.N * cfg.N * 8, "ms_per_step": e2e_s * 1e3, "steps": args.e2e_steps,
               "chunks": args.e2e_chunks, "image_seconds": e2e_s,
               "call": "rick_image_from_host_chunked" if args.e2e_chunks > 1 else "rick_image_from_host"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32" if cfg.dtype == "c64" else "f64", "data": "synthetic",
        "config": {"workload": args.config + (" (profiling subset)" if args.M or args.Nw else ""), "M": M, "M_kept": n_kept, "sort_passes": n_pass, "N": cfg.N, "Nw": cfg.Nw,
                   "support": cfg.support, "sigma": cfg.sigma, "gridding_kernel": args.kernel, "mesh": cfg.dtype,
                   "fusion_mode": int(im.fused), "rick_bin_sorted_outputs": bool(im.sorted_outputs),
                   "column_engine": "split (colsplit.cu)" if split else ("one sweep (colfft.cu)" if one_sweep else "cuFFT 2-D + K5"),
                   "mesh_rows_defined": rows_defined, "mesh_rows": rows_total, "mesh_bytes_defined_before_fft": seg_bytes,
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"inputs ({24 * M / 1e9:.2f} GB) and mesh ({mesh_bytes / 1e9:.2f} GB) exceed the 126 MB L2; no explicit flush"},
        "value_definition": "kept (gridded) visibilities of all ranks / step time; a step = rick_bin + rick_grid + rick_fft_planes + rick_wcorrect_accumulate",
        "all_input_visibilities_per_sec": job_value(M, world, ms_per_step),
        "image_seconds": ms_per_step * 1e-3,
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roofline, "stages": stages,
    }
    if world == 1 and not args.no_cpu_baseline:
        opa = dict(pa, kernel=args.kernel, beta=2.34 * cfg.support if args.kernel == "kb" else 0.0)
        fused, sorted_outputs = int(im.fused), bool(im.sorted_outputs)
        im.close()               # the timed plan's buffers make room for the one-plane plan of the parity sample
        del im
        torch.cuda.empty_cache()

        def gpu_image(pa1, hv):
            """the library, configured as the timed run, on the oracle's sample -> (host image, n_kept)"""
            kw = {k: x for k, x in pa1.items() if k not in ("kernel", "beta")}
            im1 = B.Imager(dtype=cfg.dtype, M_max=len(hv[0]), fused=fused, kernel=args.kernel, beta=2.34 * cfg.support,
                           sorted_outputs=sorted_outputs, **kw)
            assert im1.fused == fused
            img = im1.run(*(torch.from_numpy(a).to(dev) for a in hv)).cpu().numpy()
            kept = int(im1.n_kept.item())
            im1.close()
            return img, kept

        line["parity"], line["cpu_baseline"] = cpu_baseline(cfg, [h.numpy() for h in host], opa, M, n_kept, gpu_image=gpu_image)
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
