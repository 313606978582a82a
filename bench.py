#!/usr/bin/env python3
"""bench.py -- headline benchmark: real spherical harmonics, lmax = 9, fp64, on the full 128^3 grid
(BASELINE.json configs[2]), both output layouts.

One "step" = one pass of the whole hot path over the grid for each layout named by the config:
    sh_real(xyz, n, 9, out_soa, SOA) ; sh_real(xyz, n, 9, out_aos, AOS)        (2 kernel launches)
`value` counts harmonic values produced per second by the whole job (all ranks), inputs resident in HBM.
Output buffers (1.68 GB each) are far larger than L2 (126 MB); inputs and outputs rotate between
replicas so nothing is re-read from L2 between timed iterations.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
N > 1 is launched by torchrun (one rank per GPU); points are independent, so the job is a contiguous point-range
partition (inputs.shard_range) of N grids, one grid per rank, with no data-path collective ("weak" scaling);
timing is the max over ranks of CUDA-event time.

Ceilings are measured in the same run from committed code (csrc/sh_peaks.cu): write-only fills in the kernels' own
store patterns (`roofline.write_fill_gbs`) and a DFMA chain (the `alu` peak of the FP64-bound fused projection).
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

LMAX = 9
K = (LMAX + 1) ** 2
METRIC = "G harmonic values/s, real SH lmax=9 fp64 (HBM write GB/s in roofline)"
UNIT = "G values/s"
WORKLOAD = "configs[2]: real SH lmax=9 fp64, full 128^3 grid over [-6,6]^3 (2,097,152 points), SoA [100][N] + AoS [N][100]"
BYTES_PER_POINT = 24 + 8 * K  # algorithmic: xyz in + (lmax+1)^2 doubles out


def measured_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(path))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(kernel_key: str):
    """Per-launch DRAM bytes (dram__bytes_read.sum + dram__bytes_write.sum) of a kernel family from the committed ncu
    summaries (profiles/ncu_traffic.csv, one row per family, copied from the `ncu --set full` captures named in
    profiles/r2_launches.md), or None.  A profiler counter cannot be read inside an unprofiled run: this is the committed
    measurement of the same kernel on the same workload, not a live one."""
    try:
        import csv

        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "ncu_traffic.csv"))):
            if row["kernel"] == kernel_key:
                return float(row["dram_bytes_per_launch"])
    except Exception:
        pass
    return None


class ClockSampler:
    """nvidia-smi samples (the profiling recipe's clocks line) with timestamps; stop(t0, t1) keeps the samples whose
    timestamp falls inside the load window [t0, t1] (time.time() values)."""
    QUERY = "timestamp,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown," \
            "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.QUERY}", "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self, t0: float, t1: float):
        import datetime

        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                ts = datetime.datetime.strptime(c[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                if not (t0 <= ts <= t1):
                    continue
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out = {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm),
                   "power_w_max": max(pw)}
        return out


def ceilings(dev, sampler_index=None):
    """The two ceilings SURVEY.md asks the build to measure (section 6: an FP64 DFMA peak; section 8(d) denominator (ii): a
    write-only fill "measured in the same run"), from committed code (csrc/sh_peaks.cu), with the bench's own discipline:
    CUDA events on the launching stream, 3 warm-ups, median of 20, two rotating 1.68 GB buffers (far larger than L2).
      write_fill_gbs.flat        one flat stream of 32-byte evict-first stores
      write_fill_gbs.bulk_tiles  contiguous 25.6 KB tiles, one TMA bulk copy each        (the AoS kernels' store pattern)
      write_fill_gbs.soa_planes  [100][N] planes, one TMA tensor store per 128-point tile (the SoA kernels' store pattern)
      write_fill_gbs.memset      cudaMemsetAsync through torch (`zero_`), the driver's own fill
      fp64_lane_ginstr_s         DFMA chains at full occupancy for >= 1 s (so the clock is the power-capped one), with the SM clock sampled meanwhile."""
    import torch
    from paper_2510_05282_b200 import peaks

    n = 128 ** 3
    bufs = [torch.empty((K, n), dtype=torch.float64, device=dev) for _ in range(2)]
    nbytes = bufs[0].numel() * 8

    def med(fn):
        for it in range(3):
            fn(bufs[it % 2])
        torch.cuda.synchronize()
        ts = []
        for it in range(20):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            fn(bufs[it % 2])
            b.record()
            b.synchronize()
            ts.append(a.elapsed_time(b))
        return nbytes / (statistics.median(ts) * 1e-3) / 1e9

    fills = {
        "flat": med(peaks.fill_flat),
        "bulk_tiles": med(lambda o: peaks.fill_bulk_tiles(o, 32 * K * 8)),
        "soa_planes": med(lambda o: peaks.fill_soa_planes(o, 128, K)),
        "memset": med(lambda o: o.zero_()),
    }
    del bufs
    torch.cuda.empty_cache()
    # FP64 pipe: 8 CTAs of 256 threads per SM (full occupancy), launches of ~20 ms back to back for >= 1 s
    sink = torch.zeros(8, dtype=torch.float64, device=dev)
    blocks = N_SMS * 8
    iters = 1 << 16
    peaks.dfma(sink, iters, blocks)
    torch.cuda.synchronize()
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    wall0 = time.time()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    lane_instr = 0
    launches = 0
    while True:
        for _ in range(10):
            lane_instr += peaks.dfma(sink, iters, blocks)
            launches += 1
        torch.cuda.synchronize()
        if time.time() - wall0 >= 1.0:
            break
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    clocks = sampler.stop(wall0, time.time()) if sampler else None
    ginstr = lane_instr / (ms * 1e-3) / 1e9
    return {
        "write_fill_gbs": fills,
        "fp64_lane_ginstr_s": ginstr, "fp64_tflops_dfma": 2 * ginstr / 1e3,
        "fp64_measure": {"ms": ms, "launches": launches, "sm_mhz": clocks and clocks.get("sm_mhz"), "reasons": clocks and clocks.get("reasons"),
                         "lanes_per_sm_per_clk_at_sampled_clock": (ginstr * 1e3 / (N_SMS * clocks["sm_mhz"]) if clocks and clocks.get("sm_mhz") else None)},
        "how": "csrc/sh_peaks.cu through paper_2510_05282_b200/peaks.py, CUDA events, same run",
    }


def ncu_fp64_executed(kernel_key: str):
    """FP64 thread-instructions executed per launch of a kernel family on the 128^3 grid (profiles/ncu_fp64_instr.csv, from the committed
    `ncu --set full` captures), or None: what the kernel really issues, next to the algorithmic count `roofline.frac` is built on."""
    try:
        import csv

        for row in csv.DictReader(open(os.path.join(ROOT, "profiles", "ncu_fp64_instr.csv"))):
            if row["kernel"] == kernel_key:
                return float(row["fp64_thread_instr_per_launch"])
    except Exception:
        pass
    return None


def hbm_roofline(kernel, alg_bytes, written_bytes, ms, peak, peak_src, ceil, pattern, traffic_key=None):
    """`roofline` block of an HBM-bound launch: achieved = algorithmic bytes (in + out) per launch / average launch time against
    the driver-measured copy peak, plus the written bytes against the write-only fill ceiling of the kernel's own store pattern."""
    achieved = alg_bytes / (ms * 1e-3) / 1e9
    wr = written_bytes / (ms * 1e-3) / 1e9
    blk = {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
           "algorithmic_bytes_per_launch": alg_bytes, "avg_launch_ms": ms, "achieved_write": wr,
           "traffic": ncu_traffic(traffic_key) if traffic_key else None}
    if ceil:
        fill = ceil["write_fill_gbs"][pattern]
        blk.update({"write_fill_gbs": fill, "write_fill_pattern": pattern, "frac_of_write_fill": wr / fill})
    return blk


def grid_points():
    from paper_2510_05282_b200 import inputs

    return inputs.config3_full_grid()


def cpu_baseline(pts, target_seconds=12.0):
    """The oracle as it stands on this box's host cores, on a bounded prefix-sample of the same workload."""
    import oracle

    oracle.build()
    t0 = time.perf_counter()
    oracle.real(pts[: 1 << 13], LMAX)
    rate = (1 << 13) / max(time.perf_counter() - t0, 1e-9)  # points/s, calibration
    m = int(min(len(pts), max(1 << 13, rate * target_seconds)))
    t0 = time.perf_counter()
    oracle.real(pts[:m], LMAX)
    dt = time.perf_counter() - t0
    cores = oracle.threads_used()
    # one thread as well (comparable with the paper's single-core figures), on a smaller prefix
    m1 = max(1 << 12, m // (4 * max(cores, 1)))
    oracle.set_threads(1)
    try:
        t0 = time.perf_counter()
        oracle.real(pts[:m1], LMAX)
        dt1 = time.perf_counter() - t0
    finally:
        oracle.set_threads(0)
    return {
        "value": m * K / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
        "sample": f"first {m} points of the 128^3 grid, lmax=9 real, long double, one evaluation, {dt:.2f} s",
        "value_one_thread": m1 * K / dt1 / 1e9, "sample_one_thread": f"first {m1} points, {dt1:.2f} s",
    }


def cpu_method(pts):
    """The paper's own CPU scheme on this box's host cores: the generated factorized fp64 formulas compiled for
    the host (baseline/sh_cpu_method.cpp), every l <= 9 at every grid point, stored as AoS [N][100]; all cores and one thread,
    plus the compute-only (accumulate, never store: P:140) rate that is comparable with the paper's Table I."""
    import baseline

    baseline.build()
    n = len(pts)
    out = np.empty((n, K))
    res = {"unit": UNIT, "kind": "paper method: generated factorized formulas, fp64, host build (baseline/sh_cpu_method.cpp)",
           "sample": f"all {n} grid points, lmax=9 real, AoS store, second of two passes (the first touches the pages)"}
    for label, threads in (("", 0), ("_one_thread", 1)):
        baseline.set_threads(threads)
        m = n if threads == 0 else n // 8
        baseline.real(pts[:m], LMAX, out=out[:m])
        t0 = time.perf_counter()
        baseline.real(pts[:m], LMAX, out=out[:m])
        dt = time.perf_counter() - t0
        t0 = time.perf_counter()
        baseline.accumulate_l9(pts[:m])
        dta = time.perf_counter() - t0
        res["value" + label] = m * K / dt / 1e9
        res["value_accumulate_only" + label] = m * K / dta / 1e9
        if threads == 0:
            res["cores"] = baseline.threads()
    baseline.set_threads(0)
    res["sample_one_thread"] = f"first {n // 8} grid points"
    return res


def run_reference(args):
    """--impl reference: the oracle is the reference arm for this tier (no upstream code exists)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle

    oracle.build()
    pts = grid_points()
    m = 1 << 15  # bounded sample per step: 32,768 grid points, evaluated once per layout
    stride = len(pts) // m
    sample = np.ascontiguousarray(pts[::stride][:m])

    def step():
        a = oracle.real(sample, LMAX)                      # AoS [m][100]
        b = np.ascontiguousarray(oracle.real(sample, LMAX).T)  # SoA [100][m]
        return a, b

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = args.steps * 2 * m * K / dt / 1e9
    cores = oracle.threads_used()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64 result (oracle computes in x87 long double)", "data": "synthetic",
        "config": {"workload": WORKLOAD, "sample": f"every {stride}th grid point, {m} points per layout per step"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"{m} strided grid points x 2 layouts per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def extra_configs(sh, dev, only=None, ceil=None):
    """The other BASELINE.json configs, timed with CUDA events outside the headline's timed region (context, not `value`).
    `only`: run just the cases whose name contains this substring (what the ncu captures under profiles/ use)."""
    import torch
    from paper_2510_05282_b200 import inputs

    want = lambda name: only is None or only in name

    def timed(fn, reps):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(reps):
            fn()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    def timed_graph(fn, reps):
        """The same call captured `reps` times in one CUDA graph (the library allocates nothing and is asynchronous on the
        stream it is given, so it can be captured): per-call time without the Python/ctypes launch overhead."""
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            fn()
        torch.cuda.current_stream().wait_stream(side)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g):
            for _ in range(reps):
                fn()
        g.replay()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        g.replay()
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    res = {}
    peak, peak_src = measured_peak()
    # the paper's three front ends (Table I) on the headline workload, SoA
    grid = inputs.config3_full_grid()
    rr = np.linalg.norm(grid, axis=1)
    rr[rr == 0] = 1.0
    unit = np.ascontiguousarray(grid / rr[:, None])
    ang = np.ascontiguousarray(np.stack([np.arccos(np.clip(unit[:, 2], -1, 1)), np.arctan2(unit[:, 1], unit[:, 0])], axis=1))
    out = torch.empty((K, len(grid)), dtype=torch.float64, device=dev)
    for coords, arr in (("cartesian", grid), ("normalized", unit), ("angular", ang)):
        if not want(f"config3 real l9 SoA front end {coords}"):
            continue
        x = torch.from_numpy(arr).to(dev)
        ms = timed(lambda: sh.sh_real(x, LMAX, out=out, layout="soa", coords=coords), 20)
        res[f"config3 real l9 SoA front end {coords}"] = {
            "ms": ms, "write_GBps": len(grid) * K * 8 / ms / 1e6, "G_values_per_s": len(grid) * K / ms / 1e6,
            "roofline": hbm_roofline(f"sh_real lmax=9 SoA, {coords} input", len(grid) * (arr.shape[1] * 8 + 8 * K), len(grid) * 8 * K, ms, peak, peak_src, ceil, "soa_planes")}
        del x
    del out
    # the paper's own protocol (Table I: every harmonic evaluated, "accumulated and never stored"): bound by the FP64 pipe
    fp64_peak = ceil["fp64_lane_ginstr_s"] if ceil else N_SMS * FP64_LANES_PER_SM * SM_MAX_GHZ
    for coords, arr in (("cartesian", grid), ("normalized", unit), ("angular", ang)):
        name = f"config3 real l9 compute-only sum (Table I protocol) {coords}"
        if not want(name):
            continue
        x = torch.from_numpy(arr).to(dev)
        o = torch.empty(len(grid), dtype=torch.float64, device=dev)
        ms = timed(lambda: sh.sh_real_sum(x, LMAX, out=o, coords=coords), 20)
        per_point = REAL_L9_FP64_PER_POINT + K if coords == "cartesian" else None   # a2-a5 + the K additions of the sum
        res[name] = {"ms": ms, "G_values_per_s": len(grid) * K / ms / 1e6, "G_points_per_s": len(grid) / ms / 1e6}
        if per_point:
            res[name]["roofline"] = {"bound": "alu", "unit": "G FP64 lane-instr/s", "achieved": len(grid) * per_point / ms / 1e6, "peak": fp64_peak,
                                     "frac": len(grid) * per_point / ms / 1e6 / fp64_peak, "fp64_instr_per_point": per_point,
                                     "peak_source": "measured in this run (DFMA chains, csrc/sh_peaks.cu)" if ceil else "nominal 148 SMs x 64 lanes x 1.965 GHz"}
        del x, o
    cases = [
        ("config1 real l4 SoA N=10008", "real", inputs.config1_cube(), 4, ["soa"], 50),
        ("config2 real l3 SoA N=113102", "real", inputs.config2_projector_grid(), 3, ["soa"], 50),
        ("config4 complex l9 N=2^24", "complex", inputs.config4_sphere_directions(), 9, ["soa", "aos"], 3),
        ("config5 spinor l9 N=2^22", "spinor", inputs.config5_ball(), 9, ["soa", "aos"], 3),
        ("config5 real_f32 l9 N=2^22", "real_f32", inputs.config5_ball().astype(np.float32), 9, ["soa", "aos"], 20),
        # l > 9 by recurrence: ball points of config 5, first 2^20
        ("ext real l16 N=2^20", "real_ext", inputs.config5_ball(n=1 << 20), 16, ["soa"], 10),
        ("ext real l32 N=2^20", "real_ext", inputs.config5_ball(n=1 << 20), 32, ["soa"], 5),
        ("ext complex l32 N=2^20", "complex_ext", inputs.config5_ball(n=1 << 20), 32, ["soa"], 3),
    ]
    for name, kind, pts, lmax, layouts, reps in cases:
        if not any(want(f"{name} {layout}") for layout in layouts):
            continue
        x = torch.from_numpy(pts).to(dev)
        n = len(pts)
        per_point = sh.count(kind, lmax)
        esize = 4 if kind == "real_f32" else 8
        values = {"real": 1, "real_f32": 1, "real_ext": 1, "complex": 2, "complex_ext": 2, "spinor": 2}[kind]  # scalars per "value" (a complex number is one value)
        for layout in layouts:
            if not want(f"{name} {layout}"):
                continue
            out = torch.empty(sh.out_shape(kind, n, lmax, layout), dtype=x.dtype, device=dev)
            fn = getattr(sh, "sh_" + kind)
            ms = timed(lambda: fn(x, lmax, out=out, layout=layout), reps)
            res[f"{name} {layout}"] = {
                "ms": ms, "write_GBps": n * per_point * esize / ms / 1e6,
                "G_values_per_s": n * per_point / values / ms / 1e6,
            }
            if n >= (1 << 18):   # HBM-bound sizes: algorithmic bytes = xyz in + every scalar out
                res[f"{name} {layout}"]["roofline"] = hbm_roofline(
                    f"sh_{kind} lmax={lmax} {layout}", n * (3 * esize + per_point * esize), n * per_point * esize, ms, peak, peak_src, ceil,
                    "soa_planes" if layout == "soa" else "bulk_tiles", traffic_key=f"{kind}_{layout}")
            if n < (1 << 18):   # launch-bound sizes: also as CUDA-graph replays
                res[f"{name} {layout}"]["ms_in_cuda_graph"] = timed_graph(lambda: fn(x, lmax, out=out, layout=layout), 100)
            del out
        del x
        torch.cuda.empty_cache()
    res.update(projector_cases(sh, dev, timed, timed_graph, want, ceil))
    return res


# FP64 pipe peak for the ALU-bound fused projection: one DADD/DMUL/DFMA = one lane-slot of the FP64 pipe.
# The peak is MEASURED in the same run (ceilings(): DFMA chains at full occupancy for >= 1 s, csrc/sh_peaks.cu); the nominal
# figure 148 SMs x 64 lanes x 1.965 GHz (B300_MICROARCH.md unit counts x the nvidia-smi maximum clock) is printed beside it.
FP64_LANES_PER_SM = 64
N_SMS = 148
SM_MAX_GHZ = 1.965


def projector_cases(sh, dev, timed, timed_graph, want, ceil=None):
    """Fused projector consumer: sh_projectors (stores only the requested columns) and sh_project
    (contraction with weight vectors; writes nothing per point, FP64-pipe bound)."""
    import torch
    from paper_2510_05282_b200 import inputs

    res = {}
    nominal_ginstr = N_SMS * FP64_LANES_PER_SM * SM_MAX_GHZ  # G FP64 lane-instructions/s
    peak_ginstr = ceil["fp64_lane_ginstr_s"] if ceil else nominal_ginstr
    peak_src = "measured in this run (DFMA chains, csrc/sh_peaks.cu)" if ceil else "nominal 148 SMs x 64 lanes x 1.965 GHz"
    hbm_peak, hbm_src = measured_peak()
    work = [
        # name, points, (lmax, per_l, cutoff, dr), volume element
        ("config2 grid l3 x2 channels (32 cols)", inputs.config2_projector_grid(), (3, 2, 3.0, 0.01), 1e-3),
        ("128^3 grid l9 x1 channel (100 cols)", inputs.config3_full_grid(), (9, 1, 6.0, 0.02), (12.0 / 128) ** 3),
    ]
    for name, pts, (lmax, per_l, cutoff, dr), dv in work:
        if not any(want(f"{k} {name}") for k in ("projectors soa", "projectors aos", "project nvec=1", "project nvec=4", "project nvec=8")):
            continue
        n = len(pts)
        proj_l, tab, dr = inputs.projector_channels(lmax=lmax, per_l=per_l, cutoff=cutoff, dr=dr)
        ncols = sh.projector_count(proj_l)
        x = torch.from_numpy(pts).to(dev)
        t = torch.from_numpy(tab).to(dev)
        reps = 50 if n < (1 << 20) else 20
        for layout in ("soa", "aos"):
            if not want(f"projectors {layout} {name}"):
                continue
            out = torch.empty((ncols, n) if layout == "soa" else (n, ncols), dtype=torch.float64, device=dev)
            ms = timed(lambda: sh.sh_projectors(x, proj_l, t, dr, out=out, layout=layout), reps)
            res[f"projectors {layout} {name}"] = {"ms": ms, "write_GBps": n * ncols * 8 / ms / 1e6, "G_values_per_s": n * ncols / ms / 1e6}
            if n >= (1 << 18):
                res[f"projectors {layout} {name}"]["roofline"] = hbm_roofline(
                    f"sh_projectors {layout}, {ncols} columns", n * (24 + 8 * ncols), n * 8 * ncols, ms, hbm_peak, hbm_src, ceil,
                    "soa_planes" if layout == "soa" else "bulk_tiles", traffic_key=f"projectors_{layout}")
            if n < (1 << 18):
                res[f"projectors {layout} {name}"]["ms_in_cuda_graph"] = timed_graph(lambda: sh.sh_projectors(x, proj_l, t, dr, out=out, layout=layout), 100)
            del out
        for nvec in (1, 4, 8):
            if not want(f"project nvec={nvec} {name}"):
                continue
            w = torch.from_numpy(inputs.wave_weights(n, nvec, seed=8, volume_element=dv)).to(dev)
            coeff = torch.empty((nvec, ncols), dtype=torch.float64, device=dev)
            ws = torch.empty(max(sh.project_workspace_bytes(ncols, nvec), 8), dtype=torch.uint8, device=dev)
            ms = timed(lambda: sh.sh_project(x, proj_l, t, dr, w, coeff=coeff, workspace=ws), reps)
            if n < (1 << 18):   # launch-bound: the roofline below uses the CUDA-graph time
                ms_py, ms = ms, timed_graph(lambda: sh.sh_project(x, proj_l, t, dr, w, coeff=coeff, workspace=ws), 100)
            # algorithmic FP64 work per point: DESIGN.md section 6 "fused projection" (instruction counts of the evaluated blocks
            # + ncols (radial scale) + nvec x ncols (contraction)); reported against the FP64 pipe
            fp64_per_point = PROJECT_FP64_PER_POINT.get(lmax, 0) + ncols + nvec * ncols
            res[f"project nvec={nvec} {name}"] = {
                "ms": ms, "G_points_per_s": n / ms / 1e6, "G_values_per_s": n * ncols * nvec / ms / 1e6,
                "read_GBps": n * (24 + 8 * nvec) / ms / 1e6,
                "roofline": {"bound": "alu", "unit": "G FP64 lane-instr/s", "achieved": n * fp64_per_point / ms / 1e6,
                             "peak": peak_ginstr, "frac": n * fp64_per_point / ms / 1e6 / peak_ginstr, "peak_source": peak_src,
                             "peak_nominal": nominal_ginstr, "fp64_instr_per_point": fp64_per_point,
                             "what": "algorithmic FP64 work of the method (factorized forms) per second over the measured FP64 pipe peak"},
            }
            executed = ncu_fp64_executed(f"project_nv{nvec}") if n == 128 ** 3 else None
            if executed:   # the default Horner / recurrence forms issue fewer FP64 instructions than the algorithmic count
                res[f"project nvec={nvec} {name}"]["roofline"].update({
                    "fp64_instr_per_point_executed": executed / n, "frac_executed": executed / ms / 1e6 / peak_ginstr,
                    "executed_source": "profiles/ncu_fp64_instr.csv (ncu smsp__sass_thread_inst_executed_op_d*_pred_on of the same launch)"})
            if n < (1 << 18):
                res[f"project nvec={nvec} {name}"].update({"ms": ms_py, "ms_in_cuda_graph": ms})
            else:
                # the same call with the factorized root-pair forms of every other call (SH_TUNE_PROJECT_FORM = 2; the default
                # of this one FP64-bound call is Horner in z^2 + the azimuthal recurrence): the factorized-vs-Horner question of
                # the paper in the one place where arithmetic, not HBM, sets the time
                sh.set_tuning("project_form", 2)
                try:
                    res[f"project nvec={nvec} {name}"]["ms_factorized_forms"] = timed(
                        lambda: sh.sh_project(x, proj_l, t, dr, w, coeff=coeff, workspace=ws), reps)
                finally:
                    sh.set_tuning("project_form", 0)
            del w, coeff, ws
        del x, t
        torch.cuda.empty_cache()
    return res


# FP64 instructions (DADD + DMUL + DFMA in SASS, one lane-slot each) per point of steps a2-a5 for all blocks l <= lmax, as
# compiled for the store kernels (cuobjdump: 94 at lmax = 3, 566 at lmax = 9), plus the radial position (sqrt, ~12) and the
# table interpolation (3 per channel: 8 / 10 channels); DESIGN.md section 6.  Keys = lmax.
PROJECT_FP64_PER_POINT = {3: 94 + 12 + 24, 9: 566 + 12 + 30}
REAL_L9_FP64_PER_POINT = 538   # a2-a5 at lmax = 9 in the factorized forms, one warp per point group: FP64 thread-instructions EXECUTED per point
                               # (ncu smsp__sass_thread_inst_executed_op_d*_pred_on of sh_real AoS, profiles/ncu_fp64_instr.csv; the static SASS count, both
                               # branches of the range scaling included, is 566-575)


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2510_05282_b200 as sh
    from paper_2510_05282_b200.dist import env_world, max_over_ranks

    from paper_2510_05282_b200 import build as _build

    _build.ensure_built()  # compiles only if the in-tree library is absent
    sh.load()  # no fallback: fails here if libshb200.so cannot be loaded
    tune = {k: int(v) for k, v in (t.split("=", 1) for t in args.tune)}
    for knob, value in tune.items():
        sh.set_tuning(knob, value)
    rank, local, world = env_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    sampler = ClockSampler(local) if rank == 0 else None  # started early: nvidia-smi needs ~0.2 s to come up
    grid = grid_points()
    # the job is `world` grids laid end to end, cut into contiguous point ranges (inputs.shard_range): rank r owns grid r
    from paper_2510_05282_b200 import inputs as _inputs

    lo, hi = _inputs.shard_range(world * len(grid), rank, world)
    assert hi - lo == len(grid) and lo % len(grid) == 0
    pts = grid
    n = len(pts)
    nrep_in, nrep_out = 4, 2  # 4 x 50 MB inputs > L2; outputs 1.68 GB each
    xs = [torch.from_numpy(pts).to(dev) for _ in range(nrep_in)]
    out_soa = [torch.empty((K, n), dtype=torch.float64, device=dev) for _ in range(nrep_out)]
    out_aos = [torch.empty((n, K), dtype=torch.float64, device=dev) for _ in range(nrep_out)]
    stream = torch.cuda.current_stream(dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(it, marks=None):
        x = xs[it % nrep_in]
        if marks is not None:
            e0, e1, e2 = ev(), ev(), ev()
            e0.record(stream)
        sh.sh_real(x, LMAX, out=out_soa[it % nrep_out], layout="soa")
        if marks is not None:
            e1.record(stream)
        sh.sh_real(x, LMAX, out=out_aos[it % nrep_out], layout="aos")
        if marks is not None:
            e2.record(stream)
            marks.append((e0, e1, e2))

    for it in range(max(args.warmup, 3)):
        step(it)
    torch.cuda.synchronize()
    barrier()
    launches0 = sh.kernel_launch_count()
    marks = []
    start, end = ev(), ev()
    torch.cuda.synchronize()
    wall0 = time.time()
    start.record(stream)
    for it in range(args.steps):
        step(it, marks)
    end.record(stream)
    torch.cuda.synchronize()
    barrier()
    launches = sh.kernel_launch_count() - launches0
    # The timed region lasts ~0.6 ms x steps, shorter than nvidia-smi's sampling period, so the same step loop keeps
    # running (untimed) until the load window is >= 1.5 s long; clocks are the samples inside that window.
    it = args.steps
    while time.time() - wall0 < 1.5:
        for _ in range(50):
            step(it); it += 1
        torch.cuda.synchronize()
    clocks = sampler.stop(wall0, time.time()) if sampler else None
    if clocks is not None:
        clocks["window"] = "timed region + untimed continuation of the same step loop, 1.5 s in total"
    ms = start.elapsed_time(end)
    ms = max_over_ranks(ms, dev)
    t_soa = sum(a.elapsed_time(b) for a, b, _ in marks) / len(marks)
    t_aos = sum(b.elapsed_time(c) for _, b, c in marks) / len(marks)

    # end to end through the C ABI with HOST buffers (pinned): H2D of xyz and D2H of every result inside the timed region
    e2e_steps = max(1, min(args.steps, 3))
    hx = torch.from_numpy(pts).pin_memory()
    h_soa = torch.empty((K, n), dtype=torch.float64).pin_memory()
    h_aos = torch.empty((n, K), dtype=torch.float64).pin_memory()

    def e2e_step():
        sh.host_call("real", hx, LMAX, out=h_soa, layout="soa")
        sh.host_call("real", hx, LMAX, out=h_aos, layout="aos")

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dev)
    # spot-check the end-to-end result against the device-resident result
    assert torch.equal(h_aos[:1000], out_aos[(args.steps - 1) % nrep_out][:1000].cpu())
    assert torch.equal(h_soa[:, :1000], out_soa[(args.steps - 1) % nrep_out][:, :1000].cpu())

    if rank == 0:
        peak, peak_src = measured_peak()
        del out_soa, out_aos, xs
        torch.cuda.empty_cache()
        ceil = ceilings(dev, local) if (world == 1 and not args.no_ceilings) else None
        dom = ("sh_real lmax=9 SoA", t_soa, "soa") if t_soa >= t_aos else ("sh_real lmax=9 AoS", t_aos, "aos")
        values_per_step = 2 * n * K
        line = {
            "metric": METRIC, "value": world * args.steps * values_per_step / (ms * 1e-3) / 1e9, "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "points_per_gpu": n, "lmax": LMAX, "calls_per_step": ["sh_real SOA", "sh_real AOS"],
                       "l2": "outputs (1.68 GB per call) and rotating input replicas (4 x 50 MB) exceed the 126 MB L2",
                       **({"tune": tune} if tune else {})},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "kernels": {
                "sh_real_soa": {"ms": t_soa, "write_GBps": 8 * K * n / (t_soa * 1e-3) / 1e9, "G_values_per_s": n * K / (t_soa * 1e-3) / 1e9,
                                "roofline": hbm_roofline("sh_real lmax=9 SoA", BYTES_PER_POINT * n, 8 * K * n, t_soa, peak, peak_src, ceil, "soa_planes", "real_soa")},
                "sh_real_aos": {"ms": t_aos, "write_GBps": 8 * K * n / (t_aos * 1e-3) / 1e9, "G_values_per_s": n * K / (t_aos * 1e-3) / 1e9,
                                "roofline": hbm_roofline("sh_real lmax=9 AoS", BYTES_PER_POINT * n, 8 * K * n, t_aos, peak, peak_src, ceil, "bulk_tiles", "real_aos")},
            },
            "roofline": hbm_roofline(dom[0], BYTES_PER_POINT * n, 8 * K * n, dom[1], peak, peak_src, ceil,
                                     "soa_planes" if dom[2] == "soa" else "bulk_tiles", traffic_key="real_" + dom[2]),
            "e2e": {"value": world * e2e_steps * values_per_step / e2e_s / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": 2 * n * 24, "d2h_bytes_per_step": 2 * n * K * 8, "steps": e2e_steps,
                    "api": "sh_real_host (pinned host buffers)"},
        }
        if ceil:
            line["ceilings"] = ceil
        if world == 1 and not args.no_extras:
            line["other_configs"] = extra_configs(sh, dev, args.only, ceil)
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(pts)
            line["cpu_method"] = cpu_method(pts)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the untimed-by-`value` runs of the other configs")
    ap.add_argument("--no-ceilings", action="store_true", help="skip the write-fill / DFMA ceiling measurements (csrc/sh_peaks.cu)")
    ap.add_argument("--tune", action="append", default=[], metavar="KNOB=VALUE",
                    help="override a launch heuristic for the whole run (binding.TUNE names, e.g. soa_split=2); recorded in config")
    ap.add_argument("--only", default=None, help="run only the other-config cases whose name contains this substring")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
