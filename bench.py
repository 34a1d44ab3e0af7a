#!/usr/bin/env python
"""bench.py -- MSFT patterns/s on B200 (BASELINE.json metric), one JSON line.

A "step" is one pass of the whole hot path (a0-a6: q-map, [orient], column prefix, operand pack, phase
tables, tcgen05 contraction with fused epilogue, |A|^2) over one batch of synthetic input through the
C ABI (scatman_simulate).  Default workload = BASELINE.json configs[2], the 256^3 / 512x512 droplet on
which north_star quotes its target.  `--impl reference` times the FP64 CPU oracle instead.
"""
from __future__ import annotations

import argparse
import ctypes as C
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

SPLITS = 3           # FP16x3: AhBh + AlBh + AhBl
FLOP_PER_TERM = 8    # one complex MAC
# dram__bytes_read.sum + dram__bytes_write.sum of one contraction launch, from the committed `ncu --set full` capture
# (profiles/r02_contract_cfg3_full.md); only the workload that was captured has a number
NCU_DRAM_BYTES_PER_LAUNCH = {"cfg3_droplet_256": 970.813952e6 + 8.573184e6}   # profiles/r02_contract_cfg3_full.md (r01: 2.30e9, with the M_z table)
# the same for the kernels of one NUFFT pattern (strength, pack, stages X, Y, Z, interpolation; profiles/r02_nufft_tensor.md)
NCU_DRAM_BYTES_NUFFT = {"cfg3_droplet_256": (134.25 + 91.21 + 134.23 + 88.48 + 104.12 + 17.44 + 59.54 + 3.20 + 29.79 + 0.0 + 8.68 + 0.0) * 1e6}


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return {"burst": float(p["bf16_tflops"]), "sustained": float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                "source": "measured"}
    except Exception:
        return {"burst": 1590.0, "sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.gpu = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        sm.sort()
        load = [v for v in sm if mx and v > 0.3 * mx] or sm
        med = load[len(load) // 2] if load else None
        return {"sm_mhz": med, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(sm)}


def workload_for(args):
    from paper_2202_03411_b200 import workloads as W
    w = W.config(args.config)
    items = list(range(w.batch if args.batch <= 0 else min(args.batch, w.batch)))
    return w, items


def run_reference(args):
    """The oracle as it stands on the host cores, on a bounded pixel sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    from oracle import oracle as O
    from paper_2202_03411_b200 import workloads as W
    w, items = workload_for(args)
    g = w.grid(0)
    quat = None if w.quat is None else w.quat[0]
    vox = (w.dx, w.dy, w.dz)
    if args.ref_pixels > 0:
        npix_s = max(8, int(args.ref_pixels))
    else:   # ~10 s per step; two probes separate the per-call set-up from the per-pixel cost
        tp = []
        for n_probe in (16, 80):
            probe = W.sample_pixels(w.seed + 99, w.npix, n_probe)
            t0 = time.perf_counter()
            O.simulate(g, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, pixels=probe)
            tp.append((len(probe), time.perf_counter() - t0))
        per_pixel = max(1e-9, (tp[1][1] - tp[0][1]) / (tp[1][0] - tp[0][0]))
        setup = max(0.0, tp[0][1] - tp[0][0] * per_pixel)
        npix_s = int(min(8192, max(128, (10.0 - setup) / per_pixel)))
    pix = W.sample_pixels(w.seed, w.npix, npix_s)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        O.simulate(g, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, pixels=pix)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
    total = sum(times)
    frac = len(pix) / w.npix                      # of one pattern per step
    value = frac * len(times) / total             # patterns/s, exact extrapolation (work is linear in pixels)
    cores = O.num_threads()
    sample = f"{len(pix)} seeded pixels of one {w.name} pattern per step ({frac:.3e} of a pattern)"
    line = {"impl": "reference", "metric": "msft_patterns_per_s", "value": value, "unit": "patterns/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "grid": [w.nz, w.ny, w.nx], "detector": [w.npy, w.npx], "batch": 1},
            "terms_per_s": value * w.nvox * w.npix,
            "cpu_baseline": {"value": value, "unit": "patterns/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": "patterns/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_fit(args):
    """--route fit: the forward-fitting pieces on cfg4's shape of work: 256 candidate patterns of 256 x 256
    pixels against one measured pattern.  A step = scatman_discrepancy (integral-normalised L2, masked) of the whole batch; the
    Poisson deviance (FP64 log per pixel: FP64-ALU-bound) and the Ideal detector are timed beside it.  Single GPU; HBM-bound: 8 B per pixel and item (two passes over the FP32 patterns; the
    measured pattern and the mask are shared and stay in L2)."""
    import numpy as np
    import torch
    from oracle import fitting as F
    from paper_2202_03411_b200 import binding as B, build as lib_build
    lib_build.build()
    sm = B.Scatman(0)
    rng = np.random.default_rng(220203411 + 40)
    batch, npy, npx = 256, 256, 256
    npix = npy * npx
    I = (rng.uniform(0.0, 1.0, (batch, npix)) ** 6 * 1e4).astype(np.float32)       # six decades, like a wide-angle pattern
    M = rng.poisson(0.5 * I[0]).astype(np.float32)
    mask = (rng.uniform(size=npix) < 0.9).astype(np.uint8)
    d_I, d_M, d_mask = (torch.from_numpy(a).cuda() for a in (I, M, mask))
    out = torch.empty(batch, dtype=torch.float64, device="cuda")
    counts = torch.empty_like(d_I)
    flush = torch.empty(192 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()

    def timed(fn):
        for _ in range(args.warmup):
            flush.zero_()
            fn()
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev) / args.steps

    sampler = ClockSampler(0)
    sampler.start()
    time.sleep(0.25)
    ms_d = timed(lambda: sm.discrepancy(d_I, d_M, d_mask, metric=B.LOSS_L2_NORMALISED, out=out, stream=stream))
    launches = sm.last_launch_count() * args.steps
    ms_p = timed(lambda: sm.discrepancy(d_I, d_M, d_mask, metric=B.LOSS_POISSON_DEVIANCE, out=out, stream=stream))
    ms_n = timed(lambda: sm.ideal_detector(d_I, 1.0e7, seed=1, out=counts, stream=stream))
    clocks = sampler.stop()
    h_I = torch.from_numpy(I).pin_memory()
    h_out = torch.empty(batch, dtype=torch.float64).pin_memory()
    t0 = time.perf_counter()
    for _ in range(3):
        d_I.copy_(h_I, non_blocking=True)
        sm.discrepancy(d_I, d_M, d_mask, metric=B.LOSS_L2_NORMALISED, out=out, stream=stream)
        h_out.copy_(out, non_blocking=True)
        torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / 3
    t0 = time.perf_counter()
    ref = F.discrepancy_l2(I, M, mask)
    cpu_s = time.perf_counter() - t0
    parity = float(np.max(np.abs(out.cpu().numpy() - ref) / np.abs(ref)))
    peaks = load_peaks_hbm()
    bytes_step = 8.0 * batch * npix
    ach = bytes_step / (ms_d * 1e-3) / 1e9
    line = {"metric": "fit_patterns_per_s", "value": batch / (ms_d * 1e-3), "unit": "patterns/s", "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_d, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64 accumulation of f32 patterns", "data": "synthetic",
            "config": {"workload": "fit_batch_256x256x256", "detector": [npy, npx], "batch": batch, "route": "fit",
                       "metric": "l2_normalised, 90 % mask", "l2": "flushed between steps (192 MiB write)"},
            "roofline": {"bound": "hbm", "kernel": "fit_sums_kernel + fit_metric_kernel", "achieved": ach, "peak": peaks[0],
                         "unit": "GB/s", "frac": ach / peaks[0], "traffic": None, "peak_source": peaks[1],
                         "achieved_is": "8 B per pixel and item (two passes over the FP32 patterns) / CUDA-event time of the call"},
            "poisson_deviance": {"ms_per_step": ms_p, "patterns_per_s": batch / (ms_p * 1e-3), "bound": "alu (FP64 log per pixel)"},
            "ideal_detector": {"ms_per_step": ms_n, "patterns_per_s": batch / (ms_n * 1e-3), "photons_per_pattern": 1.0e7,
                               "bytes_per_pixel_item": 12, "gbps": 12.0 * batch * npix / (ms_n * 1e-3) / 1e9},
            "cpu_baseline": {"value": batch / cpu_s, "unit": "patterns/s", "cores": 1, "kind": "oracle",
                             "sample": f"oracle.fitting.discrepancy_l2 on the same {batch} patterns ({cpu_s:.2f} s)",
                             "parity_max_rel": parity},
            "e2e": {"value": batch / e2e_s, "unit": "patterns/s", "h2d_bytes_per_step": int(I.nbytes), "d2h_bytes_per_step": batch * 8},
            "gpu_launches": launches, "clocks": clocks}
    print(json.dumps(line), flush=True)


def load_peaks_hbm():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        for k in ("hbm_gbs", "hbm_gbps"):
            if k in p:
                return float(p[k]), f"MEASURED_PEAKS.json {k} (measured)"
    except Exception:
        pass
    return 6500.0, "fallback of B200_PROFILING.md"


def measure_peaks(args):
    """--measure-peaks: dense GEMM peaks of the tensor pipe for the operand types the library's tcgen05 kernels use, with
    MEASURED_PEAKS.json's protocol (torch.matmul 8192^3, 2 N^3 flop: best of 10 = burst, then back to back for 4 s =
    sustained, SM clock sampled under load).  FP16 is the type of every contraction here (kind::f16); BF16 repeats the
    driver's own measurement on this box for comparison; TF32 is the type SURVEY 8(d) sized its target on."""
    import torch
    n = 8192
    out = {"how": "torch.matmul 8192^3 (2 N^3 flop): best of 10 (burst), back to back for 4 s (sustained); CUDA events",
           "gpu": torch.cuda.get_device_name(0)}
    for name, dt, tf32 in (("fp16", torch.float16, False), ("bf16", torch.bfloat16, False), ("tf32", torch.float32, True)):
        torch.backends.cuda.matmul.allow_tf32 = tf32
        a = torch.randn(n, n, device="cuda", dtype=dt)
        b = torch.randn(n, n, device="cuda", dtype=dt)
        c = torch.empty(n, n, device="cuda", dtype=dt)
        for _ in range(5):
            torch.matmul(a, b, out=c)
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(10):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            torch.matmul(a, b, out=c)
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        sampler = ClockSampler(0)
        sampler.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0, reps = time.perf_counter(), 0
        e0.record()
        while time.perf_counter() - t0 < 4.0:
            for _ in range(20):
                torch.matmul(a, b, out=c)
            reps += 20
            torch.cuda.synchronize()
        e1.record()
        torch.cuda.synchronize()
        clocks = sampler.stop()
        out[name] = {"tflops_burst": 2.0 * n ** 3 / (best * 1e-3) / 1e12,
                     "tflops_sustained": 2.0 * n ** 3 * reps / (e0.elapsed_time(e1) * 1e-3) / 1e12, "clocks": clocks}
        del a, b, c
    torch.backends.cuda.matmul.allow_tf32 = False
    print(json.dumps(out), flush=True)


# GEMM peaks measured on this pool with MEASURED_PEAKS.json's protocol (`python bench.py --measure-peaks`, profiles/r02_peaks.md):
# the operand type of every contraction here is FP16 (kind::f16); context beside the driver-written BF16 figures.
MEASURED_FP16 = {"burst": 1466.2, "sustained": 1286.0, "sm_mhz_under_load": 1207.0, "source": "profiles/r02_peaks.md"}
PIPE_FLOP_PER_CLK_SM = 8192          # dense FP16/BF16 tensor flop per clock and SM (2250 TFLOP/s nominal = 148 SMs x 8192 x 1.855 GHz)


def tensor_roofline_extras(achieved, clocks, peaks):
    """Context for a tensor-bound roofline entry.  `frac` divides by MEASURED_PEAKS.json's bf16 BURST figure (the kernel is timed by
    its own CUDA events; kind::f16 runs at the bf16 rate).  That cuBLAS figure was measured power-capped at ~1.3 GHz, so a kernel
    that holds a higher clock can exceed it; `frac_of_pipe_ceiling` divides by what the tensor pipes can issue at the clock sampled
    during THIS run and is <= 1 by construction."""
    mhz = (clocks or {}).get("sm_mhz") or 1965.0
    ceiling = 148 * PIPE_FLOP_PER_CLK_SM * mhz * 1e6 / 1e12
    return {"peak_sustained": peaks["sustained"], "frac_of_sustained": achieved / peaks["sustained"],
            "peak_nominal": 2250.0, "frac_of_nominal": achieved / 2250.0,
            "pipe_ceiling_at_sampled_clock": ceiling, "frac_of_pipe_ceiling": achieved / ceiling, "sampled_sm_mhz": mhz,
            "peak_fp16_measured": MEASURED_FP16}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json configs (default 2: 256^3 / 512x512)")
    ap.add_argument("--batch", type=int, default=0, help="limit the batch of config 3 (0 = all)")
    ap.add_argument("--method", type=int, default=1, help="1 tensor (default), 2 simt_sincos, 3 simt_table")
    ap.add_argument("--ref-pixels", type=int, default=0, help="pixels per step of the CPU oracle sample (0 = sized for ~15 s)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--graph", action="store_true",
                    help="capture one call in a CUDA graph after the warm-up and time its replays (routes pixels, qgrid, nufft)")
    ap.add_argument("--reuse-tables", action="store_true",
                    help="time with SCATMAN_FLAG_REUSE_TABLES (q-map and phase tables kept from the previous call); the default "
                         "rebuilds them every step and reports the cached figure beside it")
    ap.add_argument("--shard", default="items", choices=["items", "pixels"],
                    help="N > 1: items = every rank runs the whole workload (weak scaling, the paper's scheme); pixels = every rank "
                         "simulates its row band of the detector and rank 0 gathers the pattern (strong scaling)")
    ap.add_argument("--e2e-batch", type=int, default=4,
                    help="patterns per end-to-end call (the host entry points overlap upload, compute and download chunk by chunk)")
    ap.add_argument("--route", default="pixels", choices=["pixels", "qgrid", "shapes", "shapes_qgrid", "fit", "nufft", "shapes_nufft"],
                    help="pixels: the flat detector of BASELINE.json (default, the headline); qgrid: the separable route on a "
                         "uniform (qx, qy) grid of the same size and angular reach (scatman_simulate_qgrid); shapes: the particles "
                         "go in as shape descriptors and are rendered on the device (scatman_simulate_shapes; not cfg5)")
    ap.add_argument("--measure-peaks", action="store_true",
                    help="measure the FP16 / BF16 / TF32 GEMM peaks with MEASURED_PEAKS.json's protocol and print them (no bench)")
    args = ap.parse_args()
    if args.measure_peaks:
        if int(os.environ.get("RANK", "0")) == 0:
            measure_peaks(args)
        return
    if args.impl == "reference":
        run_reference(args)
        return
    if args.route == "fit":
        if int(os.environ.get("RANK", "0")) == 0:
            run_fit(args)
        return

    import numpy as np
    import torch
    from paper_2202_03411_b200 import binding as B, build as lib_build
    from paper_2202_03411_b200.sharding import shard_detector_rows, shard_range
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    torch.cuda.set_device(local)
    if rank == 0:
        lib_build.build()
    if dist:
        dist.barrier()
    sm = B.Scatman(local)
    shapes_route = args.route in ("shapes", "shapes_qgrid", "shapes_nufft")
    shard_pixels = args.shard == "pixels"
    if shard_pixels and args.route not in ("pixels", "nufft"):
        raise SystemExit("--shard pixels applies to the flat-detector routes (pixels, nufft)")

    w, items = workload_for(args)
    vox = (w.dx, w.dy, w.dz)
    if shard_pixels:
        # strong scaling: every rank holds the whole (small) volume and simulates its row band of the detector
        y0, y1, cy_band = shard_detector_rows(w.npy, 0.0, rank, world)
        npy_r = y1 - y0
    else:
        # weak scaling: the global job is `world` copies of the batch; shapes shard across ranks with no collective
        global_items = [i for _ in range(world) for i in items]
        lo, hi = shard_range(len(global_items), rank, world)
        items = global_items[lo:hi]
        y0, y1, cy_band, npy_r = 0, w.npy, 0.0, w.npy
    g = w.grids(items)
    quat = None if w.quat is None else w.quat[items]
    batch = len(items)
    npix_r = npy_r * w.npx
    d_dn = torch.from_numpy(g).cuda()
    grid = B.Grid(w.nx, w.ny, w.nz, *vox)
    det = B.Detector(w.npx, npy_r, w.theta_max_deg, 0.0, cy_band)
    opts = B.Options(0, args.method, 0, 0)
    out = torch.empty((batch, npy_r, w.npx), dtype=torch.float32, device="cuda")
    flush = torch.empty(192 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()
    qmethod = args.method if args.method in (0, 1, 3) else 0
    qopts = B.Options(0, qmethod, 0, 0)
    qx = qy = qx_h = qy_h = nq = shapes = None
    need = C.c_size_t(0)
    if args.route in ("qgrid", "shapes_qgrid"):
        kk = 2 * np.pi / w.lam
        qx_h = (np.arange(w.npx) + 0.5 - 0.5 * w.npx) * (2 * kk * np.sin(np.radians(w.theta_max_deg)) / w.npx)
        qy_h = (np.arange(w.npy) + 0.5 - 0.5 * w.npy) * (2 * kk * np.sin(np.radians(w.theta_max_deg)) / w.npy)
        qx, qy = torch.from_numpy(qx_h).cuda(), torch.from_numpy(qy_h).cuda()
    if shapes_route:
        shapes = w.shapes(items)
        if shapes is None:
            raise SystemExit(f"{w.name} is not one shape per item: --route {args.route} does not apply")
    L = sm.lib
    ws_calls = {
        "pixels": lambda: L.scatman_workspace_bytes(sm._ctx, C.byref(grid), npix_r, batch, C.byref(opts), C.byref(need)),
        "qgrid": lambda: L.scatman_qgrid_workspace_bytes(sm._ctx, C.byref(grid), w.npx, w.npy, batch, C.byref(qopts), C.byref(need)),
        "nufft": lambda: L.scatman_nufft_workspace_bytes(sm._ctx, C.byref(grid), w.lam, C.byref(det), batch, C.byref(need)),
        "shapes": lambda: L.scatman_shapes_workspace_bytes(sm._ctx, C.byref(grid), npix_r, batch, C.byref(opts), C.byref(need)),
        "shapes_qgrid": lambda: L.scatman_shapes_qgrid_workspace_bytes(sm._ctx, C.byref(grid), w.npx, w.npy, batch, C.byref(qopts), C.byref(need)),
        "shapes_nufft": lambda: L.scatman_shapes_nufft_workspace_bytes(sm._ctx, C.byref(grid), w.lam, C.byref(det), batch, C.byref(need)),
    }
    sm._check(ws_calls[args.route]())
    ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")
    if args.route in ("nufft", "shapes_nufft"):
        nq = sm.nufft_grid_dims(grid, w.lam, det)
    dims = (w.nx, w.ny, w.nz)
    gathered = [torch.empty((batch, (w.npy + world - 1) // world, w.npx), dtype=torch.float32, device="cuda") for _ in range(world)] \
        if (shard_pixels and dist and rank == 0) else None
    band_pad = torch.zeros((batch, (w.npy + world - 1) // world, w.npx), dtype=torch.float32, device="cuda") if (shard_pixels and dist) else None

    def step(flags=0, st=stream):
        if args.route == "shapes":
            sm.simulate_shapes(shapes, dims, vox, w.lam, w.npx, w.npy, w.theta_max_deg, method=args.method, workspace=ws, out=out,
                               stream=st, flags=flags)
        elif args.route == "shapes_qgrid":
            sm.simulate_shapes_qgrid(shapes, dims, vox, w.lam, qx, qy, method=qmethod, workspace=ws, out=out, stream=st)
        elif args.route == "qgrid":
            sm.simulate_qgrid(d_dn, vox, w.lam, qx, qy, quat=quat, method=qmethod, workspace=ws, out=out, stream=st, flags=flags)
        elif args.route == "shapes_nufft":
            sm.simulate_shapes_nufft(shapes, dims, vox, w.lam, w.npx, w.npy, w.theta_max_deg, workspace=ws, out=out, stream=st)
        elif args.route == "nufft":
            sm.simulate_nufft(d_dn, vox, w.lam, w.npx, npy_r, w.theta_max_deg, quat=quat, cy=cy_band, workspace=ws, out=out, stream=st,
                              flags=flags)
        else:
            sm.simulate(d_dn, vox, w.lam, w.npx, npy_r, w.theta_max_deg, quat=quat, method=args.method, cy=cy_band, workspace=ws,
                        out=out, stream=st, flags=flags)
        if band_pad is not None:       # pixel sharding: rank 0 gathers the row bands (NCCL gather of equal-sized padded bands)
            band_pad[:, :npy_r] = out
            dist.gather(band_pad, gathered, dst=0)

    def timed(nsteps, flags=0, graph=None):
        """nsteps steps, L2 flushed before each (outside its events); returns (total ms, launches, contraction ms per step)."""
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
        k_ms, n = [], 0
        torch.cuda.synchronize()
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            if graph is not None:
                graph.replay()
                b.record(stream)
                continue
            step(flags)
            b.record(stream)
            n += sm.last_launch_count()
            k_ms.append(sm.last_contraction_ms())   # the library's events on the launch stream; waits for this step
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in ev), n, k_ms

    base_flags = B.FLAG_REUSE_TABLES if args.reuse_tables else 0
    for _ in range(args.warmup):
        flush.zero_()
        step(base_flags)
    torch.cuda.synchronize()
    graph = None
    graph_launches = 0
    if args.graph:
        if shapes_route or dist:
            raise SystemExit("--graph applies to the single-GPU routes pixels, qgrid, nufft")
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):      # the call only enqueues on the capturing stream: the whole step becomes one graph
            step(base_flags, st=None)
        graph_launches = sm.last_launch_count()
        graph.replay()
        torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    total_ms, launches, kernel_ms = timed(args.steps, base_flags, graph)
    if graph is not None:
        launches = graph_launches * args.steps
    if dist:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    # the same step with the phase tables of the previous call kept (SCATMAN_FLAG_REUSE_TABLES): reported beside the headline
    cached = None
    if not args.reuse_tables and graph is None and not shapes_route and not dist:
        step(B.FLAG_REUSE_TABLES)
        c_ms, _, _ = timed(min(args.steps, 5), B.FLAG_REUSE_TABLES)
        cached = {"ms_per_step": c_ms / min(args.steps, 5), "value": batch * min(args.steps, 5) / (c_ms * 1e-3), "unit": "patterns/s",
                  "what": "same step with SCATMAN_FLAG_REUSE_TABLES: q-map and phase tables kept from the previous call"}

    # ---- end to end through the host-buffer C entry points: pinned host grids in, pinned host patterns out, every step
    e2e = None
    if shapes_route:
        # the inputs ARE the descriptors (host structs, marshalled per call); the patterns come back to pinned host memory
        h_I = torch.empty((batch, npy_r, w.npx), dtype=torch.float32).pin_memory()
        e2e_steps = max(1, min(args.steps, 3))

        def e2e_step():
            step()
            h_I.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        e2e_batch = batch
        h2d = int(C.sizeof(B.Shape) * batch + sum(24 * len(sh.get("coeffs", ())) for sh in shapes))
        copy_bound = None
    else:
        e2e_batch = batch if batch >= args.e2e_batch else args.e2e_batch      # small batches are replicated: the pipeline needs chunks
        rep = (e2e_batch + batch - 1) // batch
        e2e_batch = rep * batch
        h_dn = torch.from_numpy(np.concatenate([g] * rep)).pin_memory()
        quat_e = None if quat is None else np.concatenate([quat] * rep)
        h_I = torch.empty((e2e_batch, npy_r, w.npx), dtype=torch.float32).pin_memory()
        e2e_steps = max(1, min(args.steps, 3))

        def e2e_step():
            if args.route == "qgrid":
                sm.simulate_qgrid_host(h_dn, vox, w.lam, qx_h, qy_h, quat=quat_e, method=qmethod, h_out=h_I)
            elif args.route == "nufft":
                sm.simulate_nufft_host(h_dn, vox, w.lam, w.npx, npy_r, w.theta_max_deg, quat=quat_e, h_out=h_I, cy=cy_band)
            else:
                sm.simulate_host(h_dn, vox, w.lam, w.npx, npy_r, w.theta_max_deg, quat=quat_e, method=args.method, h_out=h_I, cy=cy_band)
        h2d = int(h_dn.numel() * 4)
        # the copy bound: the same bytes through one pinned H2D copy and one D2H copy, nothing else
        d_tmp = torch.empty_like(h_dn, device="cuda")
        d_tmp.copy_(h_dn, non_blocking=True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        d_tmp.copy_(h_dn, non_blocking=True)
        torch.cuda.synchronize()
        copy_s = time.perf_counter() - t0
        del d_tmp
        copy_bound = {"h2d_s": copy_s, "h2d_gbps": h2d / copy_s / 1e9, "patterns_per_s": e2e_batch / copy_s}
    e2e_step()
    if dist:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    e2e_s = time.perf_counter() - t0
    if dist:
        t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    if rank != 0:
        return
    e2e_patterns = e2e_batch * e2e_steps * (1 if shard_pixels else world)
    e2e = {"value": e2e_patterns / e2e_s, "unit": "patterns/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": int(h_I.numel() * 4),
           "patterns_per_step": e2e_batch, "copy_bound": copy_bound,
           "through": "descriptors marshalled per call + pattern read-back" if shapes_route else
                      {"pixels": "scatman_simulate_host", "nufft": "scatman_simulate_nufft_host", "qgrid": "scatman_simulate_qgrid_host"}[args.route]}
    if copy_bound:
        e2e["frac_of_copy_bound"] = e2e["value"] / (copy_bound["patterns_per_s"] * (1 if shard_pixels else world))

    patterns = batch * args.steps * (1 if shard_pixels else world)
    value = patterns / (total_ms * 1e-3)
    terms_per_pattern = w.nvox * w.npix
    terms_issued_per_pattern = None
    peaks = load_peaks()
    # graph replays have no per-kernel events: the roofline then takes the WHOLE step (a1, a2 and tables included) as the kernel time
    k_ms = sum(kernel_ms) / len(kernel_ms) if kernel_ms else total_ms / args.steps
    dense = SPLITS * FLOP_PER_TERM * w.nvox * npix_r * batch           # tensor flop of the dense sum per launch (this rank's pixels)
    if args.route in ("qgrid", "shapes_qgrid"):
        dense_sep = 8.0 * batch * (w.nz * w.ny * w.nx * w.npx + w.nz * w.npy * w.ny * w.npx)   # both stages, 8 flop per complex MAC
        if qmethod == 3:
            # two FP32 complex GEMMs per slice on CUDA cores, dense count (vacuum rows are skipped)
            peak = 148 * 128 * 2 * 1.965e9 / 1e12      # FP32 FMA: 148 SMs x 128 lanes x 2 flop x max clock
            ach = dense_sep / (k_ms * 1e-3) / 1e12
            roofline = {"bound": "alu", "kernel": "sep_stage_x_kernel + sep_stage_yz_kernel", "achieved": ach, "peak": peak,
                        "unit": "TFLOP/s", "frac": ach / peak, "traffic": None, "kernel_ms": k_ms,
                        "achieved_is": "dense FP32 flop of both GEMM stages / their CUDA-event time; all-vacuum rows are skipped, so "
                                       "this can exceed what the ALUs executed"}
        else:
            # both stages on tcgen05, FP16x3: 24 tensor flop per complex MAC of the tiles the kernels issue.  The live tiles follow
            # from the input alone (a 64-y block of a slice is skipped iff it is all vacuum), counted here on the host:
            # stage X issues 128-y row tiles x all padded x x all padded columns, stage YZ 64-y blocks x padded rows x columns.
            pad = lambda n, m: (n + m - 1) // m * m
            NY, NXP, NPXP, NPYP = pad(w.ny, 128), pad(w.nx, 64), pad(w.npx, 64), pad(w.npy, 128)
            issued = 0.0
            for gi in g:
                occ = np.zeros((w.nz, NY), bool)
                occ[:, :w.ny] = (gi != 0).any(axis=(2, 3))
                blk = occ.reshape(w.nz, NY // 64, 64).any(axis=2)                 # live 64-y blocks
                grp = blk.reshape(w.nz, NY // 128, 2).any(axis=2)                 # live 128-y row tiles of stage X
                issued += 24.0 * (grp.sum() * 128.0 * NXP * NPXP + blk.sum() * 64.0 * NPYP * NPXP)
            ach = issued / (k_ms * 1e-3) / 1e12
            roofline = {"bound": "tensor", "kernel": "sep_tc_x2_kernel + sep_tc_yzt_kernel (stage X + stage YZ variants of sep_tensor_kernels.cu)",
                        "achieved": ach, "peak": peaks["burst"], "unit": "TFLOP/s", "frac": ach / peaks["burst"], "traffic": None, "kernel_ms": k_ms,
                        "peak_source": f"MEASURED_PEAKS.json bf16 burst ({peaks['source']}); kind::f16 runs at the bf16 rate",
                        "achieved_is": "issued tensor flop (24 per complex MAC of the live tiles: 8 flop x 3 split products) / "
                                       "CUDA-event time of the per-chunk launches (pack, stage X, stage YZ, finalize)",
                        "issued_fraction_of_dense": issued / (3.0 * dense_sep),
                        "useful_dense_tflops": dense_sep / (k_ms * 1e-3) / 1e12, **tensor_roofline_extras(ach, clocks, peaks)}
    elif args.route in ("nufft", "shapes_nufft"):
        # The route moves 8 B per voxel in and 4 B per pixel out and does ~3e-4 of the pixel route's arithmetic: its speed of light
        # is the HBM time of those bytes.  Algorithmic bytes per launch set = batch x (8 nvox + 4 npix); the GEMM stages' tensor
        # rate (24 issued flop per complex MAC of the dense transform) and the flop count are reported beside it.
        nqx, nqy, nqz = nq
        hbm, hbm_src = load_peaks_hbm()
        abytes = batch * (8.0 * w.nvox + 4.0 * npix_r)
        ach = abytes / (k_ms * 1e-3) / 1e9
        cmacs = batch * (w.nz * w.ny * w.nx * nqx + w.nz * nqx * w.ny * nqy + w.nz * nqx * nqy * nqz)     # stages X, Y, Z as run
        flop = 8.0 * cmacs + 4.0 * batch * npix_r * 10 ** 3
        roofline = {"bound": "hbm", "kernel": "strength + pack + GEMM stages X, Y, Z (tcgen05) + nufft_interp_kernel", "achieved": ach,
                    "peak": hbm, "unit": "GB/s", "frac": ach / hbm, "peak_source": hbm_src,
                    "traffic": NCU_DRAM_BYTES_NUFFT.get(w.name) if batch == 1 else None,
                    "kernel_ms": k_ms, "uniform_grid": [nqz, nqy, nqx],
                    "achieved_is": "algorithmic bytes (8 B per voxel read + 4 B per pixel written) / CUDA-event time of the per-chunk launches "
                                   "(pack, stages X, Y, Z, interpolation); the prefix kernel a2 runs before the events",
                    "gemm_stages_issued_tflops_upper": 24.0 * cmacs / (k_ms * 1e-3) / 1e12,
                    "flop_vs_pixel_route": flop / (FLOP_PER_TERM * terms_per_pattern * batch)}
    elif args.method == 1:
        # what the contraction really issued: it skips all-zero 16-y steps and narrows units to their non-empty x range.
        # One extra, untimed call with the counting flag (same inputs, same schedule).
        step(B.FLAG_COUNT_ISSUED) if args.route == "pixels" else \
            sm.simulate_shapes(shapes, dims, vox, w.lam, w.npx, w.npy, w.theta_max_deg, method=args.method, workspace=ws, out=out,
                               stream=stream, flags=B.FLAG_COUNT_ISSUED)
        blocks = sm.last_issued_blocks()
        npix_pad = (npix_r + 255) // 256 * 256
        issued = blocks * 256 * npix_pad * SPLITS * FLOP_PER_TERM         # tensor flop per contraction launch
        terms_issued_per_pattern = blocks * 256 * npix_pad / batch
        achieved = issued / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "tensor", "kernel": "msft_contract_kernel", "achieved": achieved, "peak": peaks["burst"],
                    "unit": "TFLOP/s", "frac": achieved / peaks["burst"],
                    "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(w.name) if not shard_pixels or world == 1 else None,
                    "peak_source": f"MEASURED_PEAKS.json bf16 burst ({peaks['source']}): the kernel is timed alone by its own CUDA "
                                   "events; kind::f16 runs at the bf16 rate",
                    "achieved_is": "issued tensor flop (24 per issued voxel-pixel term: 8 flop x 3 split products) / kernel time",
                    "issued_fraction_of_dense": issued / dense, "dense_equivalent_tflops": dense / (k_ms * 1e-3) / 1e12,
                    "useful_dense_tflops": dense / SPLITS / (k_ms * 1e-3) / 1e12, "kernel_ms": k_ms,
                    "kernel_share_of_step": k_ms * args.steps / total_ms, **tensor_roofline_extras(achieved, clocks, peaks)}
    elif args.method == 3:
        # FP32 FMA against phase tables: 8 flop per term (dense count; vacuum y chunks are skipped); FP32 peak as for qgrid
        peak = 148 * 128 * 2 * 1.965e9 / 1e12
        ach = FLOP_PER_TERM * w.nvox * npix_r * batch / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "simt_table_kernel", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                    "frac": ach / peak, "traffic": None, "kernel_ms": k_ms}
    else:
        # direct sincos: 2 MUFU per term; SFU peak = 148 SMs x 16 MUFU/clk x max clock
        peak = 148 * 16 * 1.965e9 / 2 / 1e12
        ach = w.nvox * npix_r * batch / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "simt_sincos_kernel", "achieved": ach, "peak": peak, "unit": "Tterm/s",
                    "frac": ach / peak, "traffic": None, "kernel_ms": k_ms}

    cpu = None
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        from paper_2202_03411_b200 import workloads as W
        # size the sample for ~15 s of host-core work from a short probe; pixels of THIS rank's band, in full-detector numbering
        g0, q0 = g[0], (None if quat is None else quat[0])
        if args.route in ("shapes", "shapes_nufft"):     # the oracle's own rendering of item 0 (already in the beam frame)
            from oracle import render as OR
            g0, q0 = OR.render(shapes[0], dims, vox), None
        # two probes separate the per-call set-up (orientation, prefix) from the per-pixel cost
        tp = []
        for n_probe in (16, 80):
            probe = W.sample_pixels(w.seed + 99, w.npix, n_probe)
            t0 = time.perf_counter()
            O.simulate(g0, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=q0, pixels=probe)
            tp.append((len(probe), time.perf_counter() - t0))
        per_pixel = max(1e-9, (tp[1][1] - tp[0][1]) / (tp[1][0] - tp[0][0]))
        setup = max(0.0, tp[0][1] - tp[0][0] * per_pixel)
        npix_s = args.ref_pixels if args.ref_pixels > 0 else int(min(8192, max(256, (15.0 - setup) / per_pixel)))
        pix = W.sample_pixels(w.seed, npix_r, npix_s) + y0 * w.npx
        t0 = time.perf_counter()
        ref = O.simulate(g0, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=q0, pixels=pix)
        dt = time.perf_counter() - t0
        if args.route == "qgrid":
            qg, okg = O.qgrid_q(qx_h, qy_h, w.lam)
            t0 = time.perf_counter()
            ref = O.simulate_q(g0, vox, w.lam, qg[pix], quat=q0) * okg[pix]
            dt = time.perf_counter() - t0
        got = out[0].flatten()[torch.from_numpy(pix - y0 * w.npx).cuda()].cpu().numpy().astype(np.float64)
        rel = float(np.sqrt(np.sum((got - ref) ** 2) / np.sum(ref ** 2)))
        m = ref > 1e-6 * ref.max()
        pixerr = float(np.max(np.abs(got[m] - ref[m]) / ref[m]))
        cpu = {"value": (len(pix) / w.npix) / dt, "unit": "patterns/s", "cores": O.num_threads(), "kind": "oracle",
               "sample": f"{len(pix)} seeded pixels of item 0 of {w.name} ({dt:.1f} s)",
               "terms_per_s": w.nvox * len(pix) / dt, "parity_rel_l2": rel, "parity_max_pixel_rel": pixerr}

    if args.route in ("nufft", "shapes_nufft"):
        dtype, method_name = "fp16x3 split GEMM stages (fp32 accumulate) + f64 interpolation", "nufft"
    elif args.route in ("qgrid", "shapes_qgrid"):
        dtype, method_name = ("f32", "separable_simt") if qmethod == 3 else ("fp16x3 split (fp32 accumulate)", "separable_tensor")
    else:
        dtype = "fp16x3 split (fp32 accumulate)" if args.method == 1 else "f32"
        method_name = {1: "tensor", 2: "simt_sincos", 3: "simt_table"}[args.method]
    parallelism = f"replicas x{world}" if not shard_pixels else f"detector row bands x{world} (rank 0: rows {y0}..{y1 - 1}), pattern gathered on rank 0"
    line = {"metric": "msft_patterns_per_s", "value": value, "unit": "patterns/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if shard_pixels else "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
            "config": {"workload": w.name, "grid": [w.nz, w.ny, w.nx], "detector": [w.npy, w.npx], "batch": batch,
                       "lambda": w.lam, "theta_max_deg": w.theta_max_deg, "route": args.route, "cuda_graph": bool(args.graph),
                       "reuse_tables": bool(args.reuse_tables), "method": method_name, "shard": args.shard,
                       "l2": "flushed between steps (192 MiB write); inputs 134 MB > L2", "parallelism": parallelism},
            # the term rate of the work really multiplied (the contraction skips vacuum); the dense-grid count of north_star beside it
            "terms_per_s": value * (terms_issued_per_pattern if terms_issued_per_pattern else terms_per_pattern),
            "terms_per_s_dense_equivalent": value * terms_per_pattern,
            "terms_counted": "issued (voxel, pixel) terms" if terms_issued_per_pattern else "dense grid (this route does not issue per-term work)",
            "roofline": roofline, "with_table_cache": cached, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "clocks": clocks}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
