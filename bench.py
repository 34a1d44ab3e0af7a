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
# (profiles/r01_contract_cfg3_full.md); only the workload that was captured has a number
NCU_DRAM_BYTES_PER_LAUNCH = {"cfg3_droplet_256": 2.295495e9 + 8.534016e6}
# the same for the four launches of one NUFFT pattern (stages Z, X, Y, interpolation; profiles/r01_nufft.md)
NCU_DRAM_BYTES_NUFFT = {"cfg3_droplet_256": (134.46 + 24.46 + 46.63 + 0.91 + 20.85 + 0.0 + 8.27 + 0.0) * 1e6}


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
    else:   # ~10 s per step from a short probe
        probe = W.sample_pixels(w.seed + 99, w.npix, 32)
        t0 = time.perf_counter()
        O.simulate(g, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, pixels=probe)
        npix_s = int(min(8192, max(128, 10.0 / ((time.perf_counter() - t0) / len(probe)))))
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
                    help="--route nufft only: capture one call in a CUDA graph after the warm-up and time its replays")
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

    w, items = workload_for(args)
    vox = (w.dx, w.dy, w.dz)
    # weak scaling: the global job is `world` copies of the batch; shapes shard across ranks with no collective
    from paper_2202_03411_b200.sharding import shard_range
    global_items = [i for _ in range(world) for i in items]
    lo, hi = shard_range(len(global_items), rank, world)
    items = global_items[lo:hi]
    g = w.grids(items)
    quat = None if w.quat is None else w.quat[items]
    batch = len(items)
    d_dn = torch.from_numpy(g).cuda()
    grid = B.Grid(w.nx, w.ny, w.nz, *vox)
    opts = B.Options(0, args.method, 0, 0)
    ws = torch.empty(sm.workspace_bytes(grid, w.npix, batch, opts), dtype=torch.uint8, device="cuda")
    out = torch.empty((batch, w.npy, w.npx), dtype=torch.float32, device="cuda")
    flush = torch.empty(192 * 1024 * 1024, dtype=torch.uint8, device="cuda")   # > 126 MB L2
    stream = torch.cuda.current_stream()

    qmethod = args.method if args.method in (0, 1, 3) else 0
    if args.route in ("qgrid", "shapes_qgrid"):
        kk = 2 * np.pi / w.lam
        qx = torch.from_numpy((np.arange(w.npx) + 0.5 - 0.5 * w.npx) * (2 * kk * np.sin(np.radians(w.theta_max_deg)) / w.npx)).cuda()
        qy = torch.from_numpy((np.arange(w.npy) + 0.5 - 0.5 * w.npy) * (2 * kk * np.sin(np.radians(w.theta_max_deg)) / w.npy)).cuda()
        need = C.c_size_t(0)
        qmethod = args.method if args.method in (0, 1, 3) else 0
        qopts = B.Options(0, qmethod, 0, 0)
        sm._check(sm.lib.scatman_qgrid_workspace_bytes(sm._ctx, C.byref(grid), w.npx, w.npy, batch, C.byref(qopts), C.byref(need)))
        ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")

    nq = None
    if args.route in ("nufft", "shapes_nufft"):      # same flat detector, same result: 3-D type-2 NUFFT instead of the pixel x voxel contraction
        det = B.Detector(w.npx, w.npy, w.theta_max_deg, 0.0, 0.0)
        need = C.c_size_t(0)
        sm._check(sm.lib.scatman_nufft_workspace_bytes(sm._ctx, C.byref(grid), w.lam, C.byref(det), batch, C.byref(need)))
        ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")
        nq = sm.nufft_grid_dims(grid, w.lam, det)

    shapes = None
    if args.route == "shapes_qgrid":
        shapes = w.shapes(items)
        if shapes is None:
            raise SystemExit(f"{w.name} is not one shape per item: --route shapes_qgrid does not apply")
        need = C.c_size_t(0)
        sm._check(sm.lib.scatman_shapes_qgrid_workspace_bytes(sm._ctx, C.byref(grid), w.npx, w.npy, batch, C.byref(qopts), C.byref(need)))
        ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")
    if args.route == "shapes_nufft":
        shapes = w.shapes(items)
        if shapes is None:
            raise SystemExit(f"{w.name} is not one shape per item: --route shapes_nufft does not apply")
        need = C.c_size_t(0)
        sm._check(sm.lib.scatman_shapes_nufft_workspace_bytes(sm._ctx, C.byref(grid), w.lam, C.byref(det), batch, C.byref(need)))
        ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")
    if args.route == "shapes":
        shapes = w.shapes(items)
        if shapes is None:
            raise SystemExit(f"{w.name} is not one shape per item: --route shapes does not apply")
        need = C.c_size_t(0)
        sm._check(sm.lib.scatman_shapes_workspace_bytes(sm._ctx, C.byref(grid), w.npix, batch, C.byref(opts), C.byref(need)))
        ws = torch.empty(int(need.value), dtype=torch.uint8, device="cuda")

    def step():
        if args.route == "shapes":
            sm.simulate_shapes(shapes, (w.nx, w.ny, w.nz), vox, w.lam, w.npx, w.npy, w.theta_max_deg, method=args.method,
                               workspace=ws, out=out, stream=stream)
            return
        if args.route == "shapes_qgrid":
            sm.simulate_shapes_qgrid(shapes, (w.nx, w.ny, w.nz), vox, w.lam, qx, qy, method=qmethod, workspace=ws, out=out,
                                     stream=stream)
            return
        if args.route == "qgrid":
            sm.simulate_qgrid(d_dn, vox, w.lam, qx, qy, quat=quat, method=qmethod, workspace=ws, out=out, stream=stream)
            return
        if args.route == "shapes_nufft":
            sm.simulate_shapes_nufft(shapes, (w.nx, w.ny, w.nz), vox, w.lam, w.npx, w.npy, w.theta_max_deg, workspace=ws, out=out,
                                     stream=stream)
            return
        if args.route == "nufft":
            sm.simulate_nufft(d_dn, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, workspace=ws, out=out, stream=stream)
            return
        sm.simulate(d_dn, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, method=args.method,
                    workspace=ws, out=out, stream=stream)

    for _ in range(args.warmup):
        flush.zero_()
        step()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kernel_ms, launches = [], 0
    torch.cuda.synchronize()
    graph = None
    if args.graph:
        if args.route != "nufft":
            raise SystemExit("--graph applies to --route nufft")
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):      # the call only enqueues on the capturing stream: the whole step becomes one graph
            sm.simulate_nufft(d_dn, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, workspace=ws, out=out)
        graph_launches = sm.last_launch_count()
        graph.replay()
        torch.cuda.synchronize()
    for i in range(args.steps):
        flush.zero_()                      # L2 flush, outside the timed events
        ev[i][0].record(stream)
        if graph is not None:
            graph.replay()
            ev[i][1].record(stream)
            launches += graph_launches
            continue
        step()
        ev[i][1].record(stream)
        launches += sm.last_launch_count()
        kernel_ms.append(sm.last_contraction_ms())   # events on the launch stream; waits for this step
    torch.cuda.synchronize()
    total_ms = sum(a.elapsed_time(b) for a, b in ev)
    if dist:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None

    # end to end through the host-buffer C entry point: pinned host grid in, pinned host intensity out
    h_dn = torch.from_numpy(g).pin_memory()
    h_I = torch.empty((batch, w.npy, w.npx), dtype=torch.float32).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))

    def e2e_step():
        if args.route in ("shapes", "shapes_qgrid", "shapes_nufft"):  # the inputs are the descriptors (host structs, marshalled per call); results to pinned host
            step()
            h_I.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        elif args.route in ("qgrid", "nufft"):   # no host-buffer C entry point for this route: the copies go through torch
            d_dn.copy_(h_dn, non_blocking=True)
            step()
            h_I.copy_(out, non_blocking=True)
            torch.cuda.synchronize()
        else:
            sm.simulate_host(h_dn, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, method=args.method, h_out=h_I)

    e2e_step()
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

    patterns = batch * args.steps * world
    value = patterns / (total_ms * 1e-3)
    terms_per_pattern = w.nvox * w.npix
    peaks = load_peaks()
    # graph replays have no per-kernel events: the roofline then takes the WHOLE step (a1, a2 and tables included) as the kernel time
    k_ms = sum(kernel_ms) / len(kernel_ms) if kernel_ms else total_ms / args.steps
    dense = SPLITS * FLOP_PER_TERM * terms_per_pattern * batch           # tensor flop of the dense sum per launch
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
            peak = peaks["sustained"]
            ach = issued / (k_ms * 1e-3) / 1e12
            roofline = {"bound": "tensor", "kernel": "sep_tc_x2_kernel + sep_tc_yzt_kernel (stage X + stage YZ variants of sep_tensor_kernels.cu)", "achieved": ach, "peak": peak,
                        "unit": "TFLOP/s", "frac": ach / peak, "traffic": None, "kernel_ms": k_ms,
                        "peak_source": f"MEASURED_PEAKS.json bf16 sustained ({peaks['source']}); kind::f16 runs at the bf16 rate",
                        "achieved_is": "issued tensor flop (24 per complex MAC of the live tiles: 8 flop x 3 split products) / "
                                       "CUDA-event time of the per-item launches (pack, stage X, stage YZ, finalize)",
                        "issued_fraction_of_dense": issued / (3.0 * dense_sep),
                        "useful_dense_tflops": dense_sep / (k_ms * 1e-3) / 1e12}
    elif args.route in ("nufft", "shapes_nufft"):
        # three FP64 complex GEMMs (slices -> g_z planes, columns -> g_x, rows -> g_y) + the 10^3-point interpolation, CUDA cores:
        # 8 flop per complex MAC of the GEMMs, 4 per (real weight x complex value) MAC of the interpolation.
        nqx, nqy, nqz = nq
        flop = batch * (8.0 * (nqz * w.nz * w.ny * w.nx + nqz * w.ny * w.nx * nqx + nqz * nqy * w.ny * nqx) + 4.0 * w.npix * 10 ** 3)
        peak = 148 * 64 * 2 * 1.965e9 / 1e12           # FP64 FMA: 148 SMs x 64 lanes x 2 flop x max clock
        ach = flop / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "nufft_zgemm_kernel (stages Z, X, Y) + nufft_interp_kernel", "achieved": ach, "peak": peak,
                    "unit": "TFLOP/s", "frac": ach / peak, "traffic": NCU_DRAM_BYTES_NUFFT.get(w.name) if batch == 1 else None,
                    "kernel_ms": k_ms, "uniform_grid": [nqz, nqy, nqx],
                    "achieved_is": "dense FP64 flop of the three GEMM stages and the interpolation / their CUDA-event time; K steps over "
                                   "vacuum are skipped, so the ALUs executed less than this (ncu: FP64 pipe 50-59 % active in the GEMMs)",
                    "flop_vs_pixel_route": flop / (FLOP_PER_TERM * terms_per_pattern * batch)}
    elif args.method == 1:
        # what the contraction really issued: it skips all-zero 16-y steps and narrows units to their non-empty x range.
        # One extra, untimed call with the counting flag (same inputs, same schedule).
        if args.route == "shapes":
            sm.simulate_shapes(shapes, (w.nx, w.ny, w.nz), vox, w.lam, w.npx, w.npy, w.theta_max_deg, method=args.method,
                               workspace=ws, out=out, stream=stream, flags=B.FLAG_COUNT_ISSUED)
        else:
            sm.simulate(d_dn, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=quat, method=args.method, workspace=ws, out=out,
                        stream=stream, flags=B.FLAG_COUNT_ISSUED)
        blocks = sm.last_issued_blocks()
        npix_pad = (w.npix + 255) // 256 * 256
        issued = blocks * 256 * npix_pad * SPLITS * FLOP_PER_TERM         # tensor flop per contraction launch
        achieved = issued / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "tensor", "kernel": "msft_contract_kernel", "achieved": achieved, "peak": peaks["sustained"],
                    "unit": "TFLOP/s", "frac": achieved / peaks["sustained"],
                    "traffic": NCU_DRAM_BYTES_PER_LAUNCH.get(w.name),
                    "peak_source": f"MEASURED_PEAKS.json bf16 sustained ({peaks['source']}); kind::f16 runs at the bf16 rate",
                    "achieved_is": "issued tensor flop (24 per issued voxel-pixel term: 8 flop x 3 split products) / kernel time",
                    "issued_fraction_of_dense": issued / dense, "dense_equivalent_tflops": dense / (k_ms * 1e-3) / 1e12,
                    "useful_dense_tflops": dense / SPLITS / (k_ms * 1e-3) / 1e12, "kernel_ms": k_ms,
                    "kernel_share_of_step": k_ms * args.steps / total_ms,
                    # context: the measured cuBLAS peak is power-limited (SM clock ~1.3 GHz under its load); this kernel skips
                    # vacuum, draws less power and holds the full clock, hence frac > 1.  Nominal dense FP16/BF16 is 2250 TFLOP/s.
                    "peak_nominal": 2250.0, "frac_of_nominal": achieved / 2250.0, "peak_burst": peaks["burst"]}
    elif args.method == 3:
        # FP32 FMA against phase tables: 8 flop per term (dense count; vacuum y chunks are skipped); FP32 peak as for qgrid
        peak = 148 * 128 * 2 * 1.965e9 / 1e12
        ach = FLOP_PER_TERM * terms_per_pattern * batch / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "simt_table_kernel", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                    "frac": ach / peak, "traffic": None, "kernel_ms": k_ms}
    else:
        # direct sincos: 2 MUFU per term; SFU peak = 148 SMs x 16 MUFU/clk x max clock
        peak = 148 * 16 * 1.965e9 / 2 / 1e12
        ach = terms_per_pattern * batch / (k_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "simt_sincos_kernel", "achieved": ach, "peak": peak, "unit": "Tterm/s",
                    "frac": ach / peak, "traffic": None, "kernel_ms": k_ms}

    cpu = None
    if not args.no_cpu_baseline:
        from oracle import oracle as O
        from paper_2202_03411_b200 import workloads as W
        # size the sample for ~15 s of host-core work from a short probe
        g0, q0 = g[0], (None if quat is None else quat[0])
        if args.route in ("shapes", "shapes_nufft"):     # the oracle's own rendering of item 0 (already in the beam frame)
            from oracle import render as OR
            g0, q0 = OR.render(shapes[0], (w.nx, w.ny, w.nz), vox), None
        probe = W.sample_pixels(w.seed + 99, w.npix, 32)
        t0 = time.perf_counter()
        O.simulate(g0, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=q0, pixels=probe)
        per_pixel = (time.perf_counter() - t0) / len(probe)
        npix_s = args.ref_pixels if args.ref_pixels > 0 else int(min(8192, max(256, 15.0 / per_pixel)))
        pix = W.sample_pixels(w.seed, w.npix, npix_s)
        t0 = time.perf_counter()
        ref = O.simulate(g0, vox, w.lam, w.npx, w.npy, w.theta_max_deg, quat=q0, pixels=pix)
        dt = time.perf_counter() - t0
        if args.route == "qgrid":
            qg, okg = O.qgrid_q(qx.cpu().numpy(), qy.cpu().numpy(), w.lam)
            t0 = time.perf_counter()
            ref = O.simulate_q(g0, vox, w.lam, qg[pix], quat=q0) * okg[pix]
            dt = time.perf_counter() - t0
        got = out[0].flatten()[torch.from_numpy(pix).cuda()].cpu().numpy().astype(np.float64)
        rel = float(np.sqrt(np.sum((got - ref) ** 2) / np.sum(ref ** 2)))
        m = ref > 1e-6 * ref.max()
        pixerr = float(np.max(np.abs(got[m] - ref[m]) / ref[m]))
        cpu = {"value": (len(pix) / w.npix) / dt, "unit": "patterns/s", "cores": O.num_threads(), "kind": "oracle",
               "sample": f"{len(pix)} seeded pixels of item 0 of {w.name} ({dt:.1f} s)",
               "terms_per_s": w.nvox * len(pix) / dt, "parity_rel_l2": rel, "parity_max_pixel_rel": pixerr}

    line = {"metric": "msft_patterns_per_s", "value": value, "unit": "patterns/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64" if args.route in ("nufft", "shapes_nufft") else "f32" if (args.route in ("qgrid", "shapes_qgrid") and qmethod == 3) or (args.route not in ("qgrid", "shapes_qgrid") and args.method != 1) else "fp16x3 split (fp32 accumulate)", "data": "synthetic",
            "config": {"workload": w.name, "grid": [w.nz, w.ny, w.nx], "detector": [w.npy, w.npx], "batch": batch,
                       "lambda": w.lam, "theta_max_deg": w.theta_max_deg, "route": args.route, "cuda_graph": bool(args.graph), "method": ("separable_simt" if qmethod == 3 else "separable_tensor") if args.route in ("qgrid", "shapes_qgrid") else "nufft_fp64" if args.route in ("nufft", "shapes_nufft") else {1: "tensor", 2: "simt_sincos", 3: "simt_table"}[args.method],
                       "l2": "flushed between steps (192 MiB write); inputs 134 MB > L2", "parallelism": f"replicas x{world}"},
            "terms_per_s": value * terms_per_pattern, "roofline": roofline, "cpu_baseline": cpu,
            "e2e": {"value": batch * e2e_steps * world / e2e_s, "unit": "patterns/s",
                    "h2d_bytes_per_step": int(h_dn.numel() * 4) if args.route not in ("shapes", "shapes_qgrid", "shapes_nufft") else int(C.sizeof(B.Shape) * batch + sum(24 * len(sh.get("coeffs", ())) for sh in shapes)),
                    "d2h_bytes_per_step": int(h_I.numel() * 4)},
            "gpu_launches": launches, "clocks": clocks}
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
