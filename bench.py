#!/usr/bin/env python
"""bench.py -- one JSON line for the gridding / degridding hot path on B200.

A "step" is one pass of the whole hot path over one batch of synthetic input:
lra_bin (index + bucket sort) -> lra_grid (tap loop + region flush + sum of weights) -> lra_degrid (model
prediction with the fused residual).  Workload at N = 1: BASELINE.json configs[2], the VLA-like W-projection
configuration the target is quoted on (40,435,200 visibility points x 2 correlations, 8192^2 grid, 128 w-planes,
supports 9..65, oversampling 8).  With N > 1 ranks every rank runs the same-sized shard (weak scaling; payload
seeded per rank) and the per-rank grids are summed with one NCCL all-reduce per step (accumulation of partial
grids).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..5] [--small]

`--gpus N` with N > 1 starts N ranks itself (torch.distributed.run on 127.0.0.1) unless it already runs under
torchrun; the other BASELINE.json configurations are `--config 1`, `2`, `4`, `5` (one line each, same script).
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2508_17187_b200 import workloads as W  # noqa: E402

FP32_PEAK_TFLOPS_NOMINAL = 148 * 128 * 2 * 1.965e9 / 1e12   # 148 SMs x 128 FP32 lanes x 2 flop x 1965 MHz
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_traffic.json")   # written from the ncu capture (profiles/r2_traffic.md)
METRIC = "visibility points per second through bin+grid+degrid"
UNIT = "vis_points/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--small", action="store_true", help="reduced config (debugging only; not a bench value)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--grid-variant", type=int, default=0)
    ap.add_argument("--tile", type=int, default=0, help="uv-tile height (0 = the config's: workloads.full_config)")
    ap.add_argument("--tile-x", type=int, default=0, help="uv-tile width (with --tile)")
    return ap.parse_args()


def source_hash():
    """sha256 over the CUDA sources: ties a stored ncu measurement to the code it was taken on (no .git on the GPU box)."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2508_17187_b200", "csrc", "*.cu*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def stored_traffic(cfg_name):
    """DRAM bytes per lra_grid call from the committed ncu capture, or None when the sources have changed since."""
    try:
        t = json.load(open(TRAFFIC_FILE))
    except Exception:
        return None, "no profiles/r2_traffic.json"
    if t.get("workload") != cfg_name:
        return None, f"profiles/r2_traffic.json is for {t.get('workload')}"
    if t.get("source_hash") != source_hash():
        return None, "profiles/r2_traffic.json was captured on other sources (hash differs): not reported"
    return t, t.get("how", "")


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.stop, self.t = index, [], threading.Event(), None

    def _run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits"],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def make_workload(args, rank):
    cfg = W.small_config(args.config) if args.small else W.full_config(args.config)
    if args.tile:
        cfg = dataclasses.replace(cfg, tile=args.tile, tile_x=args.tile_x or args.tile)
    wl = W.make_workload(cfg, with_payload=False)
    n = cfg.npoints * cfg.ncorr
    # payload seeded per rank (weak scaling: every rank grids its own shard of the same shape)
    wl.vis = W.complex_normal(cfg.cfg_id, 2 + 16 * rank, n).reshape(cfg.nrow, cfg.nchan, cfg.ncorr)
    wl.wt = W.uniform_f32(cfg.cfg_id, 3 + 16 * rank, n, 0.5, 1.0).reshape(cfg.nrow, cfg.nchan, cfg.ncorr)
    return wl


def oracle_sample(wl, args, target_taps=6.0e9, nthreads=0):
    """The oracle as it stands (oracle/lra_ref.c, fp64, OpenMP row bands) on a bounded sample of the workload: every
    k-th time sample (a uniform stride over the whole track, so the sample has the workload's w distribution; all
    baselines, channels, correlations), bin + grid + degrid.  Returns (points/s, seconds, threads, sample description,
    grid taps/s)."""
    from oracle import lra_ref as R
    cfg = wl.cfg
    per_time = max(1, wl.sum_s2() * cfg.ncorr * cfg.nterms // cfg.ntimes)          # grid taps per time sample
    nt = int(max(1, min(cfg.ntimes, target_taps // (2 * per_time))))               # grid + degrid
    if cfg.kind != "disk":
        stride = max(1, cfg.ntimes // nt)
        times = np.arange(0, cfg.ntimes, stride)[:nt]
        rows = (times[:, None] * W.N_BL + np.arange(W.N_BL)[None, :]).ravel()      # rows are time-major, baseline-minor
        what = f"every {stride}-th of {cfg.ntimes} time samples ({len(times)} samples)"
    else:
        rows = np.arange(cfg.nrow)
        what = "all rows"
    uvw, vis, wt = wl.uvw[rows], wl.vis[rows], wl.wt[rows]
    cfi = None if wl.cf_index is None else wl.cf_index[rows]
    plan = R.plan_for(wl, sort_mode=R.SORT_TILE_CF)
    threads = nthreads or R.max_threads()
    t0 = time.perf_counter()
    plan.bin(uvw, wl.freq, cfi)
    t1 = time.perf_counter()
    grid, _ = plan.grid(uvw, wl.freq, cfi, vis, wt, wl.tau, nthreads=threads)
    t2 = time.perf_counter()
    plan.degrid(uvw, wl.freq, cfi, grid, wl.tau, vis_in=vis, nthreads=threads)
    t3 = time.perf_counter()
    npts = len(rows) * cfg.nchan
    taps = (npts * int(wl.cf.support[0]) ** 2 if cfi is None else
            int((np.bincount(cfi.ravel(), minlength=len(wl.cf.support)).astype(np.int64)
                 * wl.cf.support.astype(np.int64) ** 2).sum())) * cfg.ncorr * cfg.nterms
    desc = (f"{what}, {npts} points x {cfg.ncorr} corr: bin {t1 - t0:.2f}s (1 thread) + grid {t2 - t1:.2f}s + degrid "
            f"{t3 - t2:.2f}s, fp64, {threads} OpenMP thread(s) of {os.cpu_count()} hardware threads")
    return npts / (t3 - t0), t3 - t0, threads, desc, taps / (t2 - t1)


def run_reference(args):
    """--impl reference: the oracle timed on the host cores on the same config / metric (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args, 0)
    vals, info = [], None
    for i in range(args.warmup + args.steps):
        v, secs, cores, desc, gt = oracle_sample(wl, args, target_taps=2.0e9)
        if i >= args.warmup:
            vals.append((v, secs))
        info = (cores, desc, gt)
    value = float(np.mean([v for v, _ in vals]))
    ms = float(np.mean([s for _, s in vals]) * 1e3)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": {"workload": wl.cfg.name, "note": "each step is a bounded sample: " + info[1]},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": info[0], "kind": "oracle", "sample": info[1]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2508_17187_b200 import binding as B
    from paper_2508_17187_b200 import sharding

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    B.lib()
    wl = make_workload(args, rank)
    cfg = wl.cfg
    stream = torch.cuda.current_stream()
    plan = B.lra_plan_create(cfg.nx, cfg.ny, cfg.ncorr, cfg.nterms, cfg.oversampling, wl.scale_u, wl.scale_v, wl.cf.support,
                             wl.cf.offset, wl.cf.data, tile=cfg.tile, tile_x=cfg.tile_x, sort_mode=B.LRA_SORT_TILE_CF, device=local,
                             stream=stream.cuda_stream)
    B.lra_set_variant(plan, args.grid_variant, 0)
    # host buffers (pinned) and their device copies
    h_uvw = torch.from_numpy(wl.uvw).pin_memory()
    h_cfi = None if wl.cf_index is None else torch.from_numpy(wl.cf_index).pin_memory()
    h_vis = torch.from_numpy(wl.vis).pin_memory()
    h_wt = torch.from_numpy(wl.wt).pin_memory()
    d_uvw, d_vis, d_wt = h_uvw.cuda(), h_vis.cuda(), h_wt.cuda()
    d_cfi = None if h_cfi is None else h_cfi.cuda()
    d_tau = None if wl.tau is None else torch.from_numpy(wl.tau).cuda()
    grid = torch.zeros((cfg.nterms, cfg.ncorr, cfg.ny, cfg.nx), dtype=torch.complex64, device="cuda")
    sumwt = torch.zeros((cfg.nterms, cfg.ncorr), dtype=torch.float64, device="cuda")
    res = torch.empty_like(d_vis)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    phase_ms = {"bin": [], "grid": [], "degrid": [], "allreduce": []}

    def step(record):
        e = [ev() for _ in range(5)]
        grid.zero_()
        sumwt.zero_()
        e[0].record()
        B.lra_bin(plan, d_uvw, wl.freq, d_cfi)
        e[1].record()
        B.lra_grid(plan, d_vis, d_wt, d_tau, grid, sumwt)
        e[2].record()
        sharding.reduce_grid(grid, sumwt)          # no-op on one GPU; one NCCL all-reduce over NVLink otherwise
        e[3].record()
        B.lra_degrid(plan, grid, d_tau, d_vis, res)
        e[4].record()
        if record:
            phase_ev.append(e)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    phase_ev = []
    for _ in range(args.warmup):
        step(False)
    sync_all()
    l0 = B.lra_launch_count(plan)
    with ClockSampler(local) as clk:
        t_start, t_end = ev(), ev()
        sync_all()
        t_start.record()
        for _ in range(args.steps):
            step(True)
        t_end.record()
        sync_all()
    total_ms = t_start.elapsed_time(t_end)
    launches = B.lra_launch_count(plan) - l0 + args.steps * 2      # + the two zero-fill kernels per step
    for e in phase_ev:
        phase_ms["bin"].append(e[0].elapsed_time(e[1]))
        phase_ms["grid"].append(e[1].elapsed_time(e[2]))
        phase_ms["allreduce"].append(e[2].elapsed_time(e[3]))
        phase_ms["degrid"].append(e[3].elapsed_time(e[4]))
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    n_valid, sum_s2 = B.lra_tap_count(plan)
    ms_per_step = total_ms / args.steps
    value = cfg.npoints * world / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: H2D of the step's inputs + D2H of its results ----
    e2e = None
    if not args.no_e2e:
        # Software-pipelined over the steps, the way a caller streams data through the C ABI: two sets of device inputs and
        # outputs; the H2D copy of step i+1 (copy stream) and the D2H read of step i-1 (read-back stream) run beside the
        # kernels of step i (plan's stream).  Every step still copies all of its inputs in and all of its results out.
        k = max(2, min(args.steps, 8))
        cur = torch.cuda.current_stream()
        s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
        sets = []
        for _ in range(2):
            sets.append({"uvw": torch.empty_like(d_uvw), "cfi": None if d_cfi is None else torch.empty_like(d_cfi),
                         "vis": torch.empty_like(d_vis), "wt": torch.empty_like(d_wt), "grid": torch.empty_like(grid),
                         "sumwt": torch.empty_like(sumwt), "res": torch.empty_like(res),
                         "in_ready": None, "gridded": None, "computed": None, "read_back": None})
        h_grid = torch.empty(grid.shape, dtype=torch.complex64).pin_memory()
        h_res = torch.empty(res.shape, dtype=torch.complex64).pin_memory()
        h_sw = torch.empty(sumwt.shape, dtype=torch.float64).pin_memory()

        def upload(b):
            with torch.cuda.stream(s_in):
                if b["computed"] is not None:
                    s_in.wait_event(b["computed"])          # the previous user of this input set has finished
                b["uvw"].copy_(h_uvw, non_blocking=True)
                if b["cfi"] is not None:
                    b["cfi"].copy_(h_cfi, non_blocking=True)
                b["vis"].copy_(h_vis, non_blocking=True)
                b["wt"].copy_(h_wt, non_blocking=True)
                b["in_ready"] = s_in.record_event()

        def compute(b):
            cur.wait_event(b["in_ready"])
            if b["read_back"] is not None:
                cur.wait_event(b["read_back"])              # its outputs of two steps ago have been read
            b["grid"].zero_()
            b["sumwt"].zero_()
            B.lra_bin(plan, b["uvw"], wl.freq, b["cfi"])
            B.lra_grid(plan, b["vis"], b["wt"], d_tau, b["grid"], b["sumwt"])
            sharding.reduce_grid(b["grid"], b["sumwt"])
            b["gridded"] = cur.record_event()
            B.lra_degrid(plan, b["grid"], d_tau, b["vis"], b["res"])
            b["computed"] = cur.record_event()

        def read_back(b):
            with torch.cuda.stream(s_out):
                s_out.wait_event(b["gridded"])              # the grid is final once it is reduced: its read-back runs
                h_grid.copy_(b["grid"], non_blocking=True)  # beside the degridder, which only reads it
                h_sw.copy_(b["sumwt"], non_blocking=True)
                s_out.wait_event(b["computed"])
                h_res.copy_(b["res"], non_blocking=True)
                b["read_back"] = s_out.record_event()

        def e2e_run(nsteps):
            upload(sets[0])
            for i in range(nsteps):
                if i + 1 < nsteps:
                    upload(sets[(i + 1) % 2])
                compute(sets[i % 2])
                read_back(sets[i % 2])

        e2e_run(2)
        sync_all()
        for b in sets:
            b["in_ready"] = b["gridded"] = b["computed"] = b["read_back"] = None
        t0 = time.perf_counter()
        e2e_run(k)
        sync_all()
        e_ms = (time.perf_counter() - t0) * 1e3 / k         # wall clock around k pipelined steps, all streams drained
        if world > 1:
            t = torch.tensor([e_ms], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            e_ms = float(t.item())
        h2d = h_uvw.numel() * 8 + (0 if h_cfi is None else h_cfi.numel() * 4) + h_vis.numel() * 8 + h_wt.numel() * 4
        d2h = h_grid.numel() * 8 + h_res.numel() * 8 + h_sw.numel() * 8
        e2e = {"value": cfg.npoints * world / (e_ms * 1e-3), "unit": UNIT, "ms_per_step": e_ms, "steps": k,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "how": "k steps software-pipelined over two buffer sets: H2D of step i+1 and D2H of step i-1 overlap the kernels "
                      "of step i, the grid's D2H starts when it is reduced (beside the degridder); wall clock around the k "
                      "steps with every stream drained"}

    if rank == 0:
        peaks = measured_peaks()
        med = {k: float(np.median(v)) if v else 0.0 for k, v in phase_ms.items()}
        ngrids = cfg.ncorr * cfg.nterms
        grid_taps = sum_s2 * ngrids
        grid_flops = grid_taps * 8.0
        achieved = grid_flops / (med["grid"] * 1e-3) / 1e12
        try:
            fma_peak = B.lra_diag_fma_tflops(local)       # FMA-only microbenchmark on this GPU, outside the timed region
            peak_src = ("measured on this GPU by lra_diag_fma_tflops (FP32 FMA-only kernel); nominal 148 SM x 128 lanes x 2 x "
                        "1965 MHz = %.2f; MEASURED_PEAKS.json has no FP32 entry" % FP32_PEAK_TFLOPS_NOMINAL)
        except Exception:
            fma_peak, peak_src = FP32_PEAK_TFLOPS_NOMINAL, "derived: 148 SM x 128 FP32 lanes x 2 flop x 1965 MHz"
        traffic, traffic_src = (None, "not the default launch configuration") if (args.small or args.tile) else stored_traffic(cfg.name)
        roofline = {"bound": "alu", "kernel": "lra_grid_region_kernel (all per-support-class launches of one lra_grid call, "
                                              "CUDA events on the plan's stream around the call)",
                    "achieved": achieved, "peak": fma_peak, "unit": "TFLOP/s", "frac": achieved / fma_peak,
                    "peak_source": peak_src,
                    "traffic": None if not traffic else traffic.get("region_kernels_dram_bytes"),
                    "traffic_call": None if not traffic else traffic.get("lra_grid_call_dram_bytes"),
                    "traffic_source": traffic_src, "algorithmic_bytes": 2.37e9 if cfg.cfg_id == 3 and not args.small else None,
                    "tap_updates_per_launch": grid_taps, "tap_updates_per_s": grid_taps / (med["grid"] * 1e-3),
                    "degrid_frac": (grid_flops / (med["degrid"] * 1e-3) / 1e12 / fma_peak) if med["degrid"] else None,
                    "degrid_tap_updates_per_s": grid_taps / (med["degrid"] * 1e-3) if med["degrid"] else None,
                    "hbm_gbs_measured_peak": None if not peaks else peaks.get("hbm_gbs")}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic",
                "config": {"workload": cfg.name, "points": cfg.npoints, "ncorr": cfg.ncorr, "nterms": cfg.nterms,
                           "grid": [cfg.ny, cfg.nx], "n_cf": cfg.n_cf, "oversampling": cfg.oversampling, "tile_u_x_v": [cfg.tile_x, cfg.tile], "n_valid": n_valid,
                           "sum_S2": sum_s2, "l2": "inputs larger than L2 (vis+wt 0.97 GB, grid 1.07 GB per step)",
                           "parallelism": f"dp{world}" if world > 1 else "single"},
                "phase_ms_median": med, "grid_vis_points_per_s": n_valid / (med["grid"] * 1e-3),
                "roofline": roofline, "clocks": clk.summary(), "gpu_launches": int(launches)}
        if e2e:
            line["e2e"] = e2e
        if not args.no_cpu_baseline and world == 1:
            v, secs, cores, desc, gt = oracle_sample(wl, args)
            v1, secs1, _, desc1, gt1 = oracle_sample(wl, args, target_taps=4.0e8, nthreads=1)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                                    "grid_tap_updates_per_s": gt, "hardware_threads": os.cpu_count(),
                                    "single_thread": {"value": v1, "unit": UNIT, "cores": 1, "sample": desc1,
                                                      "grid_tap_updates_per_s": gt1}}
        print(json.dumps(line))
    B.lra_plan_destroy(plan)
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` outside torchrun: start the N ranks ourselves (one process per GPU, NCCL over
    NVLink), exactly as the driver's torchrun line would; NCCL's own init lines stay on stderr."""
    import socket
    import torch
    have = torch.cuda.device_count()
    if have < args.gpus:
        raise SystemExit(f"bench.py --gpus {args.gpus}: only {have} CUDA device(s) visible")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    elif a.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(a)
    else:
        run_ours(a)
