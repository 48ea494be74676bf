#!/usr/bin/env python
"""bench.py -- FPN RoIAlign fwd+bwd throughput on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (level assignment + forward gather + backward scatter,
incl. zero-fill) over one synthetic batch of BASELINE.json configs[1] (Faster R-CNN R-50-FPN box
head, training: batch 2, 4 levels, C=256 fp32, 1024 RoIs, 7x7, sampling_ratio 2), through the C ABI.

  python bench.py --gpus N --steps K --warmup W            our arm (one rank per GPU; no collective:
                                                           the path shards by image -> weak scaling)
  python bench.py --impl reference ...                     the CPU oracle on the host cores

Prints ONE JSON line (rank 0).  See DESIGN.md section 6 for every field.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "RoIAlign fwd+bwd RoIs/sec (C=256, 7x7, FPN)"
UNIT = "RoIs/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (1-based)")
    ap.add_argument("--layout", default="cl", choices=["cl", "nchw"])
    ap.add_argument("--backward", default="auto", choices=["auto", "atomic", "deterministic", "strip", "tile"],
                    help="auto: library's choice (a pull kernel when eligible); atomic: RAF_ATOMIC; deterministic: RAF_DETERMINISTIC; "
                         "strip / tile: force one of the two pull kernels (RAF_PULL_STRIP / RAF_PULL_TILE)")
    ap.add_argument("--grad-dtype", default="f32", choices=["f32", "same"],
                    help="gradient pyramid dtype: fp32 (readings S13) or the 16-bit dtype of grad_out (roi_align_fpn_backward_ex)")
    ap.add_argument("--repack", action="store_true",
                    help="with --layout nchw: RAF_REPACK (the library repacks to channels-last inside the workspace, counted in the time)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--graph", action="store_true", help="replay each step from a CUDA graph")
    ap.add_argument("--rotate", type=int, default=0,
                    help="number of independent input/output buffer sets to rotate over (0 = cold-L2 protocol: "
                         "at least 4 and >= 2x L2; 1 = WARM single-buffer number, not the headline)")
    ap.add_argument("--op", default="align", choices=["align", "pool", "deform", "fc", "nms", "softnms"],
                    help="align: the headline FPN RoIAlign fwd+bwd (BASELINE.json metric); pool / nms / softnms: the SURVEY 8(f) "
                         "operations, one extra bench line each (not the headline)")
    ap.add_argument("--nms-n", type=int, default=2000, help="boxes for --op nms / softnms")
    ap.add_argument("--windows", type=int, default=5, help="timing windows per loop (median and min are reported)")
    ap.add_argument("--window-iters", type=int, default=200, help="back-to-back iterations per timing window")
    ap.add_argument("--sampling-ratio", type=int, default=None, help="override the config's sampling_ratio (0 = adaptive)")
    ap.add_argument("--aligned", type=int, default=None, help="override the config's aligned flag (0 / 1)")
    ap.add_argument("--roi-order", choices=["given", "level"], default="given",
                    help="given: the workload's RoI order (the headline); level: the same RoIs permuted into per-level order "
                         "(finest level first, the stable permutation roi_fpn_assign_levels returns) before the timed "
                         "region -- what a caller that extracts level by level passes; not the headline")
    ap.add_argument("--no-reuse-prep", action="store_true",
                    help="backward rebuilds its RoI buckets / tap tables instead of reusing the forward's (RAF_REUSE_PREP)")
    return ap.parse_args()


def peaks():
    """Measured peak (driver-written MEASURED_PEAKS.json) or the profiling guide's fallback."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "25",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


class OracleLeg:
    """The oracle as it stands, timed on the host cores on a bounded sample of the workload: all
    channels, the first `n` RoIs of each image of the config (fwd, + bwd when the config has one).
    `n` is chosen from a short probe so that one pass takes at most about `budget_s` seconds."""

    def __init__(self, cfg_index):
        from oracle import raf_ref as R
        from paper_1906_07155_b200 import inputs
        self.R, self.index = R, cfg_index
        self.cfg = cfg = inputs.CONFIGS[cfg_index]
        self.wl = inputs.make_workload(cfg_index)
        self.feats64 = [f.astype(np.float64) for f in self.wl.feats]
        self.gout64 = self.wl.grad_out.astype(np.float64)
        self.sel = self._pick(cfg.per_img)

    def _pick(self, n_per_img):
        c = self.cfg
        return np.concatenate([np.arange(i * c.per_img, i * c.per_img + n_per_img) for i in range(c.n_img)])

    def run(self, sel=None):
        c, R = self.cfg, self.R
        sel = self.sel if sel is None else sel
        t0 = time.perf_counter()
        R.forward(self.feats64, c.scales, self.wl.rois[sel], c.out_size, c.sampling_ratio, c.aligned, c.finest_scale)
        if c.backward:
            R.backward(c.level_shapes, c.scales, self.gout64[sel], self.wl.rois[sel], c.out_size,
                       c.sampling_ratio, c.aligned, c.finest_scale, want_abs_sum=False)
        return time.perf_counter() - t0

    def calibrate(self, budget_s):
        c = self.cfg
        probe_n = min(8, c.per_img)
        t_probe = self.run(self._pick(probe_n))
        t_fixed = self.run(self._pick(1))     # zero-fill of the double pyramid etc.
        per_roi = max((t_probe - t_fixed) / max(c.n_img * (probe_n - 1), 1), 1e-7)
        n = int(min(c.per_img, max(1, (budget_s - t_fixed) / per_roi / c.n_img)))
        self.sel = self._pick(n)
        return n

    def describe(self, t, value):
        c = self.cfg
        n = len(self.sel) // c.n_img
        return {"value": value, "unit": UNIT, "cores": self.R.num_threads(), "kind": "oracle",
                "sample": f"config {self.index}: first {n} RoIs of each of {c.n_img} images ({len(self.sel)} of {c.K} "
                          f"RoIs), all {c.channels} channels, fwd{'+bwd' if c.backward else ''}, spec mode, OpenMP; "
                          f"{t:.2f} s per pass"}


def cpu_baseline(cfg_index, budget_s=14.0):
    """The oracle on the host cores: all cores (OpenMP) on a bounded sample, then ONE thread on a smaller
    sample (both sized from a probe so that the two legs together take about 20-25 s)."""
    leg = OracleLeg(cfg_index)
    leg.calibrate(budget_s)
    t = min(leg.run() for _ in range(3 if budget_s < 5 else 1))
    d = leg.describe(t, len(leg.sel) / t)
    d["cpu_model"] = cpu_model()
    try:   # the oracle is not touched: the OpenMP runtime it links is told to use one thread
        import ctypes
        gomp = ctypes.CDLL("libgomp.so.1")
        cores = leg.R.num_threads()
        gomp.omp_set_num_threads(1)
        leg.calibrate(8.0)
        t1 = leg.run()
        d["single_thread"] = {"value": len(leg.sel) / t1, "unit": UNIT, "cores": leg.R.num_threads(),
                              "sample": f"first {len(leg.sel) // leg.cfg.n_img} RoIs of each image, {t1:.2f} s per pass"}
        gomp.omp_set_num_threads(cores)
    except Exception as e:
        d["single_thread"] = {"unavailable": str(e)}
    return d


def run_reference(args):
    """--impl reference: the oracle (kind 'oracle') on the host cores; rank 0 only.  Each step is one
    oracle pass over a bounded RoI sample sized so that steps+warmup end within about 150 s."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import build as ref_build
    ref_build.build()
    leg = OracleLeg(args.config)
    cfg = leg.cfg
    steps, warm = max(1, args.steps), max(0, args.warmup)
    leg.calibrate(150.0 / (steps + warm))
    for _ in range(warm):
        leg.run()
    times = [leg.run() for _ in range(steps)]
    t = sum(times) / len(times)
    value = len(leg.sel) / t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warm, "ms_per_step": 1e3 * t,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": f"BASELINE.json configs[{args.config - 1}]: {cfg.name}",
                                            "note": "each step = the oracle on a bounded RoI sample of the workload"},
            "cpu_baseline": leg.describe(t, value),
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def source_hash():
    """sha256 over the CUDA sources and the ABI header: identifies the build a profile was taken on."""
    import hashlib
    h = hashlib.sha256()
    csrc = os.path.join(ROOT, "paper_1906_07155_b200", "csrc")
    for f in sorted(os.listdir(csrc)) + [os.path.join("..", "..", "include", "raf.h")]:
        with open(os.path.join(csrc, f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def ncu_traffic(config, variant):
    """DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum) from profiles/traffic.json, which
    bench_traffic.py writes from an `ncu --set full` report.  Only returned when it was measured on THIS build."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        t = json.load(open(p))
    except Exception:
        return {}, True
    stale = t.get("source_hash") != source_hash()
    entry = t.get("configs", {}).get(f"{config}:{variant}", {})
    return ({} if stale else entry), stale


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def run_ours(args):
    import torch
    import torch.distributed as dist
    import bench_roofline as roofline
    from paper_1906_07155_b200 import binding as B
    from paper_1906_07155_b200 import build as raf_build
    from paper_1906_07155_b200 import inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py (our arm) needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        raf_build.build()
    if world > 1:
        dist.barrier()
    B.lib()

    cfg = inputs.CONFIGS[args.config]
    wl = inputs.make_workload(args.config)
    tdt = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[cfg.dtype]
    esz = 4 if cfg.dtype == "f32" else 2
    K, C, L = cfg.K, cfg.channels, len(cfg.level_shapes)
    PH, PW = cfg.out_size
    g, aligned, fs = cfg.sampling_ratio, cfg.aligned, cfg.finest_scale
    if args.roi_order == "level":   # permute the RoIs (and their grad_out rows) with the library's own stable per-level permutation
        d_rois = torch.from_numpy(wl.rois).cuda()
        d_perm = torch.empty((K,), dtype=torch.int32, device="cuda")
        B.roi_fpn_assign_levels(d_rois, L, fs, None, None, d_perm)
        torch.cuda.synchronize()
        perm = d_perm.cpu().numpy().astype(np.int64)
        wl.rois = np.ascontiguousarray(wl.rois[perm])
        if wl.grad_out is not None:
            wl.grad_out = np.ascontiguousarray(wl.grad_out[perm])
    if args.sampling_ratio is not None:
        g = args.sampling_ratio
    if args.aligned is not None:
        aligned = bool(args.aligned)
    flags = {"auto": 0, "atomic": B.RAF_ATOMIC, "deterministic": B.RAF_DETERMINISTIC, "strip": B.RAF_PULL_STRIP,
             "tile": B.RAF_PULL_TILE}[args.backward]
    reuse = cfg.backward and not args.no_reuse_prep and args.backward != "atomic"
    if reuse:
        flags |= B.RAF_REUSE_PREP   # a step runs the forward first, on the same RoIs and workspace: its launch
                                    # already wrote the backward's RoI buckets / tap tables (include/raf.h)
    fwd_flags = 0 if cfg.backward else B.RAF_NO_PREP   # forward-only workloads do not build the backward's tables

    def lay(t):   # logical NCHW tensor -> requested physical layout
        return t.contiguous() if args.layout == "nchw" else t.permute(0, 2, 3, 1).contiguous().permute(0, 3, 1, 2)

    pyr_bytes = sum(int(np.prod(s)) for s in cfg.level_shapes)
    ws_set = pyr_bytes * esz + pyr_bytes * 4 * cfg.backward + K * C * PH * PW * esz * (1 + cfg.backward)
    l2 = torch.cuda.get_device_properties(local_rank).L2_cache_size
    R = int(max(4, -(-2 * l2 // ws_set))) if args.rotate <= 0 else args.rotate
    base_feats = [torch.from_numpy(f).to(tdt) for f in wl.feats]
    feats = [[lay(f.cuda()) for f in base_feats] for _ in range(R)]
    rois = torch.from_numpy(wl.rois).cuda()
    outs = [lay(torch.empty((K, C, PH, PW), dtype=tdt, device="cuda")) for _ in range(R)]
    gouts = [lay(torch.from_numpy(wl.grad_out).to(tdt).cuda()) for _ in range(R)] if cfg.backward else None
    gdt = tdt if (args.grad_dtype == "same" and cfg.dtype != "f32") else torch.float32
    grads = [[lay(torch.empty(s, dtype=gdt, device="cuda")) for s in cfg.level_shapes]
             for _ in range(R)] if cfg.backward else None
    ws_bytes = B.roi_align_fpn_workspace_bytes(K, L, PH, PW, g, flags)
    repack = bool(args.repack and args.layout == "nchw")
    if repack:   # the library repacks NCHW <-> channels-last inside the (larger) workspace, inside every timed call
        ws_bytes += B.roi_align_fpn_repack_bytes(feats[0], cfg.scales, tdt, K, PH, PW)
        flags |= B.RAF_REPACK
        fwd_flags |= B.RAF_REPACK
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device="cuda")
    fdesc = [B.make_levels(f, cfg.scales) for f in feats]
    gdesc = [B.make_levels(gr, cfg.scales) for gr in grads] if cfg.backward else None
    stream = torch.cuda.current_stream()

    def fwd(j, s=stream):
        B.roi_align_fpn_forward_ex(feats[j], cfg.scales, rois, outs[j], g, aligned, fs, fwd_flags, ws, s, fdesc[j])

    def bwd(j, s=stream):
        B.roi_align_fpn_backward(grads[j], cfg.scales, gouts[j], rois, g, aligned, fs, flags, ws, s, gdesc[j])

    def step(j, s=stream):
        fwd(j, s)
        if cfg.backward:
            bwd(j, s)

    graphs = None
    if args.graph:
        graphs = []
        for j in range(R):
            step(j)
        torch.cuda.synchronize()
        for j in range(R):
            gr = torch.cuda.CUDAGraph()
            with torch.cuda.graph(gr):
                step(j, torch.cuda.current_stream())
            graphs.append(gr)

    def run_step(j):
        if graphs:
            graphs[j].replay()
        else:
            step(j)

    for i in range(args.warmup):
        run_step(i % R)
    torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.1)

    # ---- headline: EXACTLY `steps` interleaved fwd -> bwd steps between two events ----------------------
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = B.launch_count()
    e0.record(stream)
    for i in range(args.steps):
        run_step((args.warmup + i) % R)
    e1.record(stream)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches = B.launch_count() - launches0
    per_step_launches = 1 + ((1 + L) if args.backward == "atomic" else (1 if reuse else 2)) * cfg.backward
    if graphs:   # replayed launches are not seen by the library's counter: count per captured step
        launches = args.steps * per_step_launches
    total_ms = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())

    # ---- SURVEY 8(d) protocol: windows of back-to-back iterations, median of >= 5 windows + min, for the
    #      interleaved loop and for the forward-only / backward-only loops (the split) ---------------------
    def windows(fn, n_windows=args.windows, iters=args.window_iters):
        ms = []
        for w in range(n_windows):
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record(stream)
            for i in range(iters):
                fn((w * iters + i) % R)
            a1.record(stream)
            a1.synchronize()
            ms.append(a0.elapsed_time(a1) / iters)
        return {"median_ms": float(np.median(ms)), "min_ms": float(np.min(ms)), "windows": n_windows, "iters": iters}

    loops = {"step": windows(run_step), "fwd": windows(fwd)}
    if cfg.backward:
        if reuse:   # the backward-only loop reuses the tables the last forward left in the workspace
            fwd(0)
        loops["bwd"] = windows(bwd)
    clocks = sampler.stop() if rank == 0 else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline (algorithmic bytes / CUDA-event duration of the dominant call) ----
    if g > 0:
        fp = roofline.footprint(wl.rois, cfg.level_shapes, cfg.scales, cfg.out_size, g, aligned, fs)
        ab = roofline.algorithmic_bytes(fp, K, C, cfg.out_size, esz, esz, esz, grad_bytes=(esz if gdt != torch.float32 else 4))
    else:   # adaptive grid: the touched set is at least the fixed-grid one; report the dense-pyramid bound instead
        fp = {"level_hist": None}
        ab = {"fwd": pyr_bytes * esz + K * C * PH * PW * esz + 20 * K, "bwd": K * C * PH * PW * esz + pyr_bytes * 4}
    peak, peak_src = peaks()
    variant = (f"{args.layout}{'+repack' if repack else ''}{'+g16' if gdt != torch.float32 else ''}"
               f"{'+levelorder' if args.roi_order == 'level' else ''}:{args.backward}:{'reuse' if reuse else 'noreuse'}")
    traffic, traffic_stale = ncu_traffic(args.config, variant)
    legs = {"fwd": (ab["fwd"], loops["fwd"]["median_ms"])}
    if cfg.backward:
        legs["bwd"] = (ab["bwd"], loops["bwd"]["median_ms"])
    dom = max(legs, key=lambda k: legs[k][1])
    NOMINAL = 8000.0

    def roof(name):
        by, ms = legs[name]
        ach = by / (ms * 1e-3) / 1e9
        return {"bound": "hbm", "kernel": name, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "frac_nominal_8000": ach / NOMINAL,
                "traffic": traffic.get(name), "traffic_stale": bool(traffic_stale),
                "traffic_source": "profiles/traffic.json (bench_traffic.py)" if traffic.get(name) else None,
                "algorithmic_bytes": by, "ms": ms, "ms_min": loops[name]["min_ms"],
                "peak_source": peak_src,
                "note": "ms = median over windows of the CUDA-event time per C-ABI call of this leg run back to back "
                        "(fwd: gather kernel incl. the backward's prep blocks under RAF_REUSE_PREP; bwd: pull "
                        "kernel, + its prep launch otherwise); achieved = algorithmic bytes / ms"}

    step_ms = total_ms / args.steps
    step_bytes = ab["fwd"] + (ab["bwd"] if cfg.backward else 0)
    step_ach = step_bytes / (step_ms * 1e-3) / 1e9
    line = {"metric": METRIC, "value": world * K / (step_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.config - 1}]: {cfg.name}", "K": K, "C": C,
                       "out_size": [PH, PW], "levels": L, "layout": args.layout, "sampling_ratio": g, "aligned": bool(aligned),
                       "parallelism": f"{world} independent replica(s): every rank runs the whole workload on its own GPU "
                                      "(the path shards by image; no collective)",
                       "l2_protocol": (f"inputs rotate over {R} independent copies ({R * ws_set / 1e6:.0f} MB >> L2 {l2 / 1e6:.0f} MB)"
                                       if R * ws_set >= 2 * l2 else
                                       f"WARM: {R} buffer set(s), {R * ws_set / 1e6:.0f} MB vs L2 {l2 / 1e6:.0f} MB (not the headline)"),
                       "backward": args.backward if cfg.backward else "none", "repack": repack,
                       "grad_dtype": "f32" if gdt == torch.float32 else cfg.dtype,
                       "reuse_prep": bool(reuse), "cuda_graph": bool(graphs), "roi_order": args.roi_order,
                       "level_hist": fp["level_hist"]},
            "roofline": roof(dom),
            "roofline_all": {k: roof(k) for k in legs} | {"step": {
                "achieved": step_ach, "frac": step_ach / peak, "frac_nominal_8000": step_ach / NOMINAL,
                "algorithmic_bytes": step_bytes, "ms": step_ms,
                "ms_window_median": loops["step"]["median_ms"], "ms_window_min": loops["step"]["min_ms"]}},
            "loops": loops,
            "clocks": clocks, "gpu_launches": int(launches), "source_hash": source_hash()}

    # ---- e2e: HOST buffers through the C ABI, copies inside the timed region ----
    if not args.no_e2e and g > 0:
        hf = [lay(f).pin_memory() if args.layout == "nchw" else f.permute(0, 2, 3, 1).contiguous().pin_memory().permute(0, 3, 1, 2)
              for f in base_feats]
        hrois = torch.from_numpy(wl.rois).pin_memory()

        def hbuf(shape, dt):
            n, c, h, w = shape
            if args.layout == "nchw":
                return torch.empty(shape, dtype=dt).pin_memory()
            return torch.empty((n, h, w, c), dtype=dt).pin_memory().permute(0, 3, 1, 2)
        hout = hbuf((K, C, PH, PW), tdt)
        arena = torch.empty(B.roi_align_fpn_host_arena_bytes(hf, cfg.scales, tdt, K, PH, PW, g, flags),
                            dtype=torch.uint8, device="cuda")
        h2d = sum(f.numel() for f in hf) * esz + K * 20
        d2h = K * C * PH * PW * esz
        if cfg.backward:
            hgout = hbuf((K, C, PH, PW), tdt)
            hgout.copy_(torch.from_numpy(wl.grad_out).to(tdt))
            hgrads = [hbuf(s, torch.float32) for s in cfg.level_shapes]
            h2d += K * C * PH * PW * esz + K * 20
            d2h += pyr_bytes * 4

        def e2e_step():
            B.roi_align_fpn_forward_host(hf, cfg.scales, hrois, hout, g, aligned, fs, arena, stream)
            if cfg.backward:
                B.roi_align_fpn_backward_host(hgrads, cfg.scales, hgout, hrois, g, aligned, fs, flags & ~B.RAF_REUSE_PREP, arena, stream)
        n_e2e = max(1, min(args.steps, 5))
        e2e_step()
        torch.cuda.synchronize()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for _ in range(n_e2e):
            e2e_step()
        a1.record(stream)
        torch.cuda.synchronize()
        ms = a0.elapsed_time(a1) / n_e2e
        line["e2e"] = {"value": world * K / (ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                       "d2h_bytes_per_step": int(d2h), "ms_per_step": ms, "steps": n_e2e,
                       "note": "roi_align_fpn_{forward,backward}_host: pinned host buffers, copies in the timed region"}
        del arena

    if not args.no_cpu_baseline and world == 1:
        from oracle import build as ref_build
        ref_build.build()
        line["cpu_baseline"] = cpu_baseline(args.config)
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_op(args):
    """One bench line for a SURVEY 8(f) operation: RoIPool-max fwd+bwd on the config's pyramid / RoIs, greedy NMS or
    Soft-NMS on `--nms-n` synthetic proposals of one image (log-uniform sizes, 1344 x 800, scores uniform)."""
    import torch
    import bench_roofline as roofline
    from paper_1906_07155_b200 import binding as B
    from paper_1906_07155_b200 import build as raf_build
    from paper_1906_07155_b200 import inputs
    assert torch.cuda.is_available(), "bench.py needs a CUDA device; there is no CPU fallback"
    torch.cuda.set_device(0)
    raf_build.build()
    B.lib()
    stream = torch.cuda.current_stream()
    peak, peak_src = peaks()
    sampler = ClockSampler(0)

    def timed(fn, nset):
        for i in range(max(args.warmup, 3)):
            fn(i % nset)
        torch.cuda.synchronize()
        sampler.start()
        time.sleep(0.1)
        ms = []
        for w in range(args.windows):
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a0.record(stream)
            for i in range(args.window_iters):
                fn((w * args.window_iters + i) % nset)
            a1.record(stream)
            a1.synchronize()
            ms.append(a0.elapsed_time(a1) / args.window_iters)
        return float(np.median(ms)), float(np.min(ms)), sampler.stop()

    if args.op == "pool":
        cfg = inputs.CONFIGS[args.config]
        wl = inputs.make_workload(args.config)
        tdt = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[cfg.dtype]
        esz = 4 if cfg.dtype == "f32" else 2
        K, C = cfg.K, cfg.channels
        PH, PW = cfg.out_size
        lay = lambda t: t.permute(0, 2, 3, 1).contiguous().permute(0, 3, 1, 2)
        pyr = sum(int(np.prod(s)) for s in cfg.level_shapes)
        R = 4
        feats = [[lay(torch.from_numpy(f).to(tdt).cuda()) for f in wl.feats] for _ in range(R)]
        rois = torch.from_numpy(wl.rois).cuda()
        outs = [lay(torch.empty((K, C, PH, PW), dtype=tdt, device="cuda")) for _ in range(R)]
        args_ = [lay(torch.empty((K, C, PH, PW), dtype=torch.int32, device="cuda")) for _ in range(R)]
        gouts = [lay(torch.from_numpy(wl.grad_out).to(tdt).cuda()) for _ in range(R)]
        grads = [[lay(torch.empty(s, dtype=torch.float32, device="cuda")) for s in cfg.level_shapes] for _ in range(R)]

        def step(j):
            B.roi_pool_fpn_forward(feats[j], cfg.scales, rois, outs[j], args_[j], cfg.finest_scale, stream)
            B.roi_pool_fpn_backward(grads[j], cfg.scales, gouts[j], args_[j], rois, cfg.finest_scale, 0, stream)
        ms, ms_min, clocks = timed(step, R)
        fp = roofline.footprint(wl.rois, cfg.level_shapes, cfg.scales, cfg.out_size, 2, True, cfg.finest_scale)
        by = fp["union_px"] * C * esz + K * C * PH * PW * (esz + 4) + K * C * PH * PW * (esz + 4) + pyr * 4 * 2
        ach = by / (ms * 1e-3) / 1e9
        line = {"metric": "RoIPool-max fwd+bwd RoIs/sec (C=256, 7x7, FPN)", "value": K / (ms * 1e-3), "unit": UNIT,
                "n_gpus": 1, "steps": args.windows * args.window_iters, "warmup": max(args.warmup, 3), "ms_per_step": ms,
                "ms_per_step_min": ms_min, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": cfg.dtype, "data": "synthetic",
                "config": {"workload": f"RoIPool-max on BASELINE.json configs[{args.config - 1}] shapes: {cfg.name}", "K": K, "C": C,
                           "layout": "cl", "l2_protocol": f"inputs rotate over {R} independent copies"},
                "roofline": {"bound": "hbm", "kernel": "pool fwd + zero-fill + bwd", "achieved": ach, "peak": peak, "unit": "GB/s",
                             "frac": ach / peak, "frac_nominal_8000": ach / 8000.0, "traffic": None, "algorithmic_bytes": int(by),
                             "peak_source": peak_src,
                             "note": "bytes = touched-pixel union (the RoIAlign union of the same RoIs as a stand-in: RoIPool "
                                     "windows differ by at most a pixel per side) + out + argmax written + grad_out + argmax "
                                     "read + gradient pyramid zero-filled and written"},
                "clocks": clocks, "gpu_launches": args.windows * args.window_iters * (2 + len(cfg.level_shapes))}
    elif args.op == "fc":
        # RoIAlign gather fused into the box head's first FC (12544 -> 1024 for the 7 x 7 x 256 box head), bf16 features and
        # weights, fp32 accumulate.  Context number in the same line: the library's stand-alone forward + a cuBLAS product.
        cfg = inputs.CONFIGS[args.config]
        wl = inputs.make_workload(args.config)
        tdt = torch.bfloat16 if cfg.dtype == "f32" else {"f16": torch.float16, "bf16": torch.bfloat16}[cfg.dtype]
        K, C = cfg.K, cfg.channels
        PH, PW = cfg.out_size
        n_out = 1024
        lay = lambda t: t.permute(0, 2, 3, 1).contiguous().permute(0, 3, 1, 2)
        R = 4
        feats = [[lay(torch.from_numpy(f).to(tdt).cuda()) for f in wl.feats] for _ in range(R)]
        rois = torch.from_numpy(wl.rois).cuda()
        rng = np.random.default_rng(190607155 + 79)
        w = torch.from_numpy((rng.standard_normal((n_out, PH * PW * C)) / np.sqrt(PH * PW * C)).astype(np.float32)).to(tdt).cuda()
        bias = torch.from_numpy(rng.standard_normal(n_out).astype(np.float32)).cuda()
        outs = [torch.empty((K, n_out), dtype=torch.float32, device="cuda") for _ in range(R)]
        xs = [lay(torch.empty((K, C, PH, PW), dtype=tdt, device="cuda")) for _ in range(R)]

        def step(j):
            B.roi_align_fc_fpn_forward(feats[j], cfg.scales, rois, w, bias, outs[j], (PH, PW), 2, True, cfg.finest_scale, stream)

        def unfused(j):
            B.roi_align_fpn_forward_ex(feats[j], cfg.scales, rois, xs[j], 2, True, cfg.finest_scale, B.RAF_NO_PREP, None, stream)
            torch.addmm(bias.to(tdt), xs[j].permute(0, 2, 3, 1).reshape(K, -1), w.t())
        ms, ms_min, clocks = timed(step, R)
        ms_unf, _, _ = timed(unfused, R)
        flops = 2.0 * K * PH * PW * C * n_out
        tensor_peak = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json"))).get("bf16_tflops") if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else None
        tpeak = float(tensor_peak) if tensor_peak else 2250.0
        line = {"metric": "RoIAlign + first FC (12544 -> 1024) RoIs/sec, fused gather + tcgen05 GEMM", "value": K / (ms * 1e-3),
                "unit": UNIT, "n_gpus": 1, "steps": args.windows * args.window_iters, "warmup": max(args.warmup, 3),
                "ms_per_step": ms, "ms_per_step_min": ms_min, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "bf16" if tdt == torch.bfloat16 else "f16", "data": "synthetic",
                "config": {"workload": f"fused RoIAlign + FC on BASELINE.json configs[{args.config - 1}] shapes (features cast to 16 bit): {cfg.name}",
                           "K": K, "C": C, "out_size": [PH, PW], "n_out": n_out, "layout": "cl",
                           "l2_protocol": f"inputs rotate over {R} independent copies",
                           "unfused_context_ms": ms_unf,
                           "unfused_context": "roi_align_fpn_forward_ex(RAF_NO_PREP) + torch.addmm (cuBLAS), same inputs"},
                "roofline": {"bound": "tensor", "kernel": "fc_fused_kernel", "achieved": flops / (ms * 1e-3) / 1e12, "peak": tpeak,
                             "unit": "TFLOP/s", "frac": flops / (ms * 1e-3) / 1e12 / tpeak, "traffic": None,
                             "note": "flops of the matrix product only; the kernel is bound by its gathers (every RoI window "
                                     "is gathered n_out / 256 times), not by the tensor cores",
                             "peak_source": "MEASURED_PEAKS.json bf16_tflops" if tensor_peak else "nominal 2250 TFLOP/s dense bf16"},
                "clocks": clocks, "gpu_launches": args.windows * args.window_iters * 2}
    elif args.op == "deform":
        cfg = inputs.CONFIGS[args.config]
        wl = inputs.make_workload(args.config)
        tdt = {"f32": torch.float32, "f16": torch.float16, "bf16": torch.bfloat16}[cfg.dtype]
        esz = 4 if cfg.dtype == "f32" else 2
        K, C = cfg.K, cfg.channels
        PH, PW = cfg.out_size
        lay = lambda t: t.permute(0, 2, 3, 1).contiguous().permute(0, 3, 1, 2)
        pyr = sum(int(np.prod(s)) for s in cfg.level_shapes)
        R = 4
        feats = [[lay(torch.from_numpy(f).to(tdt).cuda()) for f in wl.feats] for _ in range(R)]
        rois = torch.from_numpy(wl.rois).cuda()
        offset = torch.from_numpy(np.random.default_rng(190607155 + 78).uniform(-0.5, 0.5, (K, 2, PH, PW)).astype(np.float32)).cuda()
        outs = [lay(torch.empty((K, C, PH, PW), dtype=tdt, device="cuda")) for _ in range(R)]
        gouts = [lay(torch.from_numpy(wl.grad_out).to(tdt).cuda()) for _ in range(R)]
        grads = [[lay(torch.empty(s, dtype=torch.float32, device="cuda")) for s in cfg.level_shapes] for _ in range(R)]
        goff = torch.empty((K, 2, PH, PW), dtype=torch.float32, device="cuda")

        def step(j):
            B.roi_deform_pool_fpn_forward(feats[j], cfg.scales, rois, offset, 0.1, outs[j], 2, cfg.finest_scale, stream)
            B.roi_deform_pool_fpn_backward(feats[j], grads[j], cfg.scales, gouts[j], rois, offset, 0.1, 2, cfg.finest_scale,
                                           goff, 0, stream)
        ms, ms_min, clocks = timed(step, R)
        fp = roofline.footprint(wl.rois, cfg.level_shapes, cfg.scales, cfg.out_size, 2, True, cfg.finest_scale)
        by = 2 * fp["union_px"] * C * esz + 2 * K * C * PH * PW * esz + pyr * 4 * 2 + 3 * K * 2 * PH * PW * 4
        ach = by / (ms * 1e-3) / 1e9
        line = {"metric": "deformable RoI pooling fwd+bwd RoIs/sec (C=256, 7x7, FPN)", "value": K / (ms * 1e-3), "unit": UNIT,
                "n_gpus": 1, "steps": args.windows * args.window_iters, "warmup": max(args.warmup, 3), "ms_per_step": ms,
                "ms_per_step_min": ms_min, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": cfg.dtype, "data": "synthetic",
                "config": {"workload": f"deformable RoI pooling on BASELINE.json configs[{args.config - 1}] shapes: {cfg.name}",
                           "K": K, "C": C, "layout": "cl", "gamma": 0.1, "offsets": "U(-0.5, 0.5) per bin",
                           "l2_protocol": f"inputs rotate over {R} independent copies"},
                "roofline": {"bound": "hbm", "kernel": "deform fwd + zero-fill + bwd (features and offsets)", "achieved": ach,
                             "peak": peak, "unit": "GB/s", "frac": ach / peak, "frac_nominal_8000": ach / 8000.0, "traffic": None,
                             "algorithmic_bytes": int(by), "peak_source": peak_src,
                             "note": "bytes = touched-pixel union read in the forward and again in the backward (the RoIAlign "
                                     "union of the undeformed RoIs as a stand-in) + out + grad_out + gradient pyramid "
                                     "zero-filled and written + offsets / offset gradient"},
                "clocks": clocks, "gpu_launches": args.windows * args.window_iters * (3 + len(cfg.level_shapes))}
    else:
        n = args.nms_n
        rng = np.random.default_rng(190607155 + 77)
        side = np.exp(rng.uniform(np.log(16), np.log(800), n))
        asp = np.exp(rng.uniform(np.log(0.5), np.log(2), n))
        w, h = side * np.sqrt(asp), side / np.sqrt(asp)
        cx, cy = rng.uniform(0, 1344, n), rng.uniform(0, 800, n)
        boxes = torch.from_numpy(np.stack([cx - w / 2, cy - h / 2, cx + w / 2, cy + h / 2], 1).astype(np.float32)).cuda()
        scores = torch.from_numpy(rng.uniform(0, 1, n).astype(np.float32)).cuda()
        keep = torch.empty(n, dtype=torch.int32, device="cuda")
        ns = torch.empty(n, dtype=torch.float32, device="cuda")
        nk = torch.empty(1, dtype=torch.int32, device="cuda")
        ws = torch.empty(B.roi_nms_workspace_bytes(n), dtype=torch.uint8, device="cuda")
        if args.op == "nms":
            fn = lambda j: B.roi_nms(boxes, scores, 0.7, keep, nk, ws, stream)
            name, launches = f"greedy NMS boxes/sec (n={n} proposals, IoU 0.7)", 3
        else:
            fn = lambda j: B.roi_soft_nms(boxes, scores, 0.3, 0.5, 0.05, B.RAF_SOFT_LINEAR, keep, ns, nk, stream)
            name, launches = f"Soft-NMS (linear) boxes/sec (n={n} proposals)", 1
        ms, ms_min, clocks = timed(fn, 1)
        kept = int(nk.item())
        # ALU bound: the n(n-1)/2 IoU evaluations (about 20 fp32 operations each incl. one IEEE division ~ 10)
        flops = n * (n - 1) / 2 * 30
        alu_peak = 148 * 128 * 2 * 1.965e9 / 1e12
        line = {"metric": name, "value": n / (ms * 1e-3), "unit": "boxes/s", "n_gpus": 1,
                "steps": args.windows * args.window_iters, "warmup": max(args.warmup, 3), "ms_per_step": ms, "ms_per_step_min": ms_min,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"{n} boxes of one 1344x800 image, side log-uniform 16-800 px, aspect 0.5-2, scores U(0,1); kept {kept}"},
                "roofline": {"bound": "alu", "kernel": "nms_mask_kernel" if args.op == "nms" else "soft_nms_kernel",
                             "achieved": flops / (ms * 1e-3) / 1e12, "peak": alu_peak, "unit": "TFLOP/s",
                             "frac": flops / (ms * 1e-3) / 1e12 / alu_peak, "traffic": None,
                             "note": "peak = 148 SMs x 128 fp32 lanes x 2 x 1.965 GHz; the op is latency bound (sequential "
                                     "scan over kept boxes), the fraction is reported for completeness"},
                "clocks": clocks, "gpu_launches": args.windows * args.window_iters * launches}
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.op != "align":
        run_op(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
