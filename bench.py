#!/usr/bin/env python
"""bench.py -- render throughput of the MLP-Splatting forward render on B200.

A "step" is one pass of the whole hot path (stages (a)-(e), one `ms_render`) over one view of
the workload: BASELINE.json configs[3] by default (4096 primitives, 39-128-128-128-4 bf16 MLPs,
1920x1080, K = 24 -- "the 1080p config" the north-star target is quoted on, Q21).
Prints ONE JSON line (see the contract in DESIGN.md Sec.7).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg4] [--impl ours|reference]

N > 1 (launched by torch.distributed.run): every rank owns a replica of the scene and renders
its own steps -- views are independent problems, no data-path collective ("scaling": "weak").
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded pixel sample.
"""
from __future__ import annotations

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

import numpy as np  # noqa: E402

from paper_2606_03877_b200 import synth  # noqa: E402

UNIT = "Mpixels/s"
# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel, from the committed
# `ncu --set full` capture of this very command (profiles/r1c_summary.md); null where none was taken.
NCU_TRAFFIC_BYTES = {"cfg4": 0.843211264e9 + 7.445789e9}
METRIC = "render throughput (Mpixels/s; MLP samples/s and roofline fraction alongside)"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"source": "measured", "hbm_gbs": p["hbm_gbs"], "bf16_tflops": p["bf16_tflops"],
                "bf16_tflops_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"])}
    # /opt/skills/guides/B200_PROFILING.md fallback
    return {"source": "fallback", "hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def workload_desc(cfg) -> str:
    m = cfg.mlp
    dims = "-".join(str(d) for d in [m.in_dim] + [m.width] * m.n_hidden + [m.out_dim])
    return (f"{cfg.name}: {cfg.n_prims} primitives, MLP {dims} {'bf16' if m.bf16 else 'fp32'}, "
            f"{cfg.width}x{cfg.height}, K={cfg.K}, {cfg.n_views} view(s)/step")


# ------------------------------------------------------------------------------------------------
# clocks sampling during the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# CPU oracle legs
# ------------------------------------------------------------------------------------------------
def time_oracle(cfg, sc, cams, target_s: float, seed: int = 0):
    """Times oracle/ (as it stands, all host cores) on a seeded random pixel sample of view 0,
    sized from a short calibration so the leg takes about `target_s` seconds."""
    from oracle import mso
    orc = mso.OracleScene(sc)
    H, W = cfg.height, cfg.width
    rng = np.random.default_rng(seed)
    cores = os.cpu_count() or 1
    # two calibration passes: 256 pixels (dominated by the per-call tile-list build), then ~1/8 of the target
    n, rate = min(H * W, 256), None
    for _ in range(2):
        if rate is not None:
            n = int(min(H * W, max(256, rate * target_s / 8.0)))
        pix = rng.choice(H * W, n, replace=False).astype(np.int32)
        t = time.perf_counter()
        orc.render(cams[0], H, W, cfg.K, pixels=pix, tile=cfg.tile)
        rate = n / max(time.perf_counter() - t, 1e-4)          # pixels per second
    n = int(min(H * W, max(256, rate * target_s)))
    pix = rng.choice(H * W, n, replace=False).astype(np.int32)
    t = time.perf_counter()
    _, _, _, st = orc.render(cams[0], H, W, cfg.K, pixels=pix, tile=cfg.tile)
    dt = time.perf_counter() - t
    return {"value": n / dt / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{n} seeded random pixels of view 0 of {cfg.name} ({st.n_samples} MLP samples) in {dt:.2f} s, "
                      f"OpenMP over pixels, tile lists built once per call",
            "samples_per_s": st.n_samples / dt, "seconds": dt, "n_pixels": n}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    sc = synth.make_scene(cfg)
    cams = synth.make_cameras(cfg)
    per_step = max(0.5, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        time_oracle(cfg, sc, cams, per_step)
    vals, samp = [], []
    t_all = time.perf_counter()
    for i in range(args.steps):
        r = time_oracle(cfg, sc, cams, per_step, seed=i)
        vals.append(r["value"]); samp.append(r)
    wall = time.perf_counter() - t_all
    v = float(np.mean(vals))
    px = cfg.width * cfg.height * cfg.n_views
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": px / (v * 1e6) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_desc(cfg), "note": "ms_per_step = full-frame time extrapolated from the sampled rate"},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": samp[-1]["cores"], "kind": "oracle",
                             "sample": samp[-1]["sample"]},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0, "wall_s": wall}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# our arm
# ------------------------------------------------------------------------------------------------
def algorithmic_bytes(cfg, sc) -> dict:
    """what the method must move -- the scene read once (primitives; weight matrices in the
    config's dtype, biases fp32; slot embeddings) and the image written once."""
    m = cfg.mlp
    n_w = sum(i * o for i, o in m.layer_dims)
    n_b = sum(o for _, o in m.layer_dims)
    scene = sc.n * (40 + n_w * (2 if m.bf16 else 4) + n_b * 4) + (sc.slots.nbytes if sc.slots is not None else 0)
    feat_w = cfg.c_f or m.n_feat
    out = cfg.width * cfg.height * (16 + 4 * feat_w)
    return {"scene": scene, "outputs_per_view": out, "per_view": scene + out}


def load_dram_profile():
    """dram__bytes_read.sum + dram__bytes_write.sum per view and stage, from the committed ncu captures
    (profiles/r2_dram_bytes.csv, copied by hand from the summary it names; absent workloads -> null)."""
    path = os.path.join(ROOT, "profiles", "r2_dram_bytes.csv")
    out = {}
    if os.path.exists(path):
        for ln in open(path).read().strip().split("\n")[1:]:
            w, stage, b, src = ln.split(",", 3)
            out.setdefault(w, {"source": src})[stage] = float(b)
    return out


def measure(api, cfg, args, peaks, stream, barrier, steps, warmup, sampler=None, shard=None):
    """Times `steps` steps of one workload (a step = ms_render_batch over its views: stages (a)-(e)) with CUDA
    events on the launching stream, then the same steps through ms_render_host (e2e).  Returns a dict."""
    import torch
    sc = synth.make_scene(cfg)
    cams = synth.make_cameras(cfg)
    if shard is not None:                               # this rank's share of the step's views
        cams = cams[shard[0]:shard[1]] or cams[:1]
    H, W, K, V = cfg.height, cfg.width, cfg.K, len(cams)
    t_create = time.perf_counter()
    gs = api.Scene(sc)
    create_s = time.perf_counter() - t_create
    gs.band_bytes, gs.waves = args.band_bytes, args.waves
    extra_flags = api.FLAG_TILE_ORDER if (args.tile_order and cfg.mlp.mode == 1) else 0
    if args.overlap:
        extra_flags |= api.FLAG_OVERLAP
    if not args.sync:
        extra_flags |= api.FLAG_NO_SYNC      # views sized from their predecessor: no host synchronisation inside ms_render
    tile_kw = {"tile": args.tile} if args.tile else {"tile": cfg.tile}
    kw = dict(t_stop=cfg.t_stop, **tile_kw)
    with torch.cuda.stream(stream):
        out = gs.render_batch(cams, H, W, K, flags=extra_flags, **kw)          # allocates outputs + scratch
        for _ in range(warmup):
            gs.render_batch(cams, H, W, K, out=out, flags=extra_flags, **kw)
    barrier()
    gs.stage_accum(reset=True)
    if sampler is not None:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches = api.launch_count()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(steps):
            gs.render_batch(cams, H, W, K, out=out, flags=api.FLAG_STAGE_TIMES | extra_flags, **kw)
        ev1.record(stream)
    launches = api.launch_count() - launches                # kernels this thread launched in the timed region
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if sampler is not None else None
    stage_sum, n_views_timed = gs.stage_accum()
    st = gs.stats()                                     # counts of the last view

    # ---- e2e: the same steps through ms_render_host (pinned HOST outputs, D2H inside) ----
    host_out = gs.render_host(cams, H, W, K, stream=stream.cuda_stream, flags=extra_flags, **kw)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(steps, 10))
    for _ in range(e2e_steps):
        gs.render_host(cams, H, W, K, out=host_out, stream=stream.cuda_stream, flags=extra_flags, **kw)   # synchronises the stream itself
    barrier()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    gs.close()
    del out, host_out
    torch.cuda.empty_cache()

    ms_step = ms_total / steps
    px_step = H * W * V
    n_samples_view = st.n_samples                       # last view
    n_eval_view = st.n_samples_evaluated
    flops_view = cfg.mlp.flop_per_sample * n_eval_view  # the MLP evaluations that really ran
    nv = max(1, n_views_timed)
    stage_ms = {k: v / nv for k, v in stage_sum.items()}
    mlp_ms, comp_ms = stage_ms["mlp"], stage_ms["composite"]
    achieved = flops_view / (mlp_ms * 1e-3) / 1e12 if mlp_ms > 0 else 0.0
    peak = peaks["bf16_tflops_sustained"]
    if not cfg.mlp.bf16:
        # fp32 SIMT path: 148 SMs x 128 FMA lanes x 2 FLOP at the top SM clock (guide's unit counts)
        peak = 148 * 128 * 2 * 1.965e9 / 1e12
    alg = algorithmic_bytes(cfg, sc)
    feat_w = cfg.c_f or cfg.mlp.n_feat
    feat_b = 2 if (cfg.mlp.bf16 and cfg.mlp.n_feat == 32) else 4      # the tensor path stages its features as fp16
    sample_bytes = 16 + feat_b * cfg.mlp.n_feat + (32 if cfg.c_f else 0)
    # bytes the design moves per view by construction: staging written by (d) and read by (e), both hit lists
    # written by (c) and read by (d) / (e), the outputs
    stage_bytes_design = 2 * n_eval_view * sample_bytes + 2 * st.n_intervals * 48 + alg["outputs_per_view"]
    frame_floor_ms = max(flops_view / (peak * 1e12), alg["per_view"] / (peaks["hbm_gbs"] * 1e9)) * 1e3
    dram = load_dram_profile().get(cfg.name)
    res = {
        "workload": workload_desc(cfg), "ms_per_step": ms_step, "Mpixels_per_s": px_step / (ms_step * 1e-3) / 1e6,
        "samples_per_s": n_eval_view * V / (ms_step * 1e-3), "stage_ms_per_view": stage_ms,
        "counts_per_view": {"visible": st.n_visible, "pairs": st.n_pairs, "intervals": st.n_intervals,
                            "samples": st.n_samples, "samples_evaluated": n_eval_view, "dead_rays": st.n_dead_rays,
                            "row_blocks": st.n_blocks, "bands": st.n_bands, "waves": st.n_waves,
                            "staging_MB": st.staging_bytes / 1e6, "scratch_GB": st.scratch_bytes / 1e9},
        "gpu_launches": launches, "scene_create_s": create_s, "no_sync_views": bool(st.no_sync), "overflow": bool(st.overflow),
        "e2e": {"value": px_step / (e2e_ms * 1e-3) / 1e6, "unit": UNIT, "h2d_bytes_per_step": 64 * V,
                "d2h_bytes_per_step": alg["outputs_per_view"] * V, "ms_per_step": e2e_ms},
        "roofline": {"bound": "tensor" if cfg.mlp.bf16 else "alu",
                     "kernel": "mlp_tc_kernel (stage d)" if cfg.mlp.bf16 else "mlp_f32_kernel (stage d, fp32 SIMT path)",
                     "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak if peak else None,
                     "traffic": (dram or {}).get("mlp"),
                     "traffic_unit": "bytes per view, all launches of the kernel (ncu dram read + write), " +
                                     str((dram or {}).get("source", "no capture of this workload")),
                     "algorithmic_bytes": alg["per_view"],
                     "algorithmic_bytes_note": "SURVEY.md Sec.8(d): scene read once + outputs written once, per view",
                     "stage_bytes_design": stage_bytes_design,
                     "dram_bytes_per_view": (dram or {}).get("total"),
                     "peak_kind": (f"bf16 dense, sustained, of {peaks['source']}" if cfg.mlp.bf16 else
                                   "fp32 FMA, 148 SMs x 128 lanes x 2 x 1.965 GHz (derived)"),
                     "frac_of_burst_peak": achieved / peaks["bf16_tflops"] if cfg.mlp.bf16 else None,
                     "algorithmic_flop_per_sample": cfg.mlp.flop_per_sample,
                     "kernel_ms": mlp_ms, "kernel_share_of_step": mlp_ms * V / ms_step},
        "frame_roofline": {"floor_ms_per_view": frame_floor_ms, "frac": frame_floor_ms * V / ms_step,
                           "note": "slower of the evaluated MLP FLOPs at the bf16 peak and the algorithmic bytes "
                                   "(scene + outputs) at the HBM peak, over the whole step"},
        "clocks": clocks,
    }
    if cfg.c_f and comp_ms > mlp_ms:
        # Eq.7 slot features: stage (e) dominates and is memory-bound.  Algorithmic bytes per view: staging,
        # gates and hit records once per hit (16 B each), the embeddings once, the outputs once.
        a2 = st.n_intervals * 48 + sc.slots.nbytes + alg["outputs_per_view"]
        ach = a2 / (comp_ms * 1e-3) / 1e9
        res["roofline"] = {"bound": "hbm", "kernel": "composite_kernel<2> + slot_feature_kernel (stage e, slot features)",
                           "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                           "traffic": (dram or {}).get("composite"),
                           "peak_kind": f"HBM copy bandwidth, of {peaks['source']}", "algorithmic_bytes": a2,
                           "stage_bytes_design": stage_bytes_design, "dram_bytes_per_view": (dram or {}).get("total"),
                           "kernel_ms": comp_ms, "kernel_share_of_step": comp_ms * V / ms_step,
                           "note": "the kernel re-reads each hit's four embedding rows (16 * c_f B per hit) through L1/L2; "
                                   "that traffic is not algorithmic"}
    return res, sc, cams


def measure_backward(api, cfg, args, stream, barrier, steps=5, warmup=3):
    """ms_backward (S:Sec.8(f) NEXT-4): one call = the forward stages (a)-(e) on the fp32 path + the backward kernels
    for one view, dL/dC resident in HBM.  Work counted: 3 x the forward MLP FLOPs of the samples (forward recomputed in
    the backward kernel is not counted twice: forward + dX + dW), against the fp32 FMA peak."""
    import torch
    sc = synth.make_scene(cfg)
    cam = synth.make_cameras(cfg)[0]
    H, W, K = cfg.height, cfg.width, cfg.K
    gs = api.Scene(sc)
    d_rgb = torch.randn((H, W, 3), device="cuda", dtype=torch.float32)
    with torch.cuda.stream(stream):
        grads = gs.backward(cam, H, W, K, d_rgb, tile=cfg.tile, t_stop=cfg.t_stop)
        for _ in range(warmup):
            gs.backward(cam, H, W, K, d_rgb, tile=cfg.tile, t_stop=cfg.t_stop, grads=grads)
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(steps):
            gs.backward(cam, H, W, K, d_rgb, tile=cfg.tile, t_stop=cfg.t_stop, grads=grads)
        ev1.record(stream)
    barrier()
    ms = ev0.elapsed_time(ev1) / steps
    st = gs.stats()
    gs.close()
    del grads, d_rgb
    torch.cuda.empty_cache()
    peak = 148 * 128 * 2 * 1.965e9 / 1e12
    ach = 3 * cfg.mlp.flop_per_sample * st.n_samples / (ms * 1e-3) / 1e12
    return {"workload": workload_desc(cfg) + ", fp32 path, forward + backward", "ms_per_step": ms,
            "Mpixels_per_s": H * W / (ms * 1e-3) / 1e6, "samples_per_s": st.n_samples / (ms * 1e-3),
            "samples": st.n_samples,
            "roofline": {"bound": "alu", "kernel": "whole call (forward fp32 stages + composite_bwd + mlp_bwd + interval_bwd)",
                         "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                         "peak_kind": "fp32 FMA, 148 SMs x 128 lanes x 2 x 1.965 GHz (derived)"}}


def run_backward_only(args, cfg):
    import torch
    from paper_2606_03877_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the backward pass has no CPU fallback")
    torch.cuda.set_device(0)
    stream = torch.cuda.Stream()
    out = measure_backward(api, cfg, args, stream, torch.cuda.synchronize, steps=max(1, min(args.steps, 5)),
                           warmup=max(1, min(args.warmup, 3)))
    out["config"] = args.config
    print(json.dumps(out))


def run_ours(args, cfg):
    import torch
    from paper_2606_03877_b200 import api
    from paper_2606_03877_b200 import dist as msdist

    rank, local, world = msdist.env_rank_world()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the render has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        msdist.init("nccl", torch.device("cuda", local))

    def barrier():
        msdist.barrier()
        torch.cuda.synchronize()

    peaks = load_peaks()
    stream = torch.cuda.Stream()
    sampler = ClockSampler(local) if rank == 0 else None

    # strong scaling (CFG5's batch of poses sharded over the ranks, S:Sec.8(e)): every rank renders its share
    shard = None
    if args.shard_views and world > 1:
        lo, hi = msdist.shard_range(cfg.n_views, rank, world)
        shard = (lo, hi)
    r, sc, cams = measure(api, cfg, args, peaks, stream, barrier, args.steps, args.warmup, sampler, shard=shard)
    ms_step, e2e_ms = msdist.max_over_ranks([r["ms_per_step"], r["e2e"]["ms_per_step"]], "cuda")

    others = {}
    if rank == 0 and world == 1 and args.all_configs:
        for name in ALL_CONFIGS:
            if name == cfg.name:
                continue
            o, _, _ = measure(api, synth.CONFIGS[name], args, peaks, stream, barrier, max(3, min(args.steps, 10)), 3)
            others[name] = {k: o[k] for k in ("workload", "ms_per_step", "Mpixels_per_s", "samples_per_s",
                                              "stage_ms_per_view", "counts_per_view", "gpu_launches", "scene_create_s",
                                              "no_sync_views", "overflow")}
            others[name]["e2e_Mpixels_per_s"] = o["e2e"]["value"]
            others[name]["e2e_ms_per_step"] = o["e2e"]["ms_per_step"]
            others[name]["roofline"] = {k: o["roofline"].get(k) for k in
                                        ("bound", "kernel", "achieved", "peak", "unit", "frac", "kernel_ms",
                                         "algorithmic_bytes", "stage_bytes_design", "dram_bytes_per_view")}
            others[name]["frame_roofline_frac"] = o["frame_roofline"]["frac"]
    backward = {}
    if rank == 0 and world == 1 and args.all_configs:
        for name in ("cfg1", "cfg2", "cfg3"):
            backward[name] = measure_backward(api, synth.CONFIGS[name], args, stream, barrier)
    if rank != 0:
        msdist.shutdown()
        return

    H, W, V = cfg.height, cfg.width, cfg.n_views
    strong = shard is not None
    px_job = H * W * V * (1 if strong else world)        # strong: the ranks split one step's views
    n_samp_job = r["counts_per_view"]["samples_evaluated"] * V * (1 if strong else world)
    line = {
        "metric": METRIC, "value": px_job / (ms_step * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "strong" if strong else "weak", "vs_baseline": None,
        "dtype": "bf16" if cfg.mlp.bf16 else "f32", "data": "synthetic",
        "config": {"workload": r["workload"],
                   "parallelism": (f"views sharded over {world} ranks, no collective" if strong else
                                   f"replicas x{world}, no collective"),
                   "l2": ("inputs larger than L2 (weights %.0f MB, staging %.0f MB per band)" if
                          sc.weights.nbytes / 2 + r["counts_per_view"]["staging_MB"] * 1e6 > 126e6 else
                          "working set below L2 (weights %.1f MB, staging %.1f MB): no flush, config is launch-bound")
                         % (sc.weights.nbytes / 2 / 1e6, r["counts_per_view"]["staging_MB"]),
                   "tile": args.tile or cfg.tile, "t_stop": cfg.t_stop,
                   "band_bytes": args.band_bytes, "waves": args.waves,
                   "no_sync": (not args.sync) and bool(r.get("no_sync_views")),
                   "order": "tile-centre shared order (P:109)" if args.tile_order else "exact per-ray order"},
        "samples_per_s": n_samp_job / (ms_step * 1e-3),
        "counts_per_view": r["counts_per_view"], "stage_ms_per_view": r["stage_ms_per_view"],
        "clocks": r["clocks"], "scene_create_s": r["scene_create_s"],
        "e2e": dict(r["e2e"], value=px_job / (e2e_ms * 1e-3) / 1e6, ms_per_step=e2e_ms,
                    note="ms_render_host: camera in (kernel parameters), rgb/alpha(/feat) copied to pinned host memory"),
        "gpu_launches": r["gpu_launches"], "roofline": r["roofline"], "frame_roofline": r["frame_roofline"],
    }
    if others:
        line["all_configs"] = others
    if backward:
        line["backward"] = backward
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = {k: v for k, v in time_oracle(cfg, sc, cams, args.cpu_seconds).items()
                                if k in ("value", "unit", "cores", "kind", "sample", "samples_per_s")}
    print(json.dumps(line), flush=True)
    msdist.shutdown()


ALL_CONFIGS = ["cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "next1", "next1b", "next2", "next2b", "cfg4_opaque", "cfg4_inside"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="cfg4", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--tile-order", action="store_true",
                    help="contact-mode configs: the paper's shared per-tile order (P:109) instead of the exact per-ray order")
    ap.add_argument("--tile", type=int, default=0, help="tile edge override (8, 16, 32)")
    ap.add_argument("--band-bytes", type=int, default=0,
                    help="staging budget per band in bytes (ms_opts.band_bytes): 0 = library default, -1 = one band")
    ap.add_argument("--all-configs", action="store_true", default=None,
                    help="also time every other workload (cfg1-5, next1/1b/2/2b, cfg4_opaque, cfg4_inside) in the same "
                         "run and add them as `all_configs`; default: on for the default workload at N=1")
    ap.add_argument("--no-all-configs", dest="all_configs", action="store_false")
    ap.add_argument("--shard-views", action="store_true",
                    help="N > 1: shard the workload's views over the ranks (strong scaling; cfg5's 8 poses) instead of "
                         "one replica of the whole step per rank")
    ap.add_argument("--overlap", action="store_true",
                    help="MS_FLAG_OVERLAP: stage (e) of a band runs beside stage (d) of the next on a second stream")
    ap.add_argument("--sync", action="store_true",
                    help="render without MS_FLAG_NO_SYNC (every view reads its counts back to size its scratch)")
    ap.add_argument("--waves", type=int, default=0, help="depth waves (ms_opts.waves): 0 = auto, -1 = off, C > 0 = wave size")
    ap.add_argument("--backward-only", action="store_true",
                    help="time ms_backward (forward + backward of one view, fp32) on --config alone and print its "
                         "object as one JSON line: the command behind profiles/r2d_backward.md")
    args = ap.parse_args()
    if args.backward_only:
        run_backward_only(args, synth.CONFIGS[args.config])
        return
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                  # timing rule: W >= 3
    cfg = synth.CONFIGS[args.config]
    if args.all_configs is None:
        args.all_configs = args.config == "cfg4" and args.gpus == 1
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
