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
    sc = synth.make_scene(cfg)
    cams = synth.make_cameras(cfg)
    H, W, K, V = cfg.height, cfg.width, cfg.K, cfg.n_views
    gs = api.Scene(sc)
    gs.band_bytes, gs.waves = args.band_bytes, args.waves
    stream = torch.cuda.Stream()
    out = None
    with torch.cuda.stream(stream):
        extra_flags = api.FLAG_TILE_ORDER if args.tile_order else 0
        tile_kw = {"tile": args.tile} if args.tile else {}
        out = gs.render_batch(cams, H, W, K, flags=extra_flags, **tile_kw)          # allocates outputs + scratch
        for _ in range(args.warmup):
            gs.render_batch(cams, H, W, K, out=out, flags=extra_flags, **tile_kw)
    barrier()
    gs.stage_accum(reset=True)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches = 0
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        for _ in range(args.steps):
            gs.render_batch(cams, H, W, K, out=out, flags=api.FLAG_STAGE_TIMES | extra_flags, **tile_kw)
            launches += gs.stats().n_launches * V
        ev1.record(stream)
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    stage_sum, n_views_timed = gs.stage_accum()
    st = gs.stats()                                     # counts of the last view

    # ---- e2e: the same steps through ms_render_host (pinned HOST outputs, D2H inside) ----
    host_out = gs.render_host(cams, H, W, K, stream=stream.cuda_stream, flags=extra_flags, **tile_kw)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(args.steps, 10))
    for _ in range(e2e_steps):
        gs.render_host(cams, H, W, K, out=host_out, stream=stream.cuda_stream, flags=extra_flags, **tile_kw)   # synchronises the stream itself
    barrier()
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps

    ms_total, e2e_ms = msdist.max_over_ranks([ms_total, e2e_ms], "cuda")
    if rank != 0:
        msdist.shutdown()
        return

    ms_step = ms_total / args.steps
    px_step = H * W * V
    value = world * px_step / (ms_step * 1e-3) / 1e6
    n_samples_view = st.n_samples                       # last view; equal for every step of a 1-view workload
    flops_view = cfg.mlp.flop_per_sample * n_samples_view
    mlp_ms = stage_sum["mlp"] / max(1, n_views_timed)  # mean duration of the dominant kernel, CUDA events in the timed region
    achieved = flops_view / (mlp_ms * 1e-3) / 1e12 if mlp_ms > 0 else 0.0
    peak = peaks["bf16_tflops_sustained"]
    if not cfg.mlp.bf16:
        # fp32 SIMT path: 148 SMs x 128 FMA lanes x 2 FLOP at the top SM clock (guide's unit counts)
        peak = 148 * 128 * 2 * 1.965e9 / 1e12
    feat_w = cfg.c_f or cfg.mlp.n_feat                  # Eq.7 slot features or the widened head
    out_bytes = H * W * (16 + 4 * feat_w)
    frame_floor_ms = max(flops_view / (peak * 1e12), out_bytes / (peaks["hbm_gbs"] * 1e9)) * 1e3
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16" if cfg.mlp.bf16 else "f32", "data": "synthetic",
        "config": {"workload": workload_desc(cfg), "parallelism": f"replicas x{world}, no collective",
                   "l2": ("inputs larger than L2 (weights %.0f MB, per-view staging %.1f GB)" if
                          sc.weights.nbytes / 2 + n_samples_view * 16 > 126e6 else
                          "working set below L2 (weights %.1f MB, per-view staging %.3f GB): no flush, config is launch-bound")
                         % (sc.weights.nbytes / 2 / 1e6, n_samples_view * 16 / 1e9),
                   "tile": args.tile or cfg.tile, "t_stop": cfg.t_stop,
                   "order": "tile-centre shared order (P:109)" if args.tile_order else "exact per-ray order"},
        "samples_per_s": world * n_samples_view * V / (ms_step * 1e-3),
        "counts_per_view": {"pairs": st.n_pairs, "intervals": st.n_intervals, "samples": st.n_samples,
                            "row_blocks": st.n_blocks, "scratch_GB": st.scratch_bytes / 1e9,
                            "samples_evaluated": st.n_samples_evaluated, "bands": st.n_bands, "waves": st.n_waves,
                            "staging_MB": st.staging_bytes / 1e6},
        "stage_ms_per_view": {k: v / max(1, n_views_timed) for k, v in stage_sum.items()},
        "clocks": clocks,
        "e2e": {"value": world * px_step / (e2e_ms * 1e-3) / 1e6, "unit": UNIT,
                "h2d_bytes_per_step": 64 * V, "d2h_bytes_per_step": out_bytes * V, "ms_per_step": e2e_ms,
                "note": "ms_render_host: camera in (kernel parameters), rgb/alpha(/feat) copied to pinned host memory"},
        "gpu_launches": launches,
        "roofline": {"bound": "tensor" if cfg.mlp.bf16 else "alu",
                     "kernel": "mlp_tc_kernel (stage d)" if cfg.mlp.bf16 else "mlp_f32_kernel (stage d, fp32 SIMT path)", "achieved": achieved, "peak": peak,
                     "unit": "TFLOP/s", "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get(cfg.name),
                     "traffic_unit": "bytes per launch (ncu dram read + write, profiles/r1c_summary.md)",
                     "algorithmic_bytes": n_samples_view * 16 + st.n_intervals * 32,
                     "peak_kind": (f"bf16 dense, sustained, of {peaks['source']}" if cfg.mlp.bf16 else
                                   "fp32 FMA, 148 SMs x 128 lanes x 2 x 1.965 GHz (derived)"),
                     "frac_of_burst_peak": achieved / peaks["bf16_tflops"] if cfg.mlp.bf16 else None,
                     "algorithmic_flop_per_sample": cfg.mlp.flop_per_sample,
                     "kernel_ms": mlp_ms, "kernel_share_of_step": mlp_ms * V / ms_step},
        "frame_roofline": {"floor_ms_per_view": frame_floor_ms, "frac": frame_floor_ms * V / ms_step,
                           "note": "slower of MLP FLOPs at the bf16 peak and output bytes at the HBM peak, over the whole step"},
    }
    comp_ms = stage_sum["composite"] / max(1, n_views_timed)
    if cfg.c_f and comp_ms > mlp_ms:
        # Eq.7 slot features: stage (e) dominates and is memory-bound.  Algorithmic bytes per view: staging,
        # gates and hit records once per hit (16 B each), the embeddings once, the outputs once.
        alg = st.n_intervals * 48 + sc.slots.nbytes + out_bytes
        ach = alg / (comp_ms * 1e-3) / 1e9
        line["roofline"] = {"bound": "hbm", "kernel": "composite_kernel<2> (stage e, slot features)", "achieved": ach,
                            "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"], "traffic": None,
                            "peak_kind": f"HBM copy bandwidth, of {peaks['source']}", "algorithmic_bytes": alg,
                            "kernel_ms": comp_ms, "kernel_share_of_step": comp_ms * V / ms_step,
                            "note": "the kernel re-reads each hit's four embedding rows (16 * c_f B per hit) through L1/L2; "
                                    "that traffic is not algorithmic"}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = {k: v for k, v in time_oracle(cfg, sc, cams, args.cpu_seconds).items()
                                if k in ("value", "unit", "cores", "kind", "sample", "samples_per_s")}
    print(json.dumps(line), flush=True)
    msdist.shutdown()


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
    ap.add_argument("--waves", type=int, default=0, help="depth waves (ms_opts.waves): 0 = auto, -1 = off, C > 0 = wave size")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                  # timing rule: W >= 3
    cfg = synth.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
