#!/usr/bin/env python
"""bench.py -- TPC clusters/s tracked (CA find + KF fit) on seeded synthetic time frames.

One "step" = one pass of the whole hot path (a)-(g) over one time frame (BASELINE.json config 5:
50 overlapped collisions, 1 ms frame).  `value` is device-resident throughput, `e2e` goes through
tpcca_track_host with pinned host buffers (H2D + D2H inside the timed region).
"Measurement".  `--impl reference` times the CPU oracle (the only reference this tier has).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "tpc_clusters_per_sec_tracked"
UNIT = "clusters/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback

# what each step must move once (reuse through caches is free)
BYTES_PER_CLUSTER_NEIGHBOURS = 24.0      # 8 own yz + 8 links out + ~8 bin_start/neighbour share
BYTES_PER_ROW_STEP_TRACKLETS = 22.0      # 8 bin range + ~1.2*8 candidates + 4 row_hit
BYTES_PER_TRACKLET = 112.0               # record
BYTES_PER_TRACKLET_HIT = 8.0             # weight atomic
FP32_OPS_PER_ROW_STEP = 270.0            # transport 48 + covariance 102 + update 102 + search ~18


def ncu_traffic(stage: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the stage's kernels, from the committed ncu
    --set full summary of this round (profiles/traffic.json.txt), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.json.txt")
    try:
        return float(json.load(open(p))[stage])
    except Exception:
        return None


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clocks and throttle reasons during the timed region (NVML; nvidia-smi as a fallback)."""

    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx, self.samples, self.reasons, self.max_mhz = gpu_index, [], set(), None
        self._stop = threading.Event()
        self._t = threading.Thread(target=self._run, daemon=True)
        self._nvml = None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES", "")
            phys = int(vis.split(",")[gpu_index]) if vis and vis.split(",")[gpu_index].isdigit() else gpu_index
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM))
            self._nvml = pynvml
        except Exception:
            self._nvml = None

    def _sample_nvml(self):
        n = self._nvml
        self.samples.append(float(n.nvmlDeviceGetClockInfo(self._h, n.NVML_CLOCK_SM)))
        r = n.nvmlDeviceGetCurrentClocksEventReasons(self._h)
        for name, bit in (("hw_slowdown", n.nvmlClocksEventReasonHwSlowdown),
                          ("hw_thermal_slowdown", n.nvmlClocksEventReasonHwThermalSlowdown),
                          ("sw_thermal_slowdown", n.nvmlClocksEventReasonSwThermalSlowdown),
                          ("sw_power_cap", n.nvmlClocksEventReasonSwPowerCap)):
            if r & bit:
                self.reasons.add(name)

    def _sample_smi(self):
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.idx)],
                             capture_output=True, text=True, timeout=5).stdout.strip()
        f = [x.strip() for x in out.split(",")]
        self.samples.append(float(f[0]))
        self.max_mhz = float(f[1])
        for n, v in zip(self.NAMES, f[2:6]):
            if v.lower().startswith("active"):
                self.reasons.add(n)

    def _run(self):
        while not self._stop.is_set():
            try:
                if self._nvml is not None:
                    self._sample_nvml()
                else:
                    self._sample_smi()
            except Exception:
                pass
            self._stop.wait(0.004 if self._nvml is not None else 0.1)

    def start(self):
        self._t.start()

    def stop(self) -> dict:
        self._stop.set()
        self._t.join(timeout=10)
        return {"sm_mhz": float(np.median(self.samples)) if self.samples else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples),
                "source": "nvml" if self._nvml is not None else "nvidia-smi"}


def oracle_timed(scale: float, seed: int, steps: int, warmup: int, fr=None):
    """The CPU oracle as it stands on `fr`, or on a bounded sample of the workload (config 5 at `scale` collisions)."""
    import oracle
    from paper_1811_11481_b200 import synth
    if fr is None:
        fr = synth.generate(synth.config(5, scale=scale, seed=seed))
    rx = synth.row_x()
    times, res = [], None
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        res = oracle.track(fr.clusters, fr.sector_offsets, rx)
        if i >= warmup:
            times.append(time.perf_counter() - t0)
    t = float(np.mean(times))
    return fr.n / t, t, fr.n, res


def quality(assignment, n_tracks, fr):
    """Efficiency / clone / fake rate against the generator's truth, per (track, sector) segment."""
    from paper_1811_11481_b200 import score
    q = score.score(assignment, fr.truth, score.sector_of_cluster(fr.sector_offsets, fr.n), n_tracks)
    return {k: (round(v, 5) if isinstance(v, float) else v) for k, v in q.items()}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    scale = 0.2
    v, t, n, _ = oracle_timed(scale, 5, args.steps, args.warmup)
    sample = f"config 5 at {int(round(50 * scale))} collisions in {1000 * scale:.0f} us (same occupancy), {n} clusters/step"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config5_timeframe_50_collisions (bounded sample)", "clusters_per_step": n},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def run_gpu(args):
    import torch
    from paper_1811_11481_b200 import binding, distributed, synth
    from paper_1811_11481_b200 import build as tbuild
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the tpcca path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = distributed.init(world, rank, "nccl") if world > 1 else None
    if rank == 0:
        tbuild.build()
    if dist is not None:
        dist.barrier()
    # weak scaling: every rank tracks its own time frame (one time frame per GPU)
    fr = synth.generate(synth.config(5, seed=5 + 1000 * rank))
    rx = synth.row_x()
    n = fr.n
    extra = {k: float(v) for k, v in (kv.split("=") for kv in args.params.split(",") if kv)}
    trk = binding.Tracker(rx, n_sectors=36, max_clusters=n, max_tracklets=max(1 << 16, n // 8),
                          max_tracks=max(1 << 16, n // 24), device=f"cuda:{local}", **extra)
    dev_clusters = trk.upload(fr.clusters)
    stream = torch.cuda.current_stream()

    # ---- device-resident throughput
    for _ in range(args.warmup):
        trk.track(dev_clusters, n, fr.sector_offsets)
    torch.cuda.synchronize()
    hd = trk.header()
    if hd["status"] != 0:
        raise SystemExit(f"capacity overflow in warm-up: {hd}")
    trk.set_profiling(True)
    sampler = ClockSampler(local)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        trk.track(dev_clusters, n, fr.sector_offsets)
    e1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    ms_local = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else None
    stage = trk.stage_ms()
    trk.set_profiling(False)
    launches = trk.launch_count() * args.steps
    stats = trk.stats()
    hd = trk.header()
    ms_total, n_total = distributed.aggregate(dist, ms_local, n)
    ms_per_step = ms_total / args.steps
    value = n_total / (ms_per_step * 1e-3)

    # ---- end to end through tpcca_track_host (pinned host buffers, H2D + D2H inside the timed region)
    hc = torch.from_numpy(fr.clusters.view(np.uint8).reshape(-1)).pin_memory()
    ot = torch.empty(16 + 128 * trk.max_tracks, dtype=torch.uint8).pin_memory()
    oa = torch.empty(n, dtype=torch.int32).pin_memory()
    for _ in range(max(1, args.warmup // 2)):
        trk.track_host(hc, n, fr.sector_offsets, ot, oa)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(stream)
    for _ in range(args.steps):
        trk.track_host(hc, n, fr.sector_offsets, ot, oa)
    f1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    e2e_ms, _ = distributed.aggregate(dist, f0.elapsed_time(f1), n)
    e2e_serial = n_total / (e2e_ms / args.steps * 1e-3)
    nt = int(ot[:16].numpy().view(binding.HEADER_DTYPE)["n_tracks"][0])
    h2d, d2h = n * 16, 16 + n * 4 + nt * 128

    # ---- the same calls with several frames in flight: one handle, stream and host thread per frame in
    # flight, so that one frame's copies overlap another frame's kernels.  Every step still copies its own inputs and results.
    F = max(2, args.in_flight)
    lanes = [(trk, ot, oa, torch.cuda.Stream())]
    for _ in range(F - 1):
        lanes.append((binding.Tracker(rx, n_sectors=36, max_clusters=n, max_tracklets=trk.max_tracklets,
                                      max_tracks=trk.max_tracks, device=f"cuda:{local}", **extra),
                      torch.empty(16 + 128 * trk.max_tracks, dtype=torch.uint8).pin_memory(),
                      torch.empty(n, dtype=torch.int32).pin_memory(), torch.cuda.Stream()))
    steps2 = max(F, args.steps - args.steps % F)

    def worker(tr, o_t, o_a, st, k, ev):
        torch.cuda.set_device(local)
        with torch.cuda.stream(st):
            if ev is not None:
                st.wait_event(ev)
            for _ in range(k):
                tr.track_host(hc, n, fr.sector_offsets, o_t, o_a)

    def run_pipelined(k, ev):
        ths = [threading.Thread(target=worker, args=(tr, o_t, o_a, st, k, ev)) for tr, o_t, o_a, st in lanes]
        for th in ths:
            th.start()
        for th in ths:
            th.join()

    run_pipelined(1, None)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(stream)
    run_pipelined(steps2 // F, g0)
    for _, _, _, st in lanes:
        stream.wait_stream(st)
    g1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    pipe_ms, _ = distributed.aggregate(dist, g0.elapsed_time(g1), n)
    e2e_value = n_total / (pipe_ms / steps2 * 1e-3)
    for _, _, o_a, _ in lanes[1:]:
        assert np.array_equal(o_a.numpy(), oa.numpy()), "the in-flight handles disagree"
    del lanes[1:]

    if rank != 0:
        return 0
    gpu_assignment = oa.numpy().copy()
    gpu_quality = quality(gpu_assignment, nt, fr)
    # ---- roofline of the dominant kernel (per-stage CUDA events recorded inside the timed loop)
    peak, peak_src = peaks()
    dom = max(stage, key=stage.get)
    alg = {
        "neighbours": BYTES_PER_CLUSTER_NEIGHBOURS * n,
        "tracklets": BYTES_PER_ROW_STEP_TRACKLETS * stats["row_steps"] + BYTES_PER_TRACKLET * hd["n_start_hits"]
        + BYTES_PER_TRACKLET_HIT * stats["track_hits"],
        "grid": 36.0 * n + 12.0 * stats["n_bins"],
        "clean_start": 32.0 * n,
        "select": 12.0 * stats["track_hits"] + 12.0 * n,
        "refit": 12.0 * 3 * stats["track_hits"] + 128.0 * hd["n_tracks"],
    }
    per_stage = {k: {"ms": stage[k], "alg_GBps": alg[k] / (stage[k] * 1e-3) / 1e9 if stage[k] > 0 else None,
                     "frac": alg[k] / (stage[k] * 1e-3) / 1e9 / peak if stage[k] > 0 else None} for k in stage}
    ach = alg[dom] / (stage[dom] * 1e-3) / 1e9
    # the Kalman stages are fp32-issue bound: useful fp32 operations of the section-3
    # arithmetic per row step against 148 SM x 128 lanes x SM clock (no FMA: one operation per lane and clock)
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    alu_peak = 148 * 128 * sm_mhz * 1e6 / 1e9
    alu_ops = FP32_OPS_PER_ROW_STEP * (stats["row_steps"] + 3 * stats["track_hits"])
    alu_ms = stage["tracklets"] + stage["refit"]
    alu = {"achieved": alu_ops / (alu_ms * 1e-3) / 1e9, "peak": alu_peak, "unit": "Gop/s",
           "frac": alu_ops / (alu_ms * 1e-3) / 1e9 / alu_peak, "kernels": "tracklets+refit",
           "ops_per_row_step": FP32_OPS_PER_ROW_STEP}
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": ncu_traffic(dom), "peak_source": peak_src, "algorithmic_bytes": alg[dom],
                "kernel_ms": stage[dom], "stages": per_stage, "alu": alu}
    # ---- CPU baseline: the oracle as it stands, one pass over the same frame (rank 0, N = 1 only)
    cpu_baseline = None
    if world == 1:
        cv, ct, cn, ores = oracle_timed(1.0, 5, 1, 0, fr=fr)
        cpu_baseline = {"value": cv, "unit": UNIT, "cores": 1, "kind": "oracle",
                        "sample": f"one pass over the same config-5 frame, {cn} clusters, {ct:.1f} s",
                        "quality": quality(ores.assignment, len(ores.tracks), fr),
                        "assignment_equals_cuda_path": bool(np.array_equal(ores.assignment, gpu_assignment))}
    try:
        baseline_metric = json.load(open(os.path.join(ROOT, "BASELINE.json")))["metric"]
    except Exception:
        baseline_metric = None
    line = {"metric": METRIC, "baseline_metric": baseline_metric, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "config5_timeframe_50_collisions", "clusters_per_frame": n,
                       "frames_per_step": world, "ms_per_time_frame": ms_per_step, "n_tracks": hd["n_tracks"],
                       "n_start_hits": hd["n_start_hits"], "row_steps": stats["row_steps"],
                       "quality": gpu_quality,
                       "l2": "inputs larger than L2 (cluster array %.0f MB, working set > 1 GB)" % (n * 16 / 1e6),
                       "parallelism": f"frames x{world} (no collective)"},
            "clocks": clocks, "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": pipe_ms / steps2, "steps": steps2, "frames_in_flight": F,
                    "one_in_flight": {"value": e2e_serial, "ms_per_step": e2e_ms / args.steps}},
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tpcca", choices=["tpcca", "reference"])
    ap.add_argument("--in-flight", type=int, default=3, help="frames in flight of the pipelined end-to-end leg")
    ap.add_argument("--params", default="", help="k=v,k=v overrides of tpcca_params (tuning experiments)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "tpcca" else args.warmup
    return run_reference(args) if args.impl == "reference" else run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
