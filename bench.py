#!/usr/bin/env python
"""bench.py -- TPC clusters/s tracked (CA find + KF fit) on seeded synthetic time frames.

One "step" = one pass of the whole hot path (a)-(g) over one time frame (BASELINE.json config 5:
50 overlapped collisions, 1 ms frame).  `value` is device-resident throughput, `e2e` goes through the
library's pipelined host call (tpcca_track_host_async / tpcca_wait: pinned host buffers, H2D + D2H inside
the timed region, two frames in flight in ONE workspace).  `--gpus N` starts N ranks itself (torchrun
re-exec) unless it already runs under torchrun; `--shard frames` (default, weak scaling: one frame per
rank) or `--shard sectors` (one frame split into contiguous sector ranges, strong
scaling; tpcca_merge and the leg calls then run per rank WITHOUT an exchange of boundary segments, so for N > 2 the
tracks crossing a rank boundary stay unmerged -- `config.merge.cuts_inside_a_side` counts those boundaries).  `--config k` times another BASELINE.json config (parity-test cases; the bench line is config 5).
See DESIGN.md "Measurement".  `--impl reference` times the CPU oracle (the only reference this tier has).
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
BYTES_PER_TRACKLET_HIT = 8.0             # weight atomic (every hit of every valid tracklet)
FP32_OPS_PER_ROW_STEP = 161.0            # DESIGN.md section 3 with the stated fma: transport 38 + covariance 51 + update 54 + search ~18


def ncu_traffic(stage: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel (or of a stage's kernels), from the committed
    ncu --set full summary of this round (profiles/traffic.json.txt), or None."""
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


def host_cpu() -> dict:
    """CPU model and core count of the box the oracle is timed on; the oracle itself is single-threaded."""
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    try:
        usable = len(os.sched_getaffinity(0))
    except AttributeError:
        usable = os.cpu_count() or 0
    return {"cpu_model": model, "host_cores": os.cpu_count() or 0, "host_cores_usable": usable}


def oracle_timed(cfg: int, scale: float, seed: int, steps: int, warmup: int, fr=None):
    """The CPU oracle as it stands on `fr`, or on a bounded sample of the workload (config `cfg` at `scale`)."""
    import oracle
    from paper_1811_11481_b200 import synth
    if fr is None:
        fr = synth.generate(synth.config(cfg, scale=scale, seed=seed))
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


WORKLOADS = {1: "config1_single_sector_200_primaries", 2: "config2_central_event_4000_primaries",
             3: "config3_low_pt_loopers", 4: "config4_5_collisions_100us", 5: "config5_timeframe_50_collisions"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    # bounded sample of the SAME workload: config 5 at 10 collisions in 200 us has the occupancy of the full frame
    scale = 0.2 if args.config == 5 else (0.25 if args.config == 4 else 1.0)
    v, t, n, _ = oracle_timed(args.config, scale, args.config, args.steps, args.warmup)
    sample = (f"config {args.config} at scale {scale} "
              + ("(10 collisions in 200 us: the occupancy of the full frame), " if args.config == 5 else "")
              + f"{n} clusters/step")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config] + " (bounded sample)", "clusters_per_step": n,
                       "sample_scale": scale,
                       "note": ("a bounded sample of the workload, not the full frame the CUDA arm times: the ratio of the two "
                                "arms compares clusters/s across different frame sizes" if scale != 1.0 else
                                "the same frame the CUDA arm times")},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample, **host_cpu()},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


def respawn_under_torchrun(args) -> int:
    """`python bench.py --gpus N` with N > 1 outside torchrun: start the N ranks (one process per GPU)."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_gpu(args):
    import torch
    from paper_1811_11481_b200 import binding, distributed, synth
    from paper_1811_11481_b200 import build as tbuild
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the tpcca path has no CPU fallback")
    if world > 1 and torch.cuda.device_count() < world:
        raise SystemExit(f"{world} ranks need {world} GPUs, {torch.cuda.device_count()} visible")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")       # the communicator log (nranks) stays readable
        os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
    dist = distributed.init(world, rank, "nccl") if world > 1 else None
    if rank == 0:
        tbuild.build()
    if dist is not None:
        dist.barrier()
    cfg = args.config
    rx = synth.row_x()
    if args.shard == "sectors" and world > 1:
        # strong scaling: ONE frame, rank r tracks sectors shard_sectors(36, world, r)
        whole = synth.generate(synth.config(cfg, seed=cfg))
        cl, so, lo = distributed.shard_frame(whole.clusters, whole.sector_offsets, world, rank)
        fr = synth.Frame(np.ascontiguousarray(cl), so, whole.truth[lo:lo + len(cl)], whole.track_par, whole.n_sectors,
                         f"config{cfg}/shard{rank}")
        scaling, parallelism = "strong", f"sectors x{world} of one frame (no data-path collective)"
    else:
        # weak scaling: every rank tracks its own time frame (one time frame per GPU)
        fr = synth.generate(synth.config(cfg, seed=cfg + 1000 * rank))
        scaling, parallelism = "weak", f"frames x{world} (no collective)"
    n = fr.n
    extra = {k: float(v) for k, v in (kv.split("=") for kv in args.params.split(",") if kv)}
    trk = binding.Tracker(rx, n_sectors=fr.n_sectors, max_clusters=max(n, 1024), max_tracklets=max(1 << 16, n // 8),
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
    trk.set_profiling(1)
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
    trk.set_profiling(0)
    launches = trk.launch_count() * args.steps
    stats = trk.stats()
    hd = trk.header()
    ms_total, n_total = distributed.aggregate(dist, ms_local, n)
    ms_per_step = ms_total / args.steps
    value = n_total / (ms_per_step * 1e-3)
    # global track ids of a sector split: exclusive scan of the per-rank counts (one 8-byte all-gather, outside the timed loop)
    counts = distributed.gather_counts(dist, hd["n_tracks"])
    id_offset = int(distributed.track_id_offsets(counts)[rank])

    # ---- per-kernel device times (profiling level 2: two events around each main kernel), separate short pass
    trk.set_profiling(2)
    for _ in range(3):
        trk.track(dev_clusters, n, fr.sector_offsets)
    torch.cuda.synchronize()
    kms = trk.kernel_ms()
    trk.set_profiling(0)

    # ---- the step after the path: sector-segment merger + final fit (tpcca_merge), timed on its own
    trk.track(dev_clusters, n, fr.sector_offsets)
    trk.merge()
    torch.cuda.synchronize()
    m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m0.record(stream)
    for _ in range(args.steps):
        trk.merge()
    m1.record(stream)
    torch.cuda.synchronize()
    merge_ms = m0.elapsed_time(m1) / args.steps
    mh = trk.merged_header()
    track_merged = trk.track_merged()
    dev_assign = trk.assignment()
    # ---- looper legs and cluster tags on the merged tracks (tpcca_find_legs), timed on its own
    leg_partner, leg_partner_in, leg_first, tags, leg_sum = trk.find_legs()
    torch.cuda.synchronize()
    l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0.record(stream)
    for _ in range(args.steps):
        trk.find_legs_enqueue()
    l1.record(stream)
    torch.cuda.synchronize()
    legs_ms = l0.elapsed_time(l1) / args.steps
    # ---- one fit through both legs of every pair joined at a turning point (tpcca_fit_legs), timed on its own
    leg_fits, leg_fit_failed = trk.fit_legs()
    torch.cuda.synchronize()
    k0, k1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k0.record(stream)
    for _ in range(args.steps):
        trk.fit_legs_enqueue()
    k1.record(stream)
    torch.cuda.synchronize()
    leg_fit_ms = k0.elapsed_time(k1) / args.steps

    # ---- end to end through the library's host calls (pinned host buffers, H2D + D2H inside the timed region)
    hc = torch.from_numpy(fr.clusters.view(np.uint8).reshape(-1)).pin_memory()
    outs = [(torch.empty(16 + 128 * trk.max_tracks, dtype=torch.uint8).pin_memory(),
             torch.empty(max(n, 1), dtype=torch.int32).pin_memory()) for _ in range(2)]
    ot, oa = outs[0]
    for _ in range(max(1, args.warmup // 2)):
        trk.track_host(hc, n, fr.sector_offsets, ot, oa)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record(stream)
    for _ in range(args.steps):
        trk.track_host(hc, n, fr.sector_offsets, ot, oa)   # strictly serial: copy in, track, copy out, wait
    f1.record(stream)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    e2e_ms, _ = distributed.aggregate(dist, f0.elapsed_time(f1), n)
    e2e_serial = n_total / (e2e_ms / args.steps * 1e-3)
    nt = int(ot[:16].numpy().view(binding.HEADER_DTYPE)["n_tracks"][0])
    h2d, d2h = n * 16, 16 + n * 4 + nt * 128
    # pipelined: tpcca_track_host_async / tpcca_wait, two frames in flight on ONE handle and ONE workspace:
    # the upload of frame k+1 and the download of frame k-1 overlap the kernels of frame k.  Every step still copies its
    # own input and its own results.
    for i in range(2):
        trk.track_host_async(hc, n, fr.sector_offsets, *outs[i])
    trk.wait()
    trk.wait()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record(stream)
    trk.track_host_async(hc, n, fr.sector_offsets, *outs[0])
    for i in range(1, args.steps):
        trk.track_host_async(hc, n, fr.sector_offsets, *outs[i & 1])
        trk.wait()
    trk.wait()
    g1.record(stream)
    torch.cuda.synchronize()
    wall_ms = (time.perf_counter() - t0) * 1e3
    if dist is not None:
        dist.barrier()
    # the last wait returns after the last D2H on the internal copy streams: take the larger of the device span on the
    # caller's stream and the host wall clock around the loop
    pipe_ms, _ = distributed.aggregate(dist, max(g0.elapsed_time(g1), wall_ms), n)
    e2e_value = n_total / (pipe_ms / args.steps * 1e-3)
    assert np.array_equal(outs[0][1].numpy(), outs[1][1].numpy()), "the two staging slots disagree"

    if rank != 0:
        return 0
    gpu_assignment = outs[0][1].numpy()[:n].copy()
    gpu_quality = quality(gpu_assignment, nt, fr)
    # clone rate per PARTICLE before and after the merger (a particle crossing k sectors gives k sector tracks)
    from paper_1811_11481_b200 import score
    one = np.zeros(n, np.int32)
    q_sec = score.score(dev_assign, fr.truth, one, hd["n_tracks"])
    am = np.where(dev_assign >= 0, track_merged[np.maximum(dev_assign, 0)], -1) if hd["n_tracks"] else dev_assign
    q_mrg = score.score(am, fr.truth, one, mh["n_merged"])
    # a chain of legs counts as one reconstructed particle: relabel every leg by the root of its chain (union of both kinds of link)
    leg_root = np.arange(len(leg_partner))

    def _find(x):
        while leg_root[x] != x:
            leg_root[x] = leg_root[leg_root[x]]
            x = leg_root[x]
        return x

    for lp in (leg_partner, leg_partner_in):
        for m in np.flatnonzero(lp >= 0):
            leg_root[_find(m)] = _find(int(lp[m]))
    leg_root = np.array([_find(m) for m in range(len(leg_root))], dtype=np.int64)
    al = np.where(am >= 0, leg_root[np.maximum(am, 0)], -1) if len(leg_partner) else am
    q_leg = score.score(al, fr.truth, one, mh["n_merged"])
    merge_info = {"ms": merge_ms, "api": "tpcca_merge (after the timed path, not part of `value`)", **mh,
                  "cuts_inside_a_side": (distributed.cuts_inside_a_side(36, world, 18)
                                         if args.shard == "sectors" else 0),
                  "per_particle": {"sector_tracks": {k: round(float(v), 5) for k, v in q_sec.items()},
                                   "merged_tracks": {k: round(float(v), 5) for k, v in q_mrg.items()},
                                   "merged_tracks_legs_joined": {k: round(float(v), 5) for k, v in q_leg.items()}}}
    sigma_ratio = None
    if len(leg_fits):
        okf = leg_fits["pad"][:, 2] >= 0
        c_fit = leg_fits["cov"][:, 14][okf]
        c_leg = trk.merged()["cov"][:, 14][leg_fits["pad"][:, 0][okf]]
        good = (c_fit > 0) & (c_leg > 0)
        if good.any():
            sigma_ratio = round(float(np.median(np.sqrt(c_fit[good] / c_leg[good]))), 4)
    legs_info = {"ms": legs_ms, "api": "tpcca_find_legs (after tpcca_merge, not part of `value`)", **leg_sum,
                 "tagged_fraction_of_clusters": round(float((tags > 0).mean()), 5) if n else 0.0,
                 "pair_fit": {"ms": leg_fit_ms, "api": "tpcca_fit_legs", "pairs": int(len(leg_fits)), "failed": int(leg_fit_failed),
                              "median_sigma_qpt_ratio_to_first_leg": sigma_ratio}}
    # ---- roofline (algorithmic bytes of DESIGN.md section 7 x live device counters)
    peak, peak_src = peaks()
    T = hd["n_start_hits"]
    alg_stage = {
        "neighbours": BYTES_PER_CLUSTER_NEIGHBOURS * n,
        "tracklets": BYTES_PER_ROW_STEP_TRACKLETS * stats["row_steps"] + BYTES_PER_TRACKLET * T
        + BYTES_PER_TRACKLET_HIT * stats["tracklet_hits"],
        "grid": 36.0 * n + 12.0 * stats["n_bins"],
        "clean_start": 32.0 * n,
        "select": 12.0 * stats["tracklet_hits"] + 12.0 * n,
        "refit": 12.0 * stats["track_hits"] + 128.0 * hd["n_tracks"],  # the hits are moved once, three passes reuse them
    }
    alg_kernel = {
        "k_slice_scatter": 32.0 * n, "k_slice_sort": 30.0 * n + 4.0 * stats["n_bins"],
        "k_neighbours": alg_stage["neighbours"], "k_clean": 24.0 * n,
        "k_tl_e1": BYTES_PER_ROW_STEP_TRACKLETS * stats["steps_e1"],
        "k_tl_e2": BYTES_PER_ROW_STEP_TRACKLETS * stats["steps_e2"],
        "k_tl_e3a": BYTES_PER_ROW_STEP_TRACKLETS * stats["steps_e3a"],
        "k_tl_e3b": BYTES_PER_ROW_STEP_TRACKLETS * stats["steps_e3b"] + BYTES_PER_TRACKLET * T,
        "k_tracklet_weights": (4.0 + BYTES_PER_TRACKLET_HIT) * stats["tracklet_hits"],
        "k_select_own": 12.0 * stats["tracklet_hits"], "k_assign": 12.0 * n, "k_refit": alg_stage["refit"],
    }

    def rate(b, ms):
        return b / (ms * 1e-3) / 1e9 if ms and ms > 0 else None

    per_stage = {k: {"ms": stage[k], "alg_GBps": rate(alg_stage[k], stage[k]),
                     "frac": (rate(alg_stage[k], stage[k]) or 0.0) / peak} for k in stage}
    per_kernel = {k: {"ms": kms[k], "alg_GBps": rate(alg_kernel[k], kms[k]),
                      "frac": (rate(alg_kernel[k], kms[k]) or 0.0) / peak} for k in kms}
    dom = max(kms, key=kms.get)
    # k_neighbours and k_refit are the only kernels of their stage (k_write_header aside): their time inside the timed
    # region is the stage time; any other kernel takes the per-kernel pass
    single = {"k_neighbours": "neighbours", "k_refit": "refit"}
    dom_ms = stage[single[dom]] if dom in single else kms[dom]
    dom_src = ("stage events inside the timed region (the stage is this one kernel)" if dom in single
               else "per-kernel events, separate pass after the timed region")
    ach = rate(alg_kernel[dom], dom_ms)
    # the Kalman kernels are issue bound: useful fp32 instructions of the section-3 arithmetic per
    # row step (an fma counts once) against 148 SM x 128 lanes x SM clock
    sm_mhz = (clocks or {}).get("sm_mhz") or 1965.0
    alu_peak = 148 * 128 * sm_mhz * 1e6 / 1e9
    alu_ops = FP32_OPS_PER_ROW_STEP * (stats["row_steps"] + 3 * stats["track_hits"])
    alu_ms = stage["tracklets"] + stage["refit"]
    alu = {"achieved": alu_ops / (alu_ms * 1e-3) / 1e9, "peak": alu_peak, "unit": "Ginstr/s",
           "frac": alu_ops / (alu_ms * 1e-3) / 1e9 / alu_peak, "kernels": "tracklets+refit",
           "instr_per_row_step": FP32_OPS_PER_ROW_STEP}
    whole = sum(alg_stage.values())
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": ncu_traffic(dom), "peak_source": peak_src, "algorithmic_bytes": alg_kernel[dom],
                "kernel_ms": dom_ms, "kernel_ms_source": dom_src, "stages": per_stage, "kernels": per_kernel,
                "whole_call": {"algorithmic_bytes": whole, "GBps": rate(whole, ms_local / args.steps),
                               "frac": rate(whole, ms_local / args.steps) / peak}, "alu": alu}
    # ---- CPU baseline: the oracle as it stands, one pass over the same frame (rank 0, N = 1 only)
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        cv, ct, cn, ores = oracle_timed(cfg, 1.0, cfg, 1, 0, fr=fr)
        cpu_baseline = {"value": cv, "unit": UNIT, "cores": 1, "kind": "oracle", **host_cpu(),
                        "sample": f"one pass over the same config-{cfg} frame, {cn} clusters, {ct:.1f} s",
                        "quality": quality(ores.assignment, len(ores.tracks), fr),
                        "assignment_equals_cuda_path": bool(np.array_equal(ores.assignment, gpu_assignment))}
    try:
        baseline_metric = json.load(open(os.path.join(ROOT, "BASELINE.json")))["metric"]
    except Exception:
        baseline_metric = None
    line = {"metric": METRIC, "baseline_metric": baseline_metric, "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": scaling,
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOADS[cfg], "clusters_per_frame": n, "clusters_per_step": n_total,
                       "frames_per_step": world if scaling == "weak" else 1, "ms_per_time_frame": ms_per_step,
                       "n_tracks": hd["n_tracks"], "n_tracks_all_ranks": int(counts.sum()), "track_id_offset": id_offset,
                       "n_start_hits": hd["n_start_hits"], "row_steps": stats["row_steps"], "quality": gpu_quality,
                       "l2": "inputs larger than L2 (cluster array %.0f MB, working set > 1 GB)" % (n * 16 / 1e6)
                       if n * 16 > 126e6 else "frame fits the 126 MB L2: a parity-test case, not the bench line",
                       "parallelism": parallelism, "shard": args.shard, "merge": merge_info, "legs": legs_info},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": pipe_ms / args.steps, "steps": args.steps, "frames_in_flight": 2, "handles": 1,
                    "workspaces": 1, "api": "tpcca_track_host_async + tpcca_wait",
                    "one_in_flight": {"value": e2e_serial, "ms_per_step": e2e_ms / args.steps, "api": "tpcca_track_host"}},
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu_baseline}
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="tpcca", choices=["tpcca", "reference"])
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json config (5 = the bench line; 1-4 are parity-test cases)")
    ap.add_argument("--shard", default="frames", choices=["frames", "sectors"],
                    help="N > 1: one frame per rank (weak) or one frame split by sector ranges (strong)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle leg (sweeps)")
    ap.add_argument("--params", default="", help="k=v,k=v overrides of tpcca_params (tuning experiments)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "tpcca" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "RANK" not in os.environ:
        return respawn_under_torchrun(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
