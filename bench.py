#!/usr/bin/env python
"""bench.py -- the realfast search hot path on B200: dedispersed images/s.

A "step" is one pass of the whole hot path (rf_search: dedisperse -> resample -> grid ->
2-D FFT image -> peak/sigma -> threshold over every DM trial x width x integration) over one
segment of synthetic VLA L-band visibilities (BASELINE.json:configs[1]).  Prints ONE JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config lband] [--impl ours|reference]

N > 1 (torchrun, one rank per GPU): the path shards by independent segments (PAPER.md:108,
"each segment is independent"), so every rank searches its own segment with no data-path
collective ("scaling": "weak").
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

import workloads as W  # noqa: E402

METRIC = "dedispersed images/s (grid+2D FFT+S/N)"
UNIT = "images/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self._stop, self.gpu = [], threading.Event(), gpu_index
        self._t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        try:
            p = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                  "--format=csv,noheader,nounits", "-lms", "100"],
                                 stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            return
        while not self._stop.is_set():
            line = p.stdout.readline()
            if not line:
                break
            self.rows.append([c.strip() for c in line.split(",")])
        p.terminate()

    def start(self):
        self._t.start()

    def stop(self):
        self._stop.set()
        self._t.join(timeout=2)
        sm = [int(r[0]) for r in self.rows if r and r[0].isdigit()]
        mx = [int(r[1]) for r in self.rows if len(r) > 1 and r[1].isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 6 for n, v in zip(names, r[2:6]) if v == "Active"})
        return {"sm_mhz": int(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def _setup(cfg, segment=0):
    f, uvw, dms = W.channel_freqs_hz(cfg), W.baseline_uvw_m(cfg), W.dm_list(cfg)
    return f, uvw, dms, W.default_cell_rad(cfg, uvw)


def _alg_bytes(cfg, plan):
    """A_img = 16 N_bl N_chan,w dt + 16 N_pix^2 per image, split per kernel kind
    (rf_plan_get_kernel_times): the visibility read belongs to the kernel that gathers (kind 3 `k_tree_gather` for every
    width of a plan on the boxcar-tree kernels, npix >= 256: the widths on the tree and, through their phase-decimated
    sums, the widths off it; kind 0 `k_grid_colfft` for npix < 256), the hand-off write (8 N^2) to the column FFT
    (kind 0), the hand-off read (8 N^2) to the row FFT + statistics (kind 1)."""
    c = plan.get_counters()
    images = plan.num_images()
    vis_bytes = 16.0 * c["vis_gridded"]                     # 16 B per (bl, ch) pol pair per native sample
    vis_tree = vis_bytes if cfg.npix >= 256 else 0.0
    hand = 8.0 * cfg.npix * cfg.npix * images
    return {"total": vis_bytes + 2 * hand, "kind": [vis_bytes - vis_tree + hand, hand, 0.0, vis_tree],
            "images": images, "images_device_counted": c["images"], "vis_gridded": c["vis_gridded"]}


FP32_LANES_PER_SM, N_SM = 128, 148          # B200: fp32 FMA peak = SMs x lanes x 2 flop x SM clock (B200_PROFILING.md)


def _fft_rate(cfg, plan, k_ms, sm_mhz):
    """Secondary evidence of SURVEY.md 8(d): FFT rate under the 5 N log2 N convention, counting only the transforms
    the kernels actually run (rf_plan_fft_work), per pass against the time of the kernel that holds it, and against
    the fp32 FMA peak at the SM clock seen during the run.  The 2-D FFT is the paper's dominant stage."""
    n_col, n_row = plan.fft_work()
    per = 5.0 * cfg.npix * np.log2(cfg.npix)
    peak = N_SM * FP32_LANES_PER_SM * 2 * (sm_mhz or 1965) * 1e6 / 1e12
    col = n_col * per / (k_ms[0] * 1e-3) / 1e12 if k_ms[0] > 0 else 0.0
    row = n_row * per / (k_ms[1] * 1e-3) / 1e12 if k_ms[1] > 0 else 0.0
    tot = (n_col + n_row) * per / ((k_ms[0] + k_ms[1]) * 1e-3) / 1e12 if k_ms[0] + k_ms[1] > 0 else 0.0
    return {"convention": "5 N log2 N per N-point complex transform actually run", "column_transforms": n_col,
            "row_pair_transforms": n_row, "flop_per_step": (n_col + n_row) * per, "column_pass_tflops": col,
            "row_pass_tflops": row, "both_passes_tflops": tot, "fp32_peak_tflops": peak, "frac_of_fp32_peak": tot / peak,
            "note": "the row-pass kernel also holds the statistics, the column-pass kernel the scatter and the hand-off store; "
                    "at npix >= 2048 the column pass is a pruned DFT over the occupied cells of each uv column "
                    "(k_tree_coldft), so its rate is the rate of the FFTs it replaces, not of operations executed"}


def _cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


KIND_NAMES = ["column FFT kernels (k_tree_colfft; k_grid_colfft on the per-image path)",
              "row FFT + statistics kernels (k_tree_rowfft_stats / k_rowfft_stats)",
              "Stokes-I transpose (k_stokes_transpose)",
              "gather + grid kernel (k_tree_gather)"]


def _roofline(alg, k_ms, k_n, ms_per_step, traffic=None):
    peak, peak_src = _peaks()
    dom = max((0, 1, 3), key=lambda k: k_ms[k])
    per_launch_bytes = alg["kind"][dom] / max(1, k_n[dom])
    per_launch_s = k_ms[dom] / max(1, k_n[dom]) * 1e-3
    achieved = per_launch_bytes / per_launch_s / 1e9
    path_gbs = alg["total"] / (ms_per_step * 1e-3) / 1e9
    names = ["pass1", "pass2", "prep", "gather"]
    out = {"bound": "hbm", "kernel": KIND_NAMES[dom], "achieved": achieved, "peak": peak, "unit": "GB/s",
           "frac": achieved / peak, "traffic": traffic[dom] if traffic else None, "peak_source": peak_src,
           "alg_bytes_per_launch": per_launch_bytes,
           "kernel_ms_per_step": {n: k_ms[i] for i, n in enumerate(names)},
           "kernel_launches_per_step": {n: k_n[i] for i, n in enumerate(names)},
           "kernel_alg_gbs": {n: (alg["kind"][i] / (k_ms[i] * 1e-3) / 1e9 if k_ms[i] > 0 else 0.0)
                              for i, n in enumerate(names)},
           "path": {"alg_bytes_per_step": alg["total"], "achieved": path_gbs, "frac": path_gbs / peak,
                    **_own_bytes(traffic, k_n, ms_per_step, peak)}}
    if traffic and traffic.get(dom) is not None:
        # the dominant kernel on the bytes it REALLY moves (ncu dram__bytes per launch / its live event time): the model
        # fraction above exceeds 1 because this design avoids most of the model's bytes
        own = traffic[dom] / per_launch_s / 1e9
        out["own_bytes"] = {"achieved": own, "frac_own": own / peak,
                            "note": "ncu DRAM bytes per launch / live CUDA-event time per launch / measured HBM peak"}
        out["frac_own"] = own / peak
        out["traffic_commit"] = traffic.get("commit")
        out["traffic_source"] = traffic.get("source")
    if traffic and traffic.get("limiters"):
        out["limiters_ncu"] = traffic["limiters"]     # what ncu says actually limits each kernel
    return out


def _own_bytes(traffic, k_n, ms_per_step, peak):
    """The bytes THIS design moves per step (a design that moves fewer bytes than the model reports
    its own count too): ncu DRAM bytes per launch of each tree kernel x its launches per step.  The fraction of the
    HBM peak they amount to says how far from HBM-bound the step is (the kernels are bound on chip)."""
    if not traffic or any(traffic.get(k) is None for k in (0, 1, 3)):
        return {}
    own = sum(traffic[k] * k_n[k] for k in (0, 1, 3))
    return {"dram_bytes_per_step_ncu": own, "dram_frac": own / (ms_per_step * 1e-3) / 1e9 / peak}


def _oracle_worker(args):
    (name, keys) = args
    import oracle as O
    cfg = W.get_config(name)
    f, uvw, dms, cell = _setup(cfg)
    vis = _oracle_worker.vis
    delays = O.delay_table(f, dms, cfg.inttime_s)
    wts = W.chan_weights(cfg) if cfg.n_flagged else None
    iu, iv, keep = O.cell_table(uvw, f, cfg.npix, cell, wts)
    n_w = int(keep.sum())
    out = 0
    for (d, k, j) in keys:
        s = O.dedisperse_resample(vis, delays[d], cfg.dt_list[k], j)
        img = O.image_from_grid(O.grid_visibilities(s, iu, iv, keep, cfg.npix), n_w)
        out += O.image_stats(img)[4] >= cfg.threshold
    return out


def oracle_throughput(cfg, vis, n_images_sample: int, seed: int = 11):
    """Time the float64 oracle as it stands on the host cores on a bounded uniform sample of the
    (dm, dt, j) images of the same segment.  Returns (images/s, cores, sample description)."""
    import multiprocessing as mp

    import oracle as O
    f, uvw, dms, cell = _setup(cfg)
    delays = O.delay_table(f, dms, cfg.inttime_s)
    rng = np.random.default_rng(seed)
    keys = []
    while len(keys) < n_images_sample:
        d, k = int(rng.integers(cfg.ndm)), int(rng.integers(len(cfg.dt_list)))
        nj = O.n_images(cfg.nint, int(delays[d].max()), cfg.dt_list[k])
        if nj:
            keys.append((d, k, int(rng.integers(nj))))
    cores = max(1, min(len(os.sched_getaffinity(0)), 32, n_images_sample // 4))
    os.environ.setdefault("OMP_NUM_THREADS", "1")
    _oracle_worker.vis = vis                     # inherited by fork, not pickled
    chunks = [keys[i::cores] for i in range(cores)]
    t0 = time.perf_counter()
    if cores == 1:
        _oracle_worker((cfg.name, chunks[0]))
    else:
        with mp.get_context("fork").Pool(cores) as pool:
            pool.map(_oracle_worker, [(cfg.name, c) for c in chunks])
    dt = time.perf_counter() - t0
    return n_images_sample / dt, cores, (f"{n_images_sample} images drawn uniformly over (dm, dt, j) of the same "
                                         f"segment, float64 numpy oracle, {cores} processes")


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vis = W.make_segment(cfg)
    vals = []
    cores, sample = 1, ""
    per_step = max(16, args.ref_images)
    for i in range(args.warmup + args.steps):
        v, cores, sample = oracle_throughput(cfg, vis, per_step, seed=100 + i)
        if i >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * per_step / value,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name}: BASELINE.json configs[{cfg.index}], oracle on a bounded sample "
                                   f"of {per_step} images per step"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def _ensure_built(local_rank: int) -> None:
    """A fresh checkout has no librealfast_b200.so (built artefacts are not in the history): local rank 0 compiles
    it (nvcc, sm_100a; a no-op when it is up to date), the other ranks wait for it."""
    from paper_1802_03084_b200 import build as _b
    if local_rank == 0:
        _b.build()
        return
    t0 = time.time()
    while _b.needs_build() and time.time() - t0 < 600:
        time.sleep(1.0)


class Ctx:
    """Process-wide CUDA / torch.distributed state of one bench.py run."""

    def __init__(self):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        if not torch.cuda.is_available():
            raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
        _ensure_built(self.local)
        torch.cuda.set_device(self.local)
        if self.world > 1:
            dist.init_process_group("nccl", device_id=torch.device("cuda", self.local))
        self.dev = torch.device("cuda", self.local)

    def close(self):
        if self.world > 1:
            self.dist.destroy_process_group()


def _traffic(cfg, args):
    """ncu DRAM bytes per launch of the three tree kernels in this launch configuration: numbers only a profiler run
    can provide, read from the committed capture (profiles/), which names the commit it was taken at."""
    tpath = os.path.join(ROOT, "profiles", f"r2_traffic_{cfg.name}.json.txt")
    if args.batch or args.tune or not os.path.exists(tpath):
        return None
    with open(tpath) as fh:
        tj = json.load(fh)
    return {0: tj.get("pass1_dram_bytes_per_launch"), 1: tj.get("pass2_dram_bytes_per_launch"),
            3: tj.get("gather_dram_bytes_per_launch"), "limiters": tj.get("limiters"), "commit": tj.get("commit"),
            "source": tj.get("source")}


def measure(args, cfg, ctx):
    """One config, device-resident and end to end; returns the JSON line as a dict on rank 0 (None elsewhere)."""
    import paper_1802_03084_b200 as R
    torch, dist, world, rank, local, dev = ctx.torch, ctx.dist, ctx.world, ctx.rank, ctx.local, ctx.dev

    f, uvw, dms, cell = _setup(cfg)
    # segment round-robin: rank r searches the r-th consecutive segment of the observation
    # (its own noise rows; same array, band and trial grid), no data-path collective
    import dataclasses
    vis = W.make_segment(dataclasses.replace(cfg, stride_int=cfg.nint), segment=rank) if world > 1 else W.make_segment(cfg)
    hvis = torch.from_numpy(vis).pin_memory()
    dvis = hvis.to(dev, non_blocking=True)
    plan = R.Plan(f, uvw, cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, cell, dms, cfg.dt_list, cfg.threshold)
    if cfg.n_flagged:
        plan.set_chan_weights(W.chan_weights(cfg))
    if args.batch:
        plan.set_batch(args.batch)
    if args.meansub:
        plan.set_meansub(True)
    for knob, val in args.tune:
        plan.set_tuning(knob, val)
    capacity = 1 << 17
    stream = torch.cuda.current_stream(dev)
    items = torch.empty(capacity * 32, dtype=torch.uint8, device=dev)
    count = torch.zeros(1, dtype=torch.int32, device=dev)

    def step():
        plan.search_raw(dvis.data_ptr(), stream.cuda_stream, items.data_ptr(), capacity, count.data_ptr())

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()

    for _ in range(args.warmup):
        step()
    barrier()

    # ---- device-resident timing (value); per-kernel events on for the roofline object
    plan.set_profiling(True)
    sampler = ClockSampler(local)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    barrier()
    total_ms = e0.elapsed_time(e1)
    ms, n = plan.get_kernel_times()                        # last step's kernels (all steps are identical)
    k_ms, k_n = ms, n
    clocks = sampler.stop()
    plan.set_profiling(False)
    launches = plan.get_counters()["kernel_launches"]
    n_cands = int(count.item())
    alg = _alg_bytes(cfg, plan)                            # counters of the timed searches (device-counted images)

    # ---- end to end through the C-ABI with HOST buffers (pinned input, host candidate array)
    cand_host = np.empty(capacity, dtype=R.CAND_DTYPE)
    plan.search_host(hvis, cand_host, capacity)            # warm: allocates the staging buffers
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _, n_e2e = plan.search_host(hvis, cand_host, capacity)
    torch.cuda.synchronize(dev)
    e2e_ms = (time.perf_counter() - t0) * 1e3

    # ---- optional: the periodicity search of the same segment, device-resident
    periodic = None
    if args.periodic:
        def pstep():
            plan.search_periodic_raw(dvis.data_ptr(), stream.cuda_stream, items.data_ptr(), capacity, count.data_ptr())
        pstep()
        barrier()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        p0.record(stream)
        for _ in range(args.steps):
            pstep()
        p1.record(stream)
        barrier()
        p_ms = p0.elapsed_time(p1) / args.steps
        n_freq = sum(plan.periodic_nt(d) // 2 for d in range(cfg.ndm))
        periodic = {"ms_per_step": p_ms, "frequency_images_per_step": n_freq, "value": n_freq / (p_ms * 1e-3),
                    "unit": "frequency images/s", "candidates": int(count.item()),
                    "gpu_launches": int(plan.get_counters()["kernel_launches"])}

    t_all = torch.tensor([total_ms, e2e_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(t_all, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms = float(t_all[0]), float(t_all[1])

    images = alg["images"]
    if alg["images_device_counted"] != images:
        raise SystemExit(f"the kernels finalised {alg['images_device_counted']} images, the plan lists {images}")
    ms_per_step = total_ms / args.steps
    value = world * images / (ms_per_step * 1e-3)
    e2e_value = world * images / (e2e_ms / args.steps * 1e-3)

    line = None
    if rank == 0:
        label = (f"{cfg.name}: BASELINE.json configs[{cfg.index}] ({cfg.nant} antennas, {cfg.nchan} ch, {cfg.nint} x "
                 f"{cfg.inttime_s * 1e3:g} ms, {cfg.ndm} DM x dt {list(cfg.dt_list)}, npix {cfg.npix})")
        roof = _roofline(alg, k_ms, k_n, ms_per_step, _traffic(cfg, args))
        roof["fft"] = _fft_rate(cfg, plan, k_ms, clocks.get("sm_mhz"))
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": label,
                       "images_per_step": images, "images_counted_on_device": alg["images_device_counted"],
                       "gvis_per_s": world * alg["vis_gridded"] / (ms_per_step * 1e-3) / 1e9,
                       "input_mvis_per_s": world * cfg.nint * cfg.nbl * cfg.nchan * cfg.npol / (ms_per_step * 1e-3) / 1e6,
                       "l2_policy": f"input segment {vis.nbytes / 1e9:.2f} GB is larger than L2 (126 MB); no flush",
                       "candidates": n_cands, "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                       "prep": "mean-visibility subtraction fused into the readers" if args.meansub else "none"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(vis.nbytes),
                    "d2h_bytes_per_step": int(4 + min(n_e2e, capacity) * 32)},
            "gpu_launches": int(launches) * args.steps,
            "roofline": roof,
        }
        if periodic is not None:
            line["periodic"] = periodic
        if world == 1 and not args.no_cpu_baseline:
            v, cores, sample = oracle_throughput(cfg, vis, args.ref_images)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "cpu": _cpu_model()}
    plan.destroy()
    del dvis, hvis, items, count
    torch.cuda.empty_cache()
    return line


def _stream_host_rows(cfg, nseg, torch):
    """Pinned host copy of the new integrations of every segment: segment 0 in full, then the
    cfg.stride_int integrations each later segment adds (rows [overlap, nint) of that segment)."""
    from concurrent.futures import ThreadPoolExecutor
    overlap = cfg.nint - cfg.stride_int
    row_shape = (cfg.nbl, cfg.nchan, cfg.npol)
    first = torch.empty((cfg.nint,) + row_shape, dtype=torch.complex64).pin_memory()
    new = torch.empty((max(1, nseg - 1), cfg.stride_int) + row_shape, dtype=torch.complex64).pin_memory()
    jobs = [(0, lo, min(lo + 64, cfg.nint), first.numpy()[lo:min(lo + 64, cfg.nint)]) for lo in range(0, cfg.nint, 64)]
    for s in range(1, nseg):
        for lo in range(overlap, cfg.nint, 80):
            hi = min(lo + 80, cfg.nint)
            jobs.append((s, lo, hi, new.numpy()[s - 1, lo - overlap:hi - overlap]))
    with ThreadPoolExecutor(max(1, min(32, len(os.sched_getaffinity(0))))) as ex:
        list(ex.map(lambda j: W.make_segment(cfg, j[0], rows=(j[1], j[2]), out=j[3]), jobs))
    return first, new


def run_stream(args, cfg):
    """BASELINE.json configs[4]: consecutive overlapping segments.  Each segment keeps the last
    `overlap` integrations of the previous one on the device (device-to-device copy) and uploads only
    its cfg.stride_int new integrations from pinned host memory on a side stream while the previous
    segment is searched; uvw (hour angle) changes per segment, so two plans are used alternately and
    the tables of the next segment are rebuilt on the host while the GPU searches the current one."""
    import torch

    import paper_1802_03084_b200 as R
    from workloads.generate import segment_ha_hours

    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        raise SystemExit("--config stream is a single-GPU measurement (replicas: run one per GPU)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    nseg_cfg = cfg.n_segments
    n_warm, n_timed = args.warmup, args.steps
    n_total = n_warm + n_timed
    f, dms = W.channel_freqs_hz(cfg), W.dm_list(cfg)
    geo = []
    for s in range(nseg_cfg):
        uvw = W.baseline_uvw_m(cfg, segment_ha_hours(cfg, s))
        geo.append((uvw, W.default_cell_rad(cfg, uvw)))
    first, new = _stream_host_rows(cfg, min(n_total, nseg_cfg), torch)
    overlap = cfg.nint - cfg.stride_int

    main, side = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    capacity = 1 << 19 if cfg.name == "stream1ms" else 1 << 17
    plans, bufs, items, counts, h_items, h_counts = [], [], [], [], [], []
    for b in range(2):
        pl = R.Plan(f, geo[0][0], cfg.npol, cfg.nint, cfg.inttime_s, cfg.npix, geo[0][1], dms, cfg.dt_list, cfg.threshold)
        pl.set_search_span(cfg.stride_int)
        plans.append(pl)
        bufs.append(torch.empty((cfg.nint, cfg.nbl, cfg.nchan, cfg.npol), dtype=torch.complex64, device=dev))
        items.append(torch.empty(capacity * 32, dtype=torch.uint8, device=dev))
        counts.append(torch.zeros(1, dtype=torch.int32, device=dev))
        h_items.append(torch.empty(capacity * 32, dtype=torch.uint8).pin_memory())
        h_counts.append(torch.zeros(1, dtype=torch.int32).pin_memory())
    images = plans[0].num_images()
    staged = [torch.cuda.Event() for _ in range(2)]
    searched = [torch.cuda.Event() for _ in range(2)]
    for e in searched:
        e.record(main)

    def stage(k):
        """Enqueue, on the side stream, everything that fills the device buffer of the k-th segment."""
        b, s = k % 2, k % nseg_cfg
        side.wait_event(searched[b])                       # the search that last read this buffer
        with torch.cuda.stream(side):
            if s == 0:
                bufs[b].copy_(first, non_blocking=True)
            else:
                side.wait_event(staged[1 - b])
                bufs[b][:overlap].copy_(bufs[1 - b][cfg.stride_int:], non_blocking=True)
                bufs[b][overlap:].copy_(new[s - 1], non_blocking=True)
            staged[b].record(side)

    def search(k):
        b, s = k % 2, k % nseg_cfg
        searched[b].synchronize()                          # plan b is idle: its tables may be rebuilt
        if k >= 2:
            found[0] += min(int(h_counts[b][0]), capacity)   # the host reads the result of segment k - 2
        plans[b].set_uvw(*geo[s])
        main.wait_event(staged[b])
        plans[b].search_raw(bufs[b].data_ptr(), main.cuda_stream, items[b].data_ptr(), capacity, counts[b].data_ptr())
        with torch.cuda.stream(main):
            h_counts[b].copy_(counts[b], non_blocking=True)
            h_items[b].copy_(items[b], non_blocking=True)
        searched[b].record(main)

    sampler, found = None, [0]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = 0.0
    stage(0)
    for k in range(n_total):
        if k == n_warm:
            torch.cuda.synchronize(dev)
            sampler = ClockSampler(0)
            sampler.start()
            t0 = time.perf_counter()
            e0.record(main)
        search(k)
        # staged AFTER the table rebuild of search(k): the upload of segment k + 1 waits (on the device)
        # for search k - 1, and copies queued behind a waiting copy would stall the rebuild's own uploads
        if k + 1 < n_total:
            stage(k + 1)
    e1.record(main)
    torch.cuda.synchronize(dev)
    wall_ms = (time.perf_counter() - t0) * 1e3
    dev_ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    n_last = int(h_counts[(n_total - 1) % 2].item())

    # per-kernel times of one more search of the last segment (profiling events on)
    b = (n_total - 1) % 2
    plans[b].set_profiling(True)
    plans[b].search_raw(bufs[b].data_ptr(), main.cuda_stream, items[b].data_ptr(), capacity, counts[b].data_ptr())
    main.synchronize()
    k_ms, k_n = plans[b].get_kernel_times()
    launches = plans[b].get_counters()["kernel_launches"]
    alg = _alg_bytes(cfg, plans[b])
    if alg["images_device_counted"] != images:
        raise SystemExit(f"the kernels finalised {alg['images_device_counted']} images, the plan lists {images}")
    ms_per_step = dev_ms / n_timed
    data_s = cfg.stride_int * cfg.inttime_s
    new_bytes = cfg.stride_int * cfg.nbl * cfg.nchan * cfg.npol * 8
    if cfg.name == "stream1ms":
        label = (f"stream1ms: the paper's GOAL workload (PAPER.md:94, Table 1 row L, PAPER.md:180: 1 ms sampling, 1.4 GB/s) on "
                 f"the BASELINE.json configs[4] array and trial grid ({cfg.nant} antennas, {cfg.nchan} ch, segments of {cfg.nint} x 1 ms "
                 f"with stride {cfg.stride_int} = 2.0 s, overlap = the DM 1000 sweep, {cfg.ndm} DM x dt {list(cfg.dt_list)}, npix "
                 f"{cfg.npix}); a step = one segment, pipelined")
    else:
        label = (f"stream: BASELINE.json configs[4] ({cfg.nant} antennas, {cfg.nchan} ch, segments of {cfg.nint} x "
                 f"{cfg.inttime_s * 1e3:g} ms with stride {cfg.stride_int}, {cfg.ndm} DM x dt {list(cfg.dt_list)}, npix {cfg.npix}); "
                 f"a step = one segment, pipelined")
    roof = _roofline(alg, k_ms, k_n, ms_per_step)
    roof["fft"] = _fft_rate(cfg, plans[b], k_ms, clocks.get("sm_mhz"))
    line = {
        "metric": METRIC, "value": images / (ms_per_step * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": n_timed,
        "warmup": n_warm, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": label,
                   "images_per_step": images, "images_counted_on_device": alg["images_device_counted"],
                   "realtime_factor": data_s / (ms_per_step * 1e-3),
                   "realtime_factor_wall": data_s * n_timed / (wall_ms * 1e-3),
                   "data_seconds_per_step": data_s, "input_rate_gbs": new_bytes / data_s / 1e9,
                   "h2d_gbs_sustained": new_bytes * n_timed / (wall_ms * 1e-3) / 1e9,
                   "candidates_last_segment": n_last, "candidates_read_on_host": found[0],
                   "gvis_per_s": alg["vis_gridded"] / (ms_per_step * 1e-3) / 1e9,
                   "l2_policy": f"each segment's {bufs[0].numel() * 8 / 1e9:.2f} GB buffer is larger than L2 (126 MB); no flush",
                   "overlap": "H2D of the next segment's new integrations on a side stream; table rebuild on the host",
                   "parallelism": "single GPU; on more GPUs the split is by segment (replicas, PAPER.md:108), unmeasured on hardware"},
        "clocks": clocks,
        "e2e": {"value": images * n_timed / (wall_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(new_bytes),
                "d2h_bytes_per_step": int(4 + capacity * 32)},
        "gpu_launches": int(launches) * n_timed,
        "roofline": roof,
    }
    for pl in plans:
        pl.destroy()
    del bufs, items, counts, first, new
    torch.cuda.empty_cache()
    return line


def _brief(line):
    """The part of another config's line that the default run carries as a sub-object."""
    keep = ("value", "unit", "steps", "warmup", "ms_per_step", "clocks", "gpu_launches")
    out = {k: line[k] for k in keep if k in line}
    out["config"] = line["config"]
    out["e2e"] = line["e2e"]
    r = line["roofline"]
    out["roofline"] = {"kernel_ms_per_step": r["kernel_ms_per_step"], "path_frac": r["path"]["frac"],
                       "fft_both_passes_tflops": r["fft"]["both_passes_tflops"],
                       "fft_frac_of_fp32_peak": r["fft"]["frac_of_fp32_peak"]}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed steps (default 5; 32 segments for --config stream)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default=None, choices=sorted(W.CONFIGS),
                    help="default: lband (BASELINE.json configs[1]) plus hi-res and streaming as sub-objects")
    ap.add_argument("--no-extra", action="store_true", help="default run without the hi-res / streaming sub-objects")
    ap.add_argument("--batch", type=int, default=0, help="images per batch (0 = library default)")
    ap.add_argument("--ref-images", type=int, default=512, help="oracle sample size per timing")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--periodic", action="store_true", help="also time rf_search_periodic (8f-3) on the same segment")
    ap.add_argument("--meansub", action="store_true", help="also run the prep stage (mean-visibility subtraction, 8f-1)")
    ap.add_argument("--tune", action="append", default=[], metavar="KNOB=VALUE",
                    help="rf_plan_set_tuning(knob, value) before the run (experiments; results do not change)")
    args = ap.parse_args()
    args.tune = [tuple(int(x) for x in t.split("=")) for t in args.tune]
    default_run = args.config is None
    cfg = W.get_config(args.config or "lband")
    if args.steps is None:
        args.steps = cfg.n_segments if cfg.n_segments > 1 else 5
    if args.impl == "reference":
        run_reference(args, cfg)
        return
    ctx = Ctx()
    if cfg.n_segments > 1:
        line = run_stream(args, cfg)
    else:
        line = measure(args, cfg, ctx)
    if default_run and ctx.world == 1 and line is not None and not args.no_extra:
        # the other BASELINE.json configs the metric names, as sub-objects with their own clocks: hi-res (configs[3])
        # and the streaming real-time factor (configs[4]).  S-band (configs[2]) is left to `--config sband`: its
        # 11.8 GB segment takes minutes to generate on the host.
        import copy
        extra = {}
        a = copy.copy(args)
        a.steps, a.warmup, a.no_cpu_baseline, a.periodic = 3, 3, True, False
        extra["hires"] = _brief(measure(a, W.get_config("hires"), ctx))
        a = copy.copy(args)
        a.steps, a.warmup = W.get_config("stream").n_segments, 3
        extra["stream"] = _brief(run_stream(a, W.get_config("stream")))
        line["other_configs"] = extra
    if line is not None:
        print(json.dumps(line), flush=True)
    ctx.close()


if __name__ == "__main__":
    main()
