#!/usr/bin/env python
"""bench.py -- throughput of the fused calibrate + HEALPix-resample hot path on B200 (contract in the task).

    python bench.py --gpus N --steps K --warmup W [--impl reference] [--workload config1|...|coadd|batch|segments|detect]

A step = one pass of the whole hot path over one frame: per-frame plan on the device (A0/A1, the WCS is
treated as new every step: plan cache off) + fused calibrate/resample (A2-A5) writing value + weight.
Workload at N=1: BASELINE.json configs[1] (one full 9576x6388 IMX455 frame, nside 2^17, bilinear).
Under torchrun every rank processes its own frame (frames are independent: weak scaling, no collective
on the data path; only the barrier / max-time reduction use NCCL).

`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample of the same
workload; it is a deliberately slow program and a reported baseline, not the target.
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

METRIC = "calibrated+HEALPix-resampled Mpix/s per B200; achieved HBM GB/s vs peak"
UNIT = "Mpix/s"  # input (detector) pixels per second
SAMPLE_SIDE = {"bilinear": 4096, "lanczos3": 2048}  # --impl reference / 1-thread leg: SAMPLE_SIDE^2 frame of the workload recipe
N_DISTINCT = 3   # coadd / batch: distinct synthetic frames generated on the host (61 MPix each takes ~10 s); the other
                 # frames of the batch reuse their pixels with their OWN WCS (and, for batch, their own device copies)

# B200 unit counts for the shared-memory and FP32 rooflines (B200_PROFILING.md / B300_MICROARCH.md): 148 SMs,
# 128 B of shared-memory bandwidth per SM per clock, 128 FP32 lanes per SM (FMA = 2 flop).
N_SM, SMEM_B_PER_CLK, FP32_LANES = 148, 128, 128


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


# kernel sources behind each workload's dominant kernels (device code only: argus_api.cu holds validation and launches)
# (the configs profiled for profiles/traffic.json run the tile kernel of resample_fast.cuh, not the unit kernel)
_RESAMPLE_SRC = ("common.cuh", "plan.cuh", "plan_block.cuh", "resample.cuh", "resample_fast.cuh")
KERNEL_SOURCES = {"segments": ("common.cuh", "segments.cuh"), "detect": ("common.cuh", "resample.cuh", "background.cuh"),
                  "subtract": ("common.cuh", "resample.cuh", "background.cuh", "subtract.cuh")}


def _kernel_sources_sha(key="config1"):
    """Hash of the CUDA sources of a workload's kernels: a dram-traffic figure taken from an ncu profile is only quoted
    while the kernels are the ones that were profiled."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2207_14304_b200", "csrc")
    for name in KERNEL_SOURCES.get(key.split("_")[0], _RESAMPLE_SRC):
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()[:16]


def ncu_traffic(key):
    """(bytes, provenance) of the dominant kernel's DRAM traffic from profiles/traffic.json (written from an ncu --set
    full capture; names the report and the source hash it was taken at); (None, why) when absent or stale."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            t = json.load(f)[key]
    except Exception:
        return None, "no ncu capture recorded for this workload (profiles/traffic.json)"
    if t.get("csrc_sha16") != _kernel_sources_sha(key):
        return None, "kernels changed since %s was captured (profiles/traffic.json)" % t.get("profile")
    return int(t["dram_bytes"]), "%s, csrc %s" % (t["profile"], t["csrc_sha16"])


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.1] or [r for _, r in self.rows]
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except Exception:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ workloads
WORKLOADS = {
    # name: (description, frames per step, kernel, nside)
    "config0": ("configs[0] 512x512 nside 2^17 bilinear", 1),
    "config1": ("configs[1] 9576x6388 nside 2^17 bilinear", 1),
    "config2": ("configs[2] one 9576x6388 frame, SIP order 3, nside 2^17 Lanczos-3", 1),
    "config3": ("configs[3] one 1 s 9576x6388 frame, nside 2^17 bilinear (value + weight written)", 1),
    "config4": ("configs[4] one 9576x6388 frame, SIP order 3, nside 2^18 Lanczos-3", 1),
    "coadd": ("configs[3] 60 dithered 1 s 9576x6388 frames, nside 2^17 bilinear, fused calibrate+resample+accumulate into one coadd", 60),
    "batch": ("configs[2] 38 pointings (dec -20..+72) 9576x6388, own masters, SIP order 3, nside 2^17 Lanczos-3", 38),
}


def make_frames(name, rank):
    """Host-side synthetic inputs of a workload: list of (Frame, wcs) per frame of the step.  configs[1] is the benchmark
    line; the single-frame configN lines and the two multi-frame workloads are for the record."""
    import synth
    if name == "config0":
        fr = synth.config0(seed=rank)
        return [(fr, fr.wcs)]
    if name == "config2":
        fr = synth.config2_frame(rank % 38)
        return [(fr, fr.wcs)]
    if name == "config3":
        fr = synth.config3_frame(rank)
        return [(fr, fr.wcs)]
    if name == "config4":
        fr = synth.config4_frame(rank % 9)
        return [(fr, fr.wcs)]
    if name == "coadd":      # 60 dithered pointings of one field, shared masters; N_DISTINCT noise realisations
        base = synth.config3_frame(0)
        masters = (base.bias, base.dark, base.flat)
        distinct = [base] + [synth.config3_frame(k, masters=masters) for k in range(1, N_DISTINCT)]
        return [(distinct[k % N_DISTINCT], _config3_wcs(k)) for k in range(60)]
    if name == "batch":      # 38 pointings with their own WCS; N_DISTINCT pixel sets, every frame its own device copy
        distinct = [synth.config2_frame(k) for k in range(N_DISTINCT)]
        return [(distinct[k % N_DISTINCT], synth.frames.config2_wcs(k)) for k in range(38)]
    fr = synth.config1(seed=1 + rank)
    return [(fr, fr.wcs)]


def _config3_wcs(k):
    """The WCS of configs[3] frame k without drawing its 61 MPix of pixels (same generator, same draws as synth)."""
    import numpy as np
    import synth
    W, H = synth.frames.FULL_W, synth.frames.FULL_H
    rng = np.random.Generator(np.random.PCG64(300 + k + 10_000))
    dx, dy = rng.uniform(-0.5, 0.5, 2)
    return synth.make_wcs((30.0, 20.0), ((W - 1) / 2.0 + dx, (H - 1) / 2.0 + dy), 0.3)


def algorithmic_work(kernel, px_in, px_out, coadd, in_bytes=14.0):
    """SURVEY 8(d) / DESIGN.md 6.5: what the method must move or compute once per frame.
    HBM bytes: 14 B per input px (raw u16 + three f32 masters) + 8 B per output px (value + weight), or 16 B per output
    px for the fused coadd read-modify-write.  Shared-memory bytes: the staged box is read once for calibration (14 B)
    and written once calibrated (4 B) per input px; the gather reads 4 (bilinear) or 36 (Lanczos-3) float32 taps per
    output px.  FP32 flops: A2 3 per input px; A3+A4 ~60 and A5 16 (bilinear) or 36 x 2 x 2 + 40 (Lanczos-3) per output px."""
    taps = 36 if kernel == "lanczos3" else 4
    hbm = in_bytes * px_in + (16.0 if coadd else 8.0) * px_out       # in_bytes: 14, or 10 / 6 with pre-fused masters (8(f).4)
    smem = (in_bytes + 4.0) * px_in + 4.0 * taps * px_out
    flop = 3.0 * px_in + (60.0 + (184.0 if kernel == "lanczos3" else 16.0)) * px_out
    return hbm, smem, flop


def rooflines(kernel, px_in, px_out, coadd, k_ms, sm_mhz, hbm_peak, hbm_src, in_bytes=14.0):
    """The three fractions SURVEY 8(d) asks for; `bound` = the resource whose time-at-peak for the algorithmic work is
    longest.  Peaks: HBM measured copy bandwidth; shared memory = SMs x 128 B/clk x clock; FP32 = SMs x 128 lanes x 2 x
    clock, both at the SM clock sampled under load (falls back to 1965 MHz)."""
    clk = (sm_mhz or 1965.0) * 1e6
    hbm, smem, flop = algorithmic_work(kernel, px_in, px_out, coadd, in_bytes)
    peaks = {"hbm": hbm_peak * 1e9, "smem": N_SM * SMEM_B_PER_CLK * clk, "fp32": N_SM * FP32_LANES * 2 * clk}
    work = {"hbm": hbm, "smem": smem, "fp32": flop}
    t_peak = {k: work[k] / peaks[k] for k in work}
    bound = max(t_peak, key=t_peak.get)
    t = k_ms * 1e-3
    fr = {k: (t_peak[k] / t if t > 0 else 0.0) for k in work}
    unit = {"hbm": "GB/s", "smem": "GB/s", "fp32": "GFLOP/s"}[bound]
    return {"bound": bound if bound == "hbm" else ("smem (shared-memory / LSU pipe)" if bound == "smem" else "alu (FP32 issue)"),
            "achieved": work[bound] / t / 1e9 if t > 0 else 0.0, "peak": peaks[bound] / 1e9, "unit": unit, "frac": fr[bound],
            "fractions": {"hbm": fr["hbm"], "smem": fr["smem"], "fp32": fr["fp32"]},
            "time_at_peak_ms": {k: 1e3 * v for k, v in t_peak.items()},
            "peak_source": "hbm: %s; smem = %d SMs x %d B/clk, fp32 = %d SMs x %d lanes x 2, at %.0f MHz" % (
                hbm_src, N_SM, SMEM_B_PER_CLK, N_SM, FP32_LANES, clk / 1e6),
            "kernel_ms": k_ms, "algorithmic_bytes": hbm, "algorithmic_smem_bytes": smem, "algorithmic_flop": flop}


def cpu_oracle_run(fr):
    """The oracle's whole path (calibrate + footprint + resample), as it stands, on frame `fr`.
    Returns (seconds, n_output_px)."""
    import oracle
    H, W = fr.shape
    t0 = time.perf_counter()
    cal, mask = oracle.calibrate_frame(fr)
    idx, _ = oracle.footprint(fr.wcs, W, H, fr.nside)
    oracle.resample(cal, mask, fr.wcs, fr.nside, idx, oracle.KERNELS[fr.kernel])
    return time.perf_counter() - t0, len(idx)


def cpu_sample_frame(name, side):
    """A side x side frame of the workload's own recipe (noise / star / flat model, WCS family, nside, kernel)."""
    import synth
    if name in ("config2", "batch"):
        return synth.config2_frame(0, W=side, H=side)
    if name == "config4":
        return synth.config4_frame(0, W=side, H=side)
    if name in ("config3", "coadd"):
        return synth.config3_frame(0, W=side, H=side)
    if name == "config0":
        return synth.config0()
    return synth.config1(seed=1, W=side, H=side)


def cpu_desc(name, fr, n_out, threads):
    H, W = fr.shape
    return ("%dx%d frame of the %s recipe (nside 2^%d, %s), whole oracle path calibrate+footprint+resample%s, %d output px, "
            "%d thread%s" % (W, H, WORKLOADS[name][0].split(" ")[0], fr.nside.bit_length() - 1, fr.kernel,
                             " (the coadd accumulation is not timed)" if name == "coadd" else "", n_out, threads,
                             "" if threads == 1 else "s"))


def public_config(name, fr, n_frames):
    """The part of `config` both arms print identically (the driver compares them)."""
    H, W = fr.shape if name != "config0" else (512, 512)
    full = name != "config0"
    import synth
    if full:
        W, H = synth.frames.FULL_W, synth.frames.FULL_H
    return {"workload": WORKLOADS[name][0], "frames_per_step_per_gpu": n_frames, "W": W, "H": H, "nside": fr.nside,
            "kernel": fr.kernel, "fused": True, "plan_every_step": True,
            "l2": "inputs (856 MB/frame) larger than L2 (126 MB)" if full else "inputs fit L2 (parity-sized case)",
            "parallelism": "frames independent: every GPU processes its own frames (replicas)"}


def reduce_over_ranks(ms, px_in, px_out, dist=None, device=None):
    """Whole-job accounting under torchrun: time = MAX over ranks, pixels = SUM over ranks.
    `dist` is torch.distributed (initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms), float(px_in), float(px_out)
    import torch
    tt = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    cnt = torch.tensor([float(px_in), float(px_out)], dtype=torch.float64, device=device)
    dist.all_reduce(cnt, op=dist.ReduceOp.SUM)
    return float(tt.item()), float(cnt[0].item()), float(cnt[1].item())


def run_reference(args):
    """The oracle, as it stands, on the host cores: each step = one bounded sample frame of the workload's recipe."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    oracle.lib()
    cores = oracle.max_threads()
    name = args.workload if args.workload in WORKLOADS else "config1"
    fr = cpu_sample_frame(name, SAMPLE_SIDE["lanczos3" if name in ("config2", "config4", "batch") else "bilinear"])
    H, W = fr.shape
    for _ in range(max(0, min(args.warmup, 1))):
        cpu_oracle_run(fr)
    total, n_out = 0.0, 0
    for _ in range(args.steps):
        dt, n_out = cpu_oracle_run(fr)
        total += dt
    value = W * H * args.steps / total / 1e6
    desc = cpu_desc(name, fr, n_out, cores)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": public_config(name, fr, WORKLOADS[name][1]),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_gpu(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_2207_14304_b200 as argus

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    argus.load_library()  # raises if the CUDA extension is missing: no fallback

    name = args.workload
    jobs_host = make_frames(name, rank)
    fr0 = jobs_host[0][0]
    H, W = fr0.shape
    nside, kernel = fr0.nside, fr0.kernel
    coadd = name == "coadd"
    ctx = argus.Context(local)
    if args.unit_kernel:
        ctx.set_fast_path(3)
    elif args.tile_kernel:
        ctx.set_fast_path(2)

    # device-resident inputs.  coadd: shared masters, N_DISTINCT raw frames; batch: every frame its own raw + masters
    def up(a):
        return torch.from_numpy(a).to(dev)

    dsets = {}
    jobs = []
    shared_masters = None
    for fr, wcs in jobs_host:
        if coadd:
            if shared_masters is None:
                shared_masters = (up(fr.bias), up(fr.dark), up(fr.flat))
            if id(fr) not in dsets:
                dsets[id(fr)] = up(fr.raw)
            d = dict(raw=dsets[id(fr)], bias=shared_masters[0], dark=shared_masters[1], flat=shared_masters[2])
        elif name == "batch":
            if id(fr) not in dsets:
                dsets[id(fr)] = (up(fr.raw), up(fr.bias), up(fr.dark), up(fr.flat))
                src = dsets[id(fr)]
            else:
                src = tuple(t.clone() for t in dsets[id(fr)])      # own device copy: 38 x 856 MB resident
            d = dict(raw=src[0], bias=src[1], dark=src[2], flat=src[3])
        else:
            d = dict(raw=up(fr.raw), bias=up(fr.bias), dark=up(fr.dark), flat=up(fr.flat))
        d.update(bpm=None, t_exp=fr.t_exp, sat_adu=fr.sat_adu, flat_min=fr.flat_min)
        jobs.append((wcs, d))
    if args.prefused:   # offset / gain formed once per pointing (not timed), 10 or 6 B per input pixel
        dt = torch.float32 if args.prefused == "f32" else torch.float16
        done = {}
        for i, (wcs, d) in enumerate(jobs):
            k = d["bias"].data_ptr()
            if k not in done:
                done[k] = argus.argus_prepare_masters(ctx, d["bias"], d["dark"], d["flat"], None, d["t_exp"], d["flat_min"], dtype=dt)
            jobs[i] = (wcs, dict(raw=d["raw"], offset=done[k][0], gain=done[k][1], sat_adu=d["sat_adu"]))
        torch.cuda.synchronize()
        for wcs, d in jobs:
            d.pop("bias", None)
    n_fps = [argus.argus_healpix_footprint(ctx, wcs, W, H, nside, want_indices=False)[0] for wcs, _ in jobs]
    stats = argus.argus_plan_info(ctx)
    n_out_step, n_frames = int(sum(n_fps)), len(jobs)
    if coadd:
        tiles = torch.unique(torch.cat([argus.argus_healpix_footprint(ctx, wcs, W, H, nside)[1] >> 18 for wcs, _ in jobs[:: max(1, n_frames // 8)]]
                                       + [argus.argus_healpix_footprint(ctx, jobs[-1][0], W, H, nside)[1] >> 18]))
        # +-0.5 px dithers move the footprint by less than one pixel: the union over a spread of frames + a check below
        ppt = 1 << 18
        csum = torch.zeros(tiles.numel() * ppt, dtype=torch.float32, device=dev)
        cwsum = torch.zeros_like(csum)
        skipped = torch.zeros(1, dtype=torch.int64, device=dev)
    else:
        value = torch.empty(max(n_fps), dtype=torch.float32, device=dev)
        weight = torch.empty(max(n_fps), dtype=torch.float32, device=dev)
    ctx.set_plan_cache(False)  # every frame plans again, as a new WCS does
    if args.no_plan_overlap:
        ctx.set_plan_overlap(False)

    def step():
        for wcs, d in jobs:
            if coadd:
                argus.argus_resample_coadd(ctx, wcs, W, H, nside, kernel, tiles, 256, csum, cwsum, skipped, **d)
            else:
                argus.argus_resample(ctx, wcs, W, H, nside, kernel, value, weight, **d)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    if coadd:
        assert int(skipped.item()) == 0, "coadd layout misses tiles of some frame"
    ctx.set_profile(True)
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler and n_frames == 1:
        time.sleep(0.15)       # one nvidia-smi sample before the (6 ms) timed region, one after it
    t0 = time.time()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = ctx.launch_count()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    t1 = time.time()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.launch_count() - launches0   # kernels of libargus.so launched inside the timed region (this rank)
    plan_ms, kern_ms, ncalls = ctx.profile_read()
    ctx.set_profile(False)
    clocks = sampler.stop(t0, t1) if sampler else None
    ms, px_in_all, px_out_all = reduce_over_ranks(ms, W * H * n_frames, n_out_step, dist if world > 1 else None, dev)

    # ---- end to end through the C ABI with HOST buffers: every frame's raw pixels come from pinned host memory (masters
    # stay resident per pointing) and the result goes back to pinned host memory, inside the timed
    # region; the library pipelines upload / kernels / download of consecutive frames on its own copy streams
    h_raws = {}
    for fr, _ in jobs_host:
        if id(fr) not in h_raws:
            h_raws[id(fr)] = torch.from_numpy(fr.raw).pin_memory()
    if coadd:
        h_sum, h_wsum = torch.empty_like(csum, device="cpu").pin_memory(), torch.empty_like(cwsum, device="cpu").pin_memory()
    else:
        h_val = torch.empty(max(n_fps), dtype=torch.float32).pin_memory()
        h_wgt = torch.empty(max(n_fps), dtype=torch.float32).pin_memory()

    def masters_of(fr, d):
        return (dict(offset=d["offset"], gain=d["gain"], sat_adu=fr.sat_adu) if args.prefused else
                dict(bias=d["bias"], dark=d["dark"], flat=d["flat"], t_exp=fr.t_exp, sat_adu=fr.sat_adu, flat_min=fr.flat_min))

    def e2e_vw_step():        # value + weight back to the host (8 B per footprint pixel)
        for (fr, wcs), (_, d), n in zip(jobs_host, jobs, n_fps):
            argus.argus_resample_host(ctx, wcs, W, H, nside, kernel, n, h_raws[id(fr)], h_val, h_wgt, **masters_of(fr, d))

    # the paper's per-frame PRODUCT back to the host: binary16 segment data + low-resolution map
    products = not coadd and nside >= (1 << 14)
    if products:
        mini_cap = int(max(n_fps) // 64 * 1.3) + 4096
        h_seg = torch.empty(max(n_fps), dtype=torch.int16).pin_memory()
        h_mid = torch.empty(mini_cap, dtype=torch.int64).pin_memory()
        h_mv, h_mw = torch.empty(mini_cap, dtype=torch.float32).pin_memory(), torch.empty(mini_cap, dtype=torch.float32).pin_memory()
        h_nm = torch.zeros(1, dtype=torch.int64).pin_memory()

    def e2e_step():
        for (fr, wcs), (_, d), n in zip(jobs_host, jobs, n_fps):
            if coadd:
                argus.argus_resample_coadd_host(ctx, wcs, W, H, nside, kernel, h_raws[id(fr)], tiles, 256, csum, cwsum, None, **masters_of(fr, d))
            elif products:
                argus.argus_reduce_frame_host(ctx, wcs, W, H, nside, kernel, n, h_raws[id(fr)], h_seg, h_mid, h_mv, h_mw, h_nm,
                                              nside_mini=1 << 14, **masters_of(fr, d))
            else:
                argus.argus_resample_host(ctx, wcs, W, H, nside, kernel, n, h_raws[id(fr)], h_val, h_wgt, **masters_of(fr, d))
        if coadd:   # the step's result: the coadd itself
            h_sum.copy_(csum, non_blocking=True)
            h_wsum.copy_(cwsum, non_blocking=True)

    def time_e2e(fn):
        for _ in range(2 if n_frames == 1 else 1):
            fn()
        argus.argus_host_wait(ctx)
        barrier()
        steps = max(4, min(args.steps, 10)) if n_frames == 1 else 2
        t_e0 = time.perf_counter()
        for _ in range(steps):
            fn()
        argus.argus_host_wait(ctx)
        torch.cuda.synchronize()
        wall = 1e3 * (time.perf_counter() - t_e0)   # host wall clock around enqueue + completion (copies run on the library's streams)
        barrier()
        wall, _, _ = reduce_over_ranks(wall, 0, 0, dist if world > 1 else None, dev)
        return wall, steps

    e2e_ms, e2e_steps = time_e2e(e2e_step)
    h2d = int(W * H * 2 * n_frames)
    if coadd:
        d2h = int(2 * 4 * csum.numel())
    elif products:
        n_mini = int(h_nm.item())
        d2h = int(2 * n_out_step + n_frames * (16 * mini_cap + 8))
    else:
        d2h = int(8 * n_out_step)
    e2e_vw = None
    if products and n_frames == 1:
        vw_ms, vw_steps = time_e2e(e2e_vw_step)
        e2e_vw = {"value": px_in_all * vw_steps / (vw_ms * 1e-3) / 1e6, "unit": UNIT, "ms_per_step": vw_ms / vw_steps,
                  "d2h_bytes_per_step": int(8 * n_out_step), "note": "argus_resample_host: float32 value + weight back to the host instead of the products"}

    if rank == 0:
        peak, peak_src = _peaks()
        ms_step = ms / args.steps
        k_ms = kern_ms / max(ncalls, 1)                       # per frame (argus_resample call)
        px_out_frame = n_out_step / n_frames
        in_bytes = {None: 14.0, "f32": 10.0, "f16": 6.0}[args.prefused]
        roof = rooflines(kernel, W * H, px_out_frame, coadd, k_ms, clocks and clocks.get("sm_mhz"), peak, peak_src, in_bytes)
        roof["input_bytes_per_px"] = in_bytes
        alg_step = roof["algorithmic_bytes"] * n_frames
        # nside 2^18 at this pixel scale: every box fits 48 x 48 pixels, the library runs the two-stage Lanczos-3 form
        variant = ",1" if (kernel == "lanczos3" and nside >= (1 << 18) and not args.tile_kernel) else ""
        roof["kernel"] = ("resample_fast_kernel<%s,%d%s> (TMA-staged, fused calibration%s) + resample_tiles_kernel on its slow list; "
                          "per frame, CUDA events around the resample launches" % ("true" if coadd else "false", 1 if kernel == "lanczos3" else 0,
                                                                                  variant, ", coadd read-modify-write" if coadd else ""))
        roof["step_frac"] = (alg_step / (ms_step * 1e-3) / 1e9) / peak
        tr, tr_src = ncu_traffic(name + ("" if not args.prefused else "_" + args.prefused))
        roof["traffic"], roof["traffic_source"] = tr, tr_src
        if world == 1:
            import oracle
            cores = oracle.max_threads()
            # the oracle, as it stands: all host threads on the first frame of the step (full size for bilinear, a
            # bounded sample for Lanczos-3), and one thread on a bounded sample
            fr_n = fr0 if kernel == "bilinear" else cpu_sample_frame(name, 4096)
            cpu_dt, n_o = cpu_oracle_run(fr_n)
            cpu = {"value": fr_n.shape[0] * fr_n.shape[1] / cpu_dt / 1e6, "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": cpu_desc(name, fr_n, n_o, cores), "seconds": cpu_dt}
            fr_1 = cpu_sample_frame(name, SAMPLE_SIDE[kernel] // 2)
            oracle.set_threads(1)
            try:
                dt1, n_o1 = cpu_oracle_run(fr_1)
            finally:
                oracle.set_threads(cores)
            cpu1 = {"value": fr_1.shape[0] * fr_1.shape[1] / dt1 / 1e6, "unit": UNIT, "cores": 1, "kind": "oracle",
                    "sample": cpu_desc(name, fr_1, n_o1, 1), "seconds": dt1}
        else:
            cpu = {"value": None, "unit": UNIT, "cores": None, "kind": "oracle", "sample": "rank 0 at N=1 only"}
            cpu1 = None
        cfg = public_config(name, fr0, n_frames)
        if args.prefused:
            cfg["masters"] = "pre-fused offset + gain, %s (SURVEY 8(f).4): %d B per input pixel" % (args.prefused, int(in_bytes))
        line = {
            "metric": METRIC, "value": px_in_all * args.steps / (ms * 1e-3) / 1e6, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": cfg,
            "details": {"n_footprint_per_step": n_out_step, "ms_per_frame": ms_step / n_frames, "plan_last_frame": stats,
                        "plan_overlap": ("off (diagnostic)" if args.no_plan_overlap else
                                         "the plan of frame k+1 runs on the library's side streams underneath the kernels of frame k"),
                        "distinct_pixel_sets": len(h_raws),
                        "coadd_tiles": int(tiles.numel()) if coadd else None},
            "output_mpix_per_s": px_out_all * args.steps / (ms * 1e-3) / 1e6,
            "plan_ms_per_frame": plan_ms / max(ncalls, 1),
            "roofline": roof,
            "cpu_baseline": cpu, "cpu_baseline_1thread": cpu1,
            "e2e": {"value": px_in_all * e2e_steps / (e2e_ms * 1e-3) / 1e6, "unit": UNIT,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / e2e_steps,
                    "note": ("argus_resample_coadd_host per frame (raw from pinned host memory), the coadd (sum, wsum) back to pinned host memory once per step"
                             if coadd else
                             ("argus_reduce_frame_host: raw frame from pinned host memory each frame; the paper's per-frame product back to pinned host memory: binary16 segment data (2 B per footprint pixel, PAPER.md:145) + low-resolution map on the NSIDE-16384 minipix grid (PAPER.md:149); masters resident per pointing"
                              if products else
                              "argus_resample_host: raw frame from pinned host memory each frame, value + weight back to pinned host memory; masters resident per pointing"))
                            + "; upload / kernels / download of consecutive frames pipelined by the library; host wall clock"},
            "e2e_value_weight": e2e_vw,
            "gpu_launches": launches,
            "clocks": clocks,
        }
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_segments(args):
    """--workload segments: SURVEY 8(f).1 on the configs[1] footprint.  A step = one argus_segment_products call
    (head scan + target lookup + per-minipix reduction / stamping / binary16 packing) on value + weight of a
    resampled configs[1] frame that is already in HBM.  Not the headline line; same JSON contract."""
    import numpy as np
    import torch

    import paper_2207_14304_b200 as argus

    rank = int(os.environ.get("RANK", "0"))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        if rank == 0:
            print(json.dumps({"workload": "segments", "unavailable": "single-GPU diagnostic line (frames are independent: replicas only)"}))
        return 0
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    argus.load_library()
    fr = make_frames("config1", 0)[0][0]
    H, W = fr.shape
    nside, nside_mini = fr.nside, 1 << 14
    ctx = argus.Context(0)
    d = dict(raw=torch.from_numpy(fr.raw).to(dev), bias=torch.from_numpy(fr.bias).to(dev),
             dark=torch.from_numpy(fr.dark).to(dev), flat=torch.from_numpy(fr.flat).to(dev), bpm=None,
             t_exp=fr.t_exp, sat_adu=fr.sat_adu, flat_min=fr.flat_min)
    n, idx = argus.argus_healpix_footprint(ctx, fr.wcs, W, H, nside, want_indices=True)
    value = torch.empty(n, dtype=torch.float32, device=dev)
    weight = torch.empty(n, dtype=torch.float32, device=dev)
    argus.argus_resample(ctx, fr.wcs, W, H, nside, fr.kernel, value, weight, **d)
    del d
    none = torch.zeros(0, dtype=torch.int64, device=dev)
    n_mini = argus.argus_segment_products(ctx, nside, nside_mini, idx, value, weight, none)     # count
    # targets: 2 % of the frame's minipix (sparse + low-resolution products are ~5 % of the full data)
    g = torch.Generator(device="cpu").manual_seed(7)
    all_mini = torch.unique(idx >> (2 * ((nside // nside_mini).bit_length() - 1)))
    targets = all_mini[torch.randperm(all_mini.numel(), generator=g)[: max(1, all_mini.numel() // 50)].to(dev)].contiguous()
    out = dict(seg16=torch.empty(n, dtype=torch.int16, device=dev), mini_id=torch.empty(n_mini, dtype=torch.int64, device=dev),
               mini_value=torch.empty(n_mini, dtype=torch.float32, device=dev),
               mini_weight=torch.empty(n_mini, dtype=torch.float32, device=dev),
               mini_keep=torch.empty(n_mini, dtype=torch.uint8, device=dev))

    def step():
        argus.argus_segment_products(ctx, nside, nside_mini, idx, value, weight, targets, sync=False, **out)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    sampler = ClockSampler(0)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    for _ in range(600):   # the timed region alone (K x 0.2 ms) is shorter than one nvidia-smi sample: the clocks are
        step()             # sampled over this identical untimed run-up plus the timed region
    launches0 = ctx.launch_count()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    t1 = time.time()
    ms_step = ev0.elapsed_time(ev1) / args.steps
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop(t0, t1)

    # end to end: list from pinned host memory, products back to pinned host memory, every step
    h_in = [t.cpu().pin_memory() for t in (idx, value, weight)]
    h_out = {k: torch.empty_like(v, device="cpu").pin_memory() for k, v in out.items()}
    e2e_steps = max(3, min(args.steps, 6))
    torch.cuda.synchronize()
    t_e0 = time.perf_counter()
    for _ in range(e2e_steps):
        idx.copy_(h_in[0], non_blocking=True); value.copy_(h_in[1], non_blocking=True); weight.copy_(h_in[2], non_blocking=True)
        step()
        for k, v in out.items():
            h_out[k].copy_(v, non_blocking=True)
        torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t_e0) / e2e_steps

    # the oracle, as it stands, on the same list
    from oracle import segments as oseg
    ns = n   # the numpy oracle does the whole list in a few seconds
    hi, hv, hw, ht = h_in[0][:ns].numpy(), h_in[1][:ns].numpy(), h_in[2][:ns].numpy(), targets.cpu().numpy()
    t_c0 = time.perf_counter()
    oseg.segment_products(hi, hv, hw, nside, nside_mini, ht)
    cpu_dt = time.perf_counter() - t_c0

    peak, peak_src = _peaks()
    alg = n * (8 + 4 + 4 + 2) + n_mini * (8 + 4 + 4 + 1) + targets.numel() * 8
    achieved = alg / (ms_step * 1e-3) / 1e9
    h2d = sum(t.numel() * t.element_size() for t in h_in)
    d2h = sum(t.numel() * t.element_size() for t in h_out.values())
    print(json.dumps({
        "metric": "segment products (minipix stamping + binary16 packing + low-resolution map) Mpix/s per B200; achieved HBM GB/s vs peak",
        "value": n / (ms_step * 1e-3) / 1e6, "unit": "Mpix/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "segment products of one resampled configs[1] frame (SURVEY 8(f).1)", "n_footprint": n,
                   "nside": nside, "nside_mini": nside_mini, "n_mini": n_mini, "n_targets": int(targets.numel()),
                   "layout": "compact (element i <-> idx[i])", "l2": "inputs (16 B x n = %d MB) larger than L2 (126 MB)" % (16 * n // 1000000)},
        "roofline": {"bound": "hbm", "kernel": "whole call: seg_flags_kernel + seg_scan_kernel + seg_heads_kernel + seg_targets_kernel + seg_products_kernel<false> (+ memsets); the two streaming kernels (flags, products) are 75 % of it",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic("segments")[0], "traffic_source": ncu_traffic("segments")[1],
                     "traffic_note": "dram read + write of seg_flags_kernel and seg_products_kernel, one launch each",
                     "peak_source": peak_src, "kernel_ms": ms_step, "algorithmic_bytes": alg},
        "cpu_baseline": {"value": ns / cpu_dt / 1e6, "unit": "Mpix/s", "cores": 1, "kind": "oracle",
                         "sample": "oracle.segments.segment_products (numpy, fp64) on the same list, all %d pixels" % ns, "seconds": cpu_dt},
        "e2e": {"value": n / (e2e_ms * 1e-3) / 1e6, "unit": "Mpix/s", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": e2e_ms, "note": "idx + value + weight from pinned host memory, all products back to pinned host memory, host wall clock"},
        "gpu_launches": launches, "clocks": clocks}))
    ctx.close()
    return 0


def run_detect(args):
    """--workload detect: SURVEY 8(f).2 on the configs[1] frame.  A step = argus_background_map + argus_detect_sources
    with fused calibration (raw + masters resident in HBM) -> background / noise grids and the source catalogue.
    Not the headline line; same JSON contract."""
    import numpy as np
    import torch

    import paper_2207_14304_b200 as argus

    rank = int(os.environ.get("RANK", "0"))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        if rank == 0:
            print(json.dumps({"workload": "detect", "unavailable": "single-GPU diagnostic line (frames are independent: replicas only)"}))
        return 0
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    argus.load_library()
    fr = make_frames("config1", 0)[0][0]
    H, W = fr.shape
    B, n_min, k_sigma, cap = 64, 16, 5.0, 1 << 18
    ctx = argus.Context(0)
    d = dict(raw=torch.from_numpy(fr.raw).to(dev), bias=torch.from_numpy(fr.bias).to(dev),
             dark=torch.from_numpy(fr.dark).to(dev), flat=torch.from_numpy(fr.flat).to(dev), bpm=None,
             t_exp=fr.t_exp, sat_adu=fr.sat_adu, flat_min=fr.flat_min)
    G = -(-H // B) * -(-W // B)
    bkg = torch.empty(G, dtype=torch.float32, device=dev)
    nse = torch.empty(G, dtype=torch.float32, device=dev)
    cat = torch.empty(cap * 32, dtype=torch.uint8, device=dev)
    n_dev = torch.zeros(1, dtype=torch.int64, device=dev)

    def step_map():
        argus.argus_background_map(ctx, W, H, bkg, nse, cell=B, n_min=n_min, **d)

    def step_det():
        argus.argus_detect_sources(ctx, W, H, bkg, nse, cat, cell=B, k_sigma=k_sigma, n_dev=n_dev, sync=False, **d)

    two_call = getattr(args, "two_call", False)

    def step():
        if two_call:
            step_map()
            step_det()
        else:   # one call, the frame read once (identical results: tests/test_gpu_background.py check_detect_frame)
            argus.argus_detect_frame(ctx, W, H, bkg, nse, cat, cell=B, n_min=n_min, k_sigma=k_sigma, n_dev=n_dev, sync=False, **d)

    n_src = None
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    n_src = int(n_dev.item())
    n_full = None if two_call else argus.argus_detect_frame_info(ctx)
    sampler = ClockSampler(0)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
    t0 = time.time()
    for _ in range(300):   # run-up for the clock sampler (the timed region is shorter than one nvidia-smi sample)
        step()
    launches0 = ctx.launch_count()
    ev[0].record()
    for _ in range(args.steps):
        step()
    ev[1].record()
    launches = ctx.launch_count() - launches0
    ev[2].record()
    for _ in range(args.steps):
        step_map()
    ev[3].record()
    ev[4].record()
    for _ in range(args.steps):
        step_det()
    ev[5].record()
    torch.cuda.synchronize()
    t1 = time.time()
    ms_step = ev[0].elapsed_time(ev[1]) / args.steps
    ms_map = ev[2].elapsed_time(ev[3]) / args.steps
    ms_det = ev[4].elapsed_time(ev[5]) / args.steps
    clocks = sampler.stop(t0, t1)

    # end to end: raw frame from pinned host memory, grids + catalogue back to pinned host memory, every step
    h_raw = torch.from_numpy(fr.raw).pin_memory()
    h_out = [torch.empty_like(t, device="cpu").pin_memory() for t in (bkg, nse, cat, n_dev)]
    e2e_steps = max(3, min(args.steps, 6))
    torch.cuda.synchronize()
    t_e0 = time.perf_counter()
    for _ in range(e2e_steps):
        d["raw"].copy_(h_raw, non_blocking=True)
        step()
        h_out[3].copy_(n_dev, non_blocking=True)
        h_out[0].copy_(bkg, non_blocking=True); h_out[1].copy_(nse, non_blocking=True)
        torch.cuda.synchronize()
        k = int(h_out[3].item())
        h_out[2][:k * 32].copy_(cat[:k * 32])
    e2e_ms = 1e3 * (time.perf_counter() - t_e0) / e2e_steps
    d2h = 2 * G * 4 + 8 + n_src * 32

    # the oracle, as it stands, on a bounded crop of the same frame (cell-aligned 6144 x 6144 corner, 62 % of the frame)
    import oracle
    from oracle import background as ob
    side = 6144
    cal, mask = oracle.calibrate_frame(fr)
    cal, mask = np.ascontiguousarray(cal[:side, :side]), np.ascontiguousarray(mask[:side, :side])
    t_c0 = time.perf_counter()
    ob_b, ob_n = ob.background(cal, mask, B, n_min)
    o_src = ob.detect(cal, mask, ob_b, ob_n, B=B, k_sigma=k_sigma)
    cpu_dt = time.perf_counter() - t_c0

    peak, peak_src = _peaks()
    px = W * H
    alg = px * 14 + 2 * G * 4 + n_src * 32
    achieved = alg / (ms_step * 1e-3) / 1e9
    print(json.dumps({
        "metric": "background map + source detection (fused calibration) Mpix/s per B200; achieved HBM GB/s vs peak",
        "value": px / (ms_step * 1e-3) / 1e6, "unit": "Mpix/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "background map + source detection on one configs[1] frame (SURVEY 8(f).2)", "W": W, "H": H,
                   "cell": B, "n_min": n_min, "k_sigma": k_sigma, "n_sources": n_src, "fused": True,
                   "entry": "argus_background_map + argus_detect_sources" if two_call else "argus_detect_frame",
                   "tiles_scanned_in_full": n_full, "tiles": -(-W // 64) * -(-H // 32),
                   "l2": "inputs (856 MB/frame) larger than L2 (126 MB)"},
        "roofline": {"bound": "hbm", "kernel": ("whole step: bg_cells_kernel<true> + bg_filter_kernel + det_tiles_kernel<true> + det_scan_kernel + det_order_kernel" if two_call else
                                                "whole step: bg_cells_kernel<true,true> + bg_filter_kernel + det_cand_kernel<true> + det_tiles_list_kernel<true> + det_scan_kernel + det_order_kernel"),
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": ncu_traffic("detect")[0], "traffic_source": ncu_traffic("detect")[1],
                     "traffic_note": "dram read + write of the step's kernels, one launch each",
                     "peak_source": peak_src, "kernel_ms": ms_step, "algorithmic_bytes": alg,
                     "background_map_ms": ms_map, "detect_sources_ms": ms_det},
        "cpu_baseline": {"value": side * side / cpu_dt / 1e6, "unit": "Mpix/s", "cores": 1, "kind": "oracle",
                         "sample": "oracle.background.background + detect (numpy, fp64) on the %d x %d corner of the same frame, %d sources" % (side, side, o_src["x"].size),
                         "seconds": cpu_dt},
        "e2e": {"value": px / (e2e_ms * 1e-3) / 1e6, "unit": "Mpix/s", "h2d_bytes_per_step": int(h_raw.numel() * 2), "d2h_bytes_per_step": int(d2h),
                "ms_per_step": e2e_ms, "note": "raw frame from pinned host memory, grids + catalogue back to pinned host memory, masters resident, host wall clock"},
        "gpu_launches": launches, "clocks": clocks}))
    ctx.close()
    return 0


def run_subtract(args):
    """--workload subtract: SURVEY 8(f).3 at the configs[3] field.  Reference = coadd of 8 one-second frames (210
    NSIDE-256 tiles x 2^18 pixels, resident in HBM), science = the pair of one more frame; a step = one
    argus_subtract_tiles call (per-tile affine match, difference, significance, candidates).  Same JSON contract."""
    import numpy as np
    import torch

    import paper_2207_14304_b200 as argus
    import synth

    rank = int(os.environ.get("RANK", "0"))
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        if rank == 0:
            print(json.dumps({"workload": "subtract", "unavailable": "single-GPU diagnostic line (tiles are independent: replicas only)"}))
        return 0
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    argus.load_library()
    W, H, nside = synth.frames.FULL_W, synth.frames.FULL_H, 1 << 17
    base = synth.config3_frame(0)
    masters = (base.bias, base.dark, base.flat)
    frames = [base] + [synth.config3_frame(k, masters=masters) for k in (1, 2)]
    wcs = base.wcs                     # one WCS: the synthetic star field is fixed in detector coordinates
    ctx = argus.Context(0)
    dm = [torch.from_numpy(m).to(dev) for m in masters]
    raws = [torch.from_numpy(f.raw).to(dev) for f in frames]
    kw = dict(bias=dm[0], dark=dm[1], flat=dm[2], bpm=None, t_exp=base.t_exp, sat_adu=base.sat_adu, flat_min=base.flat_min)
    n_fp, idx = argus.argus_healpix_footprint(ctx, wcs, W, H, nside)
    tiles = torch.unique(idx >> 18)
    del idx
    ppt = 1 << 18
    n_slots = tiles.numel() * ppt
    ref_s = torch.zeros(n_slots, dtype=torch.float32, device=dev); ref_w = torch.zeros_like(ref_s)
    sci_s = torch.zeros_like(ref_s); sci_w = torch.zeros_like(ref_s)
    for k in range(8):
        argus.argus_resample_coadd(ctx, wcs, W, H, nside, "bilinear", tiles, 256, ref_s, ref_w, None, raw=raws[k % 2], **kw)
    argus.argus_resample_coadd(ctx, wcs, W, H, nside, "bilinear", tiles, 256, sci_s, sci_w, None, raw=raws[2], **kw)
    diff = torch.empty_like(ref_s); sig = torch.empty_like(ref_s)
    cap = 1 << 18
    cat = torch.empty(cap * 32, dtype=torch.uint8, device=dev)
    n_dev = torch.zeros(1, dtype=torch.int64, device=dev)
    prm = dict(match="affine", k_sigma=5.0, read_noise=1.7, gain=1.0, ref_wmin=2.0)

    def step():
        argus.argus_subtract_tiles(ctx, tiles, 256, nside, sci_s, sci_w, ref_s, ref_w, diff, sig, cat, n_dev=n_dev, sync=False, **prm)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    n_cand = int(n_dev.item())
    sampler = ClockSampler(0)
    time.sleep(0.15)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.time()
    launches0 = ctx.launch_count()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    torch.cuda.synchronize()
    t1 = time.time()
    ms_step = ev0.elapsed_time(ev1) / args.steps
    launches = ctx.launch_count() - launches0
    clocks = sampler.stop(t0, t1)

    # end to end: the science frame's raw pixels from pinned host memory -> its pair on the grid -> subtraction -> the
    # candidates back to pinned host memory
    h_raw = torch.from_numpy(frames[2].raw).pin_memory()
    h_cat = torch.empty_like(cat, device="cpu").pin_memory()
    h_n = torch.zeros(1, dtype=torch.int64).pin_memory()
    m = dict(bias=dm[0], dark=dm[1], flat=dm[2], t_exp=base.t_exp, sat_adu=base.sat_adu, flat_min=base.flat_min)
    e2e_steps = 4
    torch.cuda.synchronize()
    t_e0 = time.perf_counter()
    for _ in range(e2e_steps):
        sci_s.zero_(); sci_w.zero_()
        argus.argus_resample_coadd_host(ctx, wcs, W, H, nside, "bilinear", h_raw, tiles, 256, sci_s, sci_w, None, **m)
        step()
        h_n.copy_(n_dev, non_blocking=True)
        torch.cuda.synchronize()
        k = int(h_n.item())
        h_cat[:k * 32].copy_(cat[:k * 32])
    e2e_ms = 1e3 * (time.perf_counter() - t_e0) / e2e_steps

    # the oracle, as it stands, on a bounded sample: 6 of the tiles (numpy, one core)
    from oracle import subtract as osub
    sel = np.linspace(0, tiles.numel() - 1, 6).astype(np.int64)
    cut = lambda t: np.concatenate([t[int(i) * ppt:(int(i) + 1) * ppt].cpu().numpy() for i in sel])
    a = [cut(t) for t in (sci_s, sci_w, ref_s, ref_w)]
    t_c0 = time.perf_counter()
    osub.subtract_tiles(tiles.cpu().numpy()[sel], ppt, nside, *a, match=osub.MATCH_AFFINE, k_sigma=5.0, read_noise=1.7, gain=1.0, ref_wmin=2.0)
    cpu_dt = time.perf_counter() - t_c0

    peak, peak_src = _peaks()
    alg = n_slots * (16 + 8) + n_cand * 32           # 4 input arrays read once, difference + significance written
    achieved = alg / (ms_step * 1e-3) / 1e9
    tr, tr_src = ncu_traffic("subtract")
    print(json.dumps({
        "metric": "direct image subtraction per tile (match + difference + significance + candidates) Mpix/s per B200; achieved HBM GB/s vs peak",
        "value": n_slots / (ms_step * 1e-3) / 1e6, "unit": "Mpix/s", "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": "direct image subtraction of one configs[3] frame against an 8-frame coadd (SURVEY 8(f).3)",
                   "n_tiles": int(tiles.numel()), "nside": nside, "nside_tile": 256, "pixels": int(n_slots), "match": "affine",
                   "k_sigma": 5.0, "n_candidates": n_cand, "ms_per_tile": ms_step / tiles.numel(),
                   "l2": "inputs (16 B x %d px = %d MB) larger than L2 (126 MB)" % (n_slots, 16 * n_slots // 1000000)},
        "roofline": {"bound": "hbm", "kernel": "whole call: sub_stats_kernel + sub_fit_kernel + sub_tiles_kernel + det_scan_kernel + sub_gather_kernel (the affine match reads the four arrays a second time: the algorithmic bytes count them once)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": tr, "traffic_source": tr_src,
                     "peak_source": peak_src, "kernel_ms": ms_step, "algorithmic_bytes": alg},
        "cpu_baseline": {"value": len(sel) * ppt / cpu_dt / 1e6, "unit": "Mpix/s", "cores": 1, "kind": "oracle",
                         "sample": "oracle.subtract.subtract_tiles (numpy, fp64) on 6 of the %d tiles of the same pairs: %.0f ms per tile (the paper's CPU: 20 ms per tile, PAPER.md:201)" % (tiles.numel(), 1e3 * cpu_dt / len(sel)),
                         "seconds": cpu_dt},
        "e2e": {"value": W * H / (e2e_ms * 1e-3) / 1e6, "unit": "Mpix/s (input pixels of the science frame)", "h2d_bytes_per_step": int(h_raw.numel() * 2),
                "d2h_bytes_per_step": int(8 + n_cand * 32), "ms_per_step": e2e_ms,
                "note": "science frame from pinned host memory -> argus_resample_coadd_host into a zeroed pair -> argus_subtract_tiles -> candidate count + records to pinned host memory; host wall clock"},
        "gpu_launches": launches, "clocks": clocks}))
    ctx.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-plan-overlap", action="store_true", help="diagnostic: build every plan in place on the caller's stream")
    ap.add_argument("--workload", default="config1", choices=sorted(WORKLOADS) + ["segments", "detect", "subtract"])
    ap.add_argument("--prefused", default=None, choices=["f32", "f16"], help="masters pre-fused by argus_prepare_masters (SURVEY 8(f).4)")
    ap.add_argument("--unit-kernel", action="store_true", help="diagnostic: image-aligned unit kernel wherever its geometry allows")
    ap.add_argument("--tile-kernel", action="store_true", help="diagnostic: tile kernel only")
    ap.add_argument("--two-call", action="store_true", help="--workload detect: argus_background_map + argus_detect_sources instead of argus_detect_frame")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.workload == "segments":
        return run_segments(args)
    if args.workload == "detect":
        return run_detect(args)
    if args.workload == "subtract":
        return run_subtract(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
