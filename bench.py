#!/usr/bin/env python
"""bench.py -- frames/s of the LPF hot path (qc -> detect -> associate -> flux -> append) on
seeded synthetic AARTFAAC-shaped cubes (BASELINE.json: 1024x1024x16 fp32 = config 3).

    python bench.py --gpus N --steps K --warmup W            # our CUDA path
    python bench.py --impl reference --gpus N --steps K ...  # the CPU oracle, as it stands

One JSON line on stdout (rank 0).  A "step" is one cube through the whole path.  The pool of
distinct device-resident frames is larger than L2 and cycled, so every step reads its cube from HBM.
Timing: CUDA events on a main stream that all lane streams fork from / join to; max over ranks.
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

import numpy as np

METRIC = "image-cube frames/s (whole path: qc+detect+associate+flux+dynspec)"
UNIT = "frames/s"
FALLBACK_HBM_GBS = 6650.0           # /opt/skills/guides/B200_PROFILING.md fallback
N_SM, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
ALU_PEAK_TFLOPS = N_SM * FP32_LANES * 2 * SM_MAX_GHZ / 1e3   # 74.4 TFLOP/s fp32 FMA


def env_rank():
    return int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0"))


def reduce_over_ranks(ms: float, launches: int, device, world: int):
    """Multi-rank aggregation of one timed region: the step time is the MAX over ranks (every rank ran the
    same number of steps on its own stream), the launch count the SUM.  `device` is where the scratch
    tensors live (the rank's GPU under NCCL, "cpu" under gloo)."""
    if world <= 1:
        return float(ms), int(launches)
    import torch
    import torch.distributed as dist
    tms = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(tms, op=dist.ReduceOp.MAX)
    tl = torch.tensor([launches], device=device, dtype=torch.int64)
    dist.all_reduce(tl, op=dist.ReduceOp.SUM)
    return float(tms.item()), int(tl.item())


def whole_job_value(world: int, steps: int, ms: float) -> float:
    """frames/s of the whole job: every rank processed `steps` frames of its own stream in `ms` (max over ranks)."""
    return world * steps / (ms / 1e3)


def rank_seed(rank: int) -> int:
    """Each rank streams its own seeded sky (weak scaling, no data-path collective)."""
    return int(rank)


def file_sha256(path):
    import hashlib
    try:
        return hashlib.sha256(open(path, "rb").read()).hexdigest()
    except OSError:
        return None


def traffic_from_profile(kernel: str, workload: str = None, bg: str = None):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel`, from the committed `ncu --set full`
    capture listed in profiles/traffic.json (never measured under the profiler in this run).  The entry names the CSV
    and the SHA-256 of the kernel source at capture time; a source that has changed since is reported, not hidden."""
    meta = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        e = json.load(open(meta))[kernel]
    except Exception:
        return None, {"source": None, "note": "no committed ncu capture for this kernel (profiles/traffic.json)"}
    if e.get("workload") and (workload != e["workload"] or (e.get("bg_kernel") and bg != e["bg_kernel"])):
        return None, {"source": e["csv"], "note": "the committed capture is of workload %s (%s): no per-launch figure for this one"
                      % (e["workload"], e.get("bg_kernel", "any kernel"))}
    src_now = file_sha256(os.path.join(ROOT, e["kernel_source"]))
    return float(e["dram_bytes_per_launch"]), {"source": e["csv"], "kernel_source": e["kernel_source"],
                                               "kernel_source_sha256_at_capture": e["kernel_source_sha256"],
                                               "kernel_source_unchanged": src_now == e["kernel_source_sha256"],
                                               "launch_config": e.get("launch_config")}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", d
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)", {}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the GPU is under load."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def mark(self):
        return time.time()

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons, pw = [], [], set(), []
        for (ts, ln) in self.rows:
            if t0 is not None and not (t0 <= ts <= t1 + 0.2):
                continue
            f = [x.strip() for x in ln.split(",")]
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except Exception:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples in timed region"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# algorithmic bytes / flops per launch of each kernel
def kernel_model(name: str, p: dict, n_valid: int):
    B, N = p["B"], p["Dy"] * p["Dx"]
    P = B + (1 if p["detect_sum_plane"] else 0)
    kmf, kbg = p["k_mf"], p["k_bg"]
    m = {
        "qc_pass1": (4 * B * N + 4 * N + N, 5 * B * N),     # moments + speculative sum plane: cube once, plane written, mask
        "qc_pass2": (4 * B * N + N, 6 * B * N),             # clip round: cube once, mask
        "sum_plane": (4 * B * N + 4 * N, B * N),
        "conv_mf": (8 * P * N, 2 * 2 * (2 * kmf + 1) * P * N),
        "conv_c": (8 * P * N, 2 * 2 * (2 * kbg + 1) * P * N),
        "conv_s": (12 * P * N, 2 * 2 * (2 * kbg + 1) * P * N),
        "conv_den": (5 * P * N, 2 * 2 * (2 * kbg + 1) * P * N),
        "threshold_peaks": (12 * P * N, 8 * P * N),
        # fused path: reads the cube (and the sum plane) once; flops = defined arithmetic per plane-voxel
        "fused_detect": (4 * P * N, (2 * 2 * (2 * kmf + 1) + 30) * P * N),
    }
    return m.get(name, (0, 0))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2103_15418_b200 import synth
    from paper_2103_15418_b200.binding import LPF, HostResult

    rank, world, local = env_rank()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    cfg = args.config
    s = synth.CubeStream(cfg, seed=rank_seed(rank))   # every rank: its own independent stream (weak scaling)
    p = synth.default_params(cfg, bg=args.bg, n_iter=args.n_iter)
    p["n_lanes"] = args.lanes
    p["n_back"] = args.n_back
    if args.zeta > 0:
        p.update(zeta_thr=args.zeta, zeta_nmax=8, zeta_window=64, zeta_warm=16)
    B, D = p["B"], p["Dy"]
    N = D * D
    cube_bytes = 4 * B * N
    n_pool = args.pool
    n_valid = int(s.mask.sum()) if s.mask is not None else N

    pool_h = torch.empty((n_pool, B, D, D), dtype=torch.float32, pin_memory=True)
    for i in range(n_pool):
        pool_h[i] = torch.from_numpy(s.frame(i))
    pool_d = pool_h.to(dev)
    lpf = LPF(p, s.mask, device=f"cuda:{local}")
    if s.forced_pix.size:
        lpf.add_candidates(s.forced_pix)
    lanes = args.lanes
    streams = [torch.cuda.Stream(device=dev) for _ in range(lanes)]
    main = torch.cuda.current_stream()

    def run_steps(t0, k):
        ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
        ev0.record(main)
        for st in streams:
            st.wait_event(ev0)
        for i in range(k):
            t = t0 + i
            lpf.process_frame(pool_d[t % n_pool], t, lane=t % lanes, stream=streams[t % lanes])
        for st in streams:
            e = torch.cuda.Event(); e.record(st); main.wait_event(e)
        ev1.record(main)
        return ev0, ev1

    sampler = ClockSampler(local)
    sampler.start()
    run_steps(0, args.warmup)
    t_next = args.warmup
    ts0 = sampler.mark()
    # The timed block is EXACTLY args.steps steps between a barrier + synchronize on both sides.  A short block
    # (< 100 ms: a few pipeline depths, dominated by fill and drain) is repeated and the MEDIAN block is reported
    # ("median of 5 repeats"); every repeat is bracketed the same way.
    blocks = []
    while True:
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        l0 = lpf.counters()["launches"]
        ev0, ev1 = run_steps(t_next, args.steps)
        t_next += args.steps
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        b_ms, b_l = reduce_over_ranks(ev0.elapsed_time(ev1), lpf.counters()["launches"] - l0, dev, world)
        blocks.append((b_ms, b_l))
        if len(blocks) >= args.repeats or (len(blocks) == 1 and b_ms >= 100.0 and args.repeats_auto):
            break
    ts1 = sampler.mark()
    blocks.sort()
    ms, launches = blocks[len(blocks) // 2]
    repeats = len(blocks)

    # keep the GPU under the same load until nvidia-smi has had time to sample it
    tload = time.time()
    while ms < 1500.0 and time.time() - tload < 1.6 - ms / 1e3:
        run_steps(t_next, 64); t_next += 64
        torch.cuda.synchronize()
    ts1b = sampler.mark()
    clocks = sampler.stop(ts0, max(ts1, ts1b))

    # per-kernel CUDA-event profile over the same step mix -> roofline of the dominant kernel
    # (one lane, one stream: each kernel runs alone, so its events bracket only its own execution)
    kp = min(args.steps, 200)
    torch.cuda.synchronize()
    lpf.profile_begin()
    for i in range(kp):
        lpf.process_frame(pool_d[(t_next + i) % n_pool], t_next + i, lane=0, stream=streams[0])
    t_next += kp
    prof = lpf.profile_end()
    kernels = {k: {"launches_per_step": c / kp, "us_per_launch": 1e3 * tm / c, "us_per_step": 1e3 * tm / kp}
               for k, (c, tm) in prof.items()}
    step_kernel_us = sum(v["us_per_step"] for v in kernels.values())
    dom = max(kernels, key=lambda k: kernels[k]["us_per_step"])
    hbm_peak, peak_src, _ = load_peaks()
    abytes, aflops = kernel_model(dom, p, n_valid)
    dur_s = kernels[dom]["us_per_launch"] * 1e-6
    gbs = abytes / dur_s / 1e9
    tfl = aflops / dur_s / 1e12
    t_hbm, t_alu = abytes / (hbm_peak * 1e9), aflops / (ALU_PEAK_TFLOPS * 1e12)
    if t_hbm >= t_alu:
        roof = {"bound": "hbm", "achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak}
    else:
        roof = {"bound": "alu", "achieved": tfl, "peak": ALU_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tfl / ALU_PEAK_TFLOPS}
    roof.update({"kernel": dom, "us_per_launch": kernels[dom]["us_per_launch"], "share_of_step": kernels[dom]["us_per_step"] / step_kernel_us,
                 "algorithmic_bytes": abytes, "algorithmic_flops": aflops, "hbm_gbs": gbs, "hbm_frac": gbs / hbm_peak,
                 "peak_source": peak_src, "alu_peak_source": "nominal (derived, not measured): 148 SM x 128 fp32 lanes x 2 x 1.965 GHz"})
    roof["traffic"], roof["traffic_source"] = traffic_from_profile(dom, s.c.name, args.bg)

    frames_s = whole_job_value(world, args.steps, ms)
    step_gbs = cube_bytes * frames_s / 1e9 / world
    # With several lanes in flight the plan gives one launch of the fused kernel only a share of the SMs
    # (n_sm / n_lanes: fewer, longer row segments), so a launch timed ALONE leaves most of the GPU idle.  The plain
    # per-launch figures above stand as measured; "occupancy" says how much of the GPU that launch could use, and
    # "in_timed_region" is the same kernel's work rate over the timed multi-lane region (all launches / wall time).
    if dom == "fused_detect":
        pl = lpf.plan()
        ctas = pl["ctas_per_plane"] * pl["planes"]
        smf = min(1.0, ctas / float(pl["sms"]))
        per_s = frames_s / world
        roof["occupancy"] = {"ctas_per_launch": ctas, "sms": pl["sms"], "sm_fraction": smf,
                             "frac_of_occupied_sms": roof["frac"] / smf}
        roof["in_timed_region"] = {"tflops": aflops * per_s / 1e12, "alu_frac": aflops * per_s / 1e12 / ALU_PEAK_TFLOPS,
                                   "hbm_gbs": abytes * per_s / 1e9, "hbm_frac": abytes * per_s / 1e9 / hbm_peak}

    # end to end through the host entry point: pinned host cube -> H2D -> path -> D2H of the results
    e2e = None
    if not args.no_e2e:
        # several frames in flight from the host: lane k's copy in overlaps the chain of the other lanes
        le = max(1, min(lanes, args.e2e_lanes))
        resl = [HostResult(p) for _ in range(le)]
        ke = max(3, min(args.steps, args.e2e_steps))

        def e2e_loop(k, t0):
            d2h = 0
            for i in range(k):
                ln = i % le
                if i >= le:
                    lpf.process_frame_host_end(resl[ln], lane=ln, stream=streams[ln]); d2h += resl[ln].d2h_bytes
                lpf.process_frame_host_begin(pool_h[i % n_pool], t0 + i, resl[ln], lane=ln, stream=streams[ln])
            for i in range(max(0, k - le), k):
                ln = i % le
                lpf.process_frame_host_end(resl[ln], lane=ln, stream=streams[ln]); d2h += resl[ln].d2h_bytes
            return d2h

        e2e_loop(2 * le, t_next); t_next += 2 * le
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        w0 = time.perf_counter()
        d2h = e2e_loop(ke, t_next); t_next += ke
        torch.cuda.synchronize()
        w1 = time.perf_counter()
        dt = w1 - w0
        if world > 1:
            tt = torch.tensor([dt], device=dev, dtype=torch.float64)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        e2e = {"value": world * ke / dt, "unit": UNIT, "h2d_bytes_per_step": cube_bytes, "d2h_bytes_per_step": d2h // ke,
               "steps": ke, "lanes": le,
               "api": "lpf_process_frame_host_begin/_end (pinned host cube in, results out; %d lanes in flight)" % le}

    out = {
        "metric": METRIC, "value": frames_s, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "timed_region_ms": ms, "repeats": repeats,
        "repeat_ms": [round(b[0], 4) for b in blocks], "repeat_rule": "median of the repeated timed blocks (each exactly `steps` steps)",
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": s.c.name, "cube": [B, D, D], "bg_kernel": args.bg, "n_iter": args.n_iter, "lanes": lanes, "n_back": args.n_back, "zeta_thr": args.zeta,
                   "pool_frames": n_pool, "pool_bytes": n_pool * cube_bytes,
                   "l2": "inputs larger than L2 (pool cycled, %d MB)" % (n_pool * cube_bytes >> 20),
                   "parallelism": "independent streams per GPU, no data-path collective" if world > 1 else "1 GPU"},
        "voxels_per_s": frames_s * B * N, "cube_gbs_per_gpu": step_gbs, "hbm_frac_step": step_gbs / hbm_peak,
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "kernels": kernels, "roofline": roof,
    }
    if rank == 0 and world == 1 and not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(cfg, args, seconds=args.cpu_seconds)
    lpf.close()
    if world > 1:
        dist.destroy_process_group()
    return out if rank == 0 else None


# ------------------------------------------------------------------------------------------------
def oracle_step_factory(cfg, bg, n_iter, crop):
    """One bounded sample of the workload for the CPU oracle: the whole chain on a centred crop of each frame
    (all bands).  Returns (step_fn, fraction_of_a_frame)."""
    import oracle as O
    from paper_2103_15418_b200 import synth
    s = synth.CubeStream(cfg)
    p = synth.default_params(cfg, bg=bg, n_iter=n_iter)
    D = p["Dy"]
    c = min(crop, D)
    y0 = (D - c) // 2
    p["Dy"] = p["Dx"] = c
    mask = None if s.mask is None else np.ascontiguousarray(s.mask[y0:y0 + c, y0:y0 + c])
    pipe = O.OraclePipeline(p, mask, direct=False)
    frames = [np.ascontiguousarray(s.frame(t)[:, y0:y0 + c, y0:y0 + c]) for t in range(2)]
    state = {"t": 0}

    def step():
        t = state["t"]; state["t"] += 1
        pipe.step(frames[t % len(frames)], t)
    return step, (c * c) / float(D * D), s.c.name, p


def cpu_baseline(cfg, args, seconds=12.0):
    """The oracle as it stands, one thread, on FULL frames of the workload (>= 3 of them); a crop only
    when --cpu-crop asks for one."""
    D = CONFIG_D(cfg)
    crop = D if args.cpu_crop <= 0 else min(D, args.cpu_crop)
    step, frac, name, p = oracle_step_factory(cfg, args.bg, args.n_iter, crop)
    step()
    n = 0; t0 = time.perf_counter()
    while True:
        step(); n += 1
        dt = time.perf_counter() - t0
        if (n >= 3 and dt >= seconds) or n >= 64:
            break
    what = "full %dx%d frames" % (D, D) if crop == D else "a centred %dx%d crop" % (crop, crop)
    return {"value": n * frac / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%d steps of the whole chain on %s of %s (all %d bands), float64 oracle (row-then-column form of the "
                      "window sums)%s" % (n, what, name, p["B"], "" if crop == D else ", scaled by crop/frame voxels"),
            "seconds": dt, "host_cpus": os.cpu_count()}


def run_reference(args):
    rank, world, _ = env_rank()
    if rank != 0:
        return None
    # Every step is one FULL frame of the workload when K + W of them end within ~3.5 minutes (6.5 s per 1024x1024x16
    # frame measured on the build container, cost ~ voxels); otherwise a centred crop sized to that bound.
    from paper_2103_15418_b200 import synth
    D = CONFIG_D(args.config)
    B = synth.default_params(args.config)["B"]
    n_steps = max(1, args.steps + min(args.warmup, 3))
    t_full = 6.5 * (B * D * D) / (16.0 * 1024 * 1024)
    if args.cpu_crop > 0:
        crop = min(D, args.cpu_crop)
    elif n_steps * t_full <= 210.0:
        crop = D
    else:
        crop = max(64, min(D, int(D * (210.0 / (n_steps * t_full)) ** 0.5) // 32 * 32))
    step, frac, name, p = oracle_step_factory(args.config, args.bg, args.n_iter, crop)
    for _ in range(min(args.warmup, 3)):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    v = args.steps * frac / dt
    what = "a full %dx%d frame" % (D, D) if crop == D else "a centred %dx%d crop" % (crop, crop)
    sample = ("each step = whole chain on %s of %s (all %d bands) with the float64 CPU oracle, 1 thread%s"
              % (what, name, p["B"], "" if crop == D else "; value scaled by crop/frame voxels"))
    return {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": name, "cube": [p["B"], D, D], "bg_kernel": args.bg, "n_iter": args.n_iter,
                       "sample_is_full_frame": crop == D},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}


def CONFIG_D(cfg):
    from paper_2103_15418_b200 import synth
    return synth.CONFIGS[cfg].D


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config (1-based); 3 = 1024x1024x16")
    ap.add_argument("--bg", default="box", choices=["box", "gauss"])
    ap.add_argument("--n-iter", dest="n_iter", type=int, default=1)
    ap.add_argument("--lanes", type=int, default=8)
    ap.add_argument("--pool", type=int, default=16)
    ap.add_argument("--n-back", dest="n_back", type=int, default=0,
                    help="backward fill from a device cache of the last n cubes (SURVEY 8(f1)); 0 = off (headline)")
    ap.add_argument("--zeta", type=float, default=0.0,
                    help="threshold of the per-pixel running QC of eq. A.2 (SURVEY 8(f2)); 0 = off (headline)")
    ap.add_argument("--e2e-steps", type=int, default=64)
    ap.add_argument("--e2e-lanes", dest="e2e_lanes", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--cpu-crop", dest="cpu_crop", type=int, default=0, help="0 = full frames; else the oracle runs on a centred crop")
    ap.add_argument("--repeats", type=int, default=0,
                    help="timed blocks (each exactly --steps steps); 0 = automatic: 5 when a block is shorter than 100 ms, else 1")
    args = ap.parse_args()
    args.repeats_auto = args.repeats <= 0
    if args.repeats_auto:
        args.repeats = 5
    if args.warmup < 3:
        args.warmup = 3
    out = run_reference(args) if args.impl == "reference" else run_ours(args)
    if out is not None:
        print(json.dumps(out))


if __name__ == "__main__":
    main()
