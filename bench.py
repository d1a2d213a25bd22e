#!/usr/bin/env python
"""bench.py -- PCA images/s (input frames/s) at 1024^2 x 32 uint16 (BASELINE.json metric), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--api submit|process|push]
                  [--mode 1|2|3]

A "step" is one pass of the whole hot path (A0..A6) over one stack of T frames (`--api push`: one window of the
sliding-window form, `stride` new frames).  The stream is resident in HBM before the timed region and is cycled
through; it is sized to at least 3x the 126 MB L2, so no step finds its inputs in L2 (`config.l2_policy` states
the sizes).  N > 1 (torchrun): one process per GPU, each with its own stream of stacks, no data-path collective
(weak scaling); timing is bracketed by a barrier and reported as the max over ranks.
`--impl reference` times the CPU oracle (oracle/) on host cores on a bounded sample.
"""
import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

PAPER_IMAGES_PER_S = 20.0        # "up to 20" PCA images/s, Titan RTX
L2_BYTES = 126e6                 # B200_PROFILING.md
FP32_PEAK_MEASURED_TFLOPS = 72.0 # profiles/r01_ubench_peaks.txt (register-only FFMA, csrc/ubench_peaks.cu); nominal 74.4
FP32_LANES_PER_SM = 128


def metric_name(cfg):
    return f"PCA images/s at {cfg.n}x{cfg.n}x{cfg.T} uint16 (input frames/s = {cfg.stride}x)"


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", d
    return 6650.0, "fallback (B200_PROFILING.md)", {}


# ------------------------------------------------------------------------------------------------------------
# rank / shard logic of the GPU arm (no GPU needed: tests/test_host_logic.py runs it under gloo, world_size 2)
# ------------------------------------------------------------------------------------------------------------
def rank_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0")))


def shard_plan(cfg, rank, world, stacks=None, min_resident_bytes=3 * L2_BYTES):
    """What one rank holds and cycles through.  Stacks are independent units: every rank generates its OWN stream
    (seed 1000 + rank) of the same shape -- weak scaling, no data-path collective.  The resident stream is at least
    `min_resident_bytes` long (>= 3x L2), extended beyond the config's stream length with the same generator if needed."""
    T, n = cfg.T, cfg.n
    fbytes = T * n * n * 2
    n_stacks = stacks or max(cfg.n_frames // T, int(math.ceil(min_resident_bytes / fbytes)))
    n_frames = n_stacks * T
    n_win = (n_frames - T) // cfg.stride + 1           # windows a step can start at (stride < T: overlapping)
    n_push = (n_frames - T) // cfg.stride              # pushes that fit after the first window
    return {"seed": 1000 + rank, "n_stacks": n_stacks, "n_frames": n_frames, "n_win": n_win, "n_push": n_push,
            "stack_bytes": fbytes, "resident_bytes": n_stacks * fbytes, "window_stride_bytes": cfg.stride * n * n * 2}


def reduce_max_ms(ms, dist=None, device=None):
    """Max over ranks of a device-timed duration (every rank must call)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(world, steps, ms_max):
    """Whole-job throughput: every rank did `steps` units in (at most) ms_max."""
    return world * steps / (ms_max * 1e-3)


def l2_policy(plan):
    return (f"inputs larger than L2: {plan['resident_bytes'] / 1e6:.0f} MB resident stream cycled through "
            f"({plan['resident_bytes'] / L2_BYTES:.1f}x the 126 MB L2), no flush needed")


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "50"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.06)
        self.proc.terminate()
        mhz, mx, reasons, power = [], None, set(), []
        for (ts, ln) in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                mx = float(f[1])
                if t0 - 0.02 <= ts <= t1 + 0.06:
                    mhz.append(float(f[0]))
                    power.append(float(f[2]))
                    for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[3:7]):
                        if v.lower().startswith("active"):
                            reasons.add(name)
            except ValueError:
                continue
        mhz.sort()
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": mx, "samples": len(mhz),
                "power_w_max": max(power) if power else None, "reasons": sorted(reasons)}


def stage_bytes(cfg, mode=1):
    """Algorithmic (compulsory) bytes per stack and stage, SURVEY.md 8(d) / DESIGN.md.  mode 2 (Gram from the raw
    frames, SURVEY.md 8(f)-2 stage 1) has no covariance read of the hologram stack: 20 T N_p + 12 N_p.  mode 3 (stage 2:
    no hologram stack) reads the frames three times (Gram + sum, deflation images, row pass), writes and reads the
    row-pass output once and writes the image: 22 T N_p + (16 + 8 n_rej) N_p with n_rej rejected components."""
    npix, T = cfg.n * cfg.n, cfg.T
    if mode == 3:
        nrej = (cfg.k_lo - 1) + (T - cfg.k_hi)
        d = {"sum": 2 * T * npix + 4 * npix, "defl": (2 * T * npix + 4 * npix + 4 * nrej * npix) if nrej else 0,
             "rows": 2 * T * npix + 4 * npix + 4 * nrej * npix + 8 * T * npix, "cols": 8 * T * npix + 4 * npix, "eig": 16 * T * T}
        d["total"] = d["sum"] + d["defl"] + d["rows"] + d["cols"]
        d["fft"], d["proj"], d["cov"] = d["rows"], 0, 0
        return d
    d = {"sum": 2 * T * npix + 4 * npix, "fft": 2 * T * npix + 4 * npix + 8 * T * npix,
         "cov": 8 * T * npix if mode == 1 else 0, "eig": 16 * T * T, "proj": 8 * T * npix + 4 * npix}
    d["total"] = d["sum"] + d["fft"] + d["cov"] + d["proj"]
    return d


def run_reference(args, cfg):
    """CPU oracle arm: each step = the oracle on a bounded sample (a crop of n_s x n_s pixels of one stack, all T
    frames), scaled to full-frame images/s by the pixel ratio."""
    rank, world, _ = rank_env()
    if rank != 0:
        return
    import numpy as np
    import oracle
    from gen import holo_gen as G
    steps, warmup = args.steps or 3, args.warmup if args.warmup is not None else 1
    budget_s = 150.0
    scene = G.make_scene(cfg, 0)
    frames = G.frames_np(scene, 0, cfg.T)
    c0 = frames[:, :128, :128].copy()
    t = time.time(); oracle.process(c0, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi); t128 = time.time() - t
    n_s = cfg.n
    while n_s > 128 and t128 * (n_s / 128) ** 2 * 1.15 * (steps + warmup) > budget_s:
        n_s //= 2
    crop = np.ascontiguousarray(frames[:, :n_s, :n_s])
    for _ in range(warmup):
        oracle.process(crop, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
    t0 = time.time()
    for _ in range(steps):
        oracle.process(crop, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
    dt = time.time() - t0
    frac = (n_s * n_s) / float(cfg.n * cfg.n)
    value = steps / dt * frac
    sample = f"{n_s}x{n_s}x{cfg.T} crop of one {cfg.name} stack per step ({frac:.4g} of a full stack), scaled by pixel ratio"
    cores = oracle.num_threads()
    print(json.dumps({
        "impl": "reference", "metric": metric_name(cfg), "value": value, "unit": "images/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": dt / steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": value / PAPER_IMAGES_PER_S if cfg.name.startswith("cfg3") else None,
        "vs_baseline_note": "paper's figure on another machine (Titan RTX): context, not the target",
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "nx": cfg.n, "ny": cfg.n, "T": cfg.T, "k_lo": cfg.k_lo, "k_hi": cfg.k_hi},
        "cpu_baseline": {"value": value, "unit": "images/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "images/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


KCLASS = ["sum", "fft_rows", "fft_cols", "cov_partial", "cov_reduce", "eig", "project"]


def kernel_name(cls, fused_fft, cov_real, mode, T=32, n=1024, packed=False):
    cov_tc = T > 32 or (T == 32 and n * n >= (1 << 18))      # the library's default policy (holo_tune key 13)
    if mode != 3 and packed:
        return {"sum": "k_frame_sum" if mode == 1 else "k_sum_gram", "fft_rows": f"k_rows2<{n}> (packed row pass of the stack)",
                "fft_cols": "k_cols_tiled<1024> (column pass from 8-column blocks)" if n == 1024 else "k_cols2048 (packed column pass)",
                "cov_partial": ("k_cov_tf32_tma" if cov_tc else "k_cov_partial_real") if cov_real else "k_cov_partial",
                "cov_reduce": "k_cov_reduce" if mode == 1 else "k_gram_reduce_finish", "eig": "k_eig_real" if cov_real else "k_eig",
                "project": "k_project_deflate_tma / k_project"}[cls]
    if mode == 3:
        rows = "k_rows2" if (n == 1024 and T % 2 == 0) or n == 2048 else "k_fft<rows, deflating prologue>"
        return {"sum": "k_sum_gram + k_deflate_images", "fft_rows": rows, "fft_cols": "k_col_energy",
                "cov_reduce": "k_gram_reduce_finish", "eig": "k_eig_real", "project": "k_sum_partial_images"}[cls]
    return {"sum": "k_frame_sum" if mode == 1 else "k_sum_gram", "fft_rows": "k_fresnel" if fused_fft else "k_fft<rows>",
            "fft_cols": "k_fft<cols>", "cov_partial": ("k_cov_tf32_tma" if cov_tc else "k_cov_partial_real") if cov_real else "k_cov_partial",
            "cov_reduce": "k_cov_reduce" if mode == 1 else "k_gram_reduce_finish", "eig": "k_eig_real" if cov_real else "k_eig",
            "project": "k_project_deflate_tma / k_project"}[cls]


def _traffic_table():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the round's `ncu --set full` capture
    (profiles/r02_traffic.csv: workload,kernel class,bytes; see profiles/r02.md for the command)."""
    tab = {}
    p = os.path.join(ROOT, "profiles", "r02_traffic.csv")
    if os.path.exists(p):
        for ln in open(p).read().splitlines()[1:]:
            f = ln.split(",")
            if len(f) == 3:
                tab[(f[0], f[1])] = int(f[2])
    return tab


class Runner:
    """One handle + one resident stream of one config; times K steps of one API on a stream."""

    def __init__(self, cfg, plan, dev, tune=(), mode=1, frames=None):
        import torch
        from gen import holo_gen as G
        from paper_2004_00923_b200 import Holo
        self.torch, self.cfg, self.plan, self.dev = torch, cfg, plan, dev
        self.frames = frames if frames is not None else G.stream_torch(cfg, plan["seed"], dev, n_frames=plan["n_frames"])
        torch.cuda.synchronize()
        self.h = Holo(cfg.n, cfg.n, cfg.T, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
        for kv in tune:
            k, v = kv.split("=")
            self.h.tune(int(k), int(v))
        if mode != 1:
            self.h.set_mode(mode)
        self.images = torch.empty((4, cfg.n, cfg.n), dtype=torch.float32, device=dev)
        self.st = torch.cuda.Stream(device=dev)

    def step(self, api, i):
        cfg, p, h, fr = self.cfg, self.plan, self.h, self.frames
        if api == "push":
            # sliding window: `stride` new frames per step; once per cycle of the resident stream the sequence
            # restarts with a whole window (a re-reference, counted as a step)
            k = i % (p["n_push"] + 1)
            if k == 0:
                h.push(fr.data_ptr(), cfg.T, self.images[i % 4], self.st)
            else:
                h.push(fr.data_ptr() + (cfg.T + (k - 1) * cfg.stride) * cfg.n * cfg.n * 2, cfg.stride, self.images[i % 4], self.st)
        elif api == "submit":
            h.submit(fr.data_ptr() + (i % p["n_win"]) * p["window_stride_bytes"], self.images[i % 4], self.st)
        else:
            h.process(fr.data_ptr() + (i % p["n_win"]) * p["window_stride_bytes"], self.images[i % 4], self.st)

    def timed(self, api, steps, warmup, barrier, sampler=None):
        torch = self.torch
        for i in range(warmup):
            self.step(api, i)
        self.h.flush(self.st)
        barrier()
        t0 = time.time()
        if sampler:
            sampler.start()
            time.sleep(0.12)
            t0 = time.time()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.st)
        for i in range(steps):
            self.step(api, i)
        self.h.flush(self.st)                  # the last image is part of the timed region
        e1.record(self.st)
        barrier()
        clocks = sampler.stop(t0, time.time()) if sampler else None
        return e0.elapsed_time(e1), clocks

    def image_of_first_stack(self, api):
        """The image of the first resident stack/window through the SAME entry point that was timed."""
        torch, cfg = self.torch, self.cfg
        M = torch.zeros((cfg.n, cfg.n), dtype=torch.float32, device=self.dev)
        if api == "push":
            self.h.push(self.frames.data_ptr(), cfg.T, M, self.st)
        elif api == "submit":
            self.h.submit(self.frames.data_ptr(), M, self.st)
        else:
            self.h.process(self.frames.data_ptr(), M, self.st)
        self.h.flush(self.st)
        self.st.synchronize()
        return M

    def oracle_check(self, api):
        import numpy as np
        import oracle
        torch, cfg = self.torch, self.cfg
        fr = self.frames[:cfg.T].cpu().view(torch.int16).numpy().view(np.uint16)
        t0 = time.time()
        out = oracle.process(fr, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
        dt = time.time() - t0
        Mg = self.image_of_first_stack(api).cpu().numpy()
        err = float(np.linalg.norm(Mg - out["M"]) / np.linalg.norm(out["M"]))
        return dt, err

    def close(self):
        self.h.close()


def run_ours(args, cfg):
    import torch
    from gen import holo_gen as G

    rank, world, local_rank = rank_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    steps = args.steps or 2048
    warmup = max(args.warmup if args.warmup is not None else 64, 3)
    api, mode = args.api, args.mode
    plan = shard_plan(cfg, rank, world, args.stacks)
    T, n = cfg.T, cfg.n
    R = Runner(cfg, plan, dev, args.tune, mode)
    h = R.h
    sampler = ClockSampler(local_rank if "CUDA_VISIBLE_DEVICES" not in os.environ else
                           int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
    ms, clocks = R.timed(api, steps, warmup, barrier, sampler)
    ms = reduce_max_ms(ms, dist, dev)
    rc, status = h.status(R.st)
    value = aggregate_value(world, steps, ms)

    # ---- per-kernel-class device times (library's own event brackets; second, instrumented pass).  The brackets
    # are only meaningful without kernel concurrency: the instrumented pass uses the serial entry point (same
    # kernels; in the streaming forms the projection and the eigensolver overlap other kernels on purpose)
    prof_steps = min(steps, 64)
    h.tune(5, 1)
    for i in range(prof_steps):
        R.step("process", i)
    prof = h.profile_read()
    h.tune(5, 0)
    sb = stage_bytes(cfg, mode)
    npix = n * n
    G_fft = h.fft_group()
    hbm_peak, peak_src, peaks = _peaks()
    num_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    fp32_peak_tflops = FP32_PEAK_MEASURED_TFLOPS * num_sms / 148.0
    fused_fft = prof[2][1] == 0 and mode != 3   # no separate column-pass launches: one persistent kernel does A1+A2 of all T frames
    # packed pair (1024^2, 2048^2): ONE row-pass and ONE column-pass launch per stack, the row-pass output of the whole stack
    # goes through HBM: the kernels' own compulsory bytes are frames + S + 8 T N_p (rows) and 8 T N_p + 8 T N_p (columns)
    packed = mode != 3 and not fused_fft and prof[1][1] == prof_steps and prof[2][1] == prof_steps
    cov_real = "8=0" not in args.tune
    per_launch_bytes = {"sum": sb["sum"], "fft_rows": sb["fft"] if fused_fft or packed else 2 * G_fft * npix + 4 * npix * G_fft / T,
                        "fft_cols": 16 * T * npix if packed else 8 * G_fft * npix, "cov_partial": 8 * T * npix, "cov_reduce": 0,
                        "eig": sb["eig"], "project": sb["proj"]}
    if mode == 3:       # "sum" brackets two launches (Gram + sum, deflation images): their mean; "project" is the partial-image sum
        per_launch_bytes.update({"sum": (sb["sum"] + sb["defl"]) / 2, "fft_rows": sb["rows"], "fft_cols": sb["cols"], "project": 12 * npix})
    stages = {}
    tot_ms = sum(p[0] for p in prof) or 1.0
    for name, (ms_k, cnt) in zip(KCLASS, prof):
        if cnt == 0:
            continue
        us = ms_k / cnt * 1e3
        stages[name] = {"kernel": kernel_name(name, fused_fft, cov_real, mode, T, n, packed), "us_per_launch": round(us, 2),
                        "launches_per_step": cnt / prof_steps, "share": round(ms_k / tot_ms, 4),
                        "GBps": round(per_launch_bytes[name] / (us * 1e-6) / 1e9, 1)}
    cov_flops = (2 if cov_real else 4) * T * (T + 1) * npix
    if "cov_partial" in stages:
        stages["cov_partial"]["form"] = "real part (2T(T+1) flop/pixel)" if cov_real else "complex Hermitian half (4T(T+1) flop/pixel)"
        stages["cov_partial"]["TFLOPs_fp32"] = round(cov_flops / (stages["cov_partial"]["us_per_launch"] * 1e-6) / 1e12, 2)
    fft_flops = 10.0 * T * npix * math.log2(n)          # 5 N log2 N per 1-D transform, rows + columns
    if "fft_rows" in stages and fused_fft:
        stages["fft_rows"]["TFLOPs_fp32"] = round(fft_flops / (stages["fft_rows"]["us_per_launch"] * 1e-6) / 1e12, 2)
    dom = max(stages, key=lambda k: stages[k]["share"])
    traffic = _traffic_table().get((cfg.name + ("_mode3" if mode == 3 else ""), dom))
    if dom == "cov_partial" and T <= 32 and cov_flops / (8 * T * npix) > fp32_peak_tflops * 1e12 / (hbm_peak * 1e9):
        roof = {"kernel": stages[dom]["kernel"], "bound": "alu", "achieved": stages[dom]["TFLOPs_fp32"], "peak": round(fp32_peak_tflops, 1),
                "unit": "TFLOP/s", "frac": round(stages[dom]["TFLOPs_fp32"] / fp32_peak_tflops, 4), "traffic": traffic,
                "peak_source": "measured register-only FFMA rate (profiles/r01_ubench_peaks.txt; nominal 148 SMs x 128 lanes x 2 x 1.965 GHz = 74.4)",
                "hbm_frac": round(stages[dom]["GBps"] / hbm_peak, 4)}
    else:
        roof = {"kernel": stages[dom]["kernel"], "bound": "hbm", "achieved": stages[dom]["GBps"], "peak": hbm_peak, "unit": "GB/s",
                "frac": round(stages[dom]["GBps"] / hbm_peak, 4), "traffic": traffic, "peak_source": peak_src,
                "us_per_launch": stages[dom]["us_per_launch"], "algorithmic_bytes_per_launch": per_launch_bytes[dom]}
        if dom == "fft_rows" and "TFLOPs_fp32" in stages[dom]:
            roof["alu_achieved_TFLOPs"] = stages[dom]["TFLOPs_fp32"]
            roof["alu_frac"] = round(stages[dom]["TFLOPs_fp32"] / fp32_peak_tflops, 4)
    if packed and "fft_rows" in stages and "fft_cols" in stages:
        # the Fresnel STAGE against the path's algorithmic bytes (frames + S in, holograms out); the two
        # kernels move 2.6x that, the row-pass output of the stack going through HBM
        us_st = stages["fft_rows"]["us_per_launch"] + stages["fft_cols"]["us_per_launch"]
        roof["fresnel_stage"] = {"kernels": [stages["fft_rows"]["kernel"], stages["fft_cols"]["kernel"]], "us": round(us_st, 2),
                                 "algorithmic_bytes": sb["fft"], "moved_bytes": per_launch_bytes["fft_rows"] + per_launch_bytes["fft_cols"],
                                 "frac_algorithmic": round(sb["fft"] / (us_st * 1e-6) / 1e9 / hbm_peak, 4),
                                 "frac_moved": round((per_launch_bytes["fft_rows"] + per_launch_bytes["fft_cols"]) / (us_st * 1e-6) / 1e9 / hbm_peak, 4)}
    e2e_gbps = sb["total"] * (steps / (ms * 1e-3)) / 1e9

    # ---- end to end through the host entry point (pinned host buffers, H2D + D2H inside the timed region)
    e2e = None
    streaming = api != "process"
    if not args.no_e2e:
        n_host = 2
        host_frames = torch.empty((n_host, T, n, n), dtype=torch.int16).pin_memory()
        host_frames.copy_(R.frames[:n_host * T].view(torch.int16).reshape(n_host, T, n, n).cpu())
        host_img = torch.empty((2, n, n), dtype=torch.float32).pin_memory()
        k2 = max(3, min(args.e2e_steps, steps))

        def e2e_step(i):
            if streaming:
                h.submit_host(host_frames[i % n_host], host_img[i % 2], R.st)
            else:
                h.process_host(host_frames[i % n_host], host_img[i % 2], R.st)

        for i in range(3):
            e2e_step(i)
        if streaming:
            h.flush_host(R.st)
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(R.st)
        for i in range(k2):
            e2e_step(i)
        if streaming:
            h.flush_host(R.st)                 # the last image reaches the host inside the timed region
        a1.record(R.st)
        barrier()
        ms2 = reduce_max_ms(a0.elapsed_time(a1), dist, dev)
        e2e = {"value": aggregate_value(world, k2, ms2), "unit": "images/s", "h2d_bytes_per_step": plan["stack_bytes"],
               "d2h_bytes_per_step": n * n * 4, "steps": k2, "ms_per_step": ms2 / k2,
               "api": ("holo_submit_host/holo_flush_host (pinned host frames -> host images; the H2D copy of stack i runs under "
                       "the kernels of stack i-1)") if streaming else "holo_process_host (pinned host frames -> host image, synchronous)"}

    # ---- CPU oracle on the box's host cores (rank 0, N = 1 only): a reported baseline, not the target.  The GPU image
    # it is compared with comes from the entry point that was timed.
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle
        dt, err = R.oracle_check(api)
        cpu = {"value": 1.0 / dt, "unit": "images/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"1 full stack of {cfg.name} (the first of the GPU stream), {dt:.2f} s", "rel_l2_M_vs_gpu": err,
               "gpu_api_compared": api}

    # ---- the other BASELINE.json configs and the paper's own filter window, short runs (rank 0, N = 1 only)
    side = None
    if rank == 0 and world == 1 and args.side and cfg.name.startswith("cfg3") and api == "submit":
        side = {}
        # the paper's window: ascending n1 = 1 .. n2 = 20 of 32 = descending k in [13, 32]: direct projection
        h.set_range(13, 32)
        ms_w, _ = R.timed("submit", 64, 8, barrier)
        h.set_range(cfg.k_lo, cfg.k_hi)
        side["cfg3_paper_window_k13_32"] = {"ms_per_step": ms_w / 64, "images_per_s": 64 / (ms_w * 1e-3),
                                            "note": "same stream, component window of PAPER.md:86 (direct projection kernel)"}
        # the same window through mode 3 (eigen-basis form: 20 transforms of the kept components' raw-domain images)
        R3 = Runner(cfg, plan, dev, args.tune, 3, frames=R.frames)
        R3.h.set_range(13, 32)
        ms_w3, _ = R3.timed("submit", 256, 8, barrier)
        side["cfg3_paper_window_k13_32_mode3"] = {"ms_per_step": ms_w3 / 256, "images_per_s": 256 / (ms_w3 * 1e-3), "mode": 3,
                                                  "note": "same stream and window, mode 3"}
        R3.close()
        del R3
    lib_ctx = None
    if rank == 0 and world == 1 and args.side and cfg.name.startswith("cfg3"):
        lib_ctx = library_context(torch, R, barrier)
    status_cycles = h.workspace_tensor(5).cpu().tolist()[4:7]
    launches = h.launches_per_process()
    R.close()
    del R
    torch.cuda.empty_cache()
    if side is not None:
        # (config, api, steps, resident stacks): streams of >= 3x L2, kept short so that the default run ends in minutes
        for cn, sapi, ssteps, sstacks, smode in ((3, "submit", 512, 0, 2), (3, "submit", 512, 0, 3), (2, "submit", 256, 24, 1), (2, "submit", 256, 24, 3), (4, "push", 256, 16, 1),
                                                 (5, "submit", 24, 3, 1), (5, "submit", 24, 3, 3)):
            c2 = G.CONFIGS[cn]
            p2 = shard_plan(c2, rank, world, stacks=sstacks or None)
            R2 = Runner(c2, p2, dev, mode=smode)
            ms_s, _ = R2.timed(sapi, ssteps, 6, barrier)
            sb2 = stage_bytes(c2, smode)
            ent = {"api": sapi, "mode": smode, "ms_per_step": ms_s / ssteps, "images_per_s": ssteps / (ms_s * 1e-3), "resident_bytes": p2["resident_bytes"]}
            if sapi != "push":
                ent["roofline_end_to_end_frac"] = round(sb2["total"] * (ssteps / (ms_s * 1e-3)) / 1e9 / hbm_peak, 4)
                ent["bytes_per_step"] = sb2["total"]
            else:
                ent["new_frames_per_s"] = c2.stride * ssteps / (ms_s * 1e-3)
            if not args.no_cpu:
                dt2, err2 = R2.oracle_check(sapi)
                ent["oracle_rel_l2_M_first_stack"] = err2
                ent["oracle_s_per_stack"] = round(dt2, 2)
            side[c2.name + (f"_mode{smode}" if smode != 1 else "")] = ent
            R2.close()
            del R2
            torch.cuda.empty_cache()

    if rank == 0:
        line = {
            "metric": metric_name(cfg), "value": value, "unit": "images/s", "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": value / PAPER_IMAGES_PER_S if cfg.name.startswith("cfg3") else None,
            "vs_baseline_note": "paper's 'up to 20 images/s' on a Titan RTX (PAPER.md:13,96): another machine, context only",
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "nx": n, "ny": n, "T": T, "k_lo": cfg.k_lo, "k_hi": cfg.k_hi, "mode": mode,
                       "stacks_resident": plan["n_stacks"], "windows": plan["n_win"], "stride_frames": cfg.stride,
                       "resident_input_bytes": plan["resident_bytes"], "l2_policy": l2_policy(plan),
                       "parallelism": f"replicas x{world} (independent stacks, no collective)", "fft_group": G_fft,
                       "api": {"submit": "holo_submit/holo_flush (stream of stacks, software-pipelined)",
                               "push": "holo_push (sliding window, stride %d: only the new frames are transformed)" % cfg.stride,
                               "process": "holo_process (one stack per call, strictly serial)"}[api]},
            "frames_per_s": value * cfg.stride, "clocks": clocks, "e2e": e2e,
            "gpu_launches": steps * launches, "launches_per_step": launches,
            "roofline": roof, "roofline_end_to_end": {"bound": "hbm", "achieved": round(e2e_gbps, 1), "peak": hbm_peak, "unit": "GB/s",
                                                      "frac": round(e2e_gbps / hbm_peak, 4), "bytes_per_step": sb["total"], "peak_source": peak_src},
            "stages": stages, "stages_note": "per-kernel device time from an instrumented pass of serial holo_process calls (each kernel alone on the GPU)",
            "cpu_baseline": cpu, "eig_status": status, "eig_cycles": status_cycles, "configs": side, "library_context": lib_ctx,
            "paper_context": {"images_per_s": PAPER_IMAGES_PER_S, "input_frames_per_s": 500, "hardware": "NVIDIA Titan RTX (PAPER.md:96)"},
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def library_context(torch, R, barrier):
    """Context only, never on the library path: the paper's own decomposition (cuFFT + cublasCgemm +
    cusolverDnCheevd) written with torch library calls on the same B200 and the same resident stacks."""
    cfg = R.cfg
    T, n = cfg.T, cfg.n
    try:
        qx = R.h.workspace_tensor(6)
        qy = R.h.workspace_tensor(7)
        q = (qy[:, None] * qx[None, :]).contiguous()

        def one(i):
            fr = R.frames[(i % R.plan["n_stacks"]) * T:(i % R.plan["n_stacks"] + 1) * T].view(torch.int16).to(torch.float32)
            d = fr - fr.mean(0, keepdim=True)
            H = torch.fft.fft2(d * q)
            Hm = H.reshape(T, -1)
            C = Hm.conj() @ Hm.T
            ev, V = torch.linalg.eigh(C)
            P = (Hm.T @ V[:, :T - cfg.k_lo + 1])                  # ascending order: drop the k_lo-1 largest
            return (P.real ** 2 + P.imag ** 2).sum(1).reshape(n, n)

        for i in range(3):
            one(i)
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        k = 16
        e0.record()
        for i in range(k):
            one(i)
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        return {"images_per_s": k / (ms * 1e-3), "ms_per_step": ms / k,
                "what": "torch.fft.fft2 + complex matmul + torch.linalg.eigh + matmul on the same GPU (the paper's library decomposition); context, not a target"}
    except Exception as e:                                       # a missing library must not break the bench line
        return {"unavailable": str(e)[:200]}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--mode", type=int, default=1, choices=[1, 2, 3],
                    help="1: prescribed stage decomposition (default); 2: Gram from the raw frames (SURVEY.md 8(f)-2 stage 1); "
                         "3: 2 + image without a hologram stack (stage 2)")
    ap.add_argument("--stacks", type=int, default=None, help="resident stacks (default: >= 3x L2)")
    ap.add_argument("--e2e-steps", type=int, default=24)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-side", dest="side", action="store_false", help="skip the short runs of the other configs")
    ap.add_argument("--api", default="submit", choices=["submit", "process", "push"],
                    help="submit: streaming form (default); process: one serial holo_process per stack; push: sliding window")
    ap.add_argument("--tune", action="append", default=[], help="experiment knob key=value (holo_tune), repeatable")
    args = ap.parse_args()
    from gen import holo_gen as G
    cfg = G.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
