#!/usr/bin/env python
"""bench.py -- PCA images/s (input frames/s) at 1024^2 x 32 uint16 (BASELINE.json metric), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

A "step" is one pass of the whole hot path (A0..A6, holo_process) over one stack of T frames.
The stream (BASELINE.json configs[2]: 64 stacks = 2048 frames = 4 GiB of uint16) is resident in HBM
before the timed region and is cycled through, so the inputs are far larger than L2 (126 MB).
N > 1 (torchrun): one process per GPU, each with its own stream, no data-path collective (weak
scaling); timing is bracketed by a barrier and reported as the max over ranks.
`--impl reference` times the CPU oracle (oracle/) on host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "PCA images/s at 1024x1024x32 uint16 (input frames/s = 32x)"
PAPER_IMAGES_PER_S = 20.0        # "up to 20" PCA images/s, Titan RTX


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", d
    return 6650.0, "fallback (B200_PROFILING.md)", {}


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


def stage_bytes(cfg):
    """Algorithmic (compulsory) bytes per stack and stage, SURVEY.md 8(d) / DESIGN.md."""
    npix, T = cfg.n * cfg.n, cfg.T
    return {"sum": 2 * T * npix + 4 * npix, "fft": 2 * T * npix + 4 * npix + 8 * T * npix,
            "cov": 8 * T * npix, "eig": 16 * T * T, "proj": 8 * T * npix + 4 * npix,
            "total": 28 * T * npix + 12 * npix}


def run_reference(args, cfg):
    """CPU oracle arm: each step = the oracle on a bounded sample (a centred crop of n_s x n_s pixels of
    one stack, all T frames), scaled to full-frame images/s by the pixel ratio."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import numpy as np
    import oracle
    from gen import holo_gen as G
    steps, warmup = args.steps or 3, args.warmup if args.warmup is not None else 1
    budget_s = 150.0
    scene = G.make_scene(cfg, 0)
    frames = G.frames_np(scene, 0, cfg.T)
    # calibrate on a 128^2 crop, then pick the largest power-of-two crop that fits the budget
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
        "impl": "reference", "metric": METRIC, "value": value, "unit": "images/s", "n_gpus": args.gpus,
        "steps": steps, "warmup": warmup, "ms_per_step": dt / steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": value / PAPER_IMAGES_PER_S, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "nx": cfg.n, "ny": cfg.n, "T": cfg.T, "k_lo": cfg.k_lo, "k_hi": cfg.k_hi},
        "cpu_baseline": {"value": value, "unit": "images/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "images/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


KCLASS = ["sum", "fft_rows", "fft_cols", "cov_partial", "cov_reduce", "eig", "project"]
FP32_LANES_PER_SM = 128          # B200 SM: 4 SMSP x 32 FP32 lanes (blackwell guide / B300_MICROARCH.md)


def run_ours(args, cfg):
    import numpy as np
    import torch
    from gen import holo_gen as G
    from paper_2004_00923_b200 import Holo

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    steps = args.steps or 2048
    warmup = args.warmup if args.warmup is not None else 64
    warmup = max(warmup, 3)
    T, n = cfg.T, cfg.n
    n_stacks = min(args.stacks or (cfg.n_frames // T), cfg.n_frames // T)
    frames = G.stream_torch(cfg, 1000 + rank, dev, n_frames=n_stacks * T)
    torch.cuda.synchronize()
    h = Holo(n, n, T, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
    for kv in args.tune:
        k, v = kv.split("=")
        h.tune(int(k), int(v))
    images = torch.empty((4, n, n), dtype=torch.float32, device=dev)
    st = torch.cuda.Stream(device=dev)
    fbytes = T * n * n * 2
    # stacks may overlap (config 4: stride 8 over the stream): step i starts at frame (i mod n_win) * stride
    n_win = (n_stacks * T - T) // cfg.stride + 1
    wbytes = cfg.stride * n * n * 2

    streaming = args.api == "submit"

    pushing = args.api == "push"
    n_push = (n_stacks * T - T) // cfg.stride          # pushes that fit in the resident stream after the first window

    def step(i):
        # one stack through the whole path; the streaming form delivers image i during step i+1 (or the flush)
        if pushing:
            # sliding window: only `stride` new frames per step; the stream is cycled, so once per cycle the
            # sequence restarts with a whole window (a re-reference, counted as a step)
            k = i % (n_push + 1)
            if k == 0:
                h.push(frames.data_ptr(), T, images[i % 4], st)
            else:
                h.push(frames.data_ptr() + (T + (k - 1) * cfg.stride) * n * n * 2, cfg.stride, images[i % 4], st)
        elif streaming:
            h.submit(frames.data_ptr() + (i % n_win) * wbytes, images[i % 4], st)
        else:
            h.process(frames.data_ptr() + (i % n_win) * wbytes, images[i % 4], st)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for i in range(warmup):
        step(i)
    h.flush(st)
    barrier()
    sampler = ClockSampler(local_rank if "CUDA_VISIBLE_DEVICES" not in os.environ else
                           int(os.environ["CUDA_VISIBLE_DEVICES"].split(",")[local_rank]))
    sampler.start()
    time.sleep(0.12)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_wall0 = time.time()
    e0.record(st)
    for i in range(steps):
        step(i)
    h.flush(st)                      # the last image is part of the timed region
    e1.record(st)
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)
    ms = e0.elapsed_time(e1)
    if dist is not None:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    rc, status = h.status(st)
    value = world * steps / (ms * 1e-3)

    # ---- per-kernel-class device times (library's own event brackets; second, instrumented pass)
    prof_steps = min(steps, 64)
    h.tune(5, 1)
    # the brackets are only meaningful without kernel concurrency: the instrumented pass uses the serial entry point
    # (same kernels; in the streaming form the projection and the eigensolver overlap other kernels on purpose)
    for i in range(prof_steps):
        h.process(frames.data_ptr() + (i % n_win) * wbytes, images[i % 4], st)
    prof = h.profile_read()
    h.tune(5, 0)
    sb = stage_bytes(cfg)
    npix = n * n
    G_fft = h.fft_group()
    hbm_peak, peak_src, peaks = _peaks()
    sm_clock = (clocks.get("sm_mhz") or peaks.get("sm_max_mhz") or 1965.0) * 1e6
    num_sms = torch.cuda.get_device_properties(dev).multi_processor_count
    fp32_peak_tflops = num_sms * FP32_LANES_PER_SM * 2 * (peaks.get("sm_max_mhz", 1965.0) * 1e6) / 1e12
    fused_fft = prof[2][1] == 0          # no separate column-pass launches: one persistent kernel does A1+A2 of all T frames
    per_launch_bytes = {"sum": sb["sum"], "fft_rows": sb["fft"] if fused_fft else 2 * G_fft * npix + 4 * npix * G_fft / T,
                        "fft_cols": 8 * G_fft * npix,
                        "cov_partial": sb["cov"], "cov_reduce": 0, "eig": sb["eig"], "project": sb["proj"]}
    stages = {}
    tot_ms = sum(p[0] for p in prof) or 1.0
    for name, (ms_k, cnt) in zip(KCLASS, prof):
        if cnt == 0:
            continue
        us = ms_k / cnt * 1e3
        stages[name] = {"us_per_launch": round(us, 2), "launches_per_step": cnt / prof_steps, "share": round(ms_k / tot_ms, 4),
                        "GBps": round(per_launch_bytes[name] / (us * 1e-6) / 1e9, 1)}
    # holo_process / holo_submit compute Re C only (C is real there, R21): half the complex Gram
    cov_real = "8=0" not in args.tune
    cov_flops = (2 if cov_real else 4) * T * (T + 1) * npix
    if "cov_partial" in stages:
        stages["cov_partial"]["form"] = "real part (2T(T+1) flop/pixel)" if cov_real else "complex Hermitian half (4T(T+1) flop/pixel)"
        stages["cov_partial"]["TFLOPs_fp32"] = round(cov_flops / (stages["cov_partial"]["us_per_launch"] * 1e-6) / 1e12, 2)
    import math
    fft_flops = 10.0 * T * npix * math.log2(n)          # 5 N log2 N per 1-D transform, rows + columns
    if "fft_rows" in stages and fused_fft:
        stages["fft_rows"]["TFLOPs_fp32"] = round(fft_flops / (stages["fft_rows"]["us_per_launch"] * 1e-6) / 1e12, 2)
    dom = max(stages, key=lambda k: stages[k]["share"])
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "r01c_traffic.csv")     # dram__bytes_read.sum + dram__bytes_write.sum, one ncu --set full capture
    if os.path.exists(tpath) and cfg.name.startswith("cfg3"):
        for ln in open(tpath).read().splitlines()[1:]:
            k, v = ln.split(",")
            if k == dom:
                traffic = int(v)
    if dom == "cov_partial" and cov_flops / sb["cov"] > fp32_peak_tflops * 1e12 / (hbm_peak * 1e9):
        roof = {"kernel": dom, "bound": "alu", "achieved": stages[dom]["TFLOPs_fp32"], "peak": round(fp32_peak_tflops, 1),
                "unit": "TFLOP/s", "frac": round(stages[dom]["TFLOPs_fp32"] / fp32_peak_tflops, 4), "traffic": traffic,
                "peak_source": f"{num_sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 x max SM clock (DESIGN.md)",
                "hbm_frac": round(stages[dom]["GBps"] / hbm_peak, 4)}
    else:
        roof = {"kernel": dom, "bound": "hbm", "achieved": stages[dom]["GBps"], "peak": hbm_peak, "unit": "GB/s",
                "frac": round(stages[dom]["GBps"] / hbm_peak, 4), "traffic": traffic, "peak_source": peak_src}
        if dom == "fft_rows" and "TFLOPs_fp32" in stages[dom]:
            # the Fresnel stage is balanced between HBM and the FP32 pipe: report the ALU view as well
            roof["alu_achieved_TFLOPs"] = stages[dom]["TFLOPs_fp32"]
            roof["alu_frac"] = round(stages[dom]["TFLOPs_fp32"] / fp32_peak_tflops, 4)
    e2e_gbps = sb["total"] * (steps / (ms * 1e-3)) / 1e9

    # ---- end to end through the host entry point (pinned host buffers, H2D + D2H inside the timed region)
    e2e = None
    if not args.no_e2e:
        n_host = 2
        host_frames = torch.empty((n_host, T, n, n), dtype=torch.int16).pin_memory()
        host_frames.copy_(frames[:n_host * T].view(torch.int16).reshape(n_host, T, n, n).cpu())
        host_img = torch.empty((2, n, n), dtype=torch.float32).pin_memory()
        k2 = max(3, min(args.e2e_steps, steps))

        def e2e_step(i):
            if streaming:
                h.submit_host(host_frames[i % n_host], host_img[i % 2], st)
            else:
                h.process_host(host_frames[i % n_host], host_img[i % 2], st)

        for i in range(3):
            e2e_step(i)
        if streaming:
            h.flush_host(st)
        barrier()
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(st)
        for i in range(k2):
            e2e_step(i)
        if streaming:
            h.flush_host(st)                 # the last image reaches the host inside the timed region
        a1.record(st)
        barrier()
        ms2 = a0.elapsed_time(a1)
        if dist is not None:
            t = torch.tensor([ms2], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            ms2 = float(t.item())
        e2e = {"value": world * k2 / (ms2 * 1e-3), "unit": "images/s", "h2d_bytes_per_step": fbytes,
               "d2h_bytes_per_step": n * n * 4, "steps": k2, "ms_per_step": ms2 / k2,
               "api": ("holo_submit_host/holo_flush_host (pinned host frames -> host images; the H2D copy of stack i runs under "
                       "the kernels of stack i-1)") if streaming else "holo_process_host (pinned host frames -> host image, synchronous)"}

    # ---- CPU oracle on the box's host cores (rank 0, N = 1 only): a reported baseline, not the target
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle
        fr = frames[:T].cpu().view(torch.int16).numpy().view(np.uint16)
        t0 = time.time()
        out = oracle.process(fr, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
        dt = time.time() - t0
        Mg = torch.empty((n, n), dtype=torch.float32, device=dev)
        h.process(frames.data_ptr(), Mg, st)
        st.synchronize()
        err = float(np.linalg.norm(Mg.cpu().numpy() - out["M"]) / np.linalg.norm(out["M"]))
        cpu = {"value": 1.0 / dt, "unit": "images/s", "cores": oracle.num_threads(), "kind": "oracle",
               "sample": f"1 full stack of {cfg.name} (the first of the GPU stream), {dt:.2f} s", "rel_l2_M_vs_gpu": err}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "images/s", "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": ms / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": value / PAPER_IMAGES_PER_S if cfg.name.startswith("cfg3") else None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg.name, "nx": n, "ny": n, "T": T, "k_lo": cfg.k_lo, "k_hi": cfg.k_hi,
                       "stacks_resident": n_stacks, "windows": n_win, "stride_frames": cfg.stride, "resident_input_bytes": n_stacks * fbytes,
                       "l2_policy": "inputs larger than L2 (stream cycled, no flush needed)",
                       "parallelism": f"replicas x{world} (independent stacks, no collective)", "fft_group": G_fft,
                       "api": "holo_submit/holo_flush (stream of stacks, eigensolver of stack i under the Fresnel stage of stack i+1)"
                              if streaming else ("holo_push (sliding window, stride %d: only the new frames are transformed)" % cfg.stride) if pushing
                              else "holo_process (one stack per call, strictly serial)"},
            "frames_per_s": value * cfg.stride, "clocks": clocks, "e2e": e2e,
            "gpu_launches": steps * h.launches_per_process(), "launches_per_step": h.launches_per_process(),
            "roofline": roof, "roofline_end_to_end": {"bound": "hbm", "achieved": round(e2e_gbps, 1), "peak": hbm_peak, "unit": "GB/s",
                                                      "frac": round(e2e_gbps / hbm_peak, 4), "bytes_per_step": sb["total"], "peak_source": peak_src},
            "stages": stages, "stages_note": "per-kernel device time from an instrumented pass of serial holo_process calls (each kernel alone on the GPU)", "cpu_baseline": cpu, "eig_status": status,
            "eig_cycles": h.workspace_tensor(5).cpu().tolist()[4:7],
            "paper_context": {"images_per_s": PAPER_IMAGES_PER_S, "input_frames_per_s": 500, "hardware": "NVIDIA Titan RTX (PAPER.md:96)"},
        }
        print(json.dumps(line))
    h.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--stacks", type=int, default=None, help="resident stacks (default: the whole stream)")
    ap.add_argument("--e2e-steps", type=int, default=24)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--api", default="submit", choices=["submit", "process", "push"],
                    help="submit: streaming form (default); process: one serial holo_process per stack")
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
