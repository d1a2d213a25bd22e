#!/usr/bin/env python
"""Workload for compute-sanitizer (SURVEY.md sections 4-5): BASELINE.json configs[0] (256 x 256 x 16) through every
chained entry point of the C ABI -- holo_process, holo_submit x 3 + holo_flush, holo_push x 4 + holo_flush, the same in
modes 2 and 3 (tensor-core integer Gram, deflating row pass, column energy, eigen-basis form), the host entry -- and the
per-stage calls (incl. the tensor-core Gram and projection, SVD filter, normalisation, fftshift).  Run ONE tool per process (and per gpurun call, B200_PROFILING.md):

    compute-sanitizer --tool memcheck  python tests/sanitize_driver.py
    compute-sanitizer --tool racecheck python tests/sanitize_driver.py
    compute-sanitizer --tool synccheck python tests/sanitize_driver.py
    compute-sanitizer --tool initcheck python tests/sanitize_driver.py

The summaries of these runs are kept under profiles/.  Exit code 0 = every call returned HOLO_OK and the images are
finite and reproduce the serial holo_process image (the sanitizer adds its own verdict on top).
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
from gen import holo_gen as G                      # noqa: E402
from paper_2004_00923_b200 import Holo             # noqa: E402


def main():
    small = "--small" in sys.argv                  # racecheck is ~100x slower: 64 x 64 x 16 there
    cfg = G.small_config(n=64, T=16) if small else G.CONFIGS[1]
    n, T = cfg.n, cfg.T
    scene = G.make_scene(G.Config(cfg.name, n, T, T + 4 * 8, 8, cfg.n_stripes, cfg.sigma_psi, cfg.self_beating, cfg.k_lo, cfg.k_hi), 1)
    stream = G.frames_np(scene, 0, T + 4 * 8)
    dev = torch.from_numpy(stream.view(np.int16)).cuda().view(torch.uint16)
    h = Holo(n, n, T, cfg.lam, cfg.pitch, cfg.z, cfg.k_lo, cfg.k_hi)
    st = torch.cuda.Stream()
    fbytes = n * n * 2

    def img():
        return torch.zeros((n, n), dtype=torch.float32, device="cuda")

    ref = img()
    h.process(dev, ref, st)
    st.synchronize()
    assert bool(torch.isfinite(ref).all()) and float(ref.sum()) > 0

    outs = [img() for _ in range(3)]
    for o in outs:
        h.submit(dev, o, st)
    h.flush(st)
    st.synchronize()
    for o in outs:
        err = float((o - ref).norm() / ref.norm())
        assert err <= 2e-5, err

    pouts = [img() for _ in range(5)]
    h.push(dev.data_ptr(), T, pouts[0], st)
    for k in range(4):
        h.push(dev.data_ptr() + (T + 8 * k) * fbytes, 8, pouts[k + 1], st)
    h.flush(st)
    st.synchronize()
    err = float((pouts[0] - ref).norm() / ref.norm())
    assert err <= 2e-5, err
    assert all(bool(torch.isfinite(p).all()) for p in pouts)

    # per-stage entry points (complex Gram kernel, direct projection, Fourier demodulation)
    H = torch.empty((T, n, n), dtype=torch.complex64, device="cuda")
    C = torch.empty((T, T), dtype=torch.complex64, device="cuda")
    ev = torch.empty(T, dtype=torch.float32, device="cuda")
    V = torch.empty((T, T), dtype=torch.complex64, device="cuda")
    M = img()
    with torch.cuda.stream(st):
        h.fresnel(dev, H, st)
        h.covariance(H, C, st)
        h.eig(C, ev, V, st)
        h.project(H, V, M, st)
        h.fourier_demod(H, 4, 12, M, st)                 # 9 kept components: tensor-core projection
        h.raw_covariance(dev, C, st)
        h.svd_filter(H, V, H, st)
        h.normalize(M, st)
        M2 = img()
        h.fftshift(M, M2, st)
    st.synchronize()
    rc, status = h.status(st)
    assert rc == 0, status

    # modes 2 and 3 (and the tensor-core covariance of mode 1), serial, streamed and through host buffers
    host = [torch.from_numpy(stream[:T].view(np.int16).copy()).pin_memory() for _ in range(3)]
    for mode, tf32, window in ((1, 3, None), (2, 0, None), (3, 0, None), (3, 0, (6, 12))):
        h.set_mode(mode)
        h.tune(13, tf32)
        if window:
            h.set_range(*window)                         # 9 rejected components: eigen-basis form
        r = img()
        h.process(dev, r, st)
        outs = [img() for _ in range(3)]
        for o in outs:
            h.submit(dev, o, st)
        h.flush(st)
        hout = [torch.zeros((n, n), dtype=torch.float32).pin_memory() for _ in range(3)]
        for f, o in zip(host, hout):
            h.submit_host(f, o, st)
        h.flush_host(st)
        st.synchronize()
        assert bool(torch.isfinite(r).all()) and float(r.sum()) > 0
        if not window:
            assert float((r - ref).norm() / ref.norm()) <= 2e-5
        for o in outs + [x.cuda() for x in hout]:
            assert float((o - r).norm() / r.norm()) <= 2e-5
        rc, status = h.status(st)
        assert rc == 0, status
        h.set_range(cfg.k_lo, cfg.k_hi)
    h.set_mode(1)
    h.close()
    torch.cuda.synchronize()
    print("sanitize_driver ok:", cfg.name, "sweeps", status[1])


if __name__ == "__main__":
    main()
