"""Builds paper_2004_00923_b200/libholo_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SOURCES = ["holo_api.cu", "fresnel.cu", "fresnel2.cu", "rawgram.cu", "covariance.cu", "covtf32.cu", "eig.cu", "project.cu", "project_tc.cu", "display.cu", "noalloc.cu"]
LIB = os.path.join(HERE, "libholo_b200.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
         "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets"]


def _stale(obj, src):
    if not os.path.exists(obj):
        return True
    deps = [src, os.path.join(CSRC, "holo_internal.cuh"), os.path.join(CSRC, "tma.cuh"), os.path.join(CSRC, "fft_reg.cuh"),
            os.path.join(HERE, "..", "include", "holo.h")]
    return os.path.getmtime(obj) < max(os.path.getmtime(d) for d in deps)


def build(force=False, verbose=False):
    objs = []
    procs = []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        obj = os.path.join(CSRC, s.replace(".cu", ".o"))
        objs.append(obj)
        if force or _stale(obj, src):
            cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj]
            procs.append((s, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for s, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- {s}\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed")
    if procs or not os.path.exists(LIB):
        subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-Wno-deprecated-gpu-targets",
                               "-shared", "-o", LIB] + objs + ["-cudart", "static"])
    ub_src, ub_bin = os.path.join(CSRC, "ubench_peaks.cu"), os.path.join(HERE, "ubench_peaks")
    if force or not os.path.exists(ub_bin) or os.path.getmtime(ub_bin) < os.path.getmtime(ub_src):
        subprocess.check_call([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-Wno-deprecated-gpu-targets",
                               "-o", ub_bin, ub_src])
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
