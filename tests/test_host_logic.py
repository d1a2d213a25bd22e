"""CPU-side checks of the product's host logic: the C-ABI library builds/loads and exports every
symbol include/holo.h declares (no compute calls without a GPU), bench.py's accounting helpers,
and the N>1 launch path of bench.py's reference arm under gloo (world_size 2)."""
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "holo.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(holo_[a-z_0-9]+)\s*\(", src)))


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2004_00923_b200 import build as b
    lib = b.build()
    import paper_2004_00923_b200 as pkg
    L = pkg.load_library()
    names = _declared_functions()
    assert len(names) >= 17
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/holo.h but not exported by {lib}"
    assert set(pkg.EXPORTED_SYMBOLS) == set(names)
    # ... and the other direction: the library exports no holo_* entry point that the header does not declare
    nm = subprocess.check_output(["nm", "-D", "--defined-only", lib], text=True)
    exported = sorted({ln.split()[-1] for ln in nm.splitlines() if ln.split() and ln.split()[-1].startswith("holo_") and " T " in ln})
    assert exported == names, (set(exported) ^ set(names))
    assert L.holo_version() >= 100
    out = subprocess.check_output(["cuobjdump", "-lelf", lib], text=True)
    assert "sm_100a" in out


def test_no_cpu_fallback_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2004_00923_b200 import Holo, HoloError
    with pytest.raises(HoloError):
        Holo(64, 64, 8, 785e-9, 20e-6, 0.2, 2, 8)


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2004_00923_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("oracle/", "").lower() or f.endswith((".cu", ".cuh")) and "import" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            assert "paper_2004_00923_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "never imports paper_2004_00923_b200", "").replace("under paper_2004_00923_b200/csrc/", "")


def test_stage_bytes_match_design():
    sys.path.insert(0, ROOT)
    import bench
    from gen import holo_gen as G
    sb = bench.stage_bytes(G.CONFIGS[3])
    assert sb["total"] == 28 * 32 * 1024 * 1024 + 12 * 1024 * 1024 == sb["sum"] + sb["fft"] + sb["cov"] + sb["proj"]
    assert round(sb["total"] / 1e6) == 952
    sb2 = bench.stage_bytes(G.CONFIGS[3], mode=2)          # Gram from the raw frames: no covariance read of H
    assert sb2["total"] == 20 * 32 * 1024 * 1024 + 12 * 1024 * 1024
    assert "1024x1024x32" in bench.metric_name(G.CONFIGS[3]) and "512x512x32" in bench.metric_name(G.CONFIGS[2])
    assert G.CONFIGS[3].n_stacks == 64 and G.CONFIGS[4].n_stacks == 253 and G.CONFIGS[5].n_stacks == 16


def test_reference_arm_two_ranks_env(tmp_path):
    """bench.py --impl reference with torchrun's environment for 2 ranks (no process group is needed by this arm):
    rank 0 prints one JSON line, rank 1 exits 0 silently."""
    import json
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29533", OMP_NUM_THREADS="2")
    outs = []
    for rank in (0, 1):
        e = dict(env, RANK=str(rank), LOCAL_RANK=str(rank))
        outs.append(subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                                    "--steps", "2", "--warmup", "1", "--config", "1"], env=e, capture_output=True, text=True, timeout=600))
    assert outs[0].returncode == 0 and outs[1].returncode == 0, (outs[0].stderr, outs[1].stderr)
    line = json.loads(outs[0].stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert outs[1].stdout.strip() == ""


def test_gpu_arm_rank_and_shard_logic_world_size_2_gloo():
    """bench.py's GPU arm under two ranks, up to the point where a handle would be created: every rank plans its own
    stream (different seed, same shape: weak scaling, no data-path collective), the timed duration is reduced with MAX
    over a real process group (gloo here, nccl on the GPU box) and rank 0 aggregates the whole-job value."""
    code = r'''
import os, sys, json
sys.path.insert(0, os.environ["HOLO_ROOT"])
import torch.distributed as dist
import bench
from gen import holo_gen as G
dist.init_process_group("gloo")
rank, world, local = bench.rank_env()
assert (rank, world) == (dist.get_rank(), dist.get_world_size()) and local == rank
cfg = G.CONFIGS[3]
plan = bench.shard_plan(cfg, rank, world)
assert plan["seed"] == 1000 + rank
assert plan["n_stacks"] == 64 and plan["n_win"] == 64 and plan["stack_bytes"] == 64 << 20
assert plan["resident_bytes"] >= 3 * bench.L2_BYTES
p4 = bench.shard_plan(G.CONFIGS[4], rank, world, stacks=16)          # overlapping windows, stride 8
assert p4["n_win"] == (16 * 32 - 32) // 8 + 1 and p4["n_push"] == 60 and p4["window_stride_bytes"] == 8 * 1024 * 1024 * 2
p2 = bench.shard_plan(G.CONFIGS[2], rank, world)                     # the 8-stack stream is extended to >= 3x L2
assert p2["n_stacks"] >= 23 and "larger than L2" in bench.l2_policy(p2)
ms = bench.reduce_max_ms(10.0 + 5.0 * rank, dist)                     # the slowest rank decides
assert ms == 15.0
value = bench.aggregate_value(world, 30, ms)
assert abs(value - 2 * 30 / 15e-3) < 1e-9
dist.barrier()
if rank == 0:
    print(json.dumps({"value": value, "seeds": [1000, 1001]}))
dist.destroy_process_group()
'''
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29534", WORLD_SIZE="2", HOLO_ROOT=ROOT)
    procs = [subprocess.Popen([sys.executable, "-c", code], env=dict(env, RANK=str(r), LOCAL_RANK=str(r)),
                              stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True) for r in (0, 1)]
    outs = [p.communicate(timeout=300) for p in procs]
    assert procs[0].returncode == 0 and procs[1].returncode == 0, (outs[0][1][-800:], outs[1][1][-800:])
    import json
    assert json.loads(outs[0][0].strip().splitlines()[-1])["value"] == 4000.0
    assert outs[1][0].strip() == ""
