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
    assert G.CONFIGS[3].n_stacks == 64 and G.CONFIGS[4].n_stacks == 253 and G.CONFIGS[5].n_stacks == 16


def test_reference_arm_world_size_2_gloo(tmp_path):
    """bench.py --impl reference under torchrun-style env with 2 ranks: rank 0 prints one JSON line,
    rank 1 exits 0 silently.  (The GPU arm shards stacks over ranks with no collective; its rank
    logic is the same env parsing.)"""
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


def test_gloo_max_over_ranks_timing():
    """The max-over-ranks reduction bench.py uses, on gloo with 2 processes."""
    code = r'''
import os, sys, torch, torch.distributed as dist
dist.init_process_group("gloo")
r = dist.get_rank()
t = torch.tensor([10.0 + 5.0 * r], dtype=torch.float64)
dist.barrier()
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert t.item() == 15.0
stacks = list(range(r, 64, dist.get_world_size()))      # independent units, no data-path collective
assert len(stacks) == 32
dist.destroy_process_group()
'''
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29534", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, "-c", code], env=dict(env, RANK=str(r), LOCAL_RANK=str(r))) for r in (0, 1)]
    for p in procs:
        assert p.wait(timeout=300) == 0
