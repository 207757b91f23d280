"""CPU-side checks: the C-ABI library loads and exports every symbol include/te.h declares (no
compute calls without a GPU), host-side logic of the binding, and the N>1 sharding helpers of
bench.py under a world_size-2 gloo group."""
import ctypes
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def te():
    from paper_2606_05981_b200 import build as b
    b.build()
    import paper_2606_05981_b200 as te
    return te


def test_library_exports_every_declared_symbol(te):
    L = ctypes.CDLL(te.LIB_PATH)
    for header, names in (("te.h", te.EXPORTS), ("te_debug.h", te.DEBUG_EXPORTS)):
        hdr = open(os.path.join(ROOT, "include", header)).read()
        hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
        declared = set(re.findall(r"\b(te_[a-z_0-9]+)\s*\(", hdr))
        assert declared == set(names), (header, declared ^ set(names))
        for name in declared:
            assert hasattr(L, name), name


def test_config_struct_layout_matches_header(te):
    # te_config: 9 int32, float, (pad) double, 6 int32 -> natural C layout
    assert ctypes.sizeof(te.TEConfig) == 80
    assert te.TEConfig.rope_theta.offset == 40 and te.TEConfig.max_frames.offset == 48
    assert te.TEConfig.rope_interleaved.offset == 64 and te.TEConfig.max_prefix_tokens.offset == 68 and te.TEConfig.weight_dtype.offset == 72
    assert te.TEConfig.non_causal.offset == 76
    # te_vision_config: te_config (80 bytes, 8-aligned) + 5 int32 -> 104
    assert te.TEVisionConfig.patch.offset == 80 and te.TEVisionConfig.max_frames.offset == 96
    assert ctypes.sizeof(te.TEVisionConfig) == 104


def test_vision_blob_bytes_without_gpu(te):
    import workloads as W
    for v in (W.VISION_TINY, W.VISION_FULL):
        assert te.te_vision_blob_bytes(te.make_vision_config(v, 4)) == 2 * W.vision_blob_layout(v)["total"]
    bad = te.make_vision_config(W.VISION_TINY, 4)
    bad.patch = 5                                          # image not a multiple of 2 * patch
    assert te.te_vision_blob_bytes(bad) == 0


def test_matmul_noalloc_size_limit_without_gpu(te):
    """te_matmul_noalloc (te.h) checks its arguments and the capacity of the built-in scratch array before it touches
    the device: an over-size problem is refused with TE_ERR_TOO_LARGE and bad shapes with their own codes, GPU or not."""
    L = te.lib()
    dummy = 256                                            # non-null, never dereferenced on these paths
    assert te.TE_NOALLOC_SCRATCH_BYTES == 8 << 20
    hdr = open(os.path.join(ROOT, "include", "te.h")).read()
    assert "#define TE_NOALLOC_SCRATCH_BYTES (8u << 20)" in hdr and "TE_ERR_TOO_LARGE = -7" in hdr
    # 17 tiles x 8 splits x 128 x 128 x 4 B = 8.5 MiB
    assert L.te_matmul_noalloc(0, dummy, dummy, dummy, 128, 2176, 2048, 128, 8, None) == te.TE_ERR_TOO_LARGE
    # 1 x 4 tiles x 5 splits x 128 KiB = 2.5 MiB fits, but m = 3000 makes it 24 x 4 x 5
    assert L.te_matmul_noalloc(0, dummy, dummy, dummy, 3000, 1024, 2048, 256, 5, None) == te.TE_ERR_TOO_LARGE
    assert "scratch" in L.te_strerror(te.TE_ERR_TOO_LARGE).decode()
    assert L.te_matmul_noalloc(0, None, dummy, dummy, 128, 128, 64, 128, 1, None) == te.TE_ERR_INVALID_ARG
    assert L.te_matmul_noalloc(0, dummy, dummy, dummy, 128, 128, 64, 128, 2, None) == te.TE_ERR_INVALID_ARG    # splits > k/64
    assert L.te_matmul_noalloc(0, dummy, dummy, dummy, 128, 128, 96, 128, 1, None) == te.TE_ERR_UNSUPPORTED    # k % 64
    assert L.te_matmul_noalloc(0, dummy, dummy, dummy, 128, 192, 64, 128, 1, None) == te.TE_ERR_UNSUPPORTED    # n % block_n


def test_blob_bytes_and_strerror_without_gpu(te):
    import workloads as W
    for m in (W.TINY, W.FULL1, W.FULL28):
        cfg = te.make_config(m, 4, 512)
        assert te.te_blob_bytes(cfg) == 2 * W.blob_num_elements(m)
    assert W.blob_num_elements(W.FULL28) - W.FULL28.hidden - 28 * (2 * 2048 + 2 * 128) == 1_409_286_144
    bad = te.make_config(W.TEModelConfig(1, 256, 4, 2, 32, 768, (4, 6, 6)), 2, 128)
    assert te.te_blob_bytes(bad) == 0                      # unsupported head_dim
    assert te.te_strerror(te.TE_ERR_BLOB_SIZE) == "weight blob has the wrong size"
    assert te.te_strerror(0) == "ok"


def test_create_fails_loudly_without_a_gpu(te):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import workloads as W
    with pytest.raises(te.TEError):
        te.te_create(te.make_config(W.TINY, 2, 128), 0)


def test_product_never_imports_oracle():
    """The product path must not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_05981_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("no CPU fallback", ""), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2606_05981_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(`paper_2606_05981_b200/`)", "")


def test_sharding_helpers_gloo_world2():
    """bench.py's N>1 logic (frame sharding, max-over-ranks timing, aggregate value) under gloo."""
    code = r'''
import os, sys, json
sys.path.insert(0, %r)
import torch, torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
seeds = bench.rank_seed_offset(rank)
t_local = 1.0 + rank            # rank 1 is slower
t_max = bench.max_over_ranks(t_local, device="cpu")
val = bench.aggregate_value(units_per_rank=16 * 10, world=world, seconds=t_max)
dist.barrier()
if rank == 0:
    print(json.dumps({"t_max": t_max, "val": val, "seed0": seeds}))
dist.destroy_process_group()
''' % ROOT
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29533")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
                        "--master-addr", "127.0.0.1", "--master-port", "29533", "--no-python",
                        sys.executable, "-c", code],
                       capture_output=True, text=True, env=env, timeout=240)
    assert r.returncode == 0, r.stderr[-2000:]
    import json
    line = [l for l in r.stdout.splitlines() if l.startswith("{")][-1]
    d = json.loads(line)
    assert d["t_max"] == 2.0 and abs(d["val"] - 2 * 160 / 2.0) < 1e-9
