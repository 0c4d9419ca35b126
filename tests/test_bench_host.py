"""Host-side logic of bench.py's N > 1 path on CPU: two `gloo` ranks reduce their per-rank step times to the max
and form the whole-job value of N independent replicas ("replicas only"); the reference arm
prints on rank 0 only.  No GPU, no kernels."""
import json
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import torch.distributed as dist
import bench
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")     # rank 0: 10 ms, rank 1: 15 ms
val = bench.aggregate_value(128, world, ms)
dist.barrier()
print(json.dumps({"rank": rank, "ms": ms, "value": val}), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_max_over_ranks_and_aggregate_gloo_world2(tmp_path):
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT})
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0
        outs.append(json.loads(out.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 15.0                                  # the slowest rank's time, on every rank
        assert o["value"] == pytest.approx(2 * 128 / 15e-3)     # all ranks' units / that time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.aggregate_value(128, 1, 2.0) == pytest.approx(64000.0)


def test_reference_arm_is_rank0_only():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_algorithmic_bytes_match_design_formula():
    """bench.algorithmic() sums to SURVEY.md 8(d)'s local-term formula 16(4a+4b+3nG) + 8nG + 8N/nbatch per band."""
    sys.path.insert(0, ROOT)
    import bench
    info = dict(nG=23928, a=1005 * 80, b=36 * 80 * 80, N=80 ** 3, nb=128, nproj=256, overlap_flops=0)
    nbatches = 12
    tot = sum(bench.algorithmic(info, k, nbatches) for k in ("cols_inv", "rows_inv", "planes", "rows_fwd", "cols_fwd"))
    want = 128 * (16 * (4 * info["a"] + 4 * info["b"] + 3 * info["nG"]) + 8 * info["nG"]) + nbatches * 8 * info["N"]
    assert tot == want
    assert bench.algorithmic(info, "gemm_dotk", 1) == 8 * 128 * 256 * 23928
    assert bench.algorithmic(info, "gemm_expand", 1) == 8 * 128 * 256 * 23928


def test_bench_help_renders():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--help"], capture_output=True, text=True, timeout=120)
    assert out.returncode == 0 and "--config" in out.stdout
