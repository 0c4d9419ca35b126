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


def test_committed_bench_line_has_every_contract_key():
    """The line `python bench.py` printed on the B200 (committed under profiles/bench_r02/) carries every key of the
    measurement contract: base keys, clocks, e2e with byte counts, gpu_launches, roofline, cpu_baseline."""
    import json
    path = os.path.join(ROOT, "profiles", "bench_r02", "default_run.txt")
    line = [l for l in open(path) if l.startswith("{")][-1]
    d = json.loads(line)
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["config"]["workload"] == "cfg5_bulk216_G_128^3" and d["dtype"] == "f64" and d["vs_baseline"] is None
    assert d["n_gpus"] == 1 and d["warmup"] >= 3 and d["gpu_launches"] > 0
    assert set(("sm_mhz", "sm_max_mhz", "reasons")) <= set(d["clocks"])
    assert not set(d["clocks"]["reasons"]) & {"hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown"}
    for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step"):
        assert k in d["e2e"]
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0 and d["e2e"]["value"] < d["value"]
    r = d["roofline"]
    for k in ("bound", "achieved", "peak", "unit", "frac", "traffic"):
        assert k in r
    assert r["bound"] in ("hbm", "tensor", "alu") and r["traffic"] is not None
    assert abs(r["frac"] - r["achieved"] / r["peak"]) <= 1e-9
    c = d["cpu_baseline"]
    assert c["kind"] == "oracle" and c["cores"] >= 1 and c["value"] > 0 and "sample" in c and c["unit"] == d["unit"]
    # the value is units / time
    assert abs(d["value"] - d["config"]["bands"] * d["config"]["kpoints"] / (d["ms_per_step"] * 1e-3)) <= 1e-6 * d["value"]
