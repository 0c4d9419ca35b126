"""(k-point, band) sharding glue on CPU ranks (`gloo`, world sizes 2 and 3).

The process-group logic of paper_1708_03621_b200/sharding.py (who owns which bands, the all-gather / ring schedules of
the band-sharded overlap, the all-reduce of the density) runs here with the CPU oracle standing in for the library's
local operations (`ops`); every rank checks its result against the oracle applied to the UNSHARDED arrays.
No GPU, no kernels."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_1708_03621_b200.sharding import KBLayout, shard_range  # noqa: E402

WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import numpy as np, torch
import torch.distributed as dist
from oracle import ref
from paper_1708_03621_b200 import sharding as sh

class OracleOps:   # stand-in for binding.jdft_* on CPU tensors (test infrastructure)
    @staticmethod
    def jdft_overlap(b, C1, C2):
        return torch.from_numpy(np.ascontiguousarray(b.overlap(C1.numpy(), C2.numpy())))
    @staticmethod
    def jdft_subspace(b, C1, X2):
        return torch.from_numpy(np.ascontiguousarray(b.subspace(C1.numpy(), X2.numpy())))
    @staticmethod
    def jdft_density(b, C, f):
        return torch.from_numpy(b.density(C.numpy(), f.numpy()))
    @staticmethod
    def jdft_apply_H(b, V, P, D, C, HC=None):
        return torch.from_numpy(b.apply_H(V.numpy(), P.numpy(), D.numpy(), C.numpy()))

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
nb = %(nb)d
R = np.array([[6.0, 0.3, 0.0], [0.0, 5.5, 0.2], [0.1, 0.0, 6.5]])
b = ref.RefBasis(R, [0.25, 0.0, 0.125], 4.0, [12, 12, 12])
b.S = tuple(int(s) for s in b.S)
rng = np.random.default_rng(7)
C = rng.standard_normal((nb, b.nG)) + 1j * rng.standard_normal((nb, b.nG))
X = rng.standard_normal((nb, b.nG)) + 1j * rng.standard_normal((nb, b.nG))
f = rng.uniform(0.0, 2.0, nb)
V = rng.standard_normal(b.N)
P = rng.standard_normal((3, b.nG)) + 1j * rng.standard_normal((3, b.nG))
D = rng.standard_normal(3)
lay = sh.KBLayout(1, nb, world, rank)
assert lay.group_ranks == list(range(world)) and lay.group_rank == rank
grp = lay.new_band_group()
lo, hi = sh.shard_range(nb, world, rank)
assert lay.units == ([(0, lo, hi)] if hi > lo else [])
Cl, Xl, fl = (torch.from_numpy(a[lo:hi].copy()) for a in (C, X, f))
ops = OracleOps
errs = {}
for mode in ("allgather", "ring"):
    M = sh.sharded_overlap(b, Cl, Xl, nb, group=grp, mode=mode, ops=ops)
    want = b.overlap(C, X)[:, lo:hi]
    assert tuple(M.shape) == want.shape, (M.shape, want.shape)
    errs["overlap_" + mode] = float(np.abs(M.numpy() - want).max()) if want.size else 0.0
    Mfull = sh.gather_columns(M, nb, group=grp)
    errs["gather_" + mode] = float(np.abs(Mfull.numpy() - b.overlap(C, X)).max())
    S = sh.sharded_overlap(b, Cl, Xl, nb, group=grp, mode=mode, subspace=True, ops=ops)
    errs["subspace_" + mode] = float(np.abs(S.numpy() - b.subspace(C, X)[:, lo:hi]).max()) if want.size else 0.0
n = sh.sharded_density(b, Cl, fl, group=grp, weight=0.5, ops=ops)
errs["density"] = float(np.abs(n.numpy() - 0.5 * b.density(C, f)).max())
HC = sh.sharded_apply_H(b, torch.from_numpy(V), torch.from_numpy(P), torch.from_numpy(D), Cl, ops=ops)
errs["apply_H"] = float(np.abs(HC.numpy() - b.apply_H(V, P, D, C)[lo:hi]).max()) if hi > lo else 0.0
dist.barrier()
print(json.dumps({"rank": rank, "errs": errs, "scale": float(np.abs(b.overlap(C, X)).max())}), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


@pytest.mark.parametrize("world,nb", [(2, 6), (2, 5), (3, 7), (3, 2)])
def test_band_sharded_overlap_density_gloo(tmp_path, ref, world, nb):
    """Even shards, ragged shards (5 over 2, 7 over 3) and a rank with NO bands (2 over 3)."""
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER % {"root": ROOT, "nb": nb})
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0, err[-2000:]
        o = json.loads(out.strip().splitlines()[-1])
        for name, e in o["errs"].items():
            # the sharded GEMM sums the same nG products per entry as the unsharded one; the density sum is
            # re-associated across ranks by the all-reduce
            assert e <= 1e-12 * max(1.0, o["scale"]), (name, e)


def test_shard_range_partitions():
    for n in (0, 1, 5, 128, 513):
        for parts in (1, 2, 3, 8):
            rs = [shard_range(n, parts, i) for i in range(parts)]
            assert rs[0][0] == 0 and rs[-1][1] == n
            assert all(rs[i][1] == rs[i + 1][0] for i in range(parts - 1))
            sizes = [b - a for a, b in rs]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def test_kb_layout_k_first_then_bands():
    # config 4 of BASELINE.json: 4 k-points, 384 bands
    # world <= nk: whole k-points per rank, all bands, no band group (the paper's MPI-over-k layout)
    got = [KBLayout(4, 384, 2, r).units for r in range(2)]
    assert got == [[(0, 0, 384), (1, 0, 384)], [(2, 0, 384), (3, 0, 384)]]
    assert KBLayout(4, 384, 3, 0).units == [(0, 0, 384), (1, 0, 384)] and KBLayout(4, 384, 3, 2).units == [(3, 0, 384)]
    assert all(KBLayout(4, 384, 4, r).group_size == 1 for r in range(4))
    # world > nk: one k-point per group, bands split inside the group
    lays = [KBLayout(4, 384, 8, r) for r in range(8)]
    assert [l.units for l in lays] == [[(r // 2, 192 * (r % 2), 192 * (r % 2 + 1))] for r in range(8)]
    assert lays[5].group_ranks == [4, 5] and lays[5].group_rank == 1 and lays[5].band_ranges() == [(0, 192), (192, 384)]
    # every (k, band) unit is owned exactly once, whatever the world size
    for world in (1, 2, 3, 5, 6, 8, 16):
        seen = set()
        for r in range(world):
            for k, lo, hi in KBLayout(4, 10, world, r).units:
                for bnd in range(lo, hi):
                    assert (k, bnd) not in seen
                    seen.add((k, bnd))
        assert len(seen) == 40


STEP_WORKER = r"""
import os, sys, json
sys.path.insert(0, %(root)r)
import numpy as np, torch
import torch.distributed as dist
import bench, workloads
from oracle import ref
from paper_1708_03621_b200 import sharding as sh

class OracleOps:   # stand-in for binding.jdft_* on CPU tensors (test infrastructure)
    @staticmethod
    def jdft_overlap(b, C1, C2):
        return torch.from_numpy(np.ascontiguousarray(b.overlap(C1.numpy(), C2.numpy())))
    @staticmethod
    def jdft_apply_H(b, V, P, D, C, HC=None):
        return torch.from_numpy(b.apply_H(V.numpy(), P.numpy(), D.numpy(), C.numpy()))

dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
cfg_id = %(cfg)d
cfg = workloads.get_config(cfg_id)
nk, nb = len(cfg["kpoints"]), cfg["nb"]
lay = sh.KBLayout(nk, nb, world, rank)
grp = lay.new_band_group()
def make_basis(R, k, Ecut, S):
    b = ref.RefBasis(R, k, Ecut, S)
    return b, b.iG
kdata, V, D = bench.shard_inputs(cfg_id, lay, make_basis, torch.from_numpy)
errs = {}
for mode in ("allgather", "ring"):
    out = sh.sharded_step(lay, kdata, V, D, group=grp, mode=mode, overlap=True, ops=OracleOps)
    for k, blo, bhi in lay.group_units():
        b = kdata[k]["basis"]
        inp = workloads.make_inputs(cfg_id, b.iG, ik=k)
        HC, M = out[k]
        if bhi > blo:
            want = b.apply_H(inp["Vloc"], inp["P"], inp["D"], inp["C"][blo:bhi])
            errs["H_%%s_k%%d" %% (mode, k)] = float(np.abs(HC.numpy() - want).max() / np.abs(want).max())
        wantM = b.overlap(inp["C"], inp["C"])[:, blo:bhi]
        assert tuple(M.shape) == wantM.shape
        errs["M_%%s_k%%d" %% (mode, k)] = float(np.abs(M.numpy() - wantM).max()) if wantM.size else 0.0
dist.barrier()
print(json.dumps({"rank": rank, "units": lay.group_units(), "errs": errs}), flush=True)
dist.destroy_process_group()
"""


@pytest.mark.parametrize("world,cfg", [(2, 103), (3, 103), (2, 101)])
def test_bench_shard_mode_step_gloo(tmp_path, ref, world, cfg):
    """The step `bench.py --shard kb` times (bench.shard_inputs + sharding.sharded_step), on gloo ranks with the oracle as
    the local operation: shape 103 has 2 k-points (2 ranks: one k-point each, no collective; 3 ranks: k-point 0 on one
    rank, k-point 1 band-sharded over two), shape 101 has one k-point and 5 bands over 2 ranks (ragged)."""
    import json
    script = tmp_path / "step_worker.py"
    script.write_text(STEP_WORKER % {"root": ROOT, "cfg": cfg})
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), OMP_NUM_THREADS="1")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    units = []
    for p in procs:
        out, err = p.communicate(timeout=400)
        assert p.returncode == 0, err[-3000:]
        o = json.loads(out.strip().splitlines()[-1])
        units += [tuple(u) for u in o["units"]]
        assert o["errs"], "rank did no work"
        for name, e in o["errs"].items():
            assert e <= 1e-12, (name, e)
    # every (k, band) of the job is covered exactly once
    cfgd = __import__("workloads").get_config(cfg)
    covered = sorted((k, bnd) for k, lo, hi in units for bnd in range(lo, hi))
    assert covered == [(k, bnd) for k in range(len(cfgd["kpoints"])) for bnd in range(cfgd["nb"])]
