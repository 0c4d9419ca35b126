#!/usr/bin/env python
"""bench.py -- H.psi band-applications/s (fp64) of libjdft_b200 on one BASELINE.json workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]

A "step" is one pass of the whole hot path over the workload: jdft_apply_H on every band of every k-point of the
config (config 5 also runs its 512 x 512 jdft_overlap).  Inputs are seeded synthetic data of BASELINE.json's
shapes (workloads/), resident in HBM before the timed region.  L2 is flushed (a 512 MiB memset) before every
timed step; steps are timed with CUDA events on the launch stream; N > 1 runs N independent replicas
("replicas only") and takes the max over ranks.  Prints ONE JSON line (rank 0).

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded band sample of the
same workload and prints the same line with "impl": "reference".
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "H.psi band-applications/s (fp64)"
UNIT = "band-applications/s"
KERNELS = ["cols_inv", "rows_inv", "planes", "rows_fwd", "cols_fwd", "gemm_dotk", "gemm_expand", "splitk_reduce"]
HBM_KERNELS = {"cols_inv", "rows_inv", "planes", "rows_fwd", "cols_fwd", "splitk_reduce"}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(cfg_id, kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu --set full summary (profiles/traffic.csv), or None.
    Several rows of one kernel (gemm_dotk: the projection and the overlap launch of config 5) are averaged, like the
    launches of the timed step are."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None
    vals = []
    with open(path) as f:
        for line in f:
            parts = line.strip().split(",")
            if len(parts) >= 3 and parts[0] == str(cfg_id) and (parts[1] == kernel or parts[1].startswith(kernel + "_")):
                vals.append(int(parts[2]))
    return int(sum(vals) / len(vals)) if vals else None


def fp64_peak():
    """Live DMMA / DFMA peak of this GPU from the committed micro-benchmark (csrc/fp64_peak.cu)."""
    tool = os.path.join(ROOT, "paper_1708_03621_b200", "fp64_peak")
    try:
        out = subprocess.run([tool], capture_output=True, text=True, timeout=120).stdout.strip().splitlines()[-1]
        d = json.loads(out)
        return float(d["dmma_tflops"]), float(d["dfma_tflops"]), "measured (csrc/fp64_peak.cu DMMA micro-benchmark, this run)"
    except Exception:
        return 37.2, 37.2, "nominal (148 SM x 64 FMA/clk x 2 x 1.965 GHz; micro-benchmark unavailable)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.FIELDS,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 6:
                continue
            try:
                sm.append(float(parts[0]))
                mx.append(float(parts[1]))
            except ValueError:
                continue
            for nme, v in zip(names, parts[2:6]):
                if v == "Active":
                    reasons.add(nme)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out["sm_mhz"] = float(np.median(sm))
            out["sm_max_mhz"] = float(max(mx))
        out["reasons"] = sorted(reasons)
        return out


def max_over_ranks(x, world, device="cuda"):
    """Max of a per-rank scalar over all ranks (the contract's max-over-ranks timing); identity for one rank."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(units_per_rank, world, ms_step_max):
    """Whole-job throughput of N independent replicas: all ranks' units / the slowest rank's time."""
    return world * units_per_rank / (ms_step_max * 1e-3)


def config_sizes(cfg_id):
    cfg = workloads.get_config(cfg_id)
    return cfg, len(cfg["kpoints"]), cfg["nb"], cfg["natoms"] * cfg["n_lm"]


# ------------------------------------------------------------------------------------------------ reference arm

def oracle_sample_step(rb, inp, Cs, do_overlap):
    """One pass of the oracle over a band sample of the workload: jdft_ref_apply_H on the sample and, where the step
    contains the overlap (config 5), the sample's columns of C^+ O C against ALL bands (the sample's share of it)."""
    rb.apply_H(inp["Vloc"], inp["P"], inp["D"], Cs)
    if do_overlap:
        rb.overlap(inp["C"], Cs)


def run_reference(args):
    from oracle import ref
    cfg, nk, nb, nproj = config_sizes(args.config)
    R, kpts, Ecut, S = workloads.lattice(args.config)
    do_overlap = args.config == 5
    threads = ref.threads()
    rb = ref.RefBasis(R, kpts[0], Ecut, S)
    inp = workloads.make_inputs(args.config, rb.iG, ik=0, nb=nb if do_overlap else max(threads, 1) * 4,
                                orthonormalise=not do_overlap)   # (QR of the full block is not part of the path)
    C = inp["C"]
    # calibrate: one band per thread, then size the per-step sample so the whole run stays within a few minutes
    t0 = time.perf_counter()
    oracle_sample_step(rb, inp, C[:threads], do_overlap)
    t1 = time.perf_counter() - t0
    budget = 120.0 / max(1, args.steps + args.warmup)
    nsample = int(max(threads, min(C.shape[0], threads * max(1, int(budget / max(t1, 1e-3))))))
    nsample = (nsample // threads) * threads
    Cs = np.ascontiguousarray(C[:nsample])
    for _ in range(args.warmup):
        oracle_sample_step(rb, inp, Cs, do_overlap)
    times = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        oracle_sample_step(rb, inp, Cs, do_overlap)
        times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(times))
    value = nsample / (ms * 1e-3)
    sample = "%d bands of k-point 0 of config %d per step (full P, Vloc): jdft_ref_apply_H%s" % (
        nsample, args.config, " + their %d x %d columns of jdft_ref_overlap" % (nb, nsample) if do_overlap else "")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "bands_per_step": nsample, "nproj": nproj, "fft_box": list(S),
                   "overlap_in_step": do_overlap},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def cpu_baseline(cfg_id, seconds=15.0):
    """The oracle, as it stands, on a bounded sample (about `seconds` of CPU work) of the same workload: whole passes
    of jdft_ref_apply_H over `threads x 4..8` bands of k-point 0 (full P and Vloc; config 5: plus those bands' columns
    of the 512 x 512 overlap), repeated until the time is used."""
    from oracle import ref
    R, kpts, Ecut, S = workloads.lattice(cfg_id)
    do_overlap = cfg_id == 5
    threads = ref.threads()
    rb = ref.RefBasis(R, kpts[0], Ecut, S)
    nb_cfg = workloads.get_config(cfg_id)["nb"]
    nb = min(nb_cfg, threads * (4 if do_overlap else 8))
    inp = workloads.make_inputs(cfg_id, rb.iG, ik=0, nb=nb_cfg if do_overlap else nb, orthonormalise=not do_overlap)
    Cs = np.ascontiguousarray(inp["C"][:nb])
    t0 = time.perf_counter()
    oracle_sample_step(rb, inp, Cs[:min(nb, threads)], do_overlap)      # warm-up / calibration
    t1 = time.perf_counter() - t0
    done, t0 = 0, time.perf_counter()
    while True:
        oracle_sample_step(rb, inp, Cs, do_overlap)
        done += nb
        dt = time.perf_counter() - t0
        if dt >= seconds or dt + t1 * nb / max(1, min(nb, threads)) > 2 * seconds:
            break
    return {"value": done / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "sample": "%d band-applications (%d bands of k-point 0 of config %d, repeated), jdft_ref_apply_H%s, %.1f s wall on %d threads"
                      % (done, nb, cfg_id, " + their columns of the %d^2 jdft_ref_overlap" % nb_cfg if do_overlap else "", dt, threads)}


# ------------------------------------------------------------------------------------------------ our arm

def algorithmic(cfgk, kernel, nbatches):
    """Algorithmic bytes (HBM kernels) or flops (GEMMs) of ONE step for one k-point."""
    nG, a, b, N, nb, npj = cfgk["nG"], cfgk["a"], cfgk["b"], cfgk["N"], cfgk["nb"], cfgk["nproj"]
    if kernel == "cols_inv":
        return nb * 16 * (nG + a)
    if kernel in ("rows_inv", "rows_fwd"):
        return nb * 16 * (a + b)
    if kernel == "planes":
        return nb * 32 * b + nbatches * 8 * N
    if kernel == "cols_fwd":
        return nb * (16 * (a + 2 * nG) + 8 * nG)
    if kernel == "gemm_dotk":
        return 8 * nb * npj * nG + cfgk["overlap_flops"]
    if kernel == "gemm_expand":
        return 8 * nb * npj * nG
    return 0


def overlap_flops(nb, nG):
    """Real flops counted for jdft_overlap(C, C): C^+ C is Hermitian, so only the triangle is needed (SURVEY.md 8(d):
    "half if only the Hermitian triangle is computed -- then count half"): 8 nG nb (nb + 1) / 2.  (The kernel computes
    whole 64 x 64 diagonal tiles, i.e. ~12 % more DMMAs than this at nb = 512; they are not counted.)"""
    return 8 * (nb * (nb + 1) // 2) * nG


def measure(cfg_id, args, rank, world, local, full):
    """Times one BASELINE.json workload on this rank's GPU and returns the JSON line as a dict (rank 0; None elsewhere).
    full = False: device-timed step and per-kernel rooflines only (no end-to-end leg, extras or CPU baseline)."""
    import torch
    import torch.distributed as dist
    import paper_1708_03621_b200.binding as jd

    cfg, nk, nb, nproj = config_sizes(cfg_id)
    R, kpts, Ecut, S = workloads.lattice(cfg_id)
    do_overlap = cfg_id == 5
    steps = args.steps if full else min(args.steps, 5)
    atoms = workloads.atoms_fractional(cfg_id)
    Vh = workloads.make_vloc(cfg_id, atoms).reshape(-1)
    V = torch.from_numpy(Vh).cuda()
    D_h = workloads.make_D(cfg_id)
    D = torch.from_numpy(D_h).cuda()
    ks = []
    for ik in range(nk):
        gb = jd.jdft_basis_create(R, kpts[ik], Ecut, S, device=local)
        iG, _, _ = jd.jdft_basis_export(gb)
        C_h = workloads.make_bands(cfg_id, gb.nG, ik=ik)
        P_h = workloads.make_projectors(cfg_id, iG, kpts[ik], atoms)
        jd.jdft_alloc_workspace(gb, max(args.batch, min(nb, args.ws_bands)), max(nb, nproj))
        if args.batch > 0:
            jd.jdft_set_option(gb, "band_batch", args.batch)
        if args.overlap:
            jd.jdft_set_option(gb, "overlap_gemm", 1)
        for kv in args.opt:
            key, val = kv.split("=")
            jd.jdft_set_option(gb, key, int(val))
        ks.append(dict(gb=gb, C=torch.from_numpy(C_h).cuda(), P=torch.from_numpy(P_h).cuda(),
                       HC=torch.empty((nb, gb.nG), dtype=torch.complex128, device="cuda"),
                       M=torch.empty((nb, nb), dtype=torch.complex128, device="cuda") if do_overlap else None,
                       C_h=C_h if full else None, P_h=P_h if full else None,
                       info=dict(nG=gb.nG, a=gb.ncol * S[2], b=gb.npl * S[1] * S[2], N=gb.N, nb=nb, nproj=nproj,
                                 overlap_flops=overlap_flops(nb, gb.nG) if do_overlap else 0)))
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def step():
        for k in ks:
            jd.jdft_apply_H(k["gb"], V, k["P"], D, k["C"], k["HC"])
            if do_overlap:
                jd.jdft_overlap(k["gb"], k["C"], k["C"], k["M"])

    def timed(nsteps):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(nsteps)]
        for a, b in ev:
            flush.zero_()
            a.record()
            step()
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    # warm-up; the per-kernel profile (events around every launch of one kernel at a time) runs inside it
    timed(max(args.warmup, 3))
    per_kernel = {}
    nbatches = {}
    for name in KERNELS:
        tot, launches = 0.0, 0
        for k in ks:
            jd.jdft_set_option(k["gb"], "profile_kernel", jd.KERNEL_IDS[name])
        flush.zero_()
        step()
        for k in ks:
            n, ms = jd.jdft_profile_read(k["gb"])
            tot += ms
            launches += n
            jd.jdft_set_option(k["gb"], "profile_kernel", 0)
        per_kernel[name] = (tot, launches)
        nbatches[name] = launches
    dominant = max(per_kernel, key=lambda n: per_kernel[n][0])

    # timed region: K steps, events around each; the dominant kernel's launches are bracketed by events inside it
    # (launch-bound small workloads replay a CUDA graph, inside which single kernels cannot be bracketed: config 1 keeps the
    #  dominant kernel's time from the per-kernel pass above)
    in_region_profile = nb * int(np.prod(S)) > (4 << 20)
    for k in ks:
        jd.jdft_set_option(k["gb"], "profile_kernel", jd.KERNEL_IDS[dominant] if in_region_profile else 0)
        jd.jdft_profile_read(k["gb"])
    if not in_region_profile:
        for _ in range(3):   # set_option dropped the captured CUDA graphs: re-warm so that no capture falls into the timed region
            step()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    jd.jdft_launch_count(reset=True)
    sampler = ClockSampler(local) if rank == 0 else None
    t_wall = time.perf_counter()
    times = timed(steps)
    t_wall = time.perf_counter() - t_wall
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    launches = jd.jdft_launch_count()
    dom_ms, dom_n = 0.0, 0
    for k in ks:
        n, ms = jd.jdft_profile_read(k["gb"])
        dom_ms += ms
        dom_n += n
        jd.jdft_set_option(k["gb"], "profile_kernel", 0)
    if not in_region_profile:
        dom_ms, dom_n = per_kernel[dominant][0] * steps, per_kernel[dominant][1] * steps
    ms_step = float(np.mean(times))
    ms_step = max_over_ranks(ms_step, world)
    units = nb * nk
    value = aggregate_value(units, world, ms_step)

    overlap_rec = None
    if do_overlap:   # the 512 x 512 overlap on its own (it shares the gemm_dotk kernel with the projection P^+ C)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(5)]
        for a, b in ev:
            flush.zero_()
            a.record()
            for k in ks:
                jd.jdft_overlap(k["gb"], k["C"], k["C"], k["M"])
            b.record()
        torch.cuda.synchronize()
        oms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
        ofl = sum(k["info"]["overlap_flops"] for k in ks)
        overlap_rec = {"ms": oms, "TFLOP/s_counted_as_hermitian_half": ofl / (oms * 1e-3) / 1e12}

    e2e = None
    if full:
        # end to end through the HOST-buffer ABI call: pinned host inputs -> H2D -> kernels -> D2H, every step
        Vp = torch.from_numpy(Vh).pin_memory()
        Dp = torch.from_numpy(D_h).pin_memory()
        host = [dict(C=torch.from_numpy(k["C_h"]).pin_memory(), P=torch.from_numpy(k["P_h"]).pin_memory(),
                     HC=torch.empty((nb, k["gb"].nG), dtype=torch.complex128).pin_memory(),
                     M=torch.empty((nb, nb), dtype=torch.complex128).pin_memory() if do_overlap else None) for k in ks]

        def step_host():
            for k, h in zip(ks, host):
                jd.jdft_apply_H_host(k["gb"], Vp, h["P"], Dp, h["C"], h["HC"])
                if do_overlap:   # the overlap of the bands that call just uploaded: C crosses PCIe once per step
                    jd.jdft_overlap_host_resident(k["gb"], h["M"])

        step_host()
        e2e_steps = max(1, min(steps, 5))
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step_host()
        torch.cuda.synchronize()
        e2e_ms = 1e3 * (time.perf_counter() - t0) / e2e_steps
        e2e_ms = max_over_ranks(e2e_ms, world)
        h2d = sum(h["C"].numel() * 16 + h["P"].numel() * 16 + Vp.numel() * 8 + Dp.numel() * 8 for h in host)
        d2h = sum(h["HC"].numel() * 16 + (h["M"].numel() * 16 if do_overlap else 0) for h in host)
        e2e = {"value": aggregate_value(units, world, e2e_ms), "unit": UNIT, "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms, "steps": e2e_steps,
               "note": "jdft_apply_H_host (+ jdft_overlap_host_resident on the bands it uploaded): every input is copied every step (V_loc, P, D, C in; HC, M out)"}
        # the same with V_loc, P, D resident on the device (uploaded once per SCF iteration): only C in, HC out per step
        for k, h in zip(ks, host):
            jd.jdft_host_set_operators(k["gb"], Vp, h["P"], Dp)

        def step_host_res():
            for k, h in zip(ks, host):
                jd.jdft_apply_H_host_resident(k["gb"], h["C"], h["HC"])
                if do_overlap:
                    jd.jdft_overlap_host_resident(k["gb"], h["M"])

        step_host_res()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            step_host_res()
        torch.cuda.synchronize()
        res_ms = max_over_ranks(1e3 * (time.perf_counter() - t0) / e2e_steps, world)
        e2e["resident_operators"] = {
            "value": aggregate_value(units, world, res_ms), "ms_per_step": res_ms,
            "h2d_bytes_per_step": sum(h["C"].numel() * 16 for h in host), "d2h_bytes_per_step": d2h,
            "note": "jdft_host_set_operators once, then jdft_apply_H_host_resident (+ jdft_overlap_host_resident on the block it uploaded) per step"}
        del host, Vp, Dp

    # SURVEY 8(f) rank 1 operations on the same inputs (k-point 0): density of all bands, subspace Hamiltonian C^+ (H C)
    extras = None
    if full and args.extras:
        k = ks[0]
        fo = torch.rand(nb, dtype=torch.float64, device="cuda")
        nr = torch.empty(tuple(S), dtype=torch.float64, device="cuda")
        Hs = torch.empty((nb, nb), dtype=torch.complex128, device="cuda")

        def t_op(fn, reps=5):
            fn()
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
            for a, b in ev:
                flush.zero_()
                a.record()
                fn()
                b.record()
            torch.cuda.synchronize()
            return float(np.mean([a.elapsed_time(b) for a, b in ev]))

        ms_d = t_op(lambda: jd.jdft_density(k["gb"], k["C"], fo, nr))
        ms_s = t_op(lambda: jd.jdft_subspace(k["gb"], k["C"], k["HC"], Hs))
        i = k["info"]
        nbat = (nb + 255) // 256
        dens_bytes = nb * 16 * (i["nG"] + 2 * i["a"] + 2 * i["b"]) + nbat * 2 * 8 * i["N"]
        # Listing 1 on the scalar-field basis of the density cutoff (4 x Ecut, Gamma), 16 fields per call
        gs = jd.jdft_basis_create(R, [0.0, 0.0, 0.0], 4.0 * Ecut, S, device=local)
        nf = 16
        jd.jdft_set_workspace(gs, torch.empty(jd.jdft_workspace_bytes(gs, 3 * nf, 0) + 48 * nf * gs.nG, dtype=torch.uint8, device="cuda"))
        phi = torch.randn(nf, gs.nG, dtype=torch.complex128, device="cuda")
        epsr = 1.0 + 78.0 * torch.rand(int(np.prod(S)), dtype=torch.float64, device="cuda")
        hout = torch.empty_like(phi)
        ms_h = t_op(lambda: jd.jdft_pcm_hessian(gs, epsr, phi, hout))
        a_s, b_s = gs.ncol * S[2], gs.npl * S[1] * S[2]
        hess_bytes = 3 * nf * 16 * (4 * a_s + 4 * b_s + 2 * gs.nG) + nf * 16 * 8 * gs.nG + 8 * int(np.prod(S))
        # stand-alone I and J (row a10) on 16 bands: the full real-space block is written / read once
        nbI = min(nb, 16)
        CI = k["C"][:nbI].contiguous()
        psiI = torch.empty((nbI,) + tuple(S), dtype=torch.complex128, device="cuda")
        CJ = torch.empty_like(CI)
        ms_I = t_op(lambda: jd.jdft_apply_I(k["gb"], CI, psiI))
        ms_J = t_op(lambda: jd.jdft_apply_J(k["gb"], psiI, CJ))
        ij_bytes = nbI * 16 * (i["nG"] + 2 * i["a"] + 2 * i["b"] + i["N"])
        extras = {"pcm_hessian": {"ms": ms_h, "fields": nf, "nG": gs.nG, "fields_per_s": nf / (ms_h * 1e-3),
                                  "alg_GB/s": hess_bytes / (ms_h * 1e-3) / 1e9},
                  "density": {"ms": ms_d, "bands_per_s": nb / (ms_d * 1e-3), "alg_GB/s": dens_bytes / (ms_d * 1e-3) / 1e9},
                  "subspace": {"ms": ms_s, "TFLOP/s": 8.0 * nb * nb * i["nG"] / (ms_s * 1e-3) / 1e12},
                  "apply_I": {"ms": ms_I, "bands": nbI, "alg_GB/s": ij_bytes / (ms_I * 1e-3) / 1e9},
                  "apply_J": {"ms": ms_J, "bands": nbI, "alg_GB/s": ij_bytes / (ms_J * 1e-3) / 1e9}}
        extras.update(extra_ops(jd, torch, t_op, k, V, S, nb, nproj, cfg, R, Ecut, local))
        del gs, phi, epsr, hout, psiI

    infos = [k["info"] for k in ks]
    nGs = [k["gb"].nG for k in ks]
    del ks, V, D, flush
    torch.cuda.empty_cache()
    if rank != 0:
        return None
    hbm_peak, hbm_src = measured_peaks()
    dmma_peak, dfma_peak, fp_src = fp64_peak()

    def roof(name, ms, launches_):
        if ms <= 0:
            return None
        alg = sum(algorithmic(i, name, max(1, launches_ // max(1, len(infos)))) for i in infos)
        if name in HBM_KERNELS:
            ach = alg / (ms * 1e-3) / 1e9
            return {"bound": "hbm", "achieved": ach, "peak": hbm_peak, "unit": "GB/s", "frac": ach / hbm_peak}
        ach = alg / (ms * 1e-3) / 1e12
        return {"bound": "tensor", "achieved": ach, "peak": dmma_peak, "unit": "TFLOP/s", "frac": ach / dmma_peak}

    kernels = {}
    for name, (ms, n) in per_kernel.items():
        r = roof(name, ms, n)
        kernels[name] = {"ms_per_step": ms, "launches": n}
        if r and name != "splitk_reduce":
            kernels[name].update({"achieved": r["achieved"], "unit": r["unit"], "frac": r["frac"]})
        t = ncu_traffic(cfg_id, name)
        if t is not None:
            kernels[name]["traffic_per_launch"] = t
    roofline = roof(dominant, dom_ms / steps, dom_n // steps)
    roofline.update({"kernel": dominant, "launches_per_step": dom_n // steps,
                     "avg_launch_ms": dom_ms / max(1, dom_n), "peak_source": hbm_src if roofline["bound"] == "hbm" else fp_src,
                     "traffic": None, "share_of_step": dom_ms / steps / ms_step})
    roofline["traffic"] = ncu_traffic(cfg_id, dominant)
    dom_launches_step = max(1, dom_n // steps)
    roofline["algorithmic_per_launch"] = sum(algorithmic(i, dominant, max(1, dom_launches_step // max(1, len(infos))))
                                             for i in infos) / dom_launches_step
    roofline["note"] = ("algorithmic bytes (flops) per launch = DESIGN.md section 6 per-band figure x bands per launch "
                        "(complex MAC = 8 real flops whatever the kernel executes); traffic = ncu dram bytes per launch "
                        "(profiles/traffic.csv)")
    if dominant == "gemm_dotk" or (dominant == "gemm_expand" and nproj >= 320):
        # the GEMMs run the 3M complex-product scheme (6 real flops per complex MAC on the tensor pipe): the share of the
        # DMMA issue peak the kernel actually occupies is 3/4 of the algorithmic fraction (a fraction above 1 is the
        # algorithmic saving, not a faster pipe)
        roofline["executed_frac_of_peak_3m"] = 0.75 * roofline["frac"]
    fft_names = ("cols_inv", "rows_inv", "planes", "rows_fwd", "cols_fwd")
    local_bytes = sum(sum(algorithmic(i, n, max(1, nbatches[n] // len(infos))) for n in fft_names) for i in infos)
    local_ms = sum(per_kernel[n][0] for n in fft_names)
    gemm_flops = sum(algorithmic(i, "gemm_dotk", 1) + algorithmic(i, "gemm_expand", 1) for i in infos)
    gemm_ms = per_kernel["gemm_dotk"][0] + per_kernel["gemm_expand"][0]
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": cfg["name"], "bands": nb, "kpoints": nk, "nproj": nproj, "fft_box": list(S),
                   "nG": nGs, "overlap_in_step": do_overlap, "l2": "flushed (512 MiB memset) before every timed step",
                   "parallelism": "replicas x%d" % world},
        "clocks": clocks,
        "gpu_launches": launches,
        "roofline": roofline,
        "groups": {"fft_local": {"GB/s": local_bytes / (local_ms * 1e-3) / 1e9 if local_ms else None,
                                 "frac_hbm": local_bytes / (local_ms * 1e-3) / 1e9 / hbm_peak if local_ms else None,
                                 "ms_per_step": local_ms},
                   "gemm": {"TFLOP/s": gemm_flops / (gemm_ms * 1e-3) / 1e12 if gemm_ms else None,
                            "frac_fp64_tensor": gemm_flops / (gemm_ms * 1e-3) / 1e12 / dmma_peak if gemm_ms else None,
                            "ms_per_step": gemm_ms}},
        "kernels": kernels,
        "fp64_peaks": {"dmma_tflops": dmma_peak, "dfma_tflops": dfma_peak, "source": fp_src},
        "wall_s_timed_region": t_wall,
    }
    if overlap_rec is not None:
        line["overlap"] = overlap_rec
    if e2e is not None:
        line["e2e"] = e2e
    if extras is not None:
        line["extras"] = extras
    return line


def extra_ops(jd, torch, t_op, k, V, S, nb, nproj, cfg, R, Ecut, local):
    """Timings of the SURVEY 8(f) rank 2 / 3 additions on k-point 0: ultrasoft O_us / overlap_us with per-atom Q blocks,
    H with per-atom D blocks, and Listing 1 on real fields (half-sphere storage) beside the complex variant."""
    out = {}
    gb, C, P = k["gb"], k["C"], k["P"]
    nblk = cfg["n_lm"]
    g = torch.Generator(device="cuda").manual_seed(5)
    A = torch.randn((nproj // nblk, nblk, nblk), dtype=torch.complex128, device="cuda", generator=g)
    Qb = (0.05 * (A @ A.conj().transpose(1, 2))).contiguous()
    OC = torch.empty_like(C)
    Mus = torch.empty((nb, nb), dtype=torch.complex128, device="cuda")
    ms_o = t_op(lambda: jd.jdft_apply_O_us(gb, P, Qb, C, OC))
    ms_m = t_op(lambda: jd.jdft_overlap_us(gb, P, Qb, C, C, Mus))
    ms_h = t_op(lambda: jd.jdft_apply_H(gb, V, P, Qb, C, k["HC"]))
    nG = k["info"]["nG"]
    out["apply_O_us_blockQ"] = {"ms": ms_o, "TFLOP/s": 16.0 * nb * nproj * nG / (ms_o * 1e-3) / 1e12}
    out["overlap_us_blockQ"] = {"ms": ms_m, "TFLOP/s": (8.0 * (nb * (nb + 1) // 2) * nG + 8.0 * nb * nproj * nG) / (ms_m * 1e-3) / 1e12}
    out["apply_H_blockD"] = {"ms": ms_h, "band_apps_per_s": nb / (ms_h * 1e-3)}
    # Listing 1 on real fields: the density-cutoff basis (4 x Ecut, Gamma) as the scalar-field basis, 16 fields
    gs = jd.jdft_basis_create(R, [0.0, 0.0, 0.0], 4.0 * Ecut, S, device=local)
    nf = 16
    jd.jdft_set_workspace(gs, torch.empty(jd.jdft_workspace_bytes(gs, 3 * nf, 0) + 48 * nf * gs.nG, dtype=torch.uint8, device="cuda"))
    ph = torch.randn(nf, (gs.nG + 1) // 2, dtype=torch.complex128, device="cuda")
    eps = 1.0 + 78.0 * torch.rand(int(np.prod(S)), dtype=torch.float64, device="cuda")
    oh = torch.empty_like(ph)
    ms_r = t_op(lambda: jd.jdft_pcm_hessian_real(gs, eps, ph, oh))
    a_s, b_s = gs.ncol * S[2], gs.npl * S[1] * S[2]
    npair = (3 * nf + 1) // 2
    real_bytes = npair * 16 * (4 * a_s + 4 * b_s + 2 * gs.nG) + 2 * npair * 16 * gs.nG + 2 * nf * 16 * ((gs.nG + 1) // 2) + 8 * int(np.prod(S))
    out["pcm_hessian_real"] = {"ms": ms_r, "fields": nf, "nG_half": (gs.nG + 1) // 2, "fields_per_s": nf / (ms_r * 1e-3),
                               "alg_GB/s": real_bytes / (ms_r * 1e-3) / 1e9}
    return out


def compact(line):
    """Sub-record of a non-headline config: the device-timed value and the per-kernel roofline fractions."""
    return {"workload": line["config"]["workload"], "value": line["value"], "unit": line["unit"],
            "ms_per_step": line["ms_per_step"], "steps": line["steps"], "clocks": line["clocks"],
            "roofline": {k: line["roofline"][k] for k in ("kernel", "bound", "achieved", "peak", "unit", "frac", "traffic")},
            "groups": line["groups"],
            "kernel_frac": {n: round(v["frac"], 4) for n, v in line["kernels"].items() if "frac" in v}}


def shard_inputs(cfg_id, layout, make_basis, to_dev):
    """Per-rank inputs of the (k-point, band) sharded step: for each k-point this rank works on, the basis, the full
    projector block and ITS band rows of the seeded C (rank-independent seeds, so the shards are slices of the same
    global arrays the unsharded run uses).  make_basis(R, k, Ecut, S) -> (basis, iG); to_dev(ndarray) -> tensor."""
    R, kpts, Ecut, S = workloads.lattice(cfg_id)
    atoms = workloads.atoms_fractional(cfg_id)
    kdata = {}
    for k, blo, bhi in layout.group_units():
        basis, iG = make_basis(R, kpts[k], Ecut, S)
        C = workloads.make_bands(cfg_id, len(iG), ik=k)
        kdata[k] = dict(basis=basis, P=to_dev(workloads.make_projectors(cfg_id, iG, kpts[k], atoms)),
                        C=to_dev(np.ascontiguousarray(C[blo:bhi])), nG=len(iG))
    V = to_dev(workloads.make_vloc(cfg_id, atoms).reshape(-1))
    D = to_dev(workloads.make_D(cfg_id))
    return kdata, V, D


def run_shard(args):
    """--shard kb: ONE job sharded over the ranks with paper_1708_03621_b200/sharding.py -- k-points first (the paper's
    MPI-over-k layout), bands inside a k-point when there are more ranks than k-points; per step every
    rank applies H to its band columns (no collective) and forms its column block of C^+ O C (one all-gather, or a ring
    of neighbour exchanges overlapped with the GEMM).  Fixed total work: "scaling": "strong"."""
    import torch
    import torch.distributed as dist
    import paper_1708_03621_b200.binding as jd
    from paper_1708_03621_b200 import sharding as sh

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    cfg, nk, nb, nproj = config_sizes(args.config)
    layout = sh.KBLayout(nk, nb, world, rank)
    group = layout.new_band_group() if world > 1 else None

    def make_basis(R, k, Ecut, S):
        gb = jd.jdft_basis_create(R, k, Ecut, S, device=local)
        jd.jdft_alloc_workspace(gb, min(nb, args.ws_bands), max(nb, nproj))
        return gb, jd.jdft_basis_export(gb)[0]

    kdata, V, D = shard_inputs(args.config, layout, make_basis, lambda a: torch.from_numpy(a).cuda())
    for d in kdata.values():
        d["HC"] = torch.empty_like(d["C"])
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")

    def step():
        return sh.sharded_step(layout, kdata, V, D, group=group, mode=args.shard_mode, overlap=True)

    def timed(n):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in ev:
            flush.zero_()
            a.record()
            step()
            b.record()
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    timed(max(args.warmup, 3))
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    jd.jdft_launch_count(reset=True)
    sampler = ClockSampler(local) if rank == 0 else None
    times = timed(args.steps)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    ms_step = max_over_ranks(float(np.mean(times)), world)
    if rank != 0:
        return
    line = {"metric": METRIC, "value": nb * nk / (ms_step * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "bands": nb, "kpoints": nk, "nproj": nproj,
                       "parallelism": "kb-sharded x%d (k-points first, then bands; overlap by %s)" % (world, args.shard_mode),
                       "units_of_rank0": layout.group_units(), "overlap_in_step": True,
                       "l2": "flushed (512 MiB memset) before every timed step"},
            "clocks": clocks, "gpu_launches": jd.jdft_launch_count(),
            "roofline": None, "note": "sharded mode: per-kernel rooflines are reported by the default (replica) mode"}
    print(json.dumps(line), flush=True)


def run_ours(args):
    import torch
    import torch.distributed as dist

    t_start = time.perf_counter()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    line = measure(args.config, args, rank, world, local, full=True)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(args.config)
    # compact sub-records of the other full-size workloads (device-timed only), while the time budget allows
    others = [c for c in args.also if c != args.config] if world == 1 else []
    if others:
        line["other_configs"] = {}
        for c in others:
            if time.perf_counter() - t_start > args.also_budget:
                line["other_configs"][str(c)] = "skipped (time budget of the default run)"
                continue
            line["other_configs"][str(c)] = compact(measure(c, args, rank, world, local, full=False))
    if rank == 0:
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5,
                    help="BASELINE.json workload 1..5 (default 5: the largest single-GPU one, 512 bands + the 512^2 overlap)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--batch", type=int, default=0, help="bands per FFT batch (0 = automatic)")
    ap.add_argument("--ws-bands", type=int, default=256, help="bands of FFT scratch in the workspace (= automatic batch size)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extras", action="store_true", help="also time the SURVEY 8(f) operations (density, subspace, Listing 1, ...)")
    ap.add_argument("--overlap", action="store_true",
                    help="run the projection GEMM on a side stream beside the FFT pipeline (measured +1-2 %%; off by default)")
    ap.add_argument("--shard", default="", choices=["", "kb"],
                    help="kb: ONE job sharded over the ranks by (k-point, band range) through sharding.py instead of N replicas")
    ap.add_argument("--shard-mode", default="allgather", choices=["allgather", "ring"], help="schedule of the band-sharded overlap")
    ap.add_argument("--opt", action="append", default=[], help="library option key=value (jdft_set_option), repeatable; for experiments")
    ap.add_argument("--also", type=lambda s: [int(x) for x in s.split(",") if x], default=None,
                    help="other configs to attach as compact sub-records (default: 2,3,4 when --config is 5 and all defaults)")
    ap.add_argument("--also-budget", type=float, default=150.0, help="seconds after which no further sub-record is started")
    args = ap.parse_args()
    if args.also is None:
        args.also = [2, 3, 4] if args.config == 5 else []
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args)
        return
    if args.shard:
        run_shard(args)
    else:
        run_ours(args)
    if int(os.environ.get("WORLD_SIZE", "1")) > 1:
        import torch.distributed as dist
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
