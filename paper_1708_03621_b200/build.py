"""Builds csrc/*.cu into paper_1708_03621_b200/libjdft_b200.so for sm_100a with nvcc (in-tree, no JIT cache).

Cross-compiles without a GPU.  `python -m paper_1708_03621_b200.build [--force]`.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libjdft_b200.so")
PEAK_TOOL = os.path.join(HERE, "fp64_peak")  # micro-benchmark binary bench.py runs for the FP64 roofline peak
SOURCES = ["basis.cu", "local.cu", "gemm.cu", "api.cu", "noalloc.cu"]
HEADERS = [os.path.join(CSRC, "jdft_internal.h"), os.path.join(CSRC, "fft.cuh"), os.path.join(CSRC, "cols_tuned.cuh"), os.path.join(CSRC, "planes_tma.cuh"), os.path.join(CSRC, "tma.cuh"),
           os.path.join(HERE, "..", "include", "jdft.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--expt-relaxed-constexpr", "-Xcompiler", "-fPIC", "-Wno-deprecated-gpu-targets", "-diag-suppress", "20281,177"]


def _nvcc():
    cand = os.environ.get("NVCC") or "/usr/local/cuda/bin/nvcc"
    return cand if os.path.exists(cand) else "nvcc"


def _stale(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force=False, verbose=False):
    """Compile (if stale) and return the path of libjdft_b200.so."""
    objdir = os.path.join(HERE, "build")
    os.makedirs(objdir, exist_ok=True)
    nvcc = _nvcc()
    jobs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(objdir, src.replace(".cu", ".o"))
        if force or _stale(o, [s] + HEADERS):
            jobs.append([nvcc] + NVCC_FLAGS + ["-c", s, "-o", o])
    objs = [os.path.join(objdir, s.replace(".cu", ".o")) for s in SOURCES]

    def run(cmd):
        if verbose:
            print(" ".join(cmd), flush=True)
        subprocess.check_call(cmd)

    if jobs:
        with ThreadPoolExecutor(max_workers=len(jobs)) as ex:
            list(ex.map(run, jobs))
    if force or jobs or _stale(LIB, objs):
        tmp = LIB + ".tmp%d" % os.getpid()
        run([nvcc, "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-Wno-deprecated-gpu-targets", "-o", tmp] + objs)  # static cudart (nvcc default)
        os.replace(tmp, LIB)
    peak_src = os.path.join(CSRC, "fp64_peak.cu")
    if force or _stale(PEAK_TOOL, [peak_src]):
        tmp = PEAK_TOOL + ".tmp%d" % os.getpid()
        run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-Wno-deprecated-gpu-targets", "-o", tmp, peak_src])
        os.replace(tmp, PEAK_TOOL)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
