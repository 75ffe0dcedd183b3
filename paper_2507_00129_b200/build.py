"""In-tree build of liblya.so (the product) and liblya_peaks.so (bench-only microbenchmarks)
with nvcc for sm_100a (no JIT cache, no torch extension)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblya.so")
LIB_PEAKS = os.path.join(HERE, "liblya_peaks.so")
SOURCES = ["lya_api.cu", "neighbours.cu", "prep.cu", "xi2pcf.cu", "dmat.cu", "xi3pcf.cu"]
HEADERS = sorted(f for f in os.listdir(CSRC) if f.endswith((".cuh", ".h")))
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def _stale(lib, srcs) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, s) for s in srcs] + [os.path.join(CSRC, h) for h in HEADERS]
    deps += [os.path.join(HERE, "..", "include", h) for h in ("lya.h", "lya_peaks.h")]
    return any(os.path.exists(d) and os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra_flags=()) -> str:
    """Compile csrc/*.cu into paper_2507_00129_b200/liblya.so (sm_100a, -lineinfo)."""
    if not force and not _stale(LIB, SOURCES):
        return LIB
    nvcc = _nvcc()
    objs = []
    procs = []
    for src in SOURCES:
        obj = os.path.join(CSRC, src.replace(".cu", ".o"))
        cmd = [nvcc, *NVCC_FLAGS, *extra_flags, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT)))
        objs.append(obj)
    for src, p in procs:
        out, _ = p.communicate()
        if verbose or p.returncode:
            sys.stderr.write(out.decode())
        if p.returncode:
            raise RuntimeError(f"nvcc failed on {src}")
    subprocess.check_call([nvcc, "-shared", "-o", LIB, *objs, "-lcudart"])
    return LIB


def build_peaks(force: bool = False) -> str:
    """liblya_peaks.so: roofline-denominator microbenchmarks, loaded by bench.py only."""
    if not force and not _stale(LIB_PEAKS, ["peaks.cu"]):
        return LIB_PEAKS
    subprocess.check_call([_nvcc(), *NVCC_FLAGS, "-shared", os.path.join(CSRC, "peaks.cu"), "-o", LIB_PEAKS, "-lcudart"])
    return LIB_PEAKS


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_peaks(force="--force" in sys.argv))
