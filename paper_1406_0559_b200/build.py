"""Build libmlens.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot)."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "mlens.cu")
DEPS = [SRC, os.path.join(_HERE, "csrc", "shoot_kernel.cuh"), os.path.join(_HERE, "csrc", "mapstats_kernel.cuh"), os.path.join(_HERE, "csrc", "convolve_kernel.cuh"), os.path.join(_HERE, "csrc", "shoot_umma_kernel.cuh"),
        os.path.join(os.path.dirname(_HERE), "include", "mlens.h")]
OUT = os.path.join(_HERE, "lib", "libmlens.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-shared", "-Xcompiler",
              "-fPIC", "-Xptxas", "-v", "-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64"]


MICRO_SRC = os.path.join(_HERE, "csrc", "alu_microbench.cu")
MICRO_OUT = os.path.join(_HERE, "lib", "alu_microbench")


def build_microbench(force: bool = False) -> str:
    """The pipe-rate microbenchmark executable; not on the product path."""
    os.makedirs(os.path.dirname(MICRO_OUT), exist_ok=True)
    if force or not os.path.exists(MICRO_OUT) or os.path.getmtime(MICRO_OUT) < os.path.getmtime(MICRO_SRC):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-o", MICRO_OUT, MICRO_SRC]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return MICRO_OUT


PROBE_SRC = os.path.join(_HERE, "csrc", "umma_probe.cu")
PROBE_OUT = os.path.join(_HERE, "lib", "umma_probe")


def build_umma_probe(force: bool = False) -> str:
    """The tensor-pipe probe for the next kernel generation; not on the product path."""
    os.makedirs(os.path.dirname(PROBE_OUT), exist_ok=True)
    if force or not os.path.exists(PROBE_OUT) or os.path.getmtime(PROBE_OUT) < os.path.getmtime(PROBE_SRC):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-o", PROBE_OUT, PROBE_SRC]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return PROBE_OUT


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(os.path.dirname(OUT), exist_ok=True)
    build_microbench(force)
    build_umma_probe(force)
    stale = force or not os.path.exists(OUT) or any(os.path.getmtime(OUT) < os.path.getmtime(d) for d in DEPS)
    if stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, *NVCC_FLAGS, "-o", OUT, SRC]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed: " + " ".join(cmd))
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
