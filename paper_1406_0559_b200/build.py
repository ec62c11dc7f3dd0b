"""Build the native pieces in-tree with nvcc for sm_100a (no JIT cache: the .so files travel with the repo snapshot).

  lib/libmlens.so            the product: the C ABI of include/mlens.h with the production kernels only
  lib/libmlens_ablations.so  the same sources compiled with -DMLENS_ABLATIONS: additionally holds the debug / ablation /
                             experimental shooting kernels and loop variants that `mlens_set_option` can select.  Used by
                             the tests and the profiling runs only (`mlens.lib(ablations=True)`); never by the product path.
  ../bench/alu_microbench    pipe-rate microbenchmark executable that bench.py calls for the measured FP32 peak

`build()` compiles libmlens.so FIRST and on its own, so that nothing else can break the product build.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
_CSRC = os.path.join(_HERE, "csrc")
SRC = os.path.join(_CSRC, "mlens.cu")
DEPS = [SRC, os.path.join(_ROOT, "include", "mlens.h")] + sorted(
    os.path.join(_CSRC, f) for f in os.listdir(_CSRC) if f.endswith(".cuh"))
OUT = os.path.join(_HERE, "lib", "libmlens.so")
OUT_ABLATIONS = os.path.join(_HERE, "lib", "libmlens_ablations.so")

ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
NVCC_FLAGS = [*ARCH, "-O3", "-lineinfo", "-std=c++17", "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-lcufft",
              "-Xlinker", "-rpath=/usr/local/cuda/lib64"]

MICRO_SRC = os.path.join(_ROOT, "bench", "alu_microbench.cu")
MICRO_OUT = os.path.join(_ROOT, "bench", "alu_microbench")


def _nvcc() -> str:
    return os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def _stale(out: str, deps: list[str], force: bool) -> bool:
    return force or not os.path.exists(out) or any(os.path.getmtime(out) < os.path.getmtime(d) for d in deps)


def _run(cmd: list[str], verbose: bool) -> None:
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))


def build_lib(force: bool = False, verbose: bool = False) -> str:
    """libmlens.so — the product library (production kernels only)."""
    os.makedirs(os.path.dirname(OUT), exist_ok=True)
    if _stale(OUT, DEPS, force):
        _run([_nvcc(), *NVCC_FLAGS, "-o", OUT, SRC], verbose)
    return OUT


def build_ablations(force: bool = False, verbose: bool = False) -> str:
    """libmlens_ablations.so — same ABI plus the kernels behind MLENS_ABLATIONS (tests and profiling only)."""
    os.makedirs(os.path.dirname(OUT_ABLATIONS), exist_ok=True)
    if _stale(OUT_ABLATIONS, DEPS, force):
        _run([_nvcc(), *NVCC_FLAGS, "-DMLENS_ABLATIONS", "-o", OUT_ABLATIONS, SRC], verbose)
    return OUT_ABLATIONS


def build_microbench(force: bool = False, verbose: bool = False) -> str:
    """The pipe-rate microbenchmark executable; bench.py runs it for `roofline.peak_measured`."""
    if _stale(MICRO_OUT, [MICRO_SRC], force):
        _run([_nvcc(), *ARCH, "-O3", "-lineinfo", "-std=c++17", "-o", MICRO_OUT, MICRO_SRC], verbose)
    return MICRO_OUT


def build(force: bool = False, verbose: bool = False) -> str:
    out = build_lib(force, verbose)  # the product first: a failure below cannot leave it unbuilt
    build_ablations(force, verbose)
    build_microbench(force, verbose)
    return out


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
