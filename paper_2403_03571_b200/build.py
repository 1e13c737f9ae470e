"""Builds libapd_b200.so (the C-ABI library of include/apd.h) and libapd_probe.so (include/apd_probe.h, the FP32
microbenchmark bench.py uses for its roofline denominator) in-tree with nvcc for sm_100a.

    python -m paper_2403_03571_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys

_PKG = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_PKG, "csrc")
LIB_PATH = os.path.join(_PKG, "libapd_b200.so")
PROBE_LIB_PATH = os.path.join(_PKG, "libapd_probe.so")
SOURCES = ["apd_api.cu", "apd_kernels.cu", "apd_rowpoly.cu", "apd_finalize.cu", "apd_lbfgs.cu",
           "apd_host.cu", "apd_cull.cu", "apd_lloyd.cu", "apd_points.cu", "apd_tensor.cu", "apd_shard.cu", "apd_static.cu", "apd_validate.cu"]
PROBE_SOURCES = [os.path.join("probe", "apd_probe.cu")]
HEADERS = ["apd_internal.cuh", "apd_device.cuh", "apd_epilogue.cuh", os.path.join("..", "..", "include", "apd.h"),
           os.path.join("..", "..", "include", "apd_probe.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-Xptxas", "-v"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale(lib: str, sources) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(_CSRC, s) for s in sources] + [os.path.join(_CSRC, h) for h in HEADERS]
    return any(os.path.getmtime(d) > t for d in deps if os.path.exists(d))


def needs_build() -> bool:
    return _stale(LIB_PATH, SOURCES) or _stale(PROBE_LIB_PATH, PROBE_SOURCES)


def _compile(lib: str, sources, log_name: str, verbose: bool) -> None:
    srcs = [os.path.join(_CSRC, s) for s in sources if os.path.exists(os.path.join(_CSRC, s))]
    cmd = [_nvcc()] + NVCC_FLAGS + ["-o", lib] + srcs
    proc = subprocess.run(cmd, capture_output=True, text=True)
    log = os.path.join(_PKG, log_name)
    with open(log, "w") as fh:
        fh.write(" ".join(cmd) + "\n" + proc.stdout + proc.stderr)
    if verbose or proc.returncode != 0:
        sys.stderr.write(proc.stdout + proc.stderr)
    if proc.returncode != 0:
        raise RuntimeError(f"nvcc failed (exit {proc.returncode}); see {log}")


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale(LIB_PATH, SOURCES):
        _compile(LIB_PATH, SOURCES, "build.log", verbose)
    if force or _stale(PROBE_LIB_PATH, PROBE_SOURCES):
        _compile(PROBE_LIB_PATH, PROBE_SOURCES, "build_probe.log", verbose)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
