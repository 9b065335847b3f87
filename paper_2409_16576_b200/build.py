"""Build libfann.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension).

    python -m paper_2409_16576_b200.build

`build_probe()` builds the measurement-only gather probe (csrc/fann_probe.cu, include/fann_probe.h) into its
own libfann_probe.so for bench.py; the product library carries none of it.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SOURCES = [os.path.join(HERE, "csrc", "fann_api.cu")]
DEPS = SOURCES + sorted(glob.glob(os.path.join(HERE, "csrc", "*.cuh"))) + [os.path.join(ROOT, "include", "fann.h")]
LIB = os.path.join(HERE, "libfann.so")
PROBE_SOURCES = [os.path.join(HERE, "csrc", "fann_probe.cu")]
PROBE_DEPS = PROBE_SOURCES + [os.path.join(ROOT, "include", "fann_probe.h")]
PROBE_LIB = os.path.join(HERE, "libfann_probe.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _build(lib, sources, deps, force, verbose):
    newest = max(os.path.getmtime(p) for p in deps)
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= newest:
        return lib
    nvcc = os.environ.get("NVCC", "nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib] + sources
    subprocess.check_call(cmd)
    return lib


def build(force: bool = False, verbose: bool = False) -> str:
    return _build(LIB, SOURCES, DEPS, force, verbose)


def build_probe(force: bool = False, verbose: bool = False) -> str:
    return _build(PROBE_LIB, PROBE_SOURCES, PROBE_DEPS, force, verbose)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_probe(force="--force" in sys.argv, verbose="-v" in sys.argv))
