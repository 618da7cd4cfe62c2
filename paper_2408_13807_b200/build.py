"""Build libdies.so (the C-ABI library of include/dies.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdies.so")
SOURCES = [os.path.join(CSRC, "dies_lib.cu")]
INCLUDE = os.path.join(HERE, "..", "include")


def deps() -> list[str]:
    """Everything libdies.so is compiled from: every file under csrc/ and include/ (listed at call time, so that a
    new header is a dependency without an edit here)."""
    out = []
    for d in (CSRC, INCLUDE):
        out += [os.path.join(d, f) for f in sorted(os.listdir(d)) if f.endswith((".cu", ".cuh", ".h"))]
    return out


# the tracker sources bench.py's work-per-unit constants belong to (bench.KERNEL_SHA256)
KERNEL_SOURCES = ("dies_fly.cuh", "dies_tracker.cuh")


def kernel_hash() -> str:
    """SHA-256 of the tracker sources: bench.py prints a roofline fraction only while it equals the hash its
    constants were derived at."""
    h = hashlib.sha256()
    for name in KERNEL_SOURCES:
        h.update(open(os.path.join(CSRC, name), "rb").read())
    return h.hexdigest()


def stale() -> bool:
    """True when libdies.so is missing or older than one of its sources."""
    return not os.path.exists(LIB) or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in deps())


NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a", "-shared",
              "-Xcompiler", "-fPIC", "-Xptxas", "-v",
              # single-precision division and square root of the event arithmetic at 2 ulp (R14b)
              "-prec-div=false", "-prec-sqrt=false"]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, *NVCC_FLAGS, "-o", LIB, *SOURCES]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libdies.so")
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    return LIB


if __name__ == "__main__":
    build(force=True, verbose=True)
