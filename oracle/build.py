"""Compile the C sources of the oracle with gcc (building the checker is not using it)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
TARGETS = {
    "libdies_oracle.so": ["dies_oracle.c"],
    "libtmc_check.so": ["tmc_check.c"],
}


def build(force: bool = False) -> None:
    for lib, srcs in TARGETS.items():
        out = os.path.join(HERE, lib)
        paths = [os.path.join(HERE, s) for s in srcs]
        if not all(os.path.exists(p) for p in paths):
            continue
        if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(p) for p in paths):
            continue
        cmd = ["gcc", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-ffp-contract=off", "-o", out, *paths, "-lm"]
        subprocess.check_call(cmd)


SANITIZED = "libdies_oracle_san.so"


def build_sanitized(force: bool = False) -> str:
    """dies_oracle.c under AddressSanitizer + UndefinedBehaviorSanitizer (any finding aborts): the memory-safety
    check of the checker itself.  A process loads it in place of libdies_oracle.so when
    DIES_ORACLE_LIB names it and libasan is preloaded (tests/test_oracle_sanitized.py shows how)."""
    out = os.path.join(HERE, SANITIZED)
    src = os.path.join(HERE, "dies_oracle.c")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O1", "-g", "-fPIC", "-shared", "-Wall", "-Wextra", "-ffp-contract=off",
                               "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined",
                               "-fno-omit-frame-pointer", "-o", out, src, "-lm"])
    return out


def asan_runtime() -> str:
    """Path of gcc's libasan.so, to be preloaded into an interpreter that loads the sanitized library."""
    return subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()


if __name__ == "__main__":
    build(force=True)
