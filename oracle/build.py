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


if __name__ == "__main__":
    build(force=True)
