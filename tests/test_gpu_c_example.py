"""The boundary is a C ABI: tests/c_abi/c_abi_sphere.c (plain C, cudaMalloc + the dies_* calls of include/dies.h, no
Python and no torch in the process) is built with gcc against libdies.so and run on the GPU; the same problem is then
followed by the oracle and the temperatures compared."""
import os
import re
import shutil
import subprocess

import numpy as np
import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
CUDA = os.environ.get("CUDA_HOME", "/usr/local/cuda")


def test_c_program_runs_the_hot_path_through_the_c_abi(tmp_path):
    from paper_2408_13807_b200 import build
    build.build()                                            # libdies.so must exist (fails loudly otherwise)
    pkg = os.path.join(ROOT, "paper_2408_13807_b200")
    exe = str(tmp_path / "c_abi_sphere")
    cc = shutil.which("gcc") or shutil.which("cc")
    assert cc, "no C compiler on this box"
    subprocess.run([cc, "-O2", "-I" + os.path.join(ROOT, "include"), "-I" + os.path.join(CUDA, "include"),
                    os.path.join(ROOT, "tests", "c_abi", "c_abi_sphere.c"), "-o", exe, "-L" + pkg, "-ldies",
                    "-L" + os.path.join(CUDA, "lib64"), "-lcudart", "-lm", "-Wl,-rpath," + pkg,
                    "-Wl,-rpath," + os.path.join(CUDA, "lib64")], check=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0, r.stdout + r.stderr
    assert r.stdout.strip().endswith("OK")
    # no Python runtime and no torch library in that process
    ldd = subprocess.run(["ldd", exe], capture_output=True, text=True).stdout
    assert "libdies.so" in ldd and "libtorch" not in ldd and "libpython" not in ldd and "libc10" not in ldd

    # the same sphere in the oracle: centre and surface temperatures the C program printed, within Monte Carlo noise
    from oracle import dies_oracle as orc
    from paper_2408_13807_b200 import synth
    N, K, NT, R, tau = 40, 16, 200, 3.0e17, 5.0
    k = np.arange(K)
    ka, ks, g = 100.0 * (0.2 + k / K), 50.0 * k / K, 0.6 * k / K
    J = np.where(k >= K // 2, 1e-4 * np.exp(-0.3 * (k - K // 2)), 0.0)
    Tg = 3.0 * (1000.0 / 3.0) ** (np.arange(NT) / (NT - 1))
    em = ka[None, :] * (Tg[:, None] / 100.0) ** (4.0 + 0.25 * k[None, :])
    p = synth.Problem("c_example", R * np.arange(N + 1) / N, np.full(N, tau / (ka[-1] * R)),
                      1e11 * 10.0 ** (4.0 * k / (K - 1)), ka, ks, g, Tg, em, ext_bin_intensity=J, n_packages=1_000_000)
    To = []
    for s in (1, 2, 3, 4):
        o = orc.Oracle(p)
        o.run(250_000, seed=s)
        To.append(o.temperature())
    To = np.array(To)
    mo, sd = To.mean(0), To.std(0, ddof=1)
    m = re.search(r"T\(centre\) ([0-9.]+) K\s+T\(surface\) ([0-9.]+) K", r.stdout)
    Tc, Ts = float(m.group(1)), float(m.group(2))
    assert abs(Tc - mo[0]) < max(0.01 * mo[0], 4 * sd[0]), (Tc, mo[0], sd[0])
    assert abs(Ts - mo[-1]) < max(0.01 * mo[-1], 4 * sd[-1]), (Ts, mo[-1], sd[-1])
