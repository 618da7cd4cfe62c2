"""CPU-side checks of the boundary: libdies.so loads, exports every symbol include/dies.h declares, and refuses
to compute without a device (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

from paper_2408_13807_b200 import binding, build, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "dies.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(dies_[a-z_0-9]+)\s*\(", header))
    assert len(declared) >= 19
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(binding.EXPORTS)


def test_run_opts_struct_layout():
    assert binding.dies_run_opts.k_bg.offset == 0 and binding.dies_run_opts.ffi.offset == 8
    assert binding.dies_run_opts.n_total.offset == 24
    import ctypes
    assert binding.dies_run_opts.k_A.offset == 32 and binding.dies_run_opts.k_S.offset == 48
    assert binding.dies_run_opts.g_E.offset == 56 and binding.dies_run_opts.use_g_S.offset == 72
    assert binding.dies_run_opts.reemit_in_cell.offset == 76
    assert ctypes.sizeof(binding.dies_run_opts) == 80


def test_workspace_bytes_and_argument_errors(lib):
    n1 = binding.dies_workspace_bytes(100, 200, 1000, 1)
    n2 = binding.dies_workspace_bytes(100, 200, 1000, 2)
    assert n2 > n1 > 1000 * 200 * 12
    with pytest.raises(binding.DiesError) as e:
        binding.dies_workspace_bytes(0, 200, 1000, 1)
    assert e.value.code == binding.DIES_EINVAL


def test_no_cpu_fallback(lib):
    """Without a CUDA device the library must fail loudly (DIES_ECUDA), never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(binding.DiesError) as e:
        binding.dies_device_info()
    assert e.value.code == binding.DIES_ECUDA
    with pytest.raises(binding.DiesError) as e:
        binding.dies_test_philox(1, 0, 0, 0, 4)
    assert e.value.code == binding.DIES_ECUDA


def test_product_does_not_import_oracle():
    """The product path never imports, links or executes anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2408_13807_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+\.*oracle|oracle[/.]|liboracle|libdies_oracle", txt, re.M), f


def test_synthetic_configs_have_the_stated_shapes():
    p1, p2, p3, p4 = synth.config1(), synth.config2(), synth.config3(), synth.config4()
    assert (p1.n_shells, p1.n_freq, p1.n_T, p1.n_packages) == (32, 64, 1000, 100_000)
    assert (p2.n_shells, p2.n_freq, p2.n_packages) == (100, 200, 10_000_000)
    assert (p3.n_shells, p3.n_freq, p3.r_bounds[0] > 0, p3.L_point) == (200, 200, True, 10 * synth.L_SUN)
    assert (p4.n_shells, p4.n_packages, p4.ffi) == (100, 100_000_000, 1)
    for p, tau in ((p1, 1.0), (p2, 10.0), (p3, 100.0), (p4, 0.01)):
        got = synth.kappa_ext_V() * np.sum(p.rho * np.diff(p.r_bounds))
        assert abs(got / tau - 1) < 1e-12
        assert np.all(np.diff(p.freq) > 0) and np.all(np.diff(p.emis.sum(axis=1)) > 0)
        assert np.all(np.diff(p.emis, axis=0) >= 0)
    b = synth.config5(n_models=16, n_packages=1000)
    assert b.rho.shape == (16, 64) and b.ext_bin_intensity.shape == (16, 100)
    assert 0.1 <= b.meta["tau_V"].min() and b.meta["tau_V"].max() <= 100


def test_c_example_compiles_and_links_against_the_library(tmp_path):
    """tests/c_abi/c_abi_sphere.c uses include/dies.h from plain C: it must compile without warnings about the
    declarations and link against libdies.so (it is run on the GPU by tests/test_gpu_c_example.py)."""
    import os
    import shutil
    import subprocess
    from paper_2408_13807_b200 import build
    build.build()
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    pkg = os.path.join(root, "paper_2408_13807_b200")
    cc = shutil.which("gcc") or shutil.which("cc")
    r = subprocess.run([cc, "-std=c99", "-Wall", "-Werror", "-O1", "-I" + os.path.join(root, "include"),
                        "-I" + os.path.join(cuda, "include"), os.path.join(root, "tests", "c_abi", "c_abi_sphere.c"),
                        "-o", str(tmp_path / "c_abi_sphere"), "-L" + pkg, "-ldies", "-L" + os.path.join(cuda, "lib64"),
                        "-lcudart", "-lm", "-Wl,-rpath," + pkg], capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_bench_constants_belong_to_the_kernel_sources():
    """bench.py's work-per-unit constants (INSTR) were derived from an ncu source page of ONE version of the kernel
    sources; bench.py prints a roofline fraction only while the sources still hash to KERNEL_SHA256.  This test keeps the
    two from drifting apart unnoticed: after a kernel edit, re-profile, run profile_parts and update both."""
    import bench
    assert bench.KERNEL_SHA256 == build.kernel_hash()
    assert set(bench.INSTR) == {"crossing", "scattering", "absorption", "package"}
    import hashlib
    tmc = os.path.join(ROOT, "paper_2408_13807_b200", "csrc", "dies_tmc.cuh")
    assert bench.TMC_SHA256 == hashlib.sha256(open(tmc, "rb").read()).hexdigest()


def test_build_sees_every_kernel_source(lib):
    """build.build() must rebuild after an edit to ANY file the library is compiled from (the hot kernels live in
    headers: a parity run against a stale libdies.so would be one edit away otherwise).  No compile here: a header's
    modification time is moved past the library's and back."""
    names = {os.path.basename(d) for d in build.deps()}
    csrc = os.path.join(ROOT, "paper_2408_13807_b200", "csrc")
    assert names >= {f for f in os.listdir(csrc) if f.endswith((".cu", ".cuh"))} | {"dies.h"}
    assert not build.stale()
    for name in ("dies_fly.cuh", "dies_tmc.cuh", "dies_tracker.cuh"):
        path = os.path.join(csrc, name)
        st = os.stat(path)
        try:
            newer = os.path.getmtime(build.LIB) + 10
            os.utime(path, (newer, newer))
            assert build.stale(), name
        finally:
            os.utime(path, ns=(st.st_atime_ns, st.st_mtime_ns))
    assert not build.stale()
