"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer ("host code under ASan/UBSan in
the oracle build").  compute-sanitizer is closed on this pool, so this is the memory-safety evidence there is, and it
covers the checker: every entry point the parity tests lean on runs once on config 1 (and on the edge shapes: cavity,
one shell, empty shells) in an interpreter that loads the instrumented library; any finding aborts the process."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
from oracle import dies_oracle as orc
from paper_2408_13807_b200 import synth

p = synth.config1()
o = orc.Oracle(p)
o.tables()
o.run(20000, seed=1)                                    # full IRE
T = o.temperature()
assert np.all(np.isfinite(T)) and T.max() > p.T_grid[0]
o.run(20000, seed=2, k_bg=0.2)
o.run(20000, seed=3, ffi=1)
o.set_fixed_temperature(np.linspace(12.0, 19.0, p.n_shells))
o.run(20000, seed=4, mode=1)
o.run(5000, seed=5, mode=1, k_A=3.0, k_S=2.0)
o.run(5000, seed=5, mode=1, k_A=1.0, k_A_dilute=3.0)
o.run(5000, seed=6, mode=1, g_E=0.3, g_S=0.2)
o.run(5000, seed=7, mode=1, reemit_cell=1)
for pid in range(50):
    o.trace(20000, pid, seed=5, mode=1, max_events=8)   # lists cut at max_events
    o.trace(20000, pid, seed=5, mode=1, ffi=1, max_events=512)
o.tmc_run(20000, seed=8)
_, _, mass = o.tables()
o.tmc_run(20000, seed=9, eps_cur=o.absorbed / mass)
# edge shapes: a cavity with a point source, a single shell, shells without dust
q = synth.config3(n_shells=12, n_freq=16, tau_V=5.0)
oq = orc.Oracle(q)
oq.run(5000, seed=1)
oq.tmc_run(5000, seed=1)
one = synth.config1(n_shells=1)
orc.Oracle(one).run(5000, seed=1)
e = synth.config1()
e.rho = e.rho.copy(); e.rho[::3] = 0.0
orc.Oracle(e).run(5000, seed=1)
print("sanitized oracle ok")
"""


def test_oracle_runs_clean_under_asan_and_ubsan():
    from oracle import build
    build.build_sanitized()
    env = dict(os.environ, DIES_ORACLE_LIB=build.SANITIZED, LD_PRELOAD=build.asan_runtime(),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", PYTHONPATH=ROOT)
    r = subprocess.run([sys.executable, "-c", SCRIPT], cwd=ROOT, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "sanitized oracle ok" in r.stdout
    assert "AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr, r.stderr[-3000:]
