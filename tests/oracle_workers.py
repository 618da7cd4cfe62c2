"""Oracle runs in worker processes (spawned; this module imports neither torch nor the CUDA binding), so that the
8-seed temperature parity at BASELINE.json's full package counts takes tens of seconds instead of minutes."""
import multiprocessing as mp
import os

import numpy as np


def _run(args):
    name, n, seed, kw = args
    from oracle import dies_oracle as orc
    from paper_2408_13807_b200 import synth
    p = getattr(synth, name)()
    o = orc.Oracle(p)
    o.run(n, seed=seed, **kw)
    return o.temperature(), dict(o.counters)


def oracle_temperatures(name, n, seeds, **kw):
    """T(r) of `synth.<name>()` followed with n packages for every seed; one process per seed (at most the cores)."""
    jobs = [(name, int(n), int(s), kw) for s in seeds]
    procs = max(1, min(len(jobs), os.cpu_count() or 1))
    with mp.get_context("spawn").Pool(procs) as pool:
        res = pool.map(_run, jobs)
    return np.array([r[0] for r in res]), [r[1] for r in res]
