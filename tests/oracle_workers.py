"""Oracle runs in worker processes (spawned; this module imports neither torch nor the CUDA binding), so that the
8-seed temperature parity at BASELINE.json's full package counts takes tens of seconds instead of minutes."""
import multiprocessing as mp
import os

import numpy as np


def _run(args):
    name, n, seed, kw = args
    from oracle import dies_oracle as orc
    from paper_2408_13807_b200 import synth
    if name.startswith("config5:"):
        # sphere i of the full batch of config 5: its index is word 3 of the Philox counter (RNG contract)
        i = int(name.split(":")[1])
        p = synth.config5().model(i)
        kw = dict(kw, model_index=i)
    else:
        p = getattr(synth, name)()
    o = orc.Oracle(p)
    o.run(n, seed=seed, **kw)
    return o.temperature(), dict(o.counters)


def oracle_temperatures(name, n, seeds, **kw):
    """T(r) of `synth.<name>()` followed with n packages for every seed; one process per seed (at most the cores).
    `name` may be a list of names: the result is then seeds x (names x shells), names in the given order."""
    if not isinstance(name, str):
        names = list(name)
        jobs = [(nm, int(n), int(s), kw) for s in seeds for nm in names]
        procs = max(1, min(len(jobs), os.cpu_count() or 1))
        with mp.get_context("spawn").Pool(procs) as pool:
            res = pool.map(_run, jobs, chunksize=1)
        T = np.array([r[0] for r in res]).reshape(len(list(seeds)), -1)
        return T, [r[1] for r in res]
    jobs = [(name, int(n), int(s), kw) for s in seeds]
    procs = max(1, min(len(jobs), os.cpu_count() or 1))
    with mp.get_context("spawn").Pool(procs) as pool:
        res = pool.map(_run, jobs)
    return np.array([r[0] for r in res]), [r[1] for r in res]
