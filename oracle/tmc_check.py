"""ctypes wrapper of oracle/tmc_check.c -- TEST INFRASTRUCTURE (pin d: IRE vs TMC iteration)."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_build.build()
_lib = C.CDLL(os.path.join(os.path.dirname(os.path.abspath(__file__)), "libtmc_check.so"))
_dp = C.POINTER(C.c_double)
_lib.tmc_solve.argtypes = [C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp,
                           C.c_uint64, C.c_uint64, C.c_int, C.c_double, C.c_uint64, _dp]


def tmc_solve(prob, n_src, n_dust, max_iter=20, tol=1e-3, seed=1):
    a = [np.ascontiguousarray(x, dtype=np.float64) for x in
         (prob.r_bounds, prob.rho, prob.kappa_abs, prob.kappa_sca, prob.g_hg, prob.T_grid, prob.emis,
          prob.ext_bin_intensity)]
    d = [x.ctypes.data_as(_dp) for x in a]
    T = np.zeros(prob.n_shells)
    it = _lib.tmc_solve(prob.n_shells, d[0], d[1], prob.n_freq, d[2], d[3], d[4], prob.n_T, d[5], d[6], d[7],
                        n_src, n_dust, max_iter, tol, seed, T.ctypes.data_as(_dp))
    return T, it
