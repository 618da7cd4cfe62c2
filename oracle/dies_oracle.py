"""ctypes wrapper of oracle/dies_oracle.c -- TEST INFRASTRUCTURE, not the product.

Argument marshalling only; every number is computed in dies_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

_build.build()
# DIES_ORACLE_LIB: another build of the same source (the sanitizer build of oracle/build.py) instead of the default
_lib = C.CDLL(os.path.join(os.path.dirname(os.path.abspath(__file__)),
                           os.environ.get("DIES_ORACLE_LIB", "libdies_oracle.so")))

_dp = C.POINTER(C.c_double)
_u64 = C.c_uint64
_vp = C.c_void_p

COUNTER_NAMES = ("packages", "crossings", "ffi_crossings", "scatterings", "absorptions", "escaped",
                 "uninteracted", "terminated", "extra_blocks", "clamp_hi_samples")
SUM_NAMES = ("injected", "escaped", "uninteracted", "terminated", "reweight")
EVENT_NAMES = {0: "launch", 1: "scatter", 2: "absorb", 3: "escape", 4: "terminate", 5: "uninteracted"}

_lib.dies_oracle_create.restype = _vp
_lib.dies_oracle_create.argtypes = [C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, C.c_int, _dp, _dp]
_lib.dies_oracle_free.argtypes = [_vp]
_lib.dies_oracle_set_sources.argtypes = [_vp, _dp, C.c_double, _dp]
_lib.dies_oracle_set_fixed_temperature.argtypes = [_vp, _dp]
_lib.dies_oracle_temperature.argtypes = [_vp, _dp, _dp, C.POINTER(C.c_int), C.POINTER(C.c_int)]
_lib.dies_oracle_get_tables.argtypes = [_vp, _dp, _dp, _dp]
_lib.dies_oracle_run.argtypes = [_vp, _u64, _u64, _u64, _u64, _u64, C.c_uint32, C.c_double, C.c_int, C.c_int,
                                 _dp, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _dp,
                                 C.POINTER(_u64), _dp]
_lib.dies_oracle_trace.argtypes = [_vp, _u64, _u64, _u64, C.c_uint32, C.c_double, C.c_int, C.c_int, _dp, C.c_double,
                                   C.c_double, C.c_double, C.c_int, C.c_int,
                                   _dp, C.POINTER(C.c_int32), C.c_int, C.POINTER(C.c_int), _dp]
_lib.dies_oracle_tmc_run.argtypes = [_vp, _u64, _u64, C.c_uint32, _dp, _dp, _dp, C.POINTER(_u64), _dp]
_lib.dies_oracle_hg_pdf.restype = C.c_double
_lib.dies_oracle_hg_pdf.argtypes = [C.c_double, C.c_double]
_lib.dies_oracle_kA_profile.argtypes = [_vp, C.c_double, C.c_double, _dp]
_lib.dies_oracle_chord_walk.argtypes = [C.c_int, _dp, C.c_int, C.c_double, C.c_double, C.c_int,
                                        C.POINTER(C.c_int), _dp, C.POINTER(C.c_int)]
_lib.dies_oracle_hg_cos.restype = C.c_double
_lib.dies_oracle_hg_cos.argtypes = [C.c_double, C.c_double]
_lib.dies_oracle_launch_direction.argtypes = [C.c_double, C.c_double, _dp, _dp]
_lib.dies_oracle_scatter_direction.restype = C.c_double
_lib.dies_oracle_scatter_direction.argtypes = [C.c_double, C.c_double, C.c_double]
_lib.dies_oracle_uniform.restype = C.c_double
_lib.dies_oracle_uniform.argtypes = [C.c_uint32]
_lib.dies_oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _arr(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def philox4x32_10(key, ctr):
    k = (C.c_uint32 * 2)(*key)
    c = (C.c_uint32 * 4)(*ctr)
    o = (C.c_uint32 * 4)()
    _lib.dies_oracle_philox4x32_10(k, c, o)
    return tuple(int(x) for x in o)


def uniform(word: int) -> float:
    return float(_lib.dies_oracle_uniform(word))


def hg_cos(g: float, u: float) -> float:
    return float(_lib.dies_oracle_hg_cos(g, u))


def scatter_direction(mu: float, cos_theta: float, phi: float) -> float:
    """The direction cosine after a scattering, as the package loop computes it."""
    return float(_lib.dies_oracle_scatter_direction(mu, cos_theta, phi))


def launch_direction(u: float, k_bg: float):
    mu, w = C.c_double(), C.c_double()
    _lib.dies_oracle_launch_direction(u, k_bg, C.byref(mu), C.byref(w))
    return mu.value, w.value


def chord_walk(r_bounds, shell: int, r: float, mu: float):
    rb = _arr(r_bounds)
    n = rb.size - 1
    cap = 4 * n + 8
    sh = np.zeros(cap, dtype=np.int32)
    ln = np.zeros(cap, dtype=np.float64)
    ns = C.c_int()
    nc = _lib.dies_oracle_chord_walk(n, _d(rb), shell, r, mu, cap, sh.ctypes.data_as(C.POINTER(C.c_int)), _d(ln),
                                     C.byref(ns))
    if nc < 0:
        raise RuntimeError("chord walk did not terminate")
    return sh[:ns.value].copy(), ln[:ns.value].copy(), nc


class Oracle:
    """One model (shells + dust + two possible sources) held by the C oracle."""

    def __init__(self, prob):
        self.N, self.K, self.nT = prob.n_shells, prob.n_freq, prob.n_T
        self._keep = [_arr(x) for x in (prob.r_bounds, prob.rho, prob.kappa_abs, prob.kappa_sca, prob.g_hg,
                                        prob.T_grid, prob.emis)]
        rb, rho, ka, ks, g, Tg, em = self._keep
        self._h = _lib.dies_oracle_create(self.N, _d(rb), _d(rho), self.K, _d(ka), _d(ks), _d(g), self.nT, _d(Tg),
                                          _d(em))
        if not self._h:
            raise ValueError("oracle rejected the model")
        self.set_sources(prob.ext_bin_intensity, prob.L_point, prob.point_bin_weights)
        self.reset()

    def __del__(self):
        if getattr(self, "_h", None):
            _lib.dies_oracle_free(self._h)
            self._h = None

    def set_sources(self, ext, L_point=0.0, point_w=None):
        ext, pw = _arr(ext), _arr(point_w)
        self.n_sources = _lib.dies_oracle_set_sources(self._h, _d(ext), float(L_point), _d(pw))

    def set_fixed_temperature(self, T):
        T = _arr(T)
        assert T.size == self.N
        _lib.dies_oracle_set_fixed_temperature(self._h, _d(T))

    def reset(self, reemit: bool = False, pathlen: bool = False):
        self.absorbed = np.zeros(self.N)
        self.escaped = np.zeros(self.K)
        self.reemit = np.zeros((self.N, self.K)) if reemit else None
        self.pathlen = np.zeros(self.N) if pathlen else None
        self._counters = np.zeros(len(COUNTER_NAMES), dtype=np.uint64)
        self._sums = np.zeros(len(SUM_NAMES))

    def tables(self):
        eps = np.zeros(self.nT)
        F = np.zeros((self.nT, self.K))
        mass = np.zeros(self.N)
        _lib.dies_oracle_get_tables(self._h, _d(eps), _d(F), _d(mass))
        return eps, F, mass

    def kA_profile(self, k_A=1.0, k_A_dilute=0.0):
        """Per-shell k_A (L130): k_A at the highest density, k_A_dilute at the lowest (0: k_A everywhere)."""
        k = np.zeros(self.N)
        _lib.dies_oracle_kA_profile(self._h, float(k_A), float(k_A_dilute), _d(k))
        return k

    def _weights(self, k_A, k_A_dilute, k_S):
        if k_A == 1.0 and k_A_dilute == 0.0:
            return None
        return self.kA_profile(k_A, k_A_dilute)

    def run(self, n_total, seed=1, k_bg=0.5, ffi=0, mode=0, first_id=0, n_run=None, id_stride=1, model_index=0,
            k_A=1.0, k_A_dilute=0.0, k_S=1.0, g_E=0.0, g_S=None, reemit_cell=0, fp32_tallies=0):
        """Follow packages first_id..first_id+n_run-1; tallies accumulate until reset().  g_S=None: scattering
        directions are not weighted (g_S = 0 is a weighting: isotropic sampling, L207)."""
        if n_run is None:
            n_run = n_total * max(self.n_sources, 1) - first_id
        kw = self._weights(k_A, k_A_dilute, k_S)
        rc = _lib.dies_oracle_run(self._h, n_total, first_id, n_run, id_stride, seed, model_index, k_bg, ffi, mode,
                                  _d(kw), float(k_S), float(g_E), float(g_S or 0.0), int(g_S is not None),
                                  int(reemit_cell), int(fp32_tallies), _d(self.absorbed), _d(self.escaped), _d(self.reemit), _d(self.pathlen),
                                  self._counters.ctypes.data_as(C.POINTER(_u64)), _d(self._sums))
        if rc != 0:
            raise RuntimeError(f"dies_oracle_run failed: {rc}")
        return self

    def tmc_run(self, n_total, seed=1, eps_cur=None, model_index=0):
        """One iteration of the traditional Monte Carlo (reading R22): every active source and the
        dust (cells emitting eps_cur, power per mass; None = cold dust) send n_total packages each, absorption is
        continuous along the paths.  The tallies are reset first; returns self (absorbed, escaped, counters, sums)."""
        self.reset()
        e = None if eps_cur is None else _arr(eps_cur)
        rc = _lib.dies_oracle_tmc_run(self._h, int(n_total), int(seed), int(model_index), _d(e), _d(self.absorbed),
                                      _d(self.escaped), self._counters.ctypes.data_as(C.POINTER(_u64)), _d(self._sums))
        if rc != 0:
            raise RuntimeError(f"dies_oracle_tmc_run failed: {rc}")
        return self

    def tmc_solve(self, n_total, seed=1, max_iter=30, tol=3e-3, eps0=None, skip=0):
        """TMC iterations eps <- absorbed / mass (L31) until max |dT / T| < tol over the shells from `skip` on (the
        innermost shells of an externally heated sphere stay noisy, L177); returns (T, iterations, eps)."""
        _, _, mass = self.tables()
        eps, T_old = eps0, None
        for it in range(1, max_iter + 1):
            self.tmc_run(n_total, seed=seed + it, eps_cur=eps)
            eps = np.where(mass > 0, self.absorbed / np.where(mass > 0, mass, 1.0), 0.0)
            T = self.temperature()
            if T_old is not None and np.max(np.abs(T / T_old - 1.0)[skip:]) < tol:
                return T, it, eps
            T_old = T
        return T, max_iter, eps

    @property
    def counters(self):
        return {n: int(v) for n, v in zip(COUNTER_NAMES, self._counters)}

    @property
    def sums(self):
        return {n: float(v) for n, v in zip(SUM_NAMES, self._sums)}

    def temperature(self, absorbed=None):
        a = _arr(self.absorbed if absorbed is None else absorbed)
        T = np.zeros(self.N)
        lo, hi = C.c_int(), C.c_int()
        _lib.dies_oracle_temperature(self._h, _d(a), _d(T), C.byref(lo), C.byref(hi))
        self.clamps = (lo.value, hi.value)
        return T

    def trace(self, n_total, package_id, seed=1, k_bg=0.5, ffi=0, mode=1, model_index=0, absorbed_state=None,
              max_events=4096, k_A=1.0, k_A_dilute=0.0, k_S=1.0, g_E=0.0, g_S=None, reemit_cell=0):
        ev = np.zeros((max_events, 4), dtype=np.int32)
        n, margin = C.c_int(), C.c_double()
        st = _arr(absorbed_state)
        kw = self._weights(k_A, k_A_dilute, k_S)
        rc = _lib.dies_oracle_trace(self._h, n_total, package_id, seed, model_index, k_bg, ffi, mode, _d(kw),
                                    float(k_S), float(g_E), float(g_S or 0.0), int(g_S is not None), int(reemit_cell),
                                    _d(st),
                                    ev.ctypes.data_as(C.POINTER(C.c_int32)), max_events, C.byref(n), C.byref(margin))
        if rc != 0:
            raise RuntimeError(f"dies_oracle_trace failed: {rc}")
        return ev[:min(n.value, max_events)].copy(), n.value, margin.value
