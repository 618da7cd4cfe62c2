"""Thin ctypes binding of libdies.so (include/dies.h): same names, argument marshalling only.

PyTorch is used for device memory (the workspace tensor) and the CUDA stream.  There is no CPU fallback:
a missing library raises ImportError-like RuntimeError on first use, a missing device makes every call fail with
DIES_ECUDA.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libdies.so")

DIES_OK, DIES_EINVAL, DIES_ENOMEM, DIES_ECUDA, DIES_ESTATE, DIES_EOVERFLOW = 0, -1, -2, -3, -4, -5
DIES_MODE_IRE, DIES_MODE_FIXED_T, DIES_MODE_TMC = 0, 1, 2
COUNTER_NAMES = ("packages", "crossings", "ffi_crossings", "scatterings", "absorptions", "escaped", "uninteracted",
                 "terminated", "extra_blocks", "clamp_hi_samples", "injected_raw", "terminated_raw", "reweight_raw",
                 "escaped_raw", "T_clamp_lo", "T_clamp_hi", "kernel_launches")
DIES_N_COUNTERS = len(COUNTER_NAMES)
EXPORTS = ("dies_workspace_bytes", "dies_create_model", "dies_create_batch", "dies_set_sources",
           "dies_set_sources_batch", "dies_run", "dies_run_batch", "dies_get_temperature", "dies_get_escape_spectrum",
           "dies_set_fixed_temperature", "dies_get_absorbed", "dies_get_counters", "dies_trace_packages",
           "dies_trace_package", "dies_test_philox", "dies_get_tables", "dies_destroy", "dies_last_error",
           "dies_device_info", "dies_bench_atomics", "dies_seek", "dies_set_tuning", "dies_get_tuning", "dies_set_model_offset",
           "dies_trace_packages_static")
# limits of dies_trace_packages_static (include/dies.h)
DIES_TRACE_STATIC_MAX_PACKAGES, DIES_TRACE_STATIC_MAX_EVENTS = 4096, 65536


class DiesError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libdies error {code}: {msg}")
        self.code = code


class dies_run_opts(C.Structure):
    _fields_ = [("k_bg", C.c_double), ("ffi", C.c_int32), ("mode", C.c_int32), ("accumulate", C.c_int32),
                ("fixed_shift", C.c_int32), ("n_total", C.c_uint64), ("k_A", C.c_double),
                ("k_A_dilute", C.c_double), ("k_S", C.c_double), ("g_E", C.c_double), ("g_S", C.c_double),
                ("use_g_S", C.c_int32), ("reemit_in_cell", C.c_int32)]


class dies_tuning(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("slots_uniform", "slots", "visit", "min_ready", "chunk", "pkg_per_block",
                                         "w_pool", "w_thr_hi", "w_thr_lo", "w_min_ready", "atom_stride")]


_dp = C.POINTER(C.c_double)
_lib = None


def lib():
    """Load libdies.so (built by paper_2408_13807_b200.build); fail loudly if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2408_13807_b200.build` "
                           "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, u64, i32p = C.c_void_p, C.c_uint64, C.POINTER(C.c_int32)
    L.dies_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_size_t)]
    L.dies_create_model.argtypes = [C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp, C.c_int, _dp, _dp, vp, C.c_size_t,
                                    C.POINTER(vp)]
    L.dies_create_batch.argtypes = [C.c_int, C.c_int, _dp, _dp, C.c_int, _dp, _dp, _dp, _dp, C.c_int, _dp, _dp, vp,
                                    C.c_size_t, C.POINTER(vp)]
    L.dies_set_sources.argtypes = [vp, _dp, C.c_double, _dp]
    L.dies_set_sources_batch.argtypes = [vp, _dp, _dp, _dp]
    L.dies_run.argtypes = [vp, u64, u64, C.POINTER(dies_run_opts), vp]
    L.dies_run_batch.argtypes = [vp, u64, u64, C.POINTER(dies_run_opts), vp]
    L.dies_seek.argtypes = [vp, u64]
    L.dies_set_model_offset.argtypes = [vp, C.c_uint32]
    L.dies_get_temperature.argtypes = [vp, _dp, C.c_int]
    L.dies_get_escape_spectrum.argtypes = [vp, _dp, C.c_int]
    L.dies_set_fixed_temperature.argtypes = [vp, _dp, C.c_int]
    L.dies_get_absorbed.argtypes = [vp, C.POINTER(C.c_int64), _dp, C.c_int]
    L.dies_get_counters.argtypes = [vp, C.POINTER(u64), C.c_int]
    L.dies_trace_packages.argtypes = [vp, C.c_int, u64, C.c_int, u64, u64, C.POINTER(dies_run_opts), i32p, C.c_int, i32p]
    L.dies_trace_package.argtypes = [vp, u64, u64, u64, C.POINTER(dies_run_opts), i32p, C.c_int, i32p]
    L.dies_trace_packages_static.argtypes = L.dies_trace_packages.argtypes
    L.dies_test_philox.argtypes = [u64, u64, C.c_uint32, C.c_uint32, C.c_int, C.POINTER(C.c_uint32),
                                   C.POINTER(C.c_float)]
    L.dies_get_tables.argtypes = [vp, _dp, C.POINTER(C.c_float)]
    L.dies_destroy.argtypes = [vp]
    L.dies_last_error.restype = C.c_char_p
    L.dies_device_info.argtypes = [C.POINTER(C.c_int)] * 3
    L.dies_bench_atomics.argtypes = [C.c_int, _dp, C.c_int, C.c_int, _dp, _dp]
    L.dies_set_tuning.argtypes = [C.POINTER(dies_tuning)]
    L.dies_get_tuning.argtypes = [C.POINTER(dies_tuning)]
    _lib = L
    return L


def _chk(rc):
    if rc != 0:
        raise DiesError(rc, lib().dies_last_error().decode())


def _a(x):
    return None if x is None else np.ascontiguousarray(x, dtype=np.float64)


def _p(x):
    return None if x is None else x.ctypes.data_as(_dp)


def dies_workspace_bytes(n_shells, n_freq, n_T, n_models=1) -> int:
    n = C.c_size_t()
    _chk(lib().dies_workspace_bytes(n_shells, n_freq, n_T, n_models, C.byref(n)))
    return n.value


def dies_device_info():
    a, b, c = C.c_int(), C.c_int(), C.c_int()
    _chk(lib().dies_device_info(C.byref(a), C.byref(b), C.byref(c)))
    return dict(n_sms=a.value, blocks_per_sm=b.value, threads_per_block=c.value)


def dies_set_tuning(**fields):
    """Launch tuning of the trackers (include/dies.h: dies_tuning); no fields restores the defaults."""
    if not fields:
        _chk(lib().dies_set_tuning(None))
        return
    t = dies_tuning(**{k: int(v) for k, v in fields.items()})
    _chk(lib().dies_set_tuning(C.byref(t)))


def dies_get_tuning():
    t = dies_tuning()
    _chk(lib().dies_get_tuning(C.byref(t)))
    return {n: getattr(t, n) for n, _ in dies_tuning._fields_}


def dies_bench_atomics(n_addr, weights=None, aggregate=1, iters=2000):
    """Absorptions/s and atomic instructions/s of the returning 64-bit atomicAdd pattern on n_addr tallies, drawn
    uniformly or with the probabilities `weights` (the workload's per-shell absorption histogram)."""
    a, b = C.c_double(), C.c_double()
    w = None
    if weights is not None:
        wa = np.ascontiguousarray(weights, dtype=np.float64)
        assert wa.size == n_addr
        w = wa.ctypes.data_as(_dp)
    _chk(lib().dies_bench_atomics(int(n_addr), w, int(aggregate), int(iters), C.byref(a), C.byref(b)))
    return dict(lane_ops_per_s=a.value, atomics_per_s=b.value)


def dies_test_philox(seed, first_id, block, model_index, n):
    w = np.zeros((n, 4), dtype=np.uint32)
    u = np.zeros((n, 4), dtype=np.float32)
    _chk(lib().dies_test_philox(seed, first_id, block, model_index, n, w.ctypes.data_as(C.POINTER(C.c_uint32)),
                                u.ctypes.data_as(C.POINTER(C.c_float))))
    return w, u


def _opts(k_bg=0.5, ffi=0, mode=DIES_MODE_IRE, accumulate=0, fixed_shift=24, n_total=0, k_A=1.0, k_A_dilute=0.0,
          k_S=1.0, g_E=0.0, g_S=None, reemit_cell=0):
    """g_S=None: scattering directions are not weighted (g_S = 0 is a weighting: isotropic sampling)."""
    return dies_run_opts(float(k_bg), int(ffi), int(mode), int(accumulate), int(fixed_shift), int(n_total),
                         float(k_A), float(k_A_dilute), float(k_S), float(g_E), float(g_S or 0.0),
                         int(g_S is not None), int(reemit_cell))


class Model:
    """One dies_model handle (a single model or a batch) with its torch-owned device workspace."""

    def __init__(self, prob=None, *, batch=None, device="cuda:0"):
        import torch

        if (prob is None) == (batch is None):
            raise ValueError("pass either a Problem or batch=BatchProblem")
        src = prob if prob is not None else batch
        self.n_models = 1 if prob is not None else batch.n_models
        self.N = int(src.rho.shape[-1])
        self.K, self.nT = int(src.freq.size), int(src.T_grid.size)
        nbytes = dies_workspace_bytes(self.N, self.K, self.nT, self.n_models)
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) & ~255
        arrs = [_a(x) for x in (src.r_bounds, src.rho, src.freq, src.kappa_abs, src.kappa_sca, src.g_hg, src.T_grid,
                                src.emis)]
        rb, rho, fr, ka, ks, g, Tg, em = arrs
        h = C.c_void_p()
        if prob is not None:
            _chk(lib().dies_create_model(self.N, _p(rb), _p(rho), self.K, _p(fr), _p(ka), _p(ks), _p(g), self.nT,
                                         _p(Tg), _p(em), C.c_void_p(self._ws_ptr), nbytes, C.byref(h)))
        else:
            _chk(lib().dies_create_batch(self.n_models, self.N, _p(rb), _p(rho), self.K, _p(fr), _p(ka), _p(ks),
                                         _p(g), self.nT, _p(Tg), _p(em), C.c_void_p(self._ws_ptr), nbytes,
                                         C.byref(h)))
        self._h = h
        if prob is not None:
            if prob.ext_bin_intensity is not None or prob.L_point > 0:
                self.dies_set_sources(prob.ext_bin_intensity, prob.L_point, prob.point_bin_weights)
        else:
            self.dies_set_sources_batch(batch.ext_bin_intensity, None, None)

    def close(self):
        if getattr(self, "_h", None):
            lib().dies_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/dies.h, same names
    def dies_set_sources(self, ext_bin_intensity, L_point=0.0, point_bin_weights=None):
        e, w = _a(ext_bin_intensity), _a(point_bin_weights)
        _chk(lib().dies_set_sources(self._h, _p(e), float(L_point), _p(w)))

    def dies_set_sources_batch(self, ext_bin_intensity, L_point=None, point_bin_weights=None):
        e, l, w = _a(ext_bin_intensity), _a(L_point), _a(point_bin_weights)
        _chk(lib().dies_set_sources_batch(self._h, _p(e), _p(l), _p(w)))

    def dies_run(self, n_packages, seed=1, stream=None, **opts):
        import torch

        o = _opts(**opts)
        s = torch.cuda.current_stream(self.device).cuda_stream if stream is None else stream
        _chk(lib().dies_run(self._h, int(n_packages), int(seed), C.byref(o), C.c_void_p(s)))

    dies_run_batch = dies_run

    def dies_set_model_offset(self, first_model):
        _chk(lib().dies_set_model_offset(self._h, int(first_model)))

    def dies_seek(self, first_id):
        _chk(lib().dies_seek(self._h, int(first_id)))

    def dies_get_temperature(self):
        T = np.zeros(self.n_models * self.N)
        _chk(lib().dies_get_temperature(self._h, _p(T), T.size))
        return T.reshape(self.n_models, self.N) if self.n_models > 1 else T

    def dies_get_escape_spectrum(self):
        L = np.zeros(self.n_models * self.K)
        _chk(lib().dies_get_escape_spectrum(self._h, _p(L), L.size))
        return L.reshape(self.n_models, self.K) if self.n_models > 1 else L

    def dies_set_fixed_temperature(self, T):
        T = _a(np.broadcast_to(T, (self.n_models, self.N)).reshape(-1)) if np.ndim(T) < 2 and self.n_models > 1 else _a(T).reshape(-1)
        _chk(lib().dies_set_fixed_temperature(self._h, _p(T), T.size))

    def dies_get_absorbed(self):
        """Returns (raw int64 tallies, energy per raw unit per model, absorbed energy per time = raw * unit)."""
        raw = np.zeros(self.n_models * self.N, dtype=np.int64)
        unit = np.zeros(self.n_models)
        _chk(lib().dies_get_absorbed(self._h, raw.ctypes.data_as(C.POINTER(C.c_int64)), _p(unit), raw.size))
        raw = raw.reshape(self.n_models, self.N)
        energy = raw.astype(np.float64) * unit[:, None]
        if self.n_models == 1:
            return raw[0], unit[0], energy[0]
        return raw, unit, energy

    def dies_get_counters(self):
        c = np.zeros(DIES_N_COUNTERS, dtype=np.uint64)
        _chk(lib().dies_get_counters(self._h, c.ctypes.data_as(C.POINTER(C.c_uint64)), c.size))
        d = {n: int(v) for n, v in zip(COUNTER_NAMES, c)}
        if d["reweight_raw"] >= 1 << 63:                      # signed sum in two's complement
            d["reweight_raw"] -= 1 << 64
        return d

    def dies_get_tables(self):
        eps = np.zeros(self.nT)
        F = np.zeros((self.nT, self.K), dtype=np.float32)
        _chk(lib().dies_get_tables(self._h, _p(eps), F.ctypes.data_as(C.POINTER(C.c_float))))
        return eps, F

    def dies_trace_packages(self, first_id, count, n_total, seed=1, model_index=0, max_events=256, **opts):
        opts.setdefault("mode", DIES_MODE_FIXED_T)
        o = _opts(**opts)
        ev = np.zeros((count, max_events, 4), dtype=np.int32)
        n = np.zeros(count, dtype=np.int32)
        i32p = C.POINTER(C.c_int32)
        _chk(lib().dies_trace_packages(self._h, model_index, int(first_id), count, int(n_total), int(seed),
                                       C.byref(o), ev.ctypes.data_as(i32p), max_events, n.ctypes.data_as(i32p)))
        return ev, n

    def dies_trace_packages_static(self, first_id, count, n_total, seed=1, model_index=0, max_events=256, **opts):
        """dies_trace_packages without device allocation: the scratch is a fixed array inside libdies.so.  For processes
        whose framework allocator already owns the GPU's memory, or that cannot afford the device-wide stall of
        cudaMalloc / cudaFree.  count <= DIES_TRACE_STATIC_MAX_PACKAGES and count * max_events <=
        DIES_TRACE_STATIC_MAX_EVENTS, else DiesError(DIES_EINVAL).  Calls share the array: do not overlap them."""
        opts.setdefault("mode", DIES_MODE_FIXED_T)
        o = _opts(**opts)
        # max(..., 1): a rejected size must reach the library's own check, not fail in numpy
        ev = np.zeros((max(count, 1), max(max_events, 1), 4), dtype=np.int32)
        n = np.zeros(max(count, 1), dtype=np.int32)
        i32p = C.POINTER(C.c_int32)
        _chk(lib().dies_trace_packages_static(self._h, model_index, int(first_id), count, int(n_total), int(seed),
                                              C.byref(o), ev.ctypes.data_as(i32p), max_events,
                                              n.ctypes.data_as(i32p)))
        return ev, n

    def dies_trace_package(self, package_id, n_total, seed=1, max_events=4096, **opts):
        ev, n = self.dies_trace_packages(package_id, 1, n_total, seed, 0, max_events, **opts)
        return ev[0, : min(int(n[0]), max_events)], int(n[0])
