"""Seeded synthetic inputs for the DIES hot path (arXiv 2408.13807).

This module only *generates inputs*: grids, a synthetic dust law, Planck-function
emission tables and radiation fields, shaped like the paper's workloads (PAPER.md L167:
100-shell spheres, a dust model with HG scattering, an interstellar radiation field or a
10000 K central source).  It holds none of the method's arithmetic (no CDFs, no tracking,
no temperature lookup) and is imported by both the CUDA binding's callers and the oracle's
tests.  The five configurations follow BASELINE.json `configs` and SURVEY.md section 8(d);
DESIGN.md "Input recipe" states every choice made where BASELINE.json leaves freedom.

All quantities are in cgs units.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

H_PLANCK = 6.62607015e-27
C_LIGHT = 2.99792458e10
K_BOLTZ = 1.380649e-16
PARSEC = 3.0856775814913673e18
AU = 1.495978707e13
L_SUN = 3.828e33
UM = 1.0e-4  # cm
KAPPA_UV = 3.0e4  # cm^2/g, scale of the synthetic dust law (immaterial to T and tau)
LAMBDA_V_UM = 0.55


@dataclass
class Problem:
    """Plain arrays for one model; field names follow include/dies.h."""

    name: str
    r_bounds: np.ndarray        # n_shells+1, cm, ascending
    rho: np.ndarray             # n_shells, g/cm^3 (dust mass density)
    freq: np.ndarray            # n_freq, Hz, ascending
    kappa_abs: np.ndarray       # n_freq, cm^2/g
    kappa_sca: np.ndarray       # n_freq, cm^2/g
    g_hg: np.ndarray            # n_freq
    T_grid: np.ndarray          # n_T, K, ascending
    emis: np.ndarray            # n_T x n_freq, erg/s/g per bin
    ext_bin_intensity: Optional[np.ndarray] = None   # n_freq, erg/s/cm^2/sr per bin
    L_point: float = 0.0                             # erg/s
    point_bin_weights: Optional[np.ndarray] = None   # n_freq, relative
    n_packages: int = 0
    seed: int = 1
    k_bg: float = 0.5
    ffi: int = 0
    meta: dict = field(default_factory=dict)

    @property
    def n_shells(self) -> int:
        return int(self.rho.size)

    @property
    def n_freq(self) -> int:
        return int(self.freq.size)

    @property
    def n_T(self) -> int:
        return int(self.T_grid.size)


# ----------------------------------------------------------------------------- grids
def frequency_grid(n_freq: int, lam_min_um: float = 0.1, lam_max_um: float = 3000.0):
    """K points log-spaced in wavelength, returned ascending in frequency, with trapezoid
    bin weights in frequency (SURVEY.md 8(d) 'Frequency grid')."""
    lam = np.logspace(np.log10(lam_max_um), np.log10(lam_min_um), n_freq) * UM  # descending lambda
    nu = C_LIGHT / lam                                                          # ascending nu
    w = np.empty(n_freq)
    w[1:-1] = 0.5 * (nu[2:] - nu[:-2])
    w[0] = 0.5 * (nu[1] - nu[0])
    w[-1] = 0.5 * (nu[-1] - nu[-2])
    return nu, w


def planck_nu(nu: np.ndarray, T: float | np.ndarray) -> np.ndarray:
    """B_nu(T) in erg/s/cm^2/Hz/sr."""
    nu = np.asarray(nu, dtype=np.float64)
    x = H_PLANCK * nu / (K_BOLTZ * np.asarray(T, dtype=np.float64))
    with np.errstate(over="ignore", under="ignore", divide="ignore"):
        return 2.0 * H_PLANCK * nu**3 / C_LIGHT**2 / np.expm1(x)


def kappa_abs_law(lam_um: np.ndarray) -> np.ndarray:
    """Synthetic absorption law: constant below 0.3 um, lambda^-1.2 to 100 um, lambda^-2 beyond."""
    lam_um = np.asarray(lam_um, dtype=np.float64)
    k = np.where(lam_um <= 0.3, 1.0, (np.maximum(lam_um, 0.3) / 0.3) ** -1.2)
    k100 = (100.0 / 0.3) ** -1.2
    k = np.where(lam_um > 100.0, k100 * (lam_um / 100.0) ** -2.0, k)
    return KAPPA_UV * k


def albedo_law(lam_um: np.ndarray) -> np.ndarray:
    """0.5 at 0.1 um falling linearly in log10(lambda) to 0 at >= 100 um."""
    lam_um = np.asarray(lam_um, dtype=np.float64)
    return np.clip(0.5 * (1.0 - np.log10(lam_um / 0.1) / 3.0), 0.0, 0.5)


def dust(nu: np.ndarray, g: float = 0.5):
    lam_um = C_LIGHT / nu / UM
    ka = kappa_abs_law(lam_um)
    om = albedo_law(lam_um)
    ks = ka * om / (1.0 - om)
    return ka, ks, np.full_like(ka, g)


def kappa_ext_V() -> float:
    ka = float(kappa_abs_law(np.array([LAMBDA_V_UM]))[0])
    om = float(albedo_law(np.array([LAMBDA_V_UM]))[0])
    return ka / (1.0 - om)


def temperature_grid(n_T: int = 1000, T_min: float = 3.0, T_max: float = 1600.0) -> np.ndarray:
    return np.logspace(np.log10(T_min), np.log10(T_max), n_T)


def emission_table(nu, w, kappa_abs, T_grid) -> np.ndarray:
    """emis[t][k] = 4 pi kappa_abs,k B_nu_k(T_t) w_k  (power per dust mass emitted in bin k)."""
    B = planck_nu(nu[None, :], T_grid[:, None])
    return 4.0 * np.pi * kappa_abs[None, :] * B * w[None, :]


def diluted_blackbodies(nu, w, comps) -> np.ndarray:
    """Bin-integrated mean intensity sum_j W_j B_nu(T_j) w_k for comps = [(W_j, T_j), ...]."""
    J = np.zeros_like(nu)
    for dil, T in comps:
        J += dil * planck_nu(nu, T)
    return J * w


def normalise_tau_V(rho_shape: np.ndarray, r_bounds: np.ndarray, tau_V: float) -> np.ndarray:
    """Scale a density shape so that sum_i kappa_ext(V) rho_i dr_i = tau_V (centre/inner edge -> outer edge)."""
    dr = np.diff(r_bounds)
    return rho_shape * (tau_V / (kappa_ext_V() * np.sum(rho_shape * dr)))


def _dust_tables(n_freq: int, n_T: int = 1000):
    nu, w = frequency_grid(n_freq)
    ka, ks, g = dust(nu)
    Tg = temperature_grid(n_T)
    em = emission_table(nu, w, ka, Tg)
    return nu, w, ka, ks, g, Tg, em


ISRF_LIKE = [(4e-13, 3000.0), (1e-13, 4000.0), (1e-14, 7500.0)]


# ----------------------------------------------------------------------------- configs
def config1(n_packages: int = 100_000, seed: int = 1, tau_V: float = 1.0, n_shells: int = 32,
            n_freq: int = 64, n_T: int = 1000) -> Problem:
    """Tiny IRE sphere (BASELINE.json configs[0])."""
    nu, w, ka, ks, g, Tg, em = _dust_tables(n_freq, n_T)
    R = 0.1 * PARSEC
    rb = np.linspace(0.0, R, n_shells + 1)
    rho = normalise_tau_V(np.ones(n_shells), rb, tau_V)
    ext = diluted_blackbodies(nu, w, [(1e-14, 10000.0)])
    return Problem("config1_tiny_sphere", rb, rho, nu, ka, ks, g, Tg, em, ext_bin_intensity=ext,
                   n_packages=n_packages, seed=seed, meta=dict(tau_V=tau_V, w=w))


def config2(n_packages: int = 10_000_000, seed: int = 1, k_bg: float = 0.5, tau_V: float = 10.0,
            n_shells: int = 100, n_freq: int = 200, n_T: int = 1000) -> Problem:
    """Externally heated sphere (BASELINE.json configs[1]); k_bg 0.5 = unweighted, 0.2 = paper's best (L197)."""
    nu, w, ka, ks, g, Tg, em = _dust_tables(n_freq, n_T)
    R = 0.1 * PARSEC
    rb = np.linspace(0.0, R, n_shells + 1)
    rmid = 0.5 * (rb[1:] + rb[:-1])
    r0 = R / 5.0
    rho = normalise_tau_V(1.0 / (1.0 + (rmid / r0) ** 2), rb, tau_V)
    ext = diluted_blackbodies(nu, w, ISRF_LIKE)
    return Problem("config2_external", rb, rho, nu, ka, ks, g, Tg, em, ext_bin_intensity=ext,
                   n_packages=n_packages, seed=seed, k_bg=k_bg, meta=dict(tau_V=tau_V, w=w))


def config3(n_packages: int = 10_000_000, seed: int = 1, tau_V: float = 100.0, n_shells: int = 200,
            n_freq: int = 200, n_T: int = 1000) -> Problem:
    """Internally heated protostellar envelope (BASELINE.json configs[2]); tau_V=1000 is the thick variant."""
    nu, w, ka, ks, g, Tg, em = _dust_tables(n_freq, n_T)
    rb = np.logspace(np.log10(10.0 * AU), np.log10(1.0e4 * AU), n_shells + 1)
    rgeo = np.sqrt(rb[1:] * rb[:-1])
    rho = normalise_tau_V(rgeo ** -1.5, rb, tau_V)
    pw = planck_nu(nu, 10000.0) * w
    return Problem("config3_protostar", rb, rho, nu, ka, ks, g, Tg, em, L_point=10.0 * L_SUN,
                   point_bin_weights=pw, n_packages=n_packages, seed=seed, meta=dict(tau_V=tau_V, w=w))


def config4(n_packages: int = 100_000_000, seed: int = 1, ffi: int = 1, tau_V: float = 0.01,
            n_shells: int = 100, n_freq: int = 200, n_T: int = 1000) -> Problem:
    """Optically very thin sphere (BASELINE.json configs[3]); ffi=1 forced first interaction, 0 = unweighted."""
    nu, w, ka, ks, g, Tg, em = _dust_tables(n_freq, n_T)
    R = 0.1 * PARSEC
    rb = np.linspace(0.0, R, n_shells + 1)
    rho = normalise_tau_V(np.ones(n_shells), rb, tau_V)
    ext = diluted_blackbodies(nu, w, ISRF_LIKE)
    return Problem("config4_thin", rb, rho, nu, ka, ks, g, Tg, em, ext_bin_intensity=ext,
                   n_packages=n_packages, seed=seed, ffi=ffi, meta=dict(tau_V=tau_V, w=w))


@dataclass
class BatchProblem:
    """Config 5: n_models independent spheres sharing dust and emission tables."""

    name: str
    r_bounds: np.ndarray            # n_models x (n_shells+1)
    rho: np.ndarray                 # n_models x n_shells
    freq: np.ndarray
    kappa_abs: np.ndarray
    kappa_sca: np.ndarray
    g_hg: np.ndarray
    T_grid: np.ndarray
    emis: np.ndarray
    ext_bin_intensity: np.ndarray   # n_models x n_freq
    n_packages: int                 # per model
    seed: int = 1
    meta: dict = field(default_factory=dict)

    @property
    def n_models(self) -> int:
        return int(self.rho.shape[0])

    def model(self, m: int) -> Problem:
        return Problem(f"{self.name}[{m}]", self.r_bounds[m].copy(), self.rho[m].copy(), self.freq,
                       self.kappa_abs, self.kappa_sca, self.g_hg, self.T_grid, self.emis,
                       ext_bin_intensity=self.ext_bin_intensity[m].copy(), n_packages=self.n_packages,
                       seed=self.seed, meta=dict(model_index=m, tau_V=float(self.meta["tau_V"][m])))


def config5(n_models: int = 1024, n_packages: int = 1_000_000, seed: int = 1, n_shells: int = 64,
            n_freq: int = 100, n_T: int = 1000) -> BatchProblem:
    """Parameter-study batch (BASELINE.json configs[4]): Plummer-like spheres, central tau_V log-uniform
    0.1-100 and external field scale log-uniform 0.1-10, both drawn from numpy's PCG64(seed)."""
    nu, w, ka, ks, g, Tg, em = _dust_tables(n_freq, n_T)
    rng = np.random.default_rng(seed)
    tau = 10.0 ** rng.uniform(-1.0, 2.0, n_models)
    scale = 10.0 ** rng.uniform(-1.0, 1.0, n_models)
    R = 0.1 * PARSEC
    rb = np.linspace(0.0, R, n_shells + 1)
    rmid = 0.5 * (rb[1:] + rb[:-1])
    shape = 1.0 / (1.0 + (rmid / (R / 5.0)) ** 2)
    ext0 = diluted_blackbodies(nu, w, ISRF_LIKE)
    rho = np.stack([normalise_tau_V(shape, rb, t) for t in tau])
    return BatchProblem("config5_batch", np.tile(rb, (n_models, 1)), rho, nu, ka, ks, g, Tg, em,
                        scale[:, None] * ext0[None, :], n_packages, seed=seed,
                        meta=dict(tau_V=tau, field_scale=scale, w=w))


CONFIGS = {"config1": config1, "config2": config2, "config3": config3, "config4": config4}
