"""Pins of the oracle's free-path weighting (section 2.2.2, Eq. 8; reading R17):
the biased clocks p'(tau) = k e^{-k tau} with the weight W = e^{tau (k-1)} / k must leave every expectation
unchanged.  CPU only."""
import math

import numpy as np
import pytest

from oracle import dies_oracle as orc
from paper_2408_13807_b200 import synth
from test_oracle_pins import _thin_limit_T, toy_problem


def test_unit_factors_are_the_unweighted_method():
    """k_A = k_S = 1 (also as a density-dependent profile 1..1) is the plain method, number for number."""
    p = synth.config1()
    a = orc.Oracle(p).run(20000, seed=3)
    b = orc.Oracle(p).run(20000, seed=3, k_A=1.0, k_A_dilute=1.0, k_S=1.0)
    assert np.array_equal(a.absorbed, b.absorbed) and np.array_equal(a.escaped, b.escaped)
    assert a.counters == b.counters and b.sums["reweight"] == 0.0


def test_kA_profile_is_linear_in_log_density():
    """L130 / L211: k = 3 at the lowest density, 1 at the highest, linear in log n."""
    p = synth.config2(n_shells=20)
    o = orc.Oracle(p)
    k = o.kA_profile(1.0, 3.0)
    ln = np.log(p.rho)
    assert abs(k[np.argmax(p.rho)] - 1.0) < 1e-12 and abs(k[np.argmin(p.rho)] - 3.0) < 1e-12
    np.testing.assert_allclose(k, 1.0 + 2.0 * (ln.max() - ln) / (ln.max() - ln.min()), rtol=0, atol=1e-12)
    assert np.all(o.kA_profile(2.5, 0.0) == 2.5)


@pytest.mark.parametrize("tau,k_A", [(0.01, 2.5), (0.5, 2.5), (1.0, 0.5), (0.5, 1.7)])
def test_weighted_first_flight_extinction_closed_form(tau, k_A):
    """Uniform sphere, no scattering, re-emission into a transparent bin: the absorbed ENERGY fraction is the closed
    form 1 - [1 - (1+2 tau) e^{-2 tau}]/(2 tau^2) whatever k_A; the number of absorptions follows the same formula
    at the biased depth k_A tau; every absorbed package carries W = e^{tau_A (k-1)} / k (Eq. 8)."""
    f = lambda t: 1 - (1 - (1 + 2 * t) * math.exp(-2 * t)) / (2 * t * t)
    n = 400000
    o = orc.Oracle(toy_problem(n_shells=5, tau=tau))
    o.run(n, seed=17, k_A=k_A)
    frac_n = o.counters["absorptions"] / n
    fb = f(k_A * tau)
    assert abs(frac_n - fb) < 4.5 * math.sqrt(fb * (1 - fb) / n)
    frac_e = o.absorbed.sum() / o.sums["injected"]
    # per-package weights lie in [1/k, e^{2 tau (k-1)}/k]: a generous bound of the standard error
    wmax = max(1 / k_A, math.exp(2 * tau * (k_A - 1)) / k_A)
    assert abs(frac_e - f(tau)) < 4.5 * wmax * math.sqrt(fb / n), (frac_e, f(tau))
    # exact bookkeeping: what the weights added or removed is accounted for
    s = o.sums
    assert abs(s["injected"] + s["reweight"] - s["escaped"] - s["terminated"]) < 1e-9 * s["injected"]


def test_weighted_scattering_clock_is_unbiased():
    """With scattering (albedo 0.5, g = 0.5) the absorbed energy per shell does not depend on k_S, k_A or k_A(rho)."""
    p = toy_problem(n_shells=6, tau=2.0, kappa_sca=1.0, g=0.5, rho_shape=[4, 3, 2, 1.5, 1, 0.5])
    n = 300000
    runs = []
    for kw in ({}, dict(k_S=2.0), dict(k_S=0.6, k_A=1.5), dict(k_A=1.0, k_A_dilute=3.0)):
        tot = []
        for seed in range(1, 5):
            o = orc.Oracle(p).run(n, seed=seed, **kw)
            tot.append(o.absorbed / o.sums["injected"])
            s = o.sums
            assert abs(s["injected"] + s["reweight"] - s["escaped"] - s["terminated"]) < 1e-9 * s["injected"]
        runs.append(np.array(tot))
    ref = runs[0]
    for r in runs[1:]:
        se = np.sqrt(ref.var(0, ddof=1) / 4 + r.var(0, ddof=1) / 4)
        assert np.all(np.abs(r.mean(0) - ref.mean(0)) < 5 * se + 1e-4), (r.mean(0) / ref.mean(0))


def test_weighted_temperatures_agree_and_thin_limit_noise_drops():
    """Thin sphere (tau_V = 0.01): every variant gives the analytic thin-limit temperature, and shorter absorption
    paths (k_A(rho) up to 3, L211-217) lower the noise of T at equal package count."""
    p = synth.config4(n_shells=8, n_freq=100)
    T0 = _thin_limit_T(p)
    n = 150000
    plain = np.array([orc.Oracle(p).run(n, seed=s).temperature() for s in range(1, 9)])
    fixed = np.array([orc.Oracle(p).run(n, seed=s, k_A=3.0).temperature() for s in range(1, 9)])
    assert np.max(np.abs(fixed.mean(0)[4:] / T0 - 1)) < 0.01
    # eps ~ T^5.5: compare the scatter of the outer shells
    assert fixed[:, 4:].std(0, ddof=1).mean() < 0.8 * plain[:, 4:].std(0, ddof=1).mean()


def test_weight_guard_terminates_trapped_packages():
    """L119: a package whose weight fell by ten orders of magnitude is terminated.  Albedo 0.9 at tau = 20 means
    tens of scatterings per package; with k_S = 10 each one divides the weight by 10 while the paths give back
    e^{0.9 tau'} (a factor 2.5 on average), so most packages cross the 1e-10 limit before they get out."""
    p = toy_problem(n_shells=4, tau=20.0, kappa_sca=9.0, g=0.0)
    o = orc.Oracle(p).run(5000, seed=2, k_S=10.0)
    c, s = o.counters, o.sums
    assert c["terminated"] > 100 and c["terminated"] + c["escaped"] == 5000
    assert abs(s["injected"] + s["reweight"] - s["escaped"] - s["terminated"]) < 1e-9 * s["injected"]
    assert s["terminated"] < 1e-8 * s["injected"]


def test_ffi_and_free_path_weighting_are_not_combined():
    with pytest.raises(RuntimeError):
        orc.Oracle(synth.config1()).run(100, seed=1, ffi=1, k_A=2.0)


# ------------------------------------------------------------------ directional weighting (Eq. 6-7; R19)
@pytest.mark.parametrize("g", [0.5, -0.4, 0.8])
def test_hg_density_and_reemission_weight(g):
    """Eq. 6 integrates to 1 over mu in [-1,1]; sampling mu' from HG(g_E) with the weight (1/2) / p(mu') reproduces
    the isotropic distribution: mean weight 1 and a flat weighted histogram of mu'."""
    lib = orc._lib
    mu = np.linspace(-1, 1, 20001)
    p = np.array([lib.dies_oracle_hg_pdf(g, x) for x in mu])
    assert abs(np.sum(0.5 * (p[1:] + p[:-1]) * np.diff(mu)) - 1.0) < 1e-4       # trapezoid rule
    rng = np.random.default_rng(1)
    u = rng.random(200000)
    mup = np.array([lib.dies_oracle_hg_cos(g, x) for x in u])
    w = 0.5 / np.array([lib.dies_oracle_hg_pdf(g, x) for x in mup])
    assert abs(w.mean() - 1.0) < 5 * w.std() / math.sqrt(u.size)
    h, _ = np.histogram(mup, bins=10, range=(-1, 1), weights=w)
    assert np.max(np.abs(h / h.mean() - 1)) < 0.05


def test_scattering_direction_weight_is_unbiased():
    """Absorbed energy per shell with the dust's own scattering function (g = 0.5) equals the one obtained when the
    scattering directions are drawn from HG(g_S) about the radial direction and reweighted by Eq. 7."""
    p = toy_problem(n_shells=6, tau=2.0, kappa_sca=1.0, g=0.5, rho_shape=[4, 3, 2, 1.5, 1, 0.5])
    n = 300000
    runs = []
    for kw in ({}, dict(g_S=0.3), dict(g_S=0.0), dict(g_S=-0.3)):
        tot = []
        for seed in range(1, 5):
            o = orc.Oracle(p).run(n, seed=seed, **kw)
            tot.append(o.absorbed / o.sums["injected"])
            s = o.sums
            assert abs(s["injected"] + s["reweight"] - s["escaped"] - s["terminated"]) < 1e-9 * s["injected"]
        runs.append(np.array(tot))
    ref = runs[0]
    for r in runs[1:]:
        se = np.sqrt(ref.var(0, ddof=1) / 4 + r.var(0, ddof=1) / 4)
        assert np.all(np.abs(r.mean(0) - ref.mean(0)) < 5 * se + 1e-4), (r.mean(0) / ref.mean(0))
    # g_S = 0 is a weighting (isotropic sampling), not the plain run (L207): different realisations
    assert not np.array_equal(runs[0][0], runs[2][0])


def test_reemission_direction_weight_leaves_temperatures_unchanged():
    """Full IRE on config 1 at tau_V = 3 (re-emitted packages are re-absorbed): T(r) with g_E = 0.5 and -0.5 equals
    the unweighted T(r) within the combined errors of 6 seeds."""
    p = synth.config1(tau_V=3.0)
    n = 60000
    T = {}
    for g in (0.0, 0.5, -0.5):
        T[g] = np.array([orc.Oracle(p).run(n, seed=s, g_E=g).temperature() for s in range(1, 7)])
    for g in (0.5, -0.5):
        se = np.sqrt(T[0.0].var(0, ddof=1) / 6 + T[g].var(0, ddof=1) / 6)
        d = np.abs(T[g].mean(0) - T[0.0].mean(0))
        assert np.sum(d > np.maximum(0.01 * T[0.0].mean(0), 3.5 * se)) <= 1, d / se
    a = orc.Oracle(p).run(5000, seed=1)
    b = orc.Oracle(p).run(5000, seed=1, g_E=0.0)
    assert np.array_equal(a.absorbed, b.absorbed)         # g_E = 0 is the plain method


# ------------------------------------------------------------------ re-emission position within the cell (L253; R20)
def test_reemission_from_a_random_position_of_the_cell():
    """One thick shell: packages are absorbed just below the surface and re-emitted in a transparent bin.  From the
    absorption site (the plain method) the mean way out of an isotropic package is R/2 (surface point: half the
    directions leave at once, the others cross a chord 2 R cos theta); from a position uniform in the volume it is
    3R/4.  The path-length tally sees the difference."""
    p = toy_problem(n_shells=1, tau=200.0)
    n = 200000
    res = {}
    for flag in (0, 1):
        o = orc.Oracle(p)
        o.reset(pathlen=True)
        o.run(n, seed=4, reemit_cell=flag)
        assert o.counters["absorptions"] > 0.999 * n
        res[flag] = o.pathlen.sum() / n                                   # mean path per package in units of R = 1
    assert abs(res[0] - 0.5) < 0.02, res
    assert abs(res[1] - 0.75) < 0.02, res


def test_reemission_position_leaves_temperatures_unchanged():
    """L253: "No visible differences were observed": T(r) of config 1 (32 shells) agrees within noise."""
    p = synth.config1(tau_V=3.0)
    n = 60000
    a = np.array([orc.Oracle(p).run(n, seed=s).temperature() for s in range(1, 7)])
    b = np.array([orc.Oracle(p).run(n, seed=s, reemit_cell=1).temperature() for s in range(1, 7)])
    se = np.sqrt(a.var(0, ddof=1) / 6 + b.var(0, ddof=1) / 6)
    d = np.abs(a.mean(0) - b.mean(0))
    assert np.sum(d > np.maximum(0.01 * a.mean(0), 3.5 * se)) <= 1, d / se
    assert not np.array_equal(a[0], b[0])
