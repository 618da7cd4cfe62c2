"""Accuracy behaviour the paper reports (section 3.1-3.2), checked on the GPU path with the synthetic configs:
noise ~ N^-1/2, no drift of the temperatures at 1e8 packages (the paper's fp32 counters under-estimate T there, L155,
L179-181; the 64-bit fixed-point tallies must not), k_bg = 0.2 lowers the noise in the centre (L197), forced first
interaction lowers it in an optically thin model (L217)."""
import numpy as np
import pytest

from paper_2408_13807_b200 import binding as dies
from paper_2408_13807_b200 import synth

pytestmark = pytest.mark.gpu


def _T_runs(m, n, seeds, **kw):
    out = []
    for s in seeds:
        m.dies_run(n, seed=s, **kw)
        out.append(m.dies_get_temperature())
    return np.array(out)


def test_noise_scales_as_inverse_square_root_of_packages():
    """Config 2: sigma_T of the outer half over 16 seeds at 1e5 and 1.6e6 packages differs by 4 (within 25 %)."""
    m = dies.Model(synth.config2())
    s_lo = _T_runs(m, 100_000, range(1, 17)).std(0, ddof=1)[50:].mean()
    s_hi = _T_runs(m, 1_600_000, range(1, 17)).std(0, ddof=1)[50:].mean()
    assert 3.0 < s_lo / s_hi < 5.0, s_lo / s_hi
    m.close()


def test_no_temperature_drift_at_1e8_packages():
    """Config 4 without FFI, 1e8 packages: T equals the mean of 8 runs of 1e6 packages within their scatter, with no
    systematic low bias (L179-181: fp32 counters lose updates once N >~ 1e8; integer tallies cannot)."""
    p = synth.config4(ffi=0)
    m = dies.Model(p)
    small = _T_runs(m, 1_000_000, range(1, 9))
    m.dies_run(100_000_000, seed=99)
    big = m.dies_get_temperature()
    c = m.dies_get_counters()
    assert c["injected_raw"] == c["escaped_raw"] == 100_000_000 * (1 << 24)
    mean, se = small.mean(0), small.std(0, ddof=1) / np.sqrt(8)
    outer = slice(p.n_shells // 2, None)
    z = (big - mean)[outer] / se[outer]
    assert np.abs(np.median(z)) < 1.0, np.median(z)                 # no systematic offset
    assert np.max(np.abs(z)) < 5.0, np.max(np.abs(z))               # every shell within the scatter of the small runs
    m.close()


def test_kbg_lowers_the_noise_in_the_centre():
    """L197: k_bg = 0.2 lowers the central noise by almost a factor of two at equal package count."""
    m = dies.Model(synth.config2())
    plain = _T_runs(m, 200_000, range(1, 25)).std(0, ddof=1)
    kbg = _T_runs(m, 200_000, range(1, 25), k_bg=0.2).std(0, ddof=1)
    inner = slice(2, 12)
    assert plain[inner].mean() / kbg[inner].mean() > 1.3, plain[inner].mean() / kbg[inner].mean()
    m.close()


def test_ffi_lowers_the_noise_of_a_thin_model():
    """L217: forced first interaction reduces the noise of the most diffuse models by up to an order of magnitude."""
    p = synth.config4(n_shells=50)
    m = dies.Model(p)
    plain = _T_runs(m, 1_000_000, range(1, 13)).std(0, ddof=1)
    ffi = _T_runs(m, 1_000_000, range(1, 13), ffi=1).std(0, ddof=1)
    outer = slice(25, None)
    assert plain[outer].mean() / ffi[outer].mean() > 3.0, plain[outer].mean() / ffi[outer].mean()
    m.close()
