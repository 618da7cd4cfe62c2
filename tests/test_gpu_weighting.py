"""GPU parity of the free-path weighting k_A, k_S, k_A(rho) (section 2.2.2, Eq. 8; R17, R18) against
the oracle, through the C ABI: bit-exact event lists on identical Philox streams, absorbed energy per shell in
fixed-temperature mode, IRE temperatures over 8 seeds, exact integer bookkeeping, the weight guard (L119)."""
import numpy as np
import pytest

from paper_2408_13807_b200 import binding as dies
from paper_2408_13807_b200 import synth
from test_gpu_parity import _check_T_parity, _fixed_T
from test_oracle_pins import toy_problem

pytestmark = pytest.mark.gpu

VARIANTS = [dict(k_A=2.5), dict(k_S=0.6, k_A=1.5), dict(k_A=1.0, k_A_dilute=3.0), dict(k_A=1.2, k_A_dilute=2.0, k_S=1.8, k_bg=0.3)]


@pytest.fixture(scope="module")
def orc():
    from oracle import dies_oracle as orc
    return orc


def _identity(c):
    return c["injected_raw"] + c["reweight_raw"] == c["escaped_raw"] + c["terminated_raw"]


@pytest.mark.parametrize("kw", VARIANTS)
@pytest.mark.parametrize("cfg", ["config1", "config2s", "config3s"])
def test_weighted_trace_bit_exact(orc, cfg, kw):
    if cfg == "config1":
        p = synth.config1()
    elif cfg == "config3s":
        p = synth.config3(n_shells=40, n_freq=64, tau_V=30.0)
    else:
        p = synth.config2(n_shells=50, n_freq=64)
    n_total, count, max_ev = 100000, 2000, 512
    o = orc.Oracle(p)
    o.set_fixed_temperature(_fixed_T(p.n_shells))
    m = dies.Model(p)
    m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    ev, nev = m.dies_trace_packages(0, count, n_total, seed=5, max_events=max_ev, mode=dies.DIES_MODE_FIXED_T, **kw)
    safe = same = 0
    for pid in range(count):
        ref, nref, margin = o.trace(n_total, pid, seed=5, mode=1, max_events=max_ev, **kw)
        ok = (nref == nev[pid]) and nref <= max_ev and np.array_equal(ref, ev[pid, :nref])
        same += ok
        if margin > 1e-3 and nref <= max_ev:
            safe += 1
            assert ok, (pid, margin, ref[:8], ev[pid, :8])
    assert safe > 0.4 * count
    assert same >= 0.99 * count, same / count
    m.close()


@pytest.mark.parametrize("kw", VARIANTS)
def test_weighted_fixed_T_absorbed_energy(orc, kw):
    """Identical streams, fixed temperatures: absorbed energy per shell within 1e-4 (or a few package quanta)."""
    p = synth.config2(n_shells=40, n_freq=64, tau_V=3.0)        # centrally peaked density: k_A(rho) varies by shell
    n = 400_000
    o = orc.Oracle(p)
    o.set_fixed_temperature(_fixed_T(p.n_shells))
    o.run(n, seed=3, mode=1, **kw)
    m = dies.Model(p)
    m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    m.dies_run(n, seed=3, mode=dies.DIES_MODE_FIXED_T, **kw)
    raw, unit, energy = m.dies_get_absorbed()
    c = m.dies_get_counters()
    e_pkg = o.sums["injected"] / n
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 5 * e_pkg)), \
        np.max(np.abs(energy / o.absorbed - 1))
    assert c["packages"] == n and c["terminated"] == 0 == o.counters["terminated"]
    for k in ("crossings", "scatterings", "absorptions"):
        assert abs(c[k] - o.counters[k]) <= 2e-4 * o.counters[k] + 3
    assert _identity(c)
    # the same identity in energy against the oracle's own sums
    esc = m.dies_get_escape_spectrum().sum()
    assert abs(esc / o.sums["escaped"] - 1) < 1e-4
    assert abs(c["reweight_raw"] * unit - o.sums["reweight"]) < 2e-3 * abs(o.sums["reweight"]) + 1e-5 * o.sums["injected"]
    m.close()


@pytest.mark.parametrize("kw", [dict(k_A=1.0, k_A_dilute=3.0), dict(k_S=2.0, k_A=0.7)])
def test_weighted_full_ire_temperature(orc, kw):
    p = synth.config2(n_shells=40, n_freq=64, tau_V=3.0)
    _check_T_parity(orc, p, 100_000, **kw)


def test_weighted_thin_sphere_matches_the_plain_method(orc):
    """Config 4 reduced (tau_V = 0.01): k_A(rho) up to 3 against the oracle WITHOUT weighting: same T within noise."""
    p = synth.config4(n_shells=20)
    n = 2_000_000
    m = dies.Model(p)
    T = []
    for s in range(1, 5):
        m.dies_run(n, seed=s, k_A=3.0)
        T.append(m.dies_get_temperature())
        assert _identity(m.dies_get_counters())
    T = np.array(T)
    To = np.array([orc.Oracle(p).run(400_000, seed=s, ffi=1).temperature() for s in range(1, 5)])
    se = np.sqrt(T.var(0, ddof=1) / 4 + To.var(0, ddof=1) / 4)
    assert np.all(np.abs(T.mean(0) - To.mean(0))[4:] < np.maximum(0.01 * To.mean(0), 4 * se)[4:])
    m.close()


def test_weight_guard_and_bookkeeping(orc):
    """The live weight guard: a package is terminated when its weight has fallen below 1e-10 of its
    launch weight, on the GPU exactly as in the oracle (the kernel carries the relative weight in fp32 beside the
    fixed-point quantum, R18).  Thick scattering toy sphere with k_S = 10: most packages end by the guard."""
    p = toy_problem(n_shells=4, tau=20.0, kappa_sca=9.0, g=0.0)
    n = 20000
    m = dies.Model(p)
    m.dies_run(n, seed=2, k_S=10.0)
    c = m.dies_get_counters()
    o = orc.Oracle(p).run(n, seed=2, k_S=10.0)
    assert c["packages"] == n == c["escaped"] + c["terminated"]
    assert o.counters["terminated"] > 0.2 * n
    # identical streams: the same packages are terminated, up to the fp32/fp64 flips of R14
    assert abs(c["terminated"] - o.counters["terminated"]) <= max(3, 1e-3 * o.counters["terminated"]), \
        (c["terminated"], o.counters["terminated"])
    for k in ("scatterings", "absorptions", "crossings"):
        assert abs(c[k] - o.counters[k]) <= 2e-3 * o.counters[k] + 3, (k, c[k], o.counters[k])
    assert _identity(c)
    assert c["terminated_raw"] < 1e-6 * c["injected_raw"]
    m.close()


def test_weight_guard_trace_bit_exact(orc):
    """Event lists that END WITH DIES_EV_TERMINATE, bit-exact against the oracle on identical Philox streams."""
    p = toy_problem(n_shells=4, tau=20.0, kappa_sca=9.0, g=0.0)
    n_total, count, max_ev = 20000, 1500, 4096
    Tfix = np.full(p.n_shells, 15.0)
    o = orc.Oracle(p)
    o.set_fixed_temperature(Tfix)
    m = dies.Model(p)
    m.dies_set_fixed_temperature(Tfix)
    ev, nev = m.dies_trace_packages(0, count, n_total, seed=2, max_events=max_ev, mode=dies.DIES_MODE_FIXED_T, k_S=10.0)
    safe = same = n_term = n_term_same = 0
    for pid in range(count):
        ref, nref, margin = o.trace(n_total, pid, seed=2, mode=1, max_events=max_ev, k_S=10.0)
        ok = (nref == nev[pid]) and nref <= max_ev and np.array_equal(ref, ev[pid, :nref])
        same += ok
        term = nref <= max_ev and ref[nref - 1][0] == 4          # DIES_EV_TERMINATE
        n_term += term
        n_term_same += term and ok
        if margin > 1e-3 and nref <= max_ev:
            safe += 1
            assert ok, (pid, margin, ref[:6], ev[pid, :6], nref, nev[pid])
    assert n_term > 0.2 * count, n_term                       # the guard is exercised
    assert n_term_same >= 0.98 * n_term, (n_term_same, n_term)
    assert same >= 0.98 * count, same / count
    m.close()


def test_weighting_argument_errors():
    m = dies.Model(synth.config1())
    with pytest.raises(dies.DiesError) as e:
        m.dies_run(100, ffi=1, k_A=2.0)
    assert e.value.code == dies.DIES_EINVAL
    with pytest.raises(dies.DiesError) as e:
        m.dies_run(100, k_S=-1.0)
    assert e.value.code == dies.DIES_EINVAL
    m.dies_run(1000, k_A=1.0, k_S=1.0)            # unit factors: the plain kernel
    c = m.dies_get_counters()
    assert c["reweight_raw"] == 0 and c["injected_raw"] == c["escaped_raw"]
    m.close()


# ------------------------------------------------------------------ directional weighting (Eq. 6-7; R19)
DIR_VARIANTS = [dict(g_E=0.5), dict(g_E=-0.4), dict(g_S=0.3), dict(g_S=0.0), dict(g_S=-0.3, g_E=0.3, k_A=1.5)]


@pytest.mark.parametrize("kw", DIR_VARIANTS)
@pytest.mark.parametrize("cfg", ["config1", "config3s"])
def test_directional_trace_bit_exact(orc, cfg, kw):
    p = synth.config1(tau_V=3.0) if cfg == "config1" else synth.config3(n_shells=40, n_freq=64, tau_V=30.0)
    n_total, count, max_ev = 100000, 2000, 512
    o = orc.Oracle(p)
    o.set_fixed_temperature(_fixed_T(p.n_shells))
    m = dies.Model(p)
    m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    ev, nev = m.dies_trace_packages(0, count, n_total, seed=7, max_events=max_ev, mode=dies.DIES_MODE_FIXED_T, **kw)
    safe = same = 0
    for pid in range(count):
        ref, nref, margin = o.trace(n_total, pid, seed=7, mode=1, max_events=max_ev, **kw)
        ok = (nref == nev[pid]) and nref <= max_ev and np.array_equal(ref, ev[pid, :nref])
        same += ok
        if margin > 1e-3 and nref <= max_ev:
            safe += 1
            assert ok, (pid, margin, ref[:8], ev[pid, :8])
    assert safe > 0.4 * count
    assert same >= 0.99 * count, same / count
    m.close()


@pytest.mark.parametrize("kw", DIR_VARIANTS)
def test_directional_fixed_T_absorbed_energy(orc, kw):
    p = synth.config2(n_shells=40, n_freq=64, tau_V=3.0)
    n = 400_000
    o = orc.Oracle(p)
    o.set_fixed_temperature(_fixed_T(p.n_shells))
    o.run(n, seed=3, mode=1, **kw)
    m = dies.Model(p)
    m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    m.dies_run(n, seed=3, mode=dies.DIES_MODE_FIXED_T, **kw)
    raw, unit, energy = m.dies_get_absorbed()
    c = m.dies_get_counters()
    e_pkg = o.sums["injected"] / n
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(2e-4 * o.absorbed, 8 * e_pkg)), \
        np.max(np.abs(energy / o.absorbed - 1))
    assert c["packages"] == n and c["terminated"] == 0 == o.counters["terminated"]
    for k in ("crossings", "scatterings", "absorptions"):
        assert abs(c[k] - o.counters[k]) <= 2e-4 * o.counters[k] + 3
    assert _identity(c)
    assert abs(c["reweight_raw"] * unit - o.sums["reweight"]) < 2e-3 * abs(o.sums["reweight"]) + 1e-5 * o.sums["injected"]
    m.close()


@pytest.mark.parametrize("kw", [dict(g_E=0.5), dict(g_S=0.2)])
def test_directional_full_ire_temperature(orc, kw):
    p = synth.config2(n_shells=40, n_freq=64, tau_V=3.0)
    _check_T_parity(orc, p, 100_000, **kw)


def test_directional_argument_errors():
    m = dies.Model(synth.config1())
    for kw in (dict(g_E=1.0), dict(g_S=-1.5), dict(g_E=0.3, ffi=1)):
        with pytest.raises(dies.DiesError) as e:
            m.dies_run(100, **kw)
        assert e.value.code == dies.DIES_EINVAL
    m.close()


# ------------------------------------------------------------------ re-emission position within the cell (L253; R20)
def test_reemission_in_cell_trace_and_energy(orc):
    p = synth.config2(n_shells=40, n_freq=64, tau_V=3.0)
    Tf = _fixed_T(p.n_shells)
    o = orc.Oracle(p)
    o.set_fixed_temperature(Tf)
    m = dies.Model(p)
    m.dies_set_fixed_temperature(Tf)
    n_total, count = 100000, 2000
    ev, nev = m.dies_trace_packages(0, count, n_total, seed=9, max_events=512, mode=dies.DIES_MODE_FIXED_T, reemit_cell=1)
    safe = 0
    for pid in range(count):
        ref, nref, margin = o.trace(n_total, pid, seed=9, mode=1, max_events=512, reemit_cell=1)
        ok = (nref == nev[pid]) and nref <= 512 and np.array_equal(ref, ev[pid, :nref])
        if margin > 1e-3 and nref <= 512:
            safe += 1
            assert ok, (pid, margin, ref[:8], ev[pid, :8])
    assert safe > 0.4 * count
    n = 400_000
    o.run(n, seed=3, mode=1, reemit_cell=1)
    m.dies_run(n, seed=3, mode=dies.DIES_MODE_FIXED_T, reemit_cell=1)
    raw, unit, energy = m.dies_get_absorbed()
    e_pkg = o.sums["injected"] / n
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 5 * e_pkg))
    c = m.dies_get_counters()
    assert c["injected_raw"] == c["escaped_raw"] and c["reweight_raw"] == 0
    m.close()


def test_reemission_in_cell_full_ire_temperature(orc):
    _check_T_parity(orc, synth.config2(n_shells=40, n_freq=64, tau_V=3.0), 100_000, reemit_cell=1)
