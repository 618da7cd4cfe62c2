"""GPU parity of the traditional Monte Carlo iteration with continuous absorption (DIES_MODE_TMC; PAPER.md L29-37,
L251; R22) against the oracle's dies_oracle_tmc_run, through the C ABI: identical Philox streams, so the
energy the continuous absorption leaves in every shell agrees to 1e-4 (or a few package quanta), counters to the
fp32 / fp64 flip rate of R14, and the integer bookkeeping is exact."""
import numpy as np
import pytest

from paper_2408_13807_b200 import binding as dies
from paper_2408_13807_b200 import synth
from test_oracle_pins import toy_problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def orc():
    from oracle import dies_oracle as orc
    return orc


def _identity(c, raw):
    return c["injected_raw"] == int(np.sum(raw)) + c["escaped_raw"] + c["terminated_raw"]


def _compare(m, o, n, n_src_pkgs):
    raw, unit, energy = m.dies_get_absorbed()
    c = m.dies_get_counters()
    assert c["packages"] == n_src_pkgs == o.counters["packages"]
    assert _identity(c, raw), c
    e_pkg = o.sums["injected"] / n_src_pkgs
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * e_pkg)), \
        np.max(np.abs(energy / np.maximum(o.absorbed, 1e-300) - 1))
    for k in ("crossings", "scatterings", "escaped", "terminated"):
        assert abs(c[k] - o.counters[k]) <= 2e-4 * o.counters[k] + 3, (k, c[k], o.counters[k])
    esc = m.dies_get_escape_spectrum()
    assert abs(esc.sum() / o.sums["escaped"] - 1) < 1e-4
    return raw, unit


@pytest.mark.parametrize("name", ["toy_thin", "toy_thick_scattering", "config1", "config3s"])
def test_tmc_iterations_match_the_oracle(orc, name):
    """Two iterations: cold dust (sources only), then the dust emitting what the first iteration left in it.  The
    oracle's second iteration starts from the GPU's own tallies, so both sides see the same state of the dust."""
    if name == "toy_thin":
        p, n = toy_problem(n_shells=5, tau=0.5), 200_000
    elif name == "toy_thick_scattering":
        p, n = toy_problem(n_shells=5, tau=10.0, kappa_sca=3.0, g=0.4), 200_000
    elif name == "config1":
        p, n = synth.config1(tau_V=4.0), 300_000
    else:
        p, n = synth.config3(n_shells=40, n_freq=64, tau_V=30.0), 200_000
    m = dies.Model(p)
    o = orc.Oracle(p)
    _, _, mass = o.tables()
    m.dies_run(n, seed=3, mode=dies.DIES_MODE_TMC)
    o.tmc_run(n, seed=3)
    raw, unit = _compare(m, o, n, n)
    eps = np.where(mass > 0, raw * unit / np.where(mass > 0, mass, 1.0), 0.0)
    m.dies_run(n, seed=4, mode=dies.DIES_MODE_TMC)
    o.tmc_run(n, seed=4, eps_cur=eps)
    assert o.counters["packages"] == 2 * n
    _compare(m, o, n, 2 * n)
    m.close()


def test_tmc_converges_to_the_ire_solution(orc):
    """Config 1: the TMC iteration on the GPU converges to the oracle's converged TMC and to the IRE
    temperatures (north_star check (d) on the GPU); started from an IRE run it stays there."""
    p = synth.config1(tau_V=4.0)
    n = 2_000_000
    m = dies.Model(p)
    T_old = None
    for it in range(1, 12):
        m.dies_run(n, seed=20 + it, mode=dies.DIES_MODE_TMC)
        T = m.dies_get_temperature()
        if T_old is not None and np.max(np.abs(T / T_old - 1)[4:]) < 2e-3:
            break
        T_old = T
    assert 1 < it < 11
    o = orc.Oracle(p)
    To, ito, _ = o.tmc_solve(150_000, seed=5, tol=4e-3, skip=8)
    assert np.max(np.abs(T / To - 1)[8:]) < 0.01, T / To
    m.dies_run(4_000_000, seed=2)                                   # IRE
    Ti = m.dies_get_temperature()
    assert np.max(np.abs(T / Ti - 1)[8:]) < 0.01, T / Ti
    m.dies_run(n, seed=77, mode=dies.DIES_MODE_TMC)                 # one TMC iteration from the IRE state
    Tf = m.dies_get_temperature()
    assert np.max(np.abs(Tf / Ti - 1)[8:]) < 0.01
    m.close()


def test_tmc_batch_and_errors(orc):
    b = synth.config5(n_models=3, n_packages=100_000, n_shells=16, n_freq=32, n_T=200)
    m = dies.Model(batch=b)
    m.dies_run(b.n_packages, seed=9, mode=dies.DIES_MODE_TMC)
    raw, unit, energy = m.dies_get_absorbed()
    for i in (0, 2):
        o = orc.Oracle(b.model(i))
        o.tmc_run(b.n_packages, seed=9, model_index=i)
        assert np.all(np.abs(energy[i] - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * o.sums["injected"] / b.n_packages))
    for kw in (dict(ffi=1), dict(k_bg=0.2), dict(k_A=2.0), dict(accumulate=1)):
        with pytest.raises(dies.DiesError) as e:
            m.dies_run(1000, mode=dies.DIES_MODE_TMC, **kw)
        assert e.value.code == dies.DIES_EINVAL
    # a rejected TMC call leaves the handle as it was: the pending dies_seek still applies to the next run
    m.dies_set_fixed_temperature(np.full(m.N, 15.0))
    m.dies_seek(5000)
    with pytest.raises(dies.DiesError) as e:
        m.dies_run(1000, mode=dies.DIES_MODE_TMC, fixed_shift=26)
    assert e.value.code == dies.DIES_EINVAL
    m.dies_run(1000, seed=9, mode=dies.DIES_MODE_FIXED_T, n_total=10_000)
    ev_run = m.dies_get_absorbed()[0].copy()
    m.dies_seek(5000)
    m.dies_run(1000, seed=9, mode=dies.DIES_MODE_FIXED_T, n_total=10_000)
    assert np.array_equal(ev_run, m.dies_get_absorbed()[0])
    m.dies_run(1000, seed=9, mode=dies.DIES_MODE_FIXED_T, n_total=10_000)          # ids from 0: other packages
    assert not np.array_equal(ev_run, m.dies_get_absorbed()[0])
    # the tallies of a TMC run are in the TMC energy unit: no other mode continues them, no IRE trace replays on them
    m.dies_run(10_000, seed=9, mode=dies.DIES_MODE_TMC)
    for mode in (dies.DIES_MODE_IRE, dies.DIES_MODE_FIXED_T):
        with pytest.raises(dies.DiesError) as e:
            m.dies_run(1000, seed=9, mode=mode, accumulate=1, n_total=10_000)
        assert e.value.code == dies.DIES_ESTATE
    with pytest.raises(dies.DiesError) as e:
        m.dies_trace_packages(0, 4, 10_000, mode=dies.DIES_MODE_IRE)
    assert e.value.code == dies.DIES_ESTATE
    for trace in (m.dies_trace_packages, m.dies_trace_packages_static):
        with pytest.raises(dies.DiesError) as e:
            trace(0, 4, 10_000, mode=dies.DIES_MODE_TMC)
        assert e.value.code == dies.DIES_EINVAL
    m.dies_run(1000, seed=9, mode=dies.DIES_MODE_IRE)                              # a fresh run in another mode is fine
    m.close()


@pytest.mark.parametrize("tau,bar", [(1e-6, 3e-3), (1e-8, 2e-2)])
def test_tmc_thin_sphere_deposits_are_unbiased(orc, tau, bar):
    """A nearly transparent sphere: a package leaves far less than one fixed-point unit per step (about 5 units at
    tau = 1e-6, 0.05 at 1e-8, of a quantum of 2^24).  The pieces are cut with a carried remainder that starts at a
    random offset per package, so their sum over many packages is the continuous absorption of the oracle up to the
    noise of that cut (bars: some five standard deviations of it); rounding every step to the nearest integer would
    tally exactly nothing at 1e-8."""
    p, n = toy_problem(n_shells=5, tau=tau), 1_000_000
    m = dies.Model(p)
    o = orc.Oracle(p)
    m.dies_run(n, seed=6, mode=dies.DIES_MODE_TMC)
    o.tmc_run(n, seed=6)
    raw, unit, energy = m.dies_get_absorbed()
    c = m.dies_get_counters()
    assert _identity(c, raw), c
    assert np.all(raw > 0)
    assert np.max(np.abs(energy / o.absorbed - 1)) < bar, energy / o.absorbed
    assert abs(energy.sum() / o.absorbed.sum() - 1) < bar / 2
    assert c["crossings"] == o.counters["crossings"] and c["terminated"] == 0
    m.close()


def test_tmc_weak_second_source(orc):
    """Two sources with a luminosity ratio of 1e4: the external field shines in the transparent bin (never absorbed),
    the point source, 1e-4 of it, in the absorbing bin of a thin sphere (tau = 1e-3).  Its packages carry 1e-4 of the
    reference quantum (about 1678 units) and leave a third of a unit per step: every tally comes from pieces below one
    unit of the weak source."""
    p = toy_problem(n_shells=5, tau=1e-3)
    L_ext = 4.0 * np.pi ** 2                       # 4 pi R^2 * pi * sum_k J_k with R = 1, J = (1, 0)
    p.ext_bin_intensity = np.array([1.0, 0.0])
    p.L_point, p.point_bin_weights = 1e-4 * L_ext, np.array([0.0, 1.0])
    n = 1_000_000
    m = dies.Model(p)
    o = orc.Oracle(p)
    m.dies_run(n, seed=8, mode=dies.DIES_MODE_TMC)
    o.tmc_run(n, seed=8)
    raw, unit, energy = m.dies_get_absorbed()
    c = m.dies_get_counters()
    assert c["packages"] == 2 * n == o.counters["packages"]
    assert _identity(c, raw), c
    assert np.all(raw > 0)
    assert np.max(np.abs(energy / o.absorbed - 1)) < 1e-2, energy / o.absorbed
    assert abs(energy.sum() / o.absorbed.sum() - 1) < 4e-3
    esc = m.dies_get_escape_spectrum()
    np.testing.assert_allclose(esc, o.escaped, rtol=1e-4)
    m.close()


def test_tmc_weight_guard_fires(orc):
    """PAPER.md L119 in the TMC: in a very thick, purely absorbing sphere nearly every package falls below 1e-10 of
    its launch weight before it gets out; both sides must end those packages (terminated > 0), at the same count up to
    fp32 / fp64 flips of the comparison, and the energy bookkeeping stays exact."""
    p, n = toy_problem(n_shells=5, tau=400.0), 100_000
    m = dies.Model(p)
    o = orc.Oracle(p)
    m.dies_run(n, seed=3, mode=dies.DIES_MODE_TMC)
    o.tmc_run(n, seed=3)
    raw, unit, energy = m.dies_get_absorbed()
    c = m.dies_get_counters()
    assert o.counters["terminated"] > 0.5 * n and c["terminated"] > 0.5 * n
    assert abs(c["terminated"] - o.counters["terminated"]) <= 2e-4 * n + 3
    assert c["terminated"] + c["escaped"] == n
    assert _identity(c, raw), c
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * o.sums["injected"] / n))
    m.close()
