"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (persistent grid, pools, one
launch per run): sampled packages the oracle can follow one by one (bit-exact event lists), and properties that hold
at any size (package counts, exact integer conservation, escaping = injected luminosity, temperatures against the
oracle's reduced-size profile within its own noise).  All through the C ABI."""
import numpy as np
import pytest

from paper_2408_13807_b200 import binding as dies
from paper_2408_13807_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def orc():
    from oracle import dies_oracle as orc
    return orc


def _problem(name):
    if name == "config2":
        return synth.config2(), {}
    if name == "config2_kbg":
        return synth.config2(k_bg=0.2), dict(k_bg=0.2)
    if name == "config3":
        return synth.config3(), {}
    if name == "config3_thick":
        return synth.config3(tau_V=1000.0), {}
    if name == "config4":
        return synth.config4(), dict(ffi=1)
    if name == "config4_kA":                          # free-path weighting, the comparator of FFI in Fig. 7 (Eq. 8)
        return synth.config4(ffi=0), dict(k_A=3.0, k_S=2.0)
    if name == "config3_dir":                         # directional weighting (Eq. 6-7) with sub-cell re-emission (L253)
        return synth.config3(), dict(g_E=0.5, g_S=0.2, reemit_cell=1)
    raise KeyError(name)


def _L_injected(p):
    L = 0.0
    if p.ext_bin_intensity is not None:
        L += 4 * np.pi * p.r_bounds[-1] ** 2 * np.pi * float(np.sum(p.ext_bin_intensity))
    return L + float(p.L_point)


@pytest.mark.parametrize("name", ["config2", "config2_kbg", "config3", "config4", "config4_kA", "config3_dir"])
def test_sampled_packages_at_full_size(orc, name):
    """64 packages at each of 12 places of the full id range [0, n_packages): identical event lists (type, shell,
    bin, crossings so far) for every package whose decisions sit > 1e-3 from their thresholds in the oracle."""
    p, kw = _problem(name)
    n_total, max_ev = p.n_packages, 1024
    Tfix = np.linspace(10.0, 40.0, p.n_shells)
    o = orc.Oracle(p)
    o.set_fixed_temperature(Tfix)
    m = dies.Model(p)
    m.dies_set_fixed_temperature(Tfix)
    safe = same = total = 0
    for first in np.linspace(0, n_total - 64, 12).astype(np.int64):
        ev, nev = m.dies_trace_packages(int(first), 64, n_total, seed=11, max_events=max_ev,
                                        mode=dies.DIES_MODE_FIXED_T, **kw)
        for x in range(64):
            ref, nref, margin = o.trace(n_total, int(first) + x, seed=11, mode=1, max_events=max_ev, **kw)
            ok = (nref == nev[x]) and nref <= max_ev and np.array_equal(ref, ev[x, :nref])
            total += 1
            same += ok
            if margin > 1e-3 and nref <= max_ev:
                safe += 1
                assert ok, (name, int(first) + x, margin, ref[:6], ev[x, :6])
    assert safe > 0.4 * total
    assert same >= 0.99 * total, same / total
    m.close()


@pytest.mark.parametrize("name,n_orc", [("config2", 200_000), ("config3", 60_000), ("config3_thick", 10_000),
                                        ("config4", 300_000)])
def test_full_size_run_properties(orc, name, n_orc):
    p, kw = _problem(name)
    n = p.n_packages
    m = dies.Model(p)
    m.dies_run(n, seed=21, **kw)
    c = m.dies_get_counters()
    T = m.dies_get_temperature()
    Lesc = m.dies_get_escape_spectrum()
    raw, unit, energy = m.dies_get_absorbed()
    # counts and exact conservation in integers (R13)
    assert c["packages"] == n and c["terminated"] == 0
    assert c["escaped"] + c["uninteracted"] == n
    assert c["injected_raw"] == c["escaped_raw"] + c["terminated_raw"]
    assert c["T_clamp_hi"] == 0
    # escaping luminosity = injected luminosity (north_star (b)); the fixed-point quantum is 2^-24 of a package
    assert abs(Lesc.sum() / _L_injected(p) - 1.0) < 1e-6
    if not kw:
        assert c["injected_raw"] == n * (1 << 24)
    # every absorption raised one tally by one package quantum
    if not kw:
        assert int(raw.sum()) == c["absorptions"] * (1 << 24)
    # temperatures against the oracle at reduced size: within 2 % or 4 standard errors of the oracle's 4-seed mean
    To = []
    for s in range(1, 5):
        o = orc.Oracle(p)
        o.run(n_orc, seed=s, **kw)
        To.append(o.temperature())
    To = np.array(To)
    mo, se = To.mean(0), To.std(0, ddof=1) / 2.0
    tol = np.maximum(0.02 * mo, 4 * se)
    well = To.min(0) > p.T_grid[0] * 1.001            # shells every oracle seed reached
    bad = well & (np.abs(T - mo) > tol)
    assert well.sum() > 0.5 * p.n_shells
    assert bad.sum() <= max(1, int(0.03 * p.n_shells)), (np.nonzero(bad)[0], (T / mo)[bad])
    m.close()


def _gpu_temperatures(p, n, seeds, **kw):
    m = dies.Model(p)
    T = []
    for s in seeds:
        m.dies_run(n, seed=s, **kw)
        T.append(m.dies_get_temperature())
        c = m.dies_get_counters()
        assert c["packages"] == n and c["injected_raw"] == c["escaped_raw"] and c["terminated"] == 0
    m.close()
    return np.array(T)


@pytest.mark.parametrize("name,n,kw", [("config2", 10_000_000, {}), ("config3", 10_000_000, {}),
                                       ("config4", 10_000_000, dict(ffi=1))])
def test_full_ire_temperature_at_bench_size(name, n, kw):
    """north_star's bar at the stated sizes: per-shell T(r) within 1 % or 3 combined standard errors over 8 seeds, GPU
    against the serial oracle, both following the FULL package count of config 2 (1e7, the configuration bench.py
    times) and of config 3 (1e7), and 1e7 packages of config 4 with forced first interaction (its stated 1e8 would be
    300 s per oracle seed: DESIGN.md R21).  Shells flagged on seeds 1..8 must pass on the independent seeds 9..16."""
    from oracle_workers import oracle_temperatures
    from test_gpu_parity import _two_looks
    p = getattr(synth, name)()

    def stats(seeds):
        return oracle_temperatures(name, n, seeds, **kw)[0], _gpu_temperatures(p, n, seeds, **kw)

    To, Tg = _two_looks(f"{name} n={n:g} (full size)", stats)
    # the means over all shells agree far better than any single shell
    assert abs(Tg.mean() / To.mean() - 1.0) < 2e-3


def test_full_ire_temperature_of_the_full_size_batch():
    """Config 5 at its stated size: the GPU follows the whole batch, 1024 spheres x 1e6 packages, once per seed; the
    oracle follows 16 spheres spread over the batch (0, 511 and 1023 among them) at the full 1e6 packages, each with
    its model index in the Philox counter.  Those spheres are compared at north_star's bar, 1 % or 3 combined standard
    errors over 8 seeds."""
    from oracle_workers import oracle_temperatures
    from test_gpu_parity import _two_looks
    b = synth.config5()
    picks = [0, 68, 136, 204, 272, 341, 409, 477, 511, 613, 682, 750, 818, 886, 954, 1023]
    m = dies.Model(batch=b)

    def stats(seeds):
        To, _ = oracle_temperatures([f"config5:{i}" for i in picks], b.n_packages, seeds)
        Tg = []
        for s in seeds:
            m.dies_run(b.n_packages, seed=s)
            Tg.append(m.dies_get_temperature()[picks].reshape(-1))
            c = m.dies_get_counters()
            assert c["packages"] == b.n_models * b.n_packages and c["injected_raw"] == c["escaped_raw"]
        return To, np.array(Tg)

    _two_looks("config5 full size (16 of 1024 spheres x 1e6)", stats)
    m.close()


def test_full_size_batch_properties(orc):
    """Config 5 as bench.py launches it: 1024 spheres x 1e6 packages in one launch."""
    b = synth.config5()
    m = dies.Model(batch=b)
    m.dies_run(b.n_packages, seed=31)
    c = m.dies_get_counters()
    assert c["packages"] == b.n_models * b.n_packages == c["escaped"]
    assert c["injected_raw"] == c["escaped_raw"] == b.n_models * b.n_packages * (1 << 24)
    Lesc = m.dies_get_escape_spectrum()
    T = m.dies_get_temperature()
    R = b.r_bounds[:, -1]
    L_in = 4 * np.pi * R ** 2 * np.pi * b.ext_bin_intensity.sum(1)
    assert np.max(np.abs(Lesc.sum(1) / L_in - 1.0)) < 1e-6
    raw, unit, energy = m.dies_get_absorbed()
    assert int(raw.sum()) == c["absorptions"] * (1 << 24)
    # three models against the oracle at reduced size (model index is part of the Philox counter)
    for i in (0, 511, 1023):
        o = orc.Oracle(b.model(i))
        o.run(100_000, seed=3, model_index=i)
        To = o.temperature()
        assert np.max(np.abs(T[i][24:] / To[24:] - 1)) < 0.04, i
    m.close()


def test_sampled_packages_of_the_full_size_batch(orc):
    """Config 5 (1024 spheres x 1e6 packages): 48 packages at 4 places of the id range of models 0, 511 and 1023,
    followed one by one by the oracle of that sphere (the model index is the fourth word of the Philox counter)."""
    b = synth.config5()
    m = dies.Model(batch=b)
    n_total, max_ev = b.n_packages, 1024
    Tfix = np.tile(np.linspace(10.0, 40.0, b.rho.shape[1]), (b.n_models, 1))
    m.dies_set_fixed_temperature(Tfix)
    safe = same = total = 0
    for i in (0, 511, 1023):
        o = orc.Oracle(b.model(i))
        o.set_fixed_temperature(Tfix[i])
        for first in np.linspace(0, n_total - 48, 4).astype(np.int64):
            ev, nev = m.dies_trace_packages(int(first), 48, n_total, seed=13, model_index=i, max_events=max_ev,
                                            mode=dies.DIES_MODE_FIXED_T)
            for x in range(48):
                ref, nref, margin = o.trace(n_total, int(first) + x, seed=13, mode=1, model_index=i, max_events=max_ev)
                ok = (nref == nev[x]) and nref <= max_ev and np.array_equal(ref, ev[x, :nref])
                total += 1
                same += ok
                if margin > 1e-3 and nref <= max_ev:
                    safe += 1
                    assert ok, (i, int(first) + x, margin, ref[:6], ev[x, :6])
    assert safe > 0.4 * total
    assert same >= 0.99 * total, same / total
    m.close()


def test_one_billion_packages_counters_do_not_wrap():
    """1e9 packages of config 4 without FFI in one launch: 6.7e10 crossings (beyond 2^32) are counted in 64 bits, the
    raw tallies (1.7e16 units injected) stay exact."""
    p = synth.config4(ffi=0)
    n = 1_000_000_000
    m = dies.Model(p)
    m.dies_run(n, seed=41)
    c = m.dies_get_counters()
    assert c["packages"] == n == c["escaped"]
    assert c["injected_raw"] == c["escaped_raw"] == n * (1 << 24)
    assert abs(c["crossings"] / n - 66.676) < 0.05            # straight chords through 100 equal shells: 66.67 + events
    raw, unit, energy = m.dies_get_absorbed()
    assert int(raw.sum()) == c["absorptions"] * (1 << 24)
    m.close()
