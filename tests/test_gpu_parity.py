"""GPU parity: the CUDA path (through the C ABI of include/dies.h) against the CPU oracle on the same seeded
synthetic inputs.  Bars (BASELINE.json north_star):
  * bit-exact Philox words / uniforms, package counts and event lists of the deterministic trace test;
  * fixed-temperature tracking with identical Philox streams: per-shell absorbed energy within 1e-4 relative;
  * full IRE: per-shell T within 1 % or 3 combined standard errors over 8 seeds, whichever is larger;
  * integer energy conservation exact.
"""
import math

import numpy as np
import pytest

from paper_2408_13807_b200 import binding as dies
from paper_2408_13807_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def orc():
    from oracle import dies_oracle
    return dies_oracle


def _fixed_T(n):
    return np.linspace(12.0, 19.0, n)


# ------------------------------------------------------------------ RNG and tables
def test_device_philox_and_uniforms_bit_exact(orc):
    for seed, first, blk, mi in [(1, 0, 0, 0), (0xDEADBEEF12345678, 2 ** 32 - 5, 3, 7), (42, 2 ** 40 + 11, 100, 1023)]:
        n = 4096
        w, u = dies.dies_test_philox(seed, first, blk, mi, n)
        for x in range(0, n, 37):
            pid = first + x
            ref = orc.philox4x32_10((seed & 0xFFFFFFFF, seed >> 32), (pid & 0xFFFFFFFF, pid >> 32, blk, mi))
            assert tuple(int(v) for v in w[x]) == ref
            for c in range(4):
                assert float(u[x, c]) == orc.uniform(ref[c])
        assert u.min() > 0 and u.max() < 1


def test_device_tables_match_oracle(orc):
    p = synth.config1()
    m = dies.Model(p)
    eps, F = m.dies_get_tables()
    o = orc.Oracle(p)
    eps_o, F_o, _ = o.tables()
    np.testing.assert_allclose(eps, eps_o, rtol=1e-14)
    assert np.max(np.abs(F.astype(np.float64) - F_o)) <= 6.0e-8          # one fp32 rounding of a value <= 1
    m.close()


# ------------------------------------------------------------------ deterministic trace (bit-exact)
@pytest.mark.parametrize("cfg,kw", [("config1", {}), ("config1", dict(k_bg=0.3)), ("config1", dict(ffi=1)),
                                    ("config3s", {}), ("config2s", {})])
def test_trace_bit_exact(orc, cfg, kw):
    """Same Philox streams, fixed temperatures: every package whose decisions all sit further than 1e-3 (relative)
    from their thresholds in the oracle must produce the identical event list (type, shell, bin, crossings)."""
    if cfg == "config1":
        p = synth.config1()
    elif cfg == "config3s":
        p = synth.config3(n_shells=40, n_freq=64, tau_V=30.0)
    else:
        p = synth.config2(n_shells=50, n_freq=64)
    n_total, count, max_ev = 100000, 3000, 512
    o = orc.Oracle(p)
    o.set_fixed_temperature(_fixed_T(p.n_shells))
    m = dies.Model(p)
    m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    ev, nev = m.dies_trace_packages(0, count, n_total, seed=5, max_events=max_ev, mode=dies.DIES_MODE_FIXED_T, **kw)
    safe = same = same_safe = 0
    for pid in range(count):
        ref, nref, margin = o.trace(n_total, pid, seed=5, mode=1, max_events=max_ev, **kw)
        ok = (nref == nev[pid]) and nref <= max_ev and np.array_equal(ref, ev[pid, :nref])
        same += ok
        if margin > 1e-3 and nref <= max_ev:
            safe += 1
            same_safe += ok
            assert ok, (pid, margin, ref[:8], ev[pid, :8])
    assert safe > 0.5 * count
    assert same_safe == safe
    assert same >= 0.995 * count, same / count       # the rest differ by fp32-vs-fp64 branch flips (R14)
    m.close()


# ------------------------------------------------------------------ fixed-T tracking, identical streams
def _fixed_T_pair(orc, p, n, seed=3, **kw):
    o = orc.Oracle(p)
    o.set_fixed_temperature(_fixed_T(p.n_shells))
    o.run(n, seed=seed, mode=1, **kw)
    m = dies.Model(p)
    m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    m.dies_run(n, seed=seed, mode=dies.DIES_MODE_FIXED_T, **kw)
    raw, unit, energy = m.dies_get_absorbed()
    return o, m, raw, unit, energy


@pytest.mark.parametrize("kw", [{}, dict(k_bg=0.2), dict(ffi=1)])
def test_fixed_T_absorbed_energy_config1(orc, kw):
    """Config 1 (1e5 packages): counts per shell are small, so one branch-flipped package already moves a shell by
    1e-4..1e-3; the bar here is: event totals within 2e-4 and every shell within 1e-4 relative or 3 packages."""
    p = synth.config1()
    n = p.n_packages
    o, m, raw, unit, energy = _fixed_T_pair(orc, p, n, **kw)
    c, co = m.dies_get_counters(), o.counters
    assert c["packages"] == co["packages"] == n
    for name in ("crossings", "scatterings", "absorptions", "ffi_crossings"):
        assert abs(c[name] - co[name]) <= 2e-4 * max(co[name], 1) + 3, (name, c[name], co[name])
    e_pkg = o.sums["injected"] / n
    tol = np.maximum(1e-4 * o.absorbed, 3 * e_pkg * (5 if kw.get("k_bg") else 1))
    assert np.all(np.abs(energy - o.absorbed) <= tol), np.max(np.abs(energy - o.absorbed) / e_pkg)
    assert c["injected_raw"] == c["escaped_raw"] + c["terminated_raw"]
    esc = m.dies_get_escape_spectrum()
    assert abs(esc.sum() / o.sums["escaped"] - 1) < 1e-5
    m.close()


def test_fixed_T_absorbed_energy_config2_1e4_relative(orc):
    """North-star bar at config 2's full size (1e7 packages, the launch configuration bench.py times): per-shell
    absorbed energy within 1e-4 relative with identical Philox streams wherever a shell holds >= 2e4 package
    quanta, so that one fp32-vs-fp64 branch-flipped package stays below the bar (reading R14); elsewhere within
    2 package quanta."""
    p = synth.config2()
    n = p.n_packages
    o, m, raw, unit, energy = _fixed_T_pair(orc, p, n, seed=1)
    c, co = m.dies_get_counters(), o.counters
    for name in ("crossings", "scatterings", "absorptions"):
        assert abs(c[name] / co[name] - 1) < 2e-5, (name, c[name], co[name])
    e_pkg = o.sums["injected"] / n
    cnt = o.absorbed / e_pkg
    diff = np.abs(energy - o.absorbed)
    well = cnt >= 2e4
    print("shells with >= 2e4 quanta:", int(well.sum()), "max rel there:", (diff[well] / o.absorbed[well]).max(),
          "max |diff| in packages:", diff.max() / e_pkg)
    assert abs(energy.sum() / o.absorbed.sum() - 1) < 1e-5
    assert well.sum() >= 40
    assert np.all(diff[well] < 1e-4 * o.absorbed[well])
    assert np.all(diff[~well] <= 2 * e_pkg)
    assert c["injected_raw"] == c["escaped_raw"]
    assert c["injected_raw"] == n * (1 << 24)
    m.close()


def test_fixed_T_is_deterministic_and_splittable():
    """Integer tallies: the same seed gives bit-identical tallies whatever the scheduling, and a run split into
    accumulate batches (PAPER.md L163 N_B batches) equals the single run exactly."""
    p = synth.config1()
    n = 60000
    res = []
    for parts in (1, 1, 3):
        m = dies.Model(p)
        m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
        for b in range(parts):
            m.dies_run(n // parts, seed=9, mode=dies.DIES_MODE_FIXED_T, n_total=n, accumulate=int(b > 0))
        raw, _, _ = m.dies_get_absorbed()
        res.append((raw.copy(), m.dies_get_escape_spectrum().copy(), m.dies_get_counters()))
        m.close()
    for r in res[1:]:
        assert np.array_equal(r[0], res[0][0])
        assert np.array_equal(r[1], res[0][1])
        for k in ("packages", "crossings", "scatterings", "absorptions", "injected_raw", "escaped_raw"):
            assert r[2][k] == res[0][2][k]


@pytest.mark.parametrize("kw", [{}, dict(k_bg=0.2), dict(ffi=1)])
def test_fixed_T_tallies_do_not_depend_on_tuning_or_stream(kw):
    """dies_set_tuning (pool depth, blocks per visit, batch threshold, id chunks) changes the order in which packages
    are followed, never what is computed: in fixed-temperature mode the integer tallies, the escape spectrum and the
    counters are bit-identical; the runs go through a non-default (non-blocking) CUDA stream, the first of them right
    after dies_set_sources."""
    import torch
    p = synth.config2(n_shells=50, n_freq=64, tau_V=5.0)
    n = 300_000
    res = []
    try:
        for tune in ({}, dict(visit=1, slots_uniform=1, slots=1), dict(visit=16, min_ready=1, chunk=32),
                     dict(slots_uniform=3, slots=2, min_ready=200, pkg_per_block=4096)):
            dies.dies_set_tuning()
            if tune:
                dies.dies_set_tuning(**tune)
            st = torch.cuda.Stream()
            m = dies.Model(p)
            m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
            m.dies_set_sources(p.ext_bin_intensity)
            m.dies_run(n, seed=4, mode=dies.DIES_MODE_FIXED_T, stream=st.cuda_stream, **kw)
            raw, _, _ = m.dies_get_absorbed()
            res.append((raw.copy(), m.dies_get_escape_spectrum().copy(), m.dies_get_counters()))
            m.close()
    finally:
        dies.dies_set_tuning()
    for r in res[1:]:
        assert np.array_equal(r[0], res[0][0])
        assert np.array_equal(r[1], res[0][1])
        for k in ("packages", "crossings", "ffi_crossings", "scatterings", "absorptions", "escaped", "injected_raw",
                  "escaped_raw"):
            assert r[2][k] == res[0][2][k], k
    assert res[0][2]["packages"] == n


def test_tuning_argument_errors():
    with pytest.raises(dies.DiesError) as e:
        dies.dies_set_tuning(visit=1000)
    assert e.value.code == dies.DIES_EINVAL
    t0 = dies.dies_get_tuning()
    dies.dies_set_tuning(visit=5)
    assert dies.dies_get_tuning()["visit"] == 5 and dies.dies_get_tuning()["chunk"] == t0["chunk"]
    dies.dies_set_tuning()
    assert dies.dies_get_tuning() == t0


# ------------------------------------------------------------------ full IRE, statistical
def _ire_stats(orc, p, n, seeds, model_kw=None, **kw):
    To, Tg = [], []
    for s in seeds:
        o = orc.Oracle(p)
        o.run(n, seed=s, **kw)
        To.append(o.temperature())
        m = dies.Model(p)
        m.dies_run(n, seed=s, **kw)
        Tg.append(m.dies_get_temperature())
        c = m.dies_get_counters()
        assert c["injected_raw"] + c["reweight_raw"] == c["escaped_raw"] + c["terminated_raw"]   # exact conservation
        n_src = int(p.ext_bin_intensity is not None) + int(p.L_point > 0)
        assert c["packages"] == n * n_src == o.counters["packages"] and c["terminated"] == 0
        m.close()
    return np.array(To), np.array(Tg)


def _T_outliers(To, Tg):
    """Shells where the 8-seed means differ by more than max(1 %, 3 combined standard errors) (north_star bar)."""
    mo, mg = To.mean(0), Tg.mean(0)
    se = np.sqrt(To.var(0, ddof=1) / len(To) + Tg.var(0, ddof=1) / len(Tg))
    tol = np.maximum(0.01 * mo, 3 * se)
    bad = np.abs(mg - mo) > tol
    with np.errstate(divide="ignore", invalid="ignore"):
        return bad, (np.nonzero(bad)[0], (mg / mo)[bad], (np.abs(mg - mo) / se)[bad])


def _two_looks(label, stats):
    """north_star: per-shell T(r) within 1 % or 3 combined standard errors over 8 seeds, whichever is larger.
    With the standard error estimated from 8 + 8 samples a correct implementation still exceeds 3 se in ~1 % of
    the poorly sampled shells (Student t, ~14 degrees of freedom), i.e. in one of 32..200 shells in a good share of
    runs.  So a shell flagged on seeds 1..8 is re-examined on the independent seeds 9..16 and has to pass there: a
    real bias fails twice, a fluctuation fails twice in the same shell with probability ~1e-4.  At most 5 % of the
    shells may need that second look.  `stats(seeds)` returns (oracle T, GPU T), each seeds x shells.  How many shells
    were flagged goes into the tail of the pytest run (tests/parity_notes.py), pass or fail."""
    from parity_notes import note
    To, Tg = stats(range(1, 9))
    bad, info = _T_outliers(To, Tg)
    note(f"{label}: {int(bad.sum())} of {bad.size} shells flagged"
         + (f" (shells {info[0].tolist()}, |dT|/se {np.round(info[2], 2).tolist()}): second look on seeds 9-16" if bad.any() else ""))
    if np.any(bad):
        assert bad.sum() <= max(1, int(0.05 * bad.size)), info
        To2, Tg2 = stats(range(9, 17))
        bad2, info2 = _T_outliers(To2, Tg2)
        note(f"{label}: second look flags {int(bad2.sum())} shells, {int((bad & bad2).sum())} of them again")
        assert not np.any(bad & bad2), (info, info2)
    return To, Tg


def _check_T_parity(orc, p, n, model_kw=None, **kw):
    label = f"{p.name} n={n:g}" + "".join(f" {k}={v}" for k, v in kw.items())
    _two_looks(label, lambda seeds: _ire_stats(orc, p, n, seeds, model_kw, **kw))


@pytest.mark.parametrize("name,kw", [("plain", {}), ("kbg", dict(k_bg=0.2)), ("ffi", dict(ffi=1))])
def test_full_ire_temperature_config1(orc, name, kw):
    p = synth.config1()
    _check_T_parity(orc, p, p.n_packages, **kw)


def test_full_ire_temperature_config2_reduced(orc):
    _check_T_parity(orc, synth.config2(), 200_000)


def test_full_ire_temperature_config3_reduced(orc):
    _check_T_parity(orc, synth.config3(), 30_000)


def test_full_ire_temperature_config4_reduced(orc):
    _check_T_parity(orc, synth.config4(), 300_000, ffi=1)


def test_both_sources_at_once(orc):
    p = synth.config3(n_shells=40, n_freq=64, tau_V=20.0)
    q = synth.config1(n_freq=64)
    p.ext_bin_intensity = q.ext_bin_intensity * 1e6
    _check_T_parity(orc, p, 20_000)


# ------------------------------------------------------------------ batch (config 5)
def test_batch_matches_per_model_oracle(orc):
    b = synth.config5(n_models=6, n_packages=40_000)
    m = dies.Model(batch=b)
    m.dies_set_fixed_temperature(np.tile(_fixed_T(64), (b.n_models, 1)))
    m.dies_run(b.n_packages, seed=2, mode=dies.DIES_MODE_FIXED_T)
    raw, unit, energy = m.dies_get_absorbed()
    esc = m.dies_get_escape_spectrum()
    tot = dict(crossings=0, absorptions=0, scatterings=0)
    for i in range(b.n_models):
        p = b.model(i)
        o = orc.Oracle(p)
        o.set_fixed_temperature(_fixed_T(64))
        o.run(b.n_packages, seed=2, mode=1, model_index=i)
        e_pkg = o.sums["injected"] / b.n_packages
        assert np.all(np.abs(energy[i] - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * e_pkg)), i
        assert abs(esc[i].sum() / o.sums["escaped"] - 1) < 1e-5
        for k in tot:
            tot[k] += o.counters[k]
    c = m.dies_get_counters()
    assert c["packages"] == b.n_models * b.n_packages
    for k in tot:
        assert abs(c[k] - tot[k]) <= 2e-4 * tot[k] + 3
    assert c["injected_raw"] == c["escaped_raw"]
    # full IRE on the batch: temperatures per model within noise of the oracle
    m.dies_run(b.n_packages, seed=4)
    T = m.dies_get_temperature()
    for i in (0, b.n_models - 1):
        o = orc.Oracle(b.model(i))
        o.run(b.n_packages, seed=4, model_index=i)
        To = o.temperature()
        assert np.max(np.abs(T[i][20:] / To[20:] - 1)) < 0.05
    m.close()


# ------------------------------------------------------------------ edge cases and errors
def test_edge_cases(orc):
    p = synth.config1()
    m = dies.Model(p)
    for n in (1, 31, 129, 1000):
        m.dies_run(n, seed=1)
        c = m.dies_get_counters()
        assert c["packages"] == n == c["escaped"] + c["uninteracted"]
        assert c["injected_raw"] == c["escaped_raw"] == n * (1 << 24)
    # a shell of zero density and an empty cavity
    p2 = synth.config1(n_shells=8)
    p2.rho[3] = 0.0
    p2.r_bounds = p2.r_bounds + 0.05 * p2.r_bounds[-1]
    o = orc.Oracle(p2)
    o.set_fixed_temperature(_fixed_T(8))
    o.run(50000, seed=2, mode=1)
    m2 = dies.Model(p2)
    m2.dies_set_fixed_temperature(_fixed_T(8))
    m2.dies_run(50000, seed=2, mode=dies.DIES_MODE_FIXED_T)
    raw, unit, energy = m2.dies_get_absorbed()
    assert raw[3] == 0 and o.absorbed[3] == 0
    e_pkg = o.sums["injected"] / 50000
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * e_pkg))
    c = m2.dies_get_counters()
    assert abs(c["crossings"] - o.counters["crossings"]) <= 2e-4 * o.counters["crossings"]
    T = m2.dies_get_temperature()
    assert T[3] == 0.0
    m.close(); m2.close()


def test_error_codes():
    p = synth.config1()
    p_nosrc = synth.config1()
    p_nosrc.ext_bin_intensity = None
    m = dies.Model(p_nosrc)
    with pytest.raises(dies.DiesError) as e:
        m.dies_run(10)
    assert e.value.code == dies.DIES_ESTATE
    m.close()
    m = dies.Model(p)
    with pytest.raises(dies.DiesError) as e:
        m.dies_get_temperature()
    assert e.value.code == dies.DIES_ESTATE
    with pytest.raises(dies.DiesError) as e:
        m.dies_run(10, mode=dies.DIES_MODE_FIXED_T)
    assert e.value.code == dies.DIES_ESTATE
    with pytest.raises(dies.DiesError) as e:
        m.dies_run(10, k_bg=0.0)
    assert e.value.code == dies.DIES_EINVAL
    m.dies_run(10)
    import ctypes as C
    T = np.zeros(p.n_shells + 1)
    assert dies.lib().dies_get_temperature(m._h, T.ctypes.data_as(C.POINTER(C.c_double)), T.size) == dies.DIES_EINVAL
    m.close()
    bad = synth.config1()
    bad.r_bounds[5] = bad.r_bounds[4]
    with pytest.raises(dies.DiesError) as e:
        dies.Model(bad)
    assert e.value.code == dies.DIES_EINVAL
    bad = synth.config1()
    bad.emis[10] = bad.emis[9] * 0.5
    with pytest.raises(dies.DiesError) as e:
        dies.Model(bad)
    assert e.value.code == dies.DIES_EINVAL


def test_large_dimensions(orc):
    """Many shells (1200: the unfolded table spans several KB of shared memory) and many frequency bins (1000):
    fixed-temperature parity on identical streams, and the size that no longer fits is refused."""
    p = synth.config3(n_shells=1200, n_freq=32, tau_V=5.0, n_packages=20000)
    o, m, raw, unit, energy = _fixed_T_pair(orc, p, 20000)
    e_pkg = o.sums["injected"] / 20000
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * e_pkg))
    c = m.dies_get_counters()
    assert abs(c["crossings"] - o.counters["crossings"]) <= 2e-4 * o.counters["crossings"] + 3
    assert c["injected_raw"] == c["escaped_raw"]
    m.close()
    p = synth.config1(n_freq=1000, n_packages=50000)
    o, m, raw, unit, energy = _fixed_T_pair(orc, p, 50000)
    e_pkg = o.sums["injected"] / 50000
    assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * e_pkg))
    esc = m.dies_get_escape_spectrum()
    assert abs(esc.sum() / o.sums["escaped"] - 1) < 1e-6
    assert np.all(np.abs(esc - o.escaped) <= 1e-4 * o.escaped + 3 * e_pkg)
    m.close()
    with pytest.raises(dies.DiesError) as e:
        dies.Model(synth.config3(n_shells=6000, n_freq=16))
    assert e.value.code == dies.DIES_EINVAL


def test_fixed_T_shards_add_up_bit_exactly():
    """disjoint package-id ranges followed by different handles (the ranks of a sharded run, here
    one after the other on one GPU) give integer tallies whose sum is the single run's, bit for bit."""
    from paper_2408_13807_b200 import sharding
    p = synth.config1()
    n, seed = 100_001, 8
    whole = dies.Model(p)
    whole.dies_set_fixed_temperature(_fixed_T(p.n_shells))
    whole.dies_run(n, seed=seed, mode=dies.DIES_MODE_FIXED_T)
    raw_w, _, _ = whole.dies_get_absorbed()
    c_w = whole.dies_get_counters()
    world = 3
    tot = np.zeros_like(raw_w)
    cross = 0
    for rank in range(world):
        m = dies.Model(p)
        m.dies_set_fixed_temperature(_fixed_T(p.n_shells))
        raw, esc, c = sharding.run_fixed_T_shard(m, n, seed, rank, world)
        first, count = sharding.package_range(n, rank, world)
        assert c["packages"] == count
        tot += raw
        cross += c["crossings"]
        m.close()
    assert np.array_equal(tot, raw_w)
    assert cross == c_w["crossings"]
    whole.close()


def test_batch_shards_equal_the_whole_batch_bit_for_bit():
    """Config 5 sharded over ranks: two shards of the batch, each a handle of its own with
    dies_set_model_offset, give the tallies of the one-handle batch bit for bit in fixed-temperature mode."""
    from paper_2408_13807_b200 import sharding
    b = synth.config5(n_models=7, n_packages=40_000, n_shells=24, n_freq=32, n_T=200)
    Tfix = np.linspace(8.0, 30.0, 24)

    def run(batch, first):
        m = dies.Model(batch=batch)
        m.dies_set_model_offset(first)
        m.dies_set_fixed_temperature(np.tile(Tfix, (batch.n_models, 1)))
        m.dies_run(batch.n_packages, seed=6, mode=dies.DIES_MODE_FIXED_T)
        raw, _, _ = m.dies_get_absorbed()
        esc = m.dies_get_escape_spectrum()
        c = m.dies_get_counters()
        m.close()
        return raw.reshape(batch.n_models, -1).copy(), esc.reshape(batch.n_models, -1).copy(), c

    raw, esc, c = run(b, 0)
    parts = [run(*sharding.batch_shard(b, r, 3)) for r in range(3)]
    assert np.array_equal(np.concatenate([q[0] for q in parts]), raw)
    assert np.array_equal(np.concatenate([q[1] for q in parts]), esc)
    for k in ("packages", "crossings", "scatterings", "absorptions", "escaped_raw"):
        assert sum(q[2][k] for q in parts) == c[k], k
    # without the offset the second shard would follow other packages
    m = dies.Model(batch=sharding.batch_shard(b, 1, 3)[0])
    m.dies_set_fixed_temperature(np.tile(Tfix, (m.n_models, 1)))
    m.dies_run(b.n_packages, seed=6, mode=dies.DIES_MODE_FIXED_T)
    assert not np.array_equal(m.dies_get_absorbed()[0].reshape(m.n_models, -1), parts[1][0])
    m.close()


def test_batch_full_ire_temperature_over_8_seeds(orc):
    """Config 5 reduced (4 spheres of 64 shells, one launch per seed): per-shell T of every model within 1 % or 3
    combined standard errors of the oracle's 8-seed mean; shells flagged once are re-examined on seeds 9-16."""
    b = synth.config5(n_models=4, n_packages=40_000)

    def stats(seeds):
        To = np.zeros((len(seeds), b.n_models, 64))
        Tg = np.zeros_like(To)
        m = dies.Model(batch=b)
        for a, s in enumerate(seeds):
            m.dies_run(b.n_packages, seed=s)
            Tg[a] = m.dies_get_temperature()
            c = m.dies_get_counters()
            assert c["injected_raw"] == c["escaped_raw"] and c["packages"] == b.n_models * b.n_packages
            for i in range(b.n_models):
                o = orc.Oracle(b.model(i))
                o.run(b.n_packages, seed=s, model_index=i)
                To[a, i] = o.temperature()
        m.close()
        return To.reshape(len(seeds), -1), Tg.reshape(len(seeds), -1)

    _two_looks("config5 reduced (4 spheres x 4e4)", stats)


def test_smallest_dimensions(orc):
    """One shell, two temperatures, two frequency bins (one of them transparent, zero scattering, g = 0), and a
    three-shell model with a cavity and scattering: fixed-temperature parity and exact conservation."""
    from test_oracle_pins import toy_problem
    for p in (toy_problem(n_shells=1, tau=1.5), toy_problem(n_shells=3, tau=2.0, kappa_sca=0.7, g=0.0, r_in=0.2)):
        n = 30000
        Tfix = np.full(p.n_shells, 25.0)
        o = orc.Oracle(p)
        o.set_fixed_temperature(Tfix)
        o.run(n, seed=6, mode=1)
        m = dies.Model(p)
        m.dies_set_fixed_temperature(Tfix)
        m.dies_run(n, seed=6, mode=dies.DIES_MODE_FIXED_T)
        raw, unit, energy = m.dies_get_absorbed()
        e_pkg = o.sums["injected"] / n
        assert np.all(np.abs(energy - o.absorbed) <= np.maximum(1e-4 * o.absorbed, 3 * e_pkg))
        c = m.dies_get_counters()
        assert c["packages"] == n == c["escaped"] and c["injected_raw"] == c["escaped_raw"]
        for k in ("crossings", "scatterings", "absorptions"):
            assert abs(c[k] - o.counters[k]) <= 2e-4 * o.counters[k] + 3
        m.dies_run(n, seed=6)                      # full IRE on the same tiny model
        T = m.dies_get_temperature()
        assert np.all(np.isfinite(T)) and m.dies_get_counters()["injected_raw"] == m.dies_get_counters()["escaped_raw"]
        m.close()


def test_atomic_microbenchmark_runs():
    """dies_bench_atomics (measurement support of bench.py): sane figures, merged draws issue fewer atomics."""
    r1 = dies.dies_bench_atomics(1, None, 1, iters=200)
    r0 = dies.dies_bench_atomics(1, None, 0, iters=200)
    assert r1["lane_ops_per_s"] > 5 * r0["lane_ops_per_s"] > 0       # one address: a warp merges 32 draws into one
    assert abs(r1["atomics_per_s"] / r1["lane_ops_per_s"] - 1 / 32) < 1e-6
    w = np.arange(1, 101, dtype=float)
    rw = dies.dies_bench_atomics(100, w, 1, iters=200)
    assert 0 < rw["atomics_per_s"] <= rw["lane_ops_per_s"]
    with pytest.raises(dies.DiesError):
        dies.dies_bench_atomics(100, -w, 1)


def test_ire_mode_trace_against_run_tallies(orc):
    """Full IRE decisions (table rows from the cell energy before / after the absorption, the extra Philox block when
    they differ) replayed package by package: after a GPU IRE run, packages traced in IRE mode against the run's
    tallies give the oracle's event lists computed from the same tallies."""
    p = synth.config1()
    n = p.n_packages
    m = dies.Model(p)
    m.dies_run(n, seed=12)
    raw, unit, energy = m.dies_get_absorbed()
    o = orc.Oracle(p)
    count, max_ev = 1500, 512
    ev, nev = m.dies_trace_packages(0, count, n, seed=77, max_events=max_ev, mode=dies.DIES_MODE_IRE)
    safe = same = 0
    for pid in range(count):
        ref, nref, margin = o.trace(n, pid, seed=77, mode=0, max_events=max_ev, absorbed_state=energy)
        ok = (nref == nev[pid]) and nref <= max_ev and np.array_equal(ref, ev[pid, :nref])
        same += ok
        safe += (margin > 1e-3)
    assert safe > 0.4 * count
    assert same >= 0.985 * count, same / count
    # early in a run the cells are cold and an absorption spans many table rows: replay against a young state too
    m.dies_run(2000, seed=13, n_total=n)
    raw, unit, energy = m.dies_get_absorbed()
    ev, nev = m.dies_trace_packages(5000, 500, n, seed=78, max_events=max_ev, mode=dies.DIES_MODE_IRE)
    same = 0
    for x in range(500):
        ref, nref, margin = o.trace(n, 5000 + x, seed=78, mode=0, max_events=max_ev, absorbed_state=energy)
        same += (nref == nev[x]) and nref <= max_ev and np.array_equal(ref, ev[x, :nref])
    assert same >= 0.97 * 500, same / 500
    m.close()
