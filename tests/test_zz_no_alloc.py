"""dies_trace_packages_static: the package replay for callers that cannot allocate device memory.

Some users of libdies run inside a process whose framework allocator (PyTorch's caching allocator, say) has already
claimed almost the whole GPU: a raw cudaMalloc from the library then fails even though the framework could still hand
out memory.  Others replay packages while trackers run on other streams and cannot take the device-wide stall that
cudaMalloc / cudaFree bring.  For them the library keeps the replay's scratch (event lists, event counts, package
counter) in a fixed array inside the library image, about 1 MiB per GPU, and offers dies_trace_packages_static, which
takes the same inputs and outputs as dies_trace_packages and calls no allocator at all.

The array is shared by every call and still holds the previous call's contents when the next one starts, so this test
makes two static calls back to back, the second smaller than the first and with other options, and only then asks the
allocating path for the same replays: whatever the first call left behind must not show in the second.  Event lists
are integers, so the bar is the one the other trace tests use: identical, element by element.

This file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here should
not hide the parity tests.  It does not depend on them: it passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

from paper_2408_13807_b200 import binding as dies
from paper_2408_13807_b200 import synth

pytestmark = pytest.mark.gpu

N_TOTAL = 100000


def _model():
    p = synth.config1()
    m = dies.Model(p)
    m.dies_set_fixed_temperature(np.linspace(12.0, 19.0, p.n_shells))
    return m


def _same_replay(static, plain, max_events):
    """The static path must give the event counts and the recorded events of the allocating path, and zeros after them
    (the allocating path leaves those entries undefined, so they are not compared)."""
    ev_s, n_s = static
    ev_p, n_p = plain
    assert np.array_equal(n_s, n_p)
    assert n_s.min() >= 2                       # every package is at least launched and ends
    for i in range(len(n_s)):
        k = min(int(n_s[i]), max_events)
        assert np.array_equal(ev_s[i, :k], ev_p[i, :k]), i
        assert not ev_s[i, k:].any(), i


def test_static_trace_matches_allocating_trace_on_two_calls_in_a_row():
    m = _model()
    a = dict(first_id=0, count=2000, n_total=N_TOTAL, seed=5, max_events=32)            # 64000 of the 65536 entries
    b = dict(first_id=777, count=300, n_total=N_TOTAL, seed=9, max_events=3, k_bg=0.3)  # some lists cut at max_events
    got_a = m.dies_trace_packages_static(**a)
    got_b = m.dies_trace_packages_static(**b)       # starts on the leftovers of call a
    _same_replay(got_a, m.dies_trace_packages(**a), a["max_events"])
    _same_replay(got_b, m.dies_trace_packages(**b), b["max_events"])
    assert (got_a[1] <= a["max_events"]).all()      # call a kept whole lists,
    assert (got_b[1] > b["max_events"]).any()       # call b did overflow some: the cut-off path is covered
    # a third call on the weighted tracker (free-path weighting), again on top of what the calls before left
    c = dict(first_id=123, count=500, n_total=N_TOTAL, seed=5, max_events=128, k_A=2.0)
    got_c = m.dies_trace_packages_static(**c)
    _same_replay(got_c, m.dies_trace_packages(**c), c["max_events"])
    m.close()


def test_static_trace_rejects_sizes_beyond_its_array():
    m = _model()
    with pytest.raises(dies.DiesError) as e:
        m.dies_trace_packages_static(0, dies.DIES_TRACE_STATIC_MAX_PACKAGES + 1, N_TOTAL, max_events=1)
    assert e.value.code == dies.DIES_EINVAL and "DIES_TRACE_STATIC_MAX_PACKAGES" in str(e.value)
    with pytest.raises(dies.DiesError) as e:
        m.dies_trace_packages_static(0, 1000, N_TOTAL, max_events=dies.DIES_TRACE_STATIC_MAX_EVENTS // 1000 + 1)
    assert e.value.code == dies.DIES_EINVAL and "DIES_TRACE_STATIC_MAX_EVENTS" in str(e.value)
    # the limits themselves are accepted, and a rejected call leaves the entry point usable
    full = dict(first_id=0, count=dies.DIES_TRACE_STATIC_MAX_PACKAGES, n_total=N_TOTAL, seed=2,
                max_events=dies.DIES_TRACE_STATIC_MAX_EVENTS // dies.DIES_TRACE_STATIC_MAX_PACKAGES)
    _same_replay(m.dies_trace_packages_static(**full), m.dies_trace_packages(**full), full["max_events"])
    m.close()
