"""Pins of oracle_detection_efficiency (f4; Fig. 13; readings W1-W4).  CPU only: closed forms on
regular cadences, degenerate cadences, an event-centred brute force, and the integer-day dips the figure's
caption describes."""
import numpy as np
import pytest

import oracle


def test_daily_cadence_closed_forms():
    t = np.arange(30, dtype=np.float32)                      # one epoch per day, same time every day
    # P = 1 d: the epoch always sees phase 0; detected iff the eclipse covers phase 0: fraction d/P of the phases
    cnt, eff = oracle.detection_efficiency(t, [1.0], 0.1, 1000)
    assert cnt[0] == 100 and eff[0] == 0.1
    # P = 2 d: epochs alternate between phases 0 and 1/2: two windows of width d/P -> 2 d/P = 0.1
    cnt, eff = oracle.detection_efficiency(t, [0.5], 0.1, 1000)
    assert cnt[0] == 100
    # P = 4 d, d = 0.104 d: four sampled phases, each a window of d/P = 0.026 -> 0.104 (the window edges fall
    # between the phase samples, as above, so the counts are exact); P = 0.5 d: phase 0 only, window d/P = 0.2
    assert oracle.detection_efficiency(t, [0.25], 0.104, 1000)[0][0] == 104
    assert oracle.detection_efficiency(t, [2.0], 0.1, 1000)[0][0] == 200
    # an irrational-looking period: 30 epochs sample 30 distinct phases; each phase window d/P; detection needs TWO
    # epochs in eclipse, so the efficiency is well below the one-epoch coverage but above 0
    c, e = oracle.detection_efficiency(t, [1.0 / 0.7310585], 0.1, 2000)
    assert 0 < e[0] < 30 * 0.1 / 0.7310585


def test_degenerate_cadences_never_detect():
    assert oracle.detection_efficiency(np.array([3.7], np.float32), [0.3, 1.0, 2.2], 0.2, 200)[0].sum() == 0
    # two epochs 10 minutes apart: inside the same eclipse (one event) or none -> never two events
    t = np.array([5.0, 5.0 + 10 / 1440], np.float32)
    assert oracle.detection_efficiency(t, [0.2, 0.9, 1.7], 0.05, 500)[0].sum() == 0
    # ... unless one event is enough
    c1, _ = oracle.detection_efficiency(t, [0.9], 0.05, 500, min_events=1)
    assert 0 < c1[0] < 500
    assert oracle.detection_efficiency(np.zeros(0, np.float32), [1.0], 0.1, 10)[0][0] == 0


def _event_centred(t, f, d, n_phase, min_events):
    """Independent restatement: walk the ECLIPSES of the target (not the epochs) and ask whether any epoch falls
    within d/2 of each mid-eclipse time."""
    t = np.asarray(t, dtype=np.float64)
    P = 1.0 / f
    det = 0
    for k in range(n_phase):
        T0 = (k + 0.5) / n_phase * P
        m_lo, m_hi = int(np.floor((t.min() - T0) / P)) - 1, int(np.ceil((t.max() - T0) / P)) + 1
        ev = sum(1 for m in range(m_lo, m_hi + 1) if np.any(np.abs(t - (T0 + m * P)) <= 0.5 * d * (1 + 1e-12)))
        det += ev >= min_events
    return det


def test_matches_event_centred_bruteforce():
    rng = np.random.default_rng(6)
    night = np.sort(rng.choice(40, 25, replace=False))
    t = np.sort(np.concatenate([n + 0.1 + rng.uniform(0, 0.25, 6) for n in night])).astype(np.float32)
    for f, d in ((0.37, 0.08), (1.0, 0.05), (2.71, 0.03), (0.123, 0.2)):
        c, e = oracle.detection_efficiency(t, [f], d, 240)
        b = _event_centred(t, f, d, 240, 2)
        assert abs(int(c[0]) - b) <= 2, (f, d, c[0], b)      # knife-edge phases (|x - m| == h to rounding) may differ
        assert e[0] == c[0] / 240


def test_integer_day_periods_are_the_dips_of_fig13():
    # nightly 6-hour windows over 60 nights ("low efficiencies around integer numbers of days at
    # short periods are due to the likelihood of an eclipse always occurring in daytime")
    rng = np.random.default_rng(8)
    t = np.sort(np.concatenate([n + np.arange(0.0, 0.25, 15 / 1440) for n in range(60) if rng.uniform() < 0.7])).astype(np.float32)
    periods = np.array([0.5, 1.0, 2.0, 0.37, 0.73, 1.37, 2.6])
    c, e = oracle.detection_efficiency(t, 1.0 / periods, 0.02, 400)
    assert e[3] > 0.99 and e[4] > 0.99                       # fractional-day periods: near 100 % (L426)
    assert e[1] < 0.35 and e[0] < 0.6 and e[2] < 0.35        # integer and half-integer day periods: the dips
    assert e[1] == pytest.approx(0.25 + 0.02, abs=0.03)      # P = 1 d: the nightly window plus the eclipse duration
