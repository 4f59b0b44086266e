"""The comparator itself (tests/comparator.py), on hand-made spectra and a hand-made curve: it accepts
exact matches, lists that differ from the oracle's only through PROVEN exact ties (same point set in
the best box of adjacent frequencies) and near-ties inside the 2e-6 margin, and it still rejects real
defects (an index that is no local maximum, a peak that ranks too low, a list that is not R14 applied
to the spectrum it was reported with, an SR outside 1e-4).  CPU only."""
import numpy as np
import pytest

import oracle
from comparator import (PEAK_RTOL, collapse_ties, compare_peaks, compare_spectrum, exact_tie_runs, member_set)

BASE = np.array([1.0, 2.0, 1.0, 5.0, 1.0, 3.0, 1.0, 4.0, 1.0, 2.5, 1.0]) * 1e-5   # peaks at 3, 7, 5, 9, 1


def _list(sr, k):
    return oracle.peaks(np.asarray(sr, dtype=np.float64), k)


def test_exact_match_has_no_ties():
    idx = _list(BASE, 3)
    assert list(idx) == [3, 7, 5]
    r = compare_peaks(BASE, idx, BASE[idx], 3, g_spectrum=BASE)
    assert r["exact_tie_slots"] == 0 and r["near_tie_slots"] == 0


def test_proven_tie_on_a_slope_the_collapsed_spectrum_decides():
    # oracle: samples 4 and 5 one fp64 ulp apart on a rise towards 6 (rounding noise on an exact tie)
    # -> R14 on the raw oracle row sees no peak at 4; with the tie proven, 4 and 5 are a plateau and
    # 5 < 6 does not matter: R14 makes the LEFTMOST sample of a plateau a peak iff the plateau is one
    o = np.array([1.0, 2.0, 1.0, 1.5, 3.0, np.nextafter(3.0, 4.0), 2.9, 1.0, 2.5, 1.0]) * 1e-5
    ties = np.zeros(len(o) - 1, dtype=bool)
    ties[4] = True
    g = collapse_ties(o, ties)
    assert g[4] == g[5]
    gi = _list(g, 3)
    assert list(_list(o, 3)) == [5, 8, 1] and list(gi) == [4, 8, 1]
    r = compare_peaks(o, gi, g[gi], 3, g_spectrum=g, ties=ties)
    assert r["exact_tie_slots"] == 1 and r["near_tie_slots"] == 0


def test_run_of_three_tied_samples():
    o = np.array([1.0, 2.0, 1.0, 4.0, 4.0, 4.0, 1.0, 3.0, 1.0]) * 1e-5
    o[4] = np.nextafter(o[4], 1.0)
    o[5] = np.nextafter(np.nextafter(o[5], 1.0), 1.0)      # oracle noise: strictly rising along the plateau
    ties = np.zeros(len(o) - 1, dtype=bool)
    ties[3] = ties[4] = True
    g = collapse_ties(o, ties)
    gi = _list(g, 2)
    assert list(_list(o, 2)) == [5, 7] and list(gi) == [3, 7]
    r = compare_peaks(o, gi, g[gi], 2, g_spectrum=g, ties=ties)
    assert r["exact_tie_slots"] == 1 and r["near_tie_slots"] == 0


def test_unproven_difference_inside_the_margin_is_a_counted_near_tie():
    o = BASE.copy()
    o[6] = o[7] * (1 - 0.5 * PEAK_RTOL)          # 6 and 7 nearly equal, different point sets (no tie given)
    g = o.copy()
    g[6] = g[7] * (1 + 0.5 * PEAK_RTOL)          # the reported spectrum decides the other way
    gi = _list(g, 3)
    assert 6 in gi and 7 not in gi
    r = compare_peaks(o, gi, g[gi], 3, g_spectrum=g)
    assert r["near_tie_slots"] >= 1


def test_difference_outside_the_margin_is_rejected():
    o = BASE.copy()
    o[6] = o[7] * (1 - 10 * PEAK_RTOL)
    g = o.copy()
    g[6] = g[7] * (1 + 10 * PEAK_RTOL)
    gi = _list(g, 3)
    with pytest.raises(AssertionError):
        compare_peaks(o, gi, g[gi], 3, g_spectrum=g)


def test_rejects_an_index_that_is_no_local_maximum():
    bad = np.array([3, 7, 4])
    with pytest.raises(AssertionError):
        compare_peaks(BASE, bad, BASE[bad], 3)


def test_rejects_a_peak_that_ranks_too_low():
    bad = np.array([3, 7, 1])            # 1 is a true peak but the 5th, not the 3rd
    with pytest.raises(AssertionError):
        compare_peaks(BASE, bad, BASE[bad], 3)


def test_rejects_a_list_that_is_not_r14_on_the_reported_spectrum():
    idx = np.array([3, 5, 7])            # right members, wrong order for this spectrum
    with pytest.raises(AssertionError):
        compare_peaks(BASE, idx, BASE[idx], 3, g_spectrum=BASE)
    short = np.array([3, 7, -1])         # a peak left out
    with pytest.raises(AssertionError):
        compare_peaks(BASE, short, np.array([5e-5, 4e-5, 0.0]), 3, g_spectrum=BASE)


def test_rejects_unranked_or_repeated_peaks():
    with pytest.raises(AssertionError):
        compare_peaks(BASE, np.array([7, 3, 5]), BASE[[7, 3, 5]], 3)
    with pytest.raises(AssertionError):
        compare_peaks(BASE, np.array([3, 3, 5]), BASE[[3, 3, 5]], 3)


def _curve():
    rng = np.random.default_rng(3)
    n = 40
    t = np.sort(rng.uniform(0, 10, n)).astype(np.float32)
    mag = (15 + rng.normal(0, 0.01, n) + 0.05 * (((t / 2.0) % 1.0) < 0.2)).astype(np.float32)
    sig = np.full(n, 0.01, dtype=np.float32)
    return t, mag, sig


def test_exact_tie_runs_proves_ties_from_member_sets():
    t, mag, sig = _curve()
    nb, kmin, kmax = 16, 1, 4
    # frequencies 1e-9 apart fold every point into the same bin -> identical member sets -> proven ties;
    # the last one is far away -> a different point set
    freqs = np.array([0.5, 0.5 + 1e-9, 0.5 + 2e-9, 0.61])
    st, sr, a, k, dp = oracle.spectrum(t, mag, sig, freqs, nb, kmin, kmax)
    assert st == 0
    m0 = member_set(t, freqs[0], nb, a[0], k[0])
    assert 0 < m0.size < len(t)
    # the member set is what the oracle's own fold puts in the box: its weight and residual sums give SR back
    _, w, x = oracle.prepare(t, mag, sig)
    r, s = w[m0].sum(), (w[m0] * x[m0]).sum()
    assert sr[0] == pytest.approx(s * s / (r * (1 - r)), rel=1e-12)
    tied, ncand = exact_tie_runs(t, freqs, nb, sr, a, k)
    assert list(tied) == [True, True, False] and ncand >= 2
    flat = collapse_ties(sr, tied)
    assert flat[0] == flat[1] == flat[2] == sr[0] and flat[3] == sr[3]


def test_candidate_tie_with_different_point_sets_is_not_collapsed():
    t, mag, sig = _curve()
    nb = 16
    freqs = np.array([0.5, 0.61])
    st, sr, a, k, dp = oracle.spectrum(t, mag, sig, freqs, nb, 1, 4)
    fake = np.array([sr[0], sr[0] * (1 + 1e-13)])      # values that LOOK tied
    tied, ncand = exact_tie_runs(t, freqs, nb, fake, a, k)
    assert ncand == 1 and not tied[0]


def test_compare_spectrum_asserts_1e4_directly():
    t, mag, sig = _curve()
    nb, kmin, kmax = 16, 1, 4
    freqs = np.linspace(0.3, 0.7, 9)
    orc = oracle.spectrum(t, mag, sig, freqs, nb, kmin, kmax)
    _, sr, a, k, dp = orc
    r = compare_spectrum(t, mag, sig, freqs, nb, kmin, kmax, sr * (1 + 5e-5), a, k, dp * (1 + 5e-5), orc=orc)
    assert r["max_rel_err"] == pytest.approx(5e-5, rel=1e-3) and r["box_near_ties"] == 0
    with pytest.raises(AssertionError):
        compare_spectrum(t, mag, sig, freqs, nb, kmin, kmax, sr * (1 + 3e-4), a, k, dp, orc=orc)
    # a different box is only accepted as a near-tie below 1e-6
    a2 = a.copy()
    a2[4] = (a2[4] + 5) % nb
    with pytest.raises(AssertionError):
        compare_spectrum(t, mag, sig, freqs, nb, kmin, kmax, sr, a2, k, dp, orc=orc)
