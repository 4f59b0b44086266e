"""The peak-list comparator itself (tests/comparator.py: compare_peaks), on hand-made spectra:
it accepts exact matches and the rounding-decided plateau ties of readings R14 + R15, and it still
rejects real defects (an index that is no local maximum, a peak that ranks too low, a list that is not
R14 applied to the spectrum it was reported with).  CPU only."""
import numpy as np
import pytest

import oracle
from comparator import compare_peaks

BASE = np.array([1.0, 2.0, 1.0, 5.0, 1.0, 3.0, 1.0, 4.0, 1.0, 2.5, 1.0]) * 1e-5   # peaks at 3, 7, 5, 9, 1


def _list(sr, k):
    return oracle.peaks(np.asarray(sr, dtype=np.float64), k)


def test_exact_match_has_no_near_ties():
    idx = _list(BASE, 3)
    assert list(idx) == [3, 7, 5]
    r = compare_peaks(BASE, idx, BASE[idx], 3, g_spectrum=BASE)
    assert r["peak_near_ties"] == 0


def test_plateau_on_a_slope_either_side_may_call_it_a_peak():
    # oracle: samples 4 and 5 one fp64 ulp apart on a rise towards 6 -> no peak at 4;
    # reported spectrum: equal in fp32 -> R14 makes 4 a peak (C4 curve 34 in miniature)
    o = np.array([1.0, 2.0, 1.0, 1.5, 3.0, np.nextafter(3.0, 4.0), 6.0, 1.0, 2.5, 1.0]) * 1e-5
    g = o.astype(np.float32).astype(np.float64)
    assert g[4] == g[5] and o[4] < o[5]
    gi = _list(g, 3)
    assert 4 in gi and 4 not in _list(o, 3)
    r = compare_peaks(o, gi, g[gi], 3, g_spectrum=g)
    assert r["peak_near_ties"] >= 1


def test_plateau_peak_of_the_oracle_may_be_missing():
    # oracle: exact plateau 3,4 then a rise -> 3 is a peak by the plateau clause only (C4 curve 63);
    # reported spectrum: rounding made sample 4 an ulp higher -> 3 is no peak, a lower peak moves up
    o = np.array([1.0, 2.0, 1.0, 4.0, 4.0, 5.0, 1.0, 3.0, 1.0, 2.5, 1.0, 2.2, 1.0]) * 1e-5
    g = o.copy()
    g[4] = np.nextafter(g[4], 1.0)
    oi, gi = _list(o, 3), _list(g, 3)
    assert 3 in oi and 3 not in gi
    r = compare_peaks(o, gi, g[gi], 3, g_spectrum=g)
    assert r["peak_near_ties"] >= 1


def test_run_of_tied_samples_reaches_the_oracle_peak():
    # exact 3-sample plateau (C4 curve 45): oracle takes the leftmost, the reported spectrum the rightmost
    o = np.array([1.0, 2.0, 1.0, 4.0, 4.0, 4.0, 1.0, 3.0, 1.0]) * 1e-5
    g = o.copy()
    g[4] = np.nextafter(g[4], 1.0)                       # one ulp up
    g[5] = np.nextafter(np.nextafter(g[5], 1.0), 1.0)    # two ulps up: strictly rising along the plateau
    gi = _list(g, 2)
    assert list(_list(o, 2)) == [3, 7] and list(gi) == [5, 7]
    compare_peaks(o, gi, g[gi], 2, g_spectrum=g)


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
