"""Pins for the oracle's peak picking (O5, reading R14): hand-made spectra, answers written out."""
import numpy as np

import oracle


def pk(sr, k):
    return list(oracle.peaks(np.asarray(sr, dtype=np.float64), k))


def test_simple_local_maxima_ranked_by_sr():
    #            0    1    2    3    4    5    6    7    8
    sr = [1.0, 3.0, 2.0, 5.0, 4.0, 4.5, 1.0, 0.5, 0.7]
    # local maxima: 1 (3.0), 3 (5.0), 5 (4.5), 8 (0.7, right end > left neighbour)
    assert pk(sr, 5) == [3, 5, 1, 8, -1]
    assert pk(sr, 2) == [3, 5]
    assert pk(sr, 1) == [3]


def test_plateau_resolves_to_leftmost_and_endpoints():
    sr = [2.0, 2.0, 1.0, 3.0, 3.0, 3.0, 0.5, 4.0]
    # index 0: no left neighbour, >= right -> peak.  index 1: not > left.  3: > left, >= right -> peak;
    # 4, 5: not > left.  7: right end, > left -> peak
    assert pk(sr, 4) == [7, 3, 0, -1]


def test_equal_sr_peaks_keep_index_order():
    sr = [0.0, 2.0, 0.0, 2.0, 0.0, 2.0, 0.0]
    assert pk(sr, 2) == [1, 3]
    assert pk(sr, 5) == [1, 3, 5, -1, -1]


def test_zero_and_monotone_spectra():
    assert pk([0.0, 0.0, 0.0], 3) == [-1, -1, -1]         # SR must be > 0
    assert pk([1.0, 2.0, 3.0], 2) == [2, -1]              # rising: only the right end
    assert pk([3.0, 2.0, 1.0], 2) == [0, -1]              # falling: only the left end
    assert pk([5.0], 2) == [0, -1]
    assert pk([0.0, 1.0, 0.0, 0.0, 2.0], 3) == [4, 1, -1]
