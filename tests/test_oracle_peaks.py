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


# ---- reading R14 with a minimum separation (oracle_peaks_sep): answers written out by hand -------------

def pks(sr, k, sep):
    return list(oracle.peaks_sep(np.asarray(sr, dtype=np.float64), k, sep))


def test_separation_answers_written_out():
    #     0  1  2  3  4  5  6  7  8
    sr = [1, 5, 1, 4, 1, 3, 1, 2, 1]                       # peaks at 1, 3, 5, 7 worth 5, 4, 3, 2
    assert pks(sr, 4, 0) == [1, 3, 5, 7]
    assert pks(sr, 4, 1) == [1, 3, 5, 7]                   # neighbours are 2 apart: "more than 1"
    assert pks(sr, 4, 2) == [1, 5, -1, -1]                 # 3 is exactly 2 from 1: not MORE than 2; 7 is 2 from 5
    assert pks(sr, 4, 3) == [1, 5, -1, -1]
    assert pks(sr, 4, 4) == [1, 7, -1, -1]                 # 5 is exactly 4 from 1; 7 is 6 from 1
    assert pks(sr, 4, 6) == [1, -1, -1, -1]
    assert pks(sr, 1, 2) == [1]


def test_a_rejected_peak_suppresses_nothing():
    #     0   1  2  3  4  5  6
    sr = [0, 10, 0, 9, 0, 8, 0]
    # 3 is rejected (2 from the accepted 1); 5 is 2 from the REJECTED 3 but 4 from 1: accepted
    assert pks(sr, 3, 2) == [1, 5, -1]
    # ranking decides who is accepted first, not position: the highest peak sits on the right here
    sr = [0, 8, 0, 9, 0, 10, 0]
    assert pks(sr, 3, 2) == [5, 1, -1]
    assert pks(sr, 3, 1) == [5, 3, 1]


def test_equal_values_and_plateaus_with_separation():
    sr = [0.0, 2.0, 0.0, 2.0, 0.0, 2.0, 0.0, 2.0]          # equal peaks: index order; 7 is the right end
    assert pks(sr, 4, 2) == [1, 5, -1, -1]
    assert pks(sr, 4, 3) == [1, 5, -1, -1]
    assert pks(sr, 4, 5) == [1, 7, -1, -1]
    sr = [2.0, 2.0, 1.0, 3.0, 3.0, 3.0, 0.5, 4.0]          # plateaus resolve to their leftmost sample first
    assert pks(sr, 4, 0) == [7, 3, 0, -1]
    assert pks(sr, 4, 3) == [7, 3, -1, -1]                 # 3 is 4 from 7; 0 is exactly 3 from 3
    assert pks(sr, 4, 4) == [7, 0, -1, -1]


def test_separation_zero_is_the_plain_rule_and_brute_force_agrees():
    rng = np.random.default_rng(14)
    for trial in range(300):
        nf = int(rng.integers(1, 14))
        sr = np.round(rng.uniform(0, 4, nf), 0 if trial % 2 else 1)            # many exact ties and zeros
        k = int(rng.integers(1, 6))
        assert pks(sr, k, 0) == pk(sr, k)
        sep = int(rng.integers(0, 5))
        got = [q for q in pks(sr, k, sep) if q >= 0]
        # brute force from the definition, stated differently: the accepted list is the one obtained by repeatedly
        # taking, among the peaks farther than sep from everything taken so far OR already passed over, ... i.e. by
        # sorting the peaks once and filtering; here: enumerate ranks, keep a peak iff no EARLIER-RANKED KEPT peak is
        # within sep, computed by dynamic programming over the ranked list
        peaks_all = [q for q in range(nf) if sr[q] > 0 and (q == 0 or sr[q] > sr[q - 1]) and (q == nf - 1 or sr[q] >= sr[q + 1])]
        ranked = sorted(peaks_all, key=lambda q: (-sr[q], q))
        kept = []
        for q in ranked:
            if all(abs(q - p) > sep for p in kept):
                kept.append(q)
        assert got == kept[:k], (list(sr), k, sep, got, kept)
        # properties that hold for any correct answer: pairwise separation, and maximality (every peak left out that
        # ranks before the last accepted one is within sep of an accepted one ranked before it)
        assert all(abs(a - b) > sep for i, a in enumerate(got) for b in got[i + 1:])
        if got:
            last_rank = ranked.index(got[-1])
            for r, q in enumerate(ranked[:last_rank]):
                if q not in got:
                    assert any(abs(q - p) <= sep for p in got if ranked.index(p) < r)
