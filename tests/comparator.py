"""Comparator between the CUDA path's outputs and the fp64 oracle.

Tolerances are BASELINE.json north_star's:
  * per-frequency SR maximum: |SR_gpu - SR_orc| <= 1e-4 * SR_orc (+ an absolute floor of
    1e-6 * sum_i w_i x_i^2 for frequencies where the oracle's SR is rounding noise);
  * best (start, width): identical, except at documented near-ties: the oracle's SR of the box the
    CUDA path chose is within 1e-6 relative of the oracle's maximum (boxes holding the same or
    complementary point sets tie mathematically);
  * top-k peak lists: matching (a flip between adjacent near-flat samples or between peaks whose SR
    differ by < 2e-4 relative is a near-tie, counted and reported).
Every use of a tolerance branch is counted in the returned report.
"""
from __future__ import annotations

import numpy as np

import oracle

SR_RTOL = 1e-4
TIE_RTOL = 1e-6
PEAK_RTOL = 2e-4
ABS_FLOOR = 1e-6


def total_variance(t, mag, sig) -> float:
    st, w, x = oracle.prepare(t, mag, sig)
    return float(np.sum(w * x * x)) if st == 0 else 0.0


def compare_spectrum(t, mag, sig, freqs, nb, kmin, kmax, g_sr, g_a, g_k, g_depth, orc=None, label=""):
    """Element-by-element comparison of one curve's spectrum.  Returns a report dict; raises
    AssertionError on a violation."""
    if orc is None:
        orc = oracle.spectrum(t, mag, sig, freqs, nb, kmin, kmax)
    st, o_sr, o_a, o_k, o_dp = orc
    assert st == 0
    tot = total_variance(t, mag, sig)
    g_sr = np.asarray(g_sr, dtype=np.float64)
    err = np.abs(g_sr - o_sr)
    tol = SR_RTOL * o_sr + ABS_FLOOR * tot
    bad = np.nonzero(err > tol)[0]
    assert bad.size == 0, "%s SR mismatch at %d freqs, first %d: gpu %.9g orc %.9g" % (
        label, bad.size, bad[0], g_sr[bad[0]], o_sr[bad[0]])
    with np.errstate(divide="ignore", invalid="ignore"):
        rel = np.where(o_sr > ABS_FLOOR * tot, err / o_sr, 0.0)
    diff = np.nonzero((np.asarray(g_a) != o_a) | (np.asarray(g_k) != o_k))[0]
    near = 0
    worst_tie = 0.0
    for q in diff:
        if o_sr[q] <= ABS_FLOOR * tot:          # nothing to fit here: any box is as good
            near += 1
            continue
        v, _ = oracle.sr_at(t, mag, sig, freqs[q], nb, int(g_a[q]), int(g_k[q]))
        gap = (o_sr[q] - v) / o_sr[q]
        worst_tie = max(worst_tie, gap)
        assert gap <= TIE_RTOL, "%s box mismatch beyond a near-tie at freq %d: gpu (a=%d,k=%d) scores %.12g, " \
            "oracle (a=%d,k=%d) %.12g, gap %.3g" % (label, q, g_a[q], g_k[q], v, o_a[q], o_k[q], o_sr[q], gap)
        near += 1
    same = np.setdiff1d(np.arange(len(freqs)), diff)
    if g_depth is not None and same.size:
        gd = np.asarray(g_depth, dtype=np.float64)[same]
        od = o_dp[same]
        big = o_sr[same] > ABS_FLOOR * tot
        assert np.all(np.abs(gd[big] - od[big]) <= 1e-4 * np.abs(od[big]) + 1e-9), label + " depth mismatch"
    return dict(max_rel_err=float(rel.max()) if rel.size else 0.0, box_near_ties=int(near),
                worst_tie_gap=float(worst_tie), n_freq=len(freqs), oracle=orc)


def compare_peaks(o_sr, g_idx, g_srs, k, label=""):
    """g_idx: the CUDA path's peak indices (length k, -1 padded) against the oracle's spectrum."""
    o_idx = oracle.peaks(o_sr, k)
    n_o = int((o_idx >= 0).sum())
    g_idx = np.asarray(g_idx)
    n_g = int((g_idx >= 0).sum())
    # all oracle local maxima, for membership tests
    allpk = oracle.peaks(o_sr, len(o_sr))
    allpk = set(int(i) for i in allpk if i >= 0)
    near = 0
    if n_g != n_o:
        # the only legitimate cause: a near-flat sample flipped peak status when fewer than k exist
        assert abs(n_g - n_o) <= 1 and min(n_g, n_o) < k, "%s peak count %d vs %d" % (label, n_g, n_o)
        near += 1
    kth = o_sr[o_idx[n_o - 1]] if n_o else 0.0
    g_valid = g_idx[:n_g]
    assert np.all(g_valid[:-1] != g_valid[1:]) if n_g > 1 else True
    gs = np.asarray(g_srs, dtype=np.float64)[:n_g]
    assert np.all(gs[:-1] >= gs[1:]), label + " peaks not ranked"
    for j, q in enumerate(g_valid):
        q = int(q)
        if j < n_o and q == int(o_idx[j]):
            continue
        near += 1
        ok_member = q in allpk
        if not ok_member:
            for nbq in (q - 1, q + 1):
                if nbq in allpk and abs(o_sr[nbq] - o_sr[q]) <= PEAK_RTOL * o_sr[nbq]:
                    ok_member = True
        assert ok_member, "%s gpu peak %d is not an oracle local maximum" % (label, q)
        assert o_sr[q] >= kth * (1 - PEAK_RTOL), "%s gpu peak %d ranks below the oracle's k-th peak" % (label, q)
    return dict(peak_near_ties=near, n_peaks=n_g)
