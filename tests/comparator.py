"""Comparator between the CUDA path's outputs and the fp64 oracle.

Tolerances are BASELINE.json north_star's:
  * per-frequency SR maximum: |SR_gpu - SR_orc| <= 1e-4 * SR_orc (+ an absolute floor of
    1e-6 * sum_i w_i x_i^2 for frequencies where the oracle's SR is rounding noise);
  * best (start, width): identical, except at documented near-ties: the oracle's SR of the box the
    CUDA path chose is within 1e-6 relative of the oracle's maximum (boxes holding the same or
    complementary point sets tie mathematically);
  * top-k peak lists: matching (a flip between adjacent near-flat samples or a swap between peaks
    whose SR differ by < 2e-4 relative is a near-tie; so is a peak of the oracle's spectrum rounded to
    fp32, the reported precision (R14 + R15: a plateau below fp32 resolution).  Each is counted).
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


def compare_peaks(o_sr, g_idx, g_srs, k, label="", g_spectrum=None):
    """g_idx: the CUDA path's peak indices (length k, -1 padded) against the oracle's spectrum o_sr.

    What "matching" means (readings R14, R15).  R14's plateau clause (the
    leftmost of equal samples is a peak) is decided by rounding wherever adjacent frequencies hold the
    SAME point set in their best box: those SR values are mathematically equal, the fp64 oracle gets
    them 0-1 ulp apart depending on how the points fell into bins, the fp32 CUDA path likewise.  Such
    samples are exact ties, so the two peak lists can differ there in either direction.  The check is
    therefore in two parts:
      (a) EXACT, when g_spectrum (the CUDA path's own SR row) is given: the reported list must equal
          the oracle's peak picker run on that row, index for index -- the peak stage has no freedom;
          with the per-frequency SR parity of compare_spectrum this says the list is the oracle's list
          for a spectrum within the SR tolerance of the oracle's;
      (b) against the oracle's own spectrum: every reported peak must be an oracle peak, or be tied to
          one along a run of samples within PEAK_RTOL, or be a peak of the oracle's spectrum rounded to
          the reported precision (fp32); and must not rank below the oracle's k-th ROBUST peak (one
          whose two neighbours are lower by more than PEAK_RTOL, i.e. a peak under any rounding).
    Every departure from the oracle's list is counted as a near-tie in the report."""
    o_sr = np.asarray(o_sr, dtype=np.float64)
    g_idx = np.asarray(g_idx)
    n_g = int((g_idx >= 0).sum())
    if g_spectrum is not None:                                   # (a)
        want = oracle.peaks(np.asarray(g_spectrum, dtype=np.float64), k)
        assert np.array_equal(want, g_idx), "%s peak list is not R14 applied to the reported spectrum: %s vs %s" % (
            label, g_idx, want)
    o_idx = oracle.peaks(o_sr, k)
    n_o = int((o_idx >= 0).sum())
    allpk = oracle.peaks(o_sr, len(o_sr))
    allpk = [int(i) for i in allpk if i >= 0]                    # ranked by SR
    o_sr32 = o_sr.astype(np.float32).astype(np.float64)          # the reported precision (R15)
    allpk32 = set(int(i) for i in oracle.peaks(o_sr32, len(o_sr32)) if i >= 0)
    nfq = len(o_sr)
    nbr = lambda p: max(o_sr[p - 1] if p > 0 else -np.inf, o_sr[p + 1] if p + 1 < nfq else -np.inf)
    robust = [p for p in allpk if nbr(p) < o_sr[p] * (1 - PEAK_RTOL)]
    kth_robust = o_sr[robust[k - 1]] if len(robust) >= k else 0.0
    allpk = set(allpk)
    near = 0
    if n_g != n_o:
        assert min(n_g, n_o) < k, "%s peak count %d vs %d" % (label, n_g, n_o)
        near += 1
    g_valid = g_idx[:n_g]
    assert len(set(int(q) for q in g_valid)) == n_g, label + " repeated peak"
    gs = np.asarray(g_srs, dtype=np.float64)[:n_g]
    assert np.all(gs[:-1] >= gs[1:]), label + " peaks not ranked"
    for j, q in enumerate(g_valid):
        q = int(q)
        if j < n_o and q == int(o_idx[j]):
            continue
        near += 1
        ok_member = q in allpk or q in allpk32
        for step in (-1, 1):                                     # tied to an oracle peak along a near-flat run
            i = q + step
            while not ok_member and 0 <= i < nfq and abs(o_sr[i] - o_sr[q]) <= PEAK_RTOL * o_sr[q]:
                ok_member = i in allpk
                i += step
        assert ok_member, "%s gpu peak %d is not an oracle local maximum" % (label, q)
        assert o_sr[q] >= kth_robust * (1 - PEAK_RTOL), "%s gpu peak %d ranks below the oracle's k-th robust peak" % (label, q)
    return dict(peak_near_ties=near, n_peaks=n_g)
