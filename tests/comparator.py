"""Comparator between the CUDA path's outputs and the fp64 oracle (DESIGN.md section 3 "Tolerances").

Tolerances are BASELINE.json north_star's:
  * per-frequency SR maximum: |SR_gpu - SR_orc| <= 1e-4 * SR_orc, asserted directly; the absolute floor
    is SURVEY.md 8(c)'s 1e-12 * sum_i w_i x_i^2 (only a curve whose residuals are rounding noise gets
    near it);
  * best (start, width): identical, except at documented near-ties: the oracle's SR of the box the
    CUDA path chose is within 1e-6 relative of the oracle's maximum (each is counted);
  * top-k peak lists: matching.  Adjacent trial frequencies whose best boxes hold the SAME point set
    have mathematically equal SR; the fp64 oracle computes such values 0-1 ulp apart (its bins are
    summed in a different order at the two frequencies), so its own plateau decisions (reading R14)
    there are rounding noise.  `exact_tie_runs` PROVES each such tie from the member sets (rebuilt with
    oracle.bins_many), `collapse_ties` gives every proven run one common value, and the CUDA path's
    list must equal R14 applied to that spectrum.  What is left -- decisions between DIFFERENT point
    sets whose SR differ by less than PEAK_RTOL = 2e-6 relative (fp32 output, reading R15) -- is
    accepted only with that margin shown, and counted.
Every use of a tolerance branch is counted in the returned report.
"""
from __future__ import annotations

import numpy as np

import oracle

SR_RTOL = 1e-4
TIE_RTOL = 1e-6
PEAK_RTOL = 2e-6
ABS_FLOOR = 1e-12
TIE_CANDIDATE_RTOL = 1e-10      # adjacent oracle values closer than this are CANDIDATE exact ties (then proven)


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
    floor = ABS_FLOOR * total_variance(t, mag, sig)
    g_sr = np.asarray(g_sr, dtype=np.float64)
    err = np.abs(g_sr - o_sr)
    bad = np.nonzero(err > SR_RTOL * o_sr + floor)[0]
    assert bad.size == 0, "%s SR mismatch at %d freqs, first %d: gpu %.9g orc %.9g" % (
        label, bad.size, bad[0], g_sr[bad[0]], o_sr[bad[0]])
    with np.errstate(divide="ignore", invalid="ignore"):
        rel = np.where(o_sr > floor, err / o_sr, 0.0)
    diff = np.nonzero((np.asarray(g_a) != o_a) | (np.asarray(g_k) != o_k))[0]
    near = 0
    worst_tie = 0.0
    for q in diff:
        if o_sr[q] <= floor:                     # nothing to fit here (SR = 0 up to rounding): any box is as good
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
        big = o_sr[same] > floor
        assert np.all(np.abs(gd[big] - od[big]) <= 1e-4 * np.abs(od[big])), label + " depth mismatch"
    return dict(max_rel_err=float(rel.max()) if rel.size else 0.0, box_near_ties=int(near),
                worst_tie_gap=float(worst_tie), n_freq=len(freqs), oracle=orc)


# ---- peak lists ------------------------------------------------------------------------------------

def member_set(t, f, nb, a, k):
    """Indices of the points inside box (start a, width k) at frequency f -- from the oracle's own bin rule."""
    t64 = np.ascontiguousarray(t, dtype=np.float64)
    b = oracle.bins_many(np.full(t64.size, float(f)), t64, nb)
    return np.nonzero(((b - int(a)) % nb) < int(k))[0]


def exact_tie_runs(t, freqs, nb, o_sr, o_a, o_k):
    """Adjacent frequencies q, q+1 whose oracle values are candidate ties (closer than
    TIE_CANDIDATE_RTOL) AND whose best boxes hold the same points or complementary point sets (a box
    and its complement have equal SR).  Returns (tied, n_candidates): tied[q] is True iff q ~ q+1 is
    a PROVEN exact tie."""
    o_sr = np.asarray(o_sr, dtype=np.float64)
    nf = len(o_sr)
    tied = np.zeros(max(nf - 1, 0), dtype=bool)
    if nf < 2:
        return tied, 0
    close = (np.abs(o_sr[1:] - o_sr[:-1]) <= TIE_CANDIDATE_RTOL * np.maximum(o_sr[1:], o_sr[:-1])) & (o_sr[1:] > 0)
    cand = np.nonzero(close)[0]
    n = len(t)
    for q in cand:
        m0 = member_set(t, freqs[q], nb, o_a[q], o_k[q])
        m1 = member_set(t, freqs[q + 1], nb, o_a[q + 1], o_k[q + 1])
        same = m0.size == m1.size and np.array_equal(m0, m1)
        if not same and m0.size + m1.size == n:
            same = np.array_equal(np.sort(np.concatenate([m0, m1])), np.arange(n))
        tied[q] = same
    return tied, int(cand.size)


def collapse_ties(o_sr, tied):
    """Every run of proven-tied samples takes the value of its first sample: the spectrum exact
    arithmetic would give there, up to rounding that no longer decides anything."""
    s = np.array(o_sr, dtype=np.float64)
    for q in np.nonzero(tied)[0]:            # ascending, so a run propagates its first value
        s[q + 1] = s[q]
    return s


def compare_peaks(o_sr, g_idx, g_srs, k, label="", g_spectrum=None, ties=None):
    """g_idx: the CUDA path's peak indices (length k, -1 padded) against the oracle's spectrum o_sr.

      (a) EXACT, when g_spectrum (the CUDA path's own SR row) is given: the reported list must equal
          the oracle's peak picker (R14) run on that row, index for index.
      (b) against the oracle: with `ties` = exact_tie_runs(...)[0] the reference list is R14 applied to
          collapse_ties(o_sr, ties); the reported list must equal it.  A departure is accepted only as
          a near-tie of margin PEAK_RTOL between different point sets (see module docstring):
          a reported index outside the reference list must be a local maximum within the margin and
          rank no lower than the reference's last peak within the margin; a reference index that is
          not reported must be within the margin of a neighbour or of the last reported peak.
    Returns counts: exact_tie_slots (reference list differs from the raw oracle list: explained by a
    proven tie), near_tie_slots (accepted with the margin), unexplained is always 0 (else it raises)."""
    o_sr = np.asarray(o_sr, dtype=np.float64)
    g_idx = np.asarray(g_idx).astype(np.int64)
    nfq = len(o_sr)
    n_g = int((g_idx >= 0).sum())
    assert np.all(g_idx[n_g:] == -1), label + " padding inside the list"
    g_valid = g_idx[:n_g]
    assert len(set(int(q) for q in g_valid)) == n_g, label + " repeated peak"
    gs = np.asarray(g_srs, dtype=np.float64)[:n_g]
    assert np.all(gs[:-1] >= gs[1:]), label + " peaks not ranked"
    if g_spectrum is not None:                                   # (a)
        want = oracle.peaks(np.asarray(g_spectrum, dtype=np.float64), k)
        assert np.array_equal(want, g_idx), "%s peak list is not R14 applied to the reported spectrum: %s vs %s" % (
            label, g_idx, want)
    raw = oracle.peaks(o_sr, k)
    ref_sr = collapse_ties(o_sr, ties) if ties is not None else o_sr
    ref = oracle.peaks(ref_sr, k)
    exact_tie_slots = int((raw != ref).sum())
    if np.array_equal(ref, g_idx):
        return dict(exact_tie_slots=exact_tie_slots, near_tie_slots=0, n_peaks=n_g)
    # departures: every one needs its margin
    n_r = int((ref >= 0).sum())
    ref_valid = [int(q) for q in ref[:n_r]]
    tau = PEAK_RTOL
    last_ref = ref_sr[ref_valid[-1]] if n_r == k else 0.0
    last_g = ref_sr[int(g_valid[-1])] if n_g == k else 0.0
    nbr_max = lambda p: max(ref_sr[p - 1] if p > 0 else -np.inf, ref_sr[p + 1] if p + 1 < nfq else -np.inf)
    near = 0
    for q in (int(x) for x in g_valid):
        if q in ref_valid:
            continue
        near += 1
        assert ref_sr[q] > 0 and ref_sr[q] >= nbr_max(q) * (1 - tau), \
            "%s gpu peak %d is not a local maximum of the oracle's spectrum within %.0e" % (label, q, tau)
        assert ref_sr[q] >= last_ref * (1 - tau), "%s gpu peak %d ranks below the oracle's k-th peak" % (label, q)
    for p in ref_valid:
        if p in g_valid:
            continue
        near += 1
        flat = ref_sr[p] <= nbr_max(p) * (1 + tau)
        pushed = n_g == k and ref_sr[p] <= last_g * (1 + tau)
        assert flat or pushed, "%s oracle peak %d (SR %.9g) is missing from the gpu list %s" % (label, p, ref_sr[p], g_idx)
    common_g = [int(q) for q in g_valid if int(q) in ref_valid]
    common_r = [p for p in ref_valid if p in common_g]
    for x, y in zip(common_g, common_r):                           # same peaks in another order: near-equal SR only
        if x != y:
            near += 1
            assert abs(ref_sr[x] - ref_sr[y]) <= tau * max(ref_sr[x], ref_sr[y]), \
                "%s peaks %d and %d are ranked differently from the oracle" % (label, x, y)
    assert near > 0
    return dict(exact_tie_slots=exact_tie_slots, near_tie_slots=near, n_peaks=n_g)
