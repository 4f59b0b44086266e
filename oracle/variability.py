"""fp64 oracle of the high-variability pre-filter -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md section 2.2.1 (L131): "We estimate the value and scatter of the locally expected photometric
stability as a function of stellar magnitude in 0.1-mag bins, using a sigma-clipped average of the stars
detected on each chip.  Objects that show a more than 2 sigma increased variability compared to the
ensemble expectation are flagged for further review."

The paper gives no formula; the readings (V1-V5) are:
  V1  a star's "photometric stability" is the weighted RMS of its magnitudes about their weighted mean,
      rms = sqrt(sum_i w_i x_i^2) with the BLS weights w_i = sigma_i^-2 / sum_j sigma_j^-2 (Fig. 2 plots
      RMS against magnitude, L117-121); its magnitude is the weighted mean mu;
  V2  magnitude bin b = floor((mu - mag_lo) / mag_bin), mag_bin = 0.1; stars outside
      [mag_lo, mag_lo + n_mag_bins * mag_bin) or with a data fault belong to no ensemble and are never flagged;
  V3  an ensemble is one (group, magnitude bin) cell; group = the chip the star was detected on
      (caller-supplied integer per star; one group if absent);
  V4  sigma-clipped average: start from all members; repeat at most max_iter times: E = mean, S = population
      standard deviation of the members' rms; drop members with |rms - E| > clip * S; stop when nothing is
      dropped.  E and S of the last member set are the expected value and its scatter;
  V5  a star is flagged iff its cell kept at least min_members stars and rms > E + nsig * S (nsig = 2:
      "more than 2 sigma increased variability").
Plain numpy/python loops in index order, nothing blocked or reordered.  Pins: tests/test_variability_oracle.py
(hand-made ensembles with known outliers, the clip written out step by step, invariances).
Only tests/, __graft_entry__.smoke() and bench.py may import this module; it imports nothing from the
CUDA package.
"""
from __future__ import annotations

import math

import numpy as np

import oracle


def star_stats(offsets, t, mag, sigma):
    """V1 per star: (status, mu, rms) in fp64, sums in index order (oracle.prepare)."""
    n = len(offsets) - 1
    st = np.zeros(n, dtype=np.int32)
    mu = np.zeros(n)
    rms = np.zeros(n)
    for c in range(n):
        a, b = int(offsets[c]), int(offsets[c + 1])
        s, w, x = oracle.prepare(t[a:b], mag[a:b], sigma[a:b])
        st[c] = s
        if s != 0:
            continue
        m = 0.0
        for i in range(b - a):
            m += w[i] * float(mag[a + i])
        mu[c] = m
        v = 0.0
        for i in range(b - a):
            v += w[i] * x[i] * x[i]
        rms[c] = math.sqrt(v)
    return st, mu, rms


def cell_of(status, mu, group, mag_lo, mag_bin, n_mag_bins):
    """V2 + V3: cell index group * n_mag_bins + bin, or -1."""
    if status != 0:
        return -1
    b = math.floor((mu - mag_lo) / mag_bin)
    if b < 0 or b >= n_mag_bins:
        return -1
    return int(group) * n_mag_bins + int(b)


def sigma_clip(values, clip, max_iter):
    """V4 on one ensemble (values in member order).  Returns (E, S, kept mask)."""
    vals = [float(v) for v in values]
    keep = [True] * len(vals)
    E = S = 0.0
    for _ in range(max_iter + 1):
        m = [v for v, k in zip(vals, keep) if k]
        if not m:
            return 0.0, 0.0, keep
        E = sum(m) / len(m)
        S = math.sqrt(sum((v - E) * (v - E) for v in m) / len(m))
        if _ == max_iter:
            break
        dropped = False
        for i, v in enumerate(vals):
            if keep[i] and abs(v - E) > clip * S:
                keep[i] = False
                dropped = True
        if not dropped:
            break
    return E, S, keep


def variability_flags(offsets, t, mag, sigma, group=None, *, mag_lo=12.0, mag_bin=0.1, n_mag_bins=80,
                      clip=3.0, nsig=2.0, max_iter=5, min_members=5):
    """V1-V5 for a CSR batch.  Returns dict(status, mean_mag, rms, cell, expected, scatter, kept, flag)."""
    n = len(offsets) - 1
    if group is None:
        group = np.zeros(n, dtype=np.int32)
    st, mu, rms = star_stats(offsets, t, mag, sigma)
    cell = np.array([cell_of(st[c], mu[c], group[c], mag_lo, mag_bin, n_mag_bins) for c in range(n)], dtype=np.int64)
    expected = np.zeros(n)
    scatter = np.zeros(n)
    kept = np.zeros(n, dtype=np.int32)
    flag = np.zeros(n, dtype=np.int32)
    for ce in sorted(set(int(x) for x in cell if x >= 0)):
        members = [c for c in range(n) if cell[c] == ce]           # index order
        E, S, keep = sigma_clip([rms[c] for c in members], clip, max_iter)
        nk = sum(1 for k in keep if k)
        for c in members:
            expected[c], scatter[c], kept[c] = E, S, nk
            if nk >= min_members and rms[c] > E + nsig * S:
                flag[c] = 1
    return dict(status=st, mean_mag=mu, rms=rms, cell=cell, expected=expected, scatter=scatter, kept=kept, flag=flag)
