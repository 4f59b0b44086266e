"""Pins of oracle/variability.py (section 2.2.1; readings V1-V5).  CPU only.

None of these retype the oracle's loops: the per-star statistics are checked against numpy's weighted
average / std, the sigma clip against scipy.stats.sigmaclip and against hand-made ensembles whose answer
is known in closed form, the flag rule on ensembles with planted outliers."""
import numpy as np
import pytest
import scipy.stats

from oracle import variability as V


def _batch(curves):
    offs = np.zeros(len(curves) + 1, dtype=np.int64)
    for i, c in enumerate(curves):
        offs[i + 1] = offs[i] + len(c[0])
    cat = lambda j: np.concatenate([np.asarray(c[j], dtype=np.float32) for c in curves])
    return offs, cat(0), cat(1), cat(2)


def _star(rng, n, m0, rms, sig=0.01):
    return (np.sort(rng.uniform(0, 30, n)), m0 + rng.normal(0, rms, n), np.full(n, sig))


def test_star_stats_are_the_weighted_mean_and_rms():
    rng = np.random.default_rng(1)
    curves = [_star(rng, 50, 15.0, 0.02), (np.arange(40.0), 16 + rng.normal(0, 0.05, 40), rng.uniform(0.01, 0.05, 40))]
    offs, t, mag, sig = _batch(curves)
    st, mu, rms = V.star_stats(offs, t, mag, sig)
    assert list(st) == [0, 0]
    m0 = mag[:50].astype(np.float64)
    assert mu[0] == pytest.approx(np.mean(m0), rel=1e-14) and rms[0] == pytest.approx(np.std(m0), rel=1e-9)
    m1, w1 = mag[50:].astype(np.float64), 1.0 / sig[50:].astype(np.float64) ** 2
    mu1 = np.average(m1, weights=w1)
    assert mu[1] == pytest.approx(mu1, rel=1e-14)
    assert rms[1] == pytest.approx(np.sqrt(np.average((m1 - mu1) ** 2, weights=w1)), rel=1e-9)


def test_sigma_clip_closed_form_single_outlier():
    # nineteen 1.0 and one 100: z = 19/sqrt(20) = 4.2 > 3 -> dropped, then E = 1, S = 0 and nothing else goes.
    # (with ten values a single outlier can never exceed (n-1)/sqrt(n) = 2.85 sigma: nothing is dropped)
    E, S, keep = V.sigma_clip([1.0] * 19 + [100.0], 3.0, 5)
    assert (E, S) == (1.0, 0.0) and keep == [True] * 19 + [False]
    E, S, keep = V.sigma_clip([1.0] * 9 + [100.0], 3.0, 5)
    assert all(keep) and E == pytest.approx(10.9) and S == pytest.approx(29.7)


def test_sigma_clip_two_rounds_by_hand():
    # round 1: the 50 hides the 3; round 2 (without the 50) drops the 3; round 3 drops nothing
    vals = [1.0, 1.1, 0.9, 1.05, 0.95, 1.0, 1.1, 0.9, 1.0, 1.0, 1.05, 0.95, 1.0, 1.0, 1.1, 0.9, 1.0, 1.0, 3.0, 50.0]
    a = np.array(vals)
    m1, s1 = a.mean(), a.std()
    assert abs(50 - m1) > 3 * s1 and abs(3 - m1) < 3 * s1
    b = a[:-1]
    assert abs(3 - b.mean()) > 3 * b.std()
    c = a[:-2]
    assert np.all(np.abs(c - c.mean()) <= 3 * c.std())
    E, S, keep = V.sigma_clip(vals, 3.0, 5)
    assert keep == [True] * 18 + [False, False]
    assert E == pytest.approx(c.mean(), rel=1e-14) and S == pytest.approx(c.std(), rel=1e-12)
    # max_iter = 1: only the first round of rejection happens
    E1, S1, keep1 = V.sigma_clip(vals, 3.0, 1)
    assert keep1 == [True] * 19 + [False] and E1 == pytest.approx(b.mean(), rel=1e-14)


def test_sigma_clip_matches_scipy_on_random_ensembles():
    rng = np.random.default_rng(5)
    for trial in range(20):
        v = np.concatenate([rng.normal(0.01, 0.001, 150), rng.uniform(0.02, 0.2, rng.integers(0, 12))])
        rng.shuffle(v)
        E, S, keep = V.sigma_clip(v, 3.0, 100)
        kept, lo, hi = scipy.stats.sigmaclip(v, 3.0, 3.0)
        assert int(np.sum(keep)) == kept.size
        assert E == pytest.approx(kept.mean(), rel=1e-12) and S == pytest.approx(kept.std(), rel=1e-10)


def test_planted_outliers_are_flagged_and_cells_do_not_mix():
    rng = np.random.default_rng(9)
    curves, group, planted = [], [], []
    for g in range(2):
        for i in range(120):
            big = i in (7, 63, 99)
            # group 1 is a noisier chip: its ordinary stars must not be judged by group 0's ensemble
            base = 0.01 if g == 0 else 0.03
            curves.append(_star(rng, 80, 15.02 + 0.06 * rng.uniform(), base * (5.0 if big else 1.0)))
            group.append(g)
            if big:
                planted.append(len(curves) - 1)
    curves.append(_star(rng, 80, 19.95, 0.3))          # alone in its magnitude bin: no ensemble, no flag
    group.append(0)
    offs, t, mag, sig = _batch(curves)
    r = V.variability_flags(offs, t, mag, sig, np.array(group), mag_lo=12.0, mag_bin=0.1, n_mag_bins=80)
    assert all(r["flag"][p] == 1 for p in planted)
    assert r["flag"][-1] == 0 and r["kept"][-1] == 1
    assert set(r["cell"][:120]) == {30} and set(r["cell"][120:240]) == {80 + 30}
    # independent restatement per cell with scipy's clip
    for g in range(2):
        idx = np.arange(120) + 120 * g
        kept, _, _ = scipy.stats.sigmaclip(r["rms"][idx], 3.0, 3.0)
        thr = kept.mean() + 2.0 * kept.std()
        assert np.array_equal(r["flag"][idx] == 1, r["rms"][idx] > thr)
        assert r["expected"][idx[0]] == pytest.approx(kept.mean(), rel=1e-12)
    # group 1's ordinary stars (rms 0.03) would all be > 2 sigma outliers of group 0's ensemble (0.01)
    assert r["flag"][120:240].sum() < 15


def test_magnitude_offset_and_group_split_invariance_and_faults():
    rng = np.random.default_rng(11)
    curves = [_star(rng, 60, 16.33 + 0.03 * rng.uniform(), 0.01 * (4.0 if i == 5 else 1.0)) for i in range(40)]
    bad = _star(rng, 60, 16.35, 0.01)
    bad[1][3] = np.nan
    curves.append(bad)
    curves.append((np.zeros(1), np.full(1, 16.3), np.full(1, 0.01)))     # one point: status 1
    offs, t, mag, sig = _batch(curves)
    r0 = V.variability_flags(offs, t, mag, sig, mag_lo=12.0)
    assert r0["flag"][5] == 1 and list(r0["status"][-2:]) == [2, 1] and list(r0["cell"][-2:]) == [-1, -1]
    assert r0["flag"][-2:].sum() == 0
    # magnitudes and mag_lo shifted by the same exactly representable amount: same cells, same flags
    r1 = V.variability_flags(offs, t, mag - np.float32(2.0), sig, mag_lo=10.0)
    assert np.array_equal(r1["flag"], r0["flag"]) and np.array_equal(r1["cell"], r0["cell"])
    # out of the magnitude range: no cell
    r2 = V.variability_flags(offs, t, mag, sig, mag_lo=17.0)
    assert (r2["cell"] == -1).all() and r2["flag"].sum() == 0
    # fewer than min_members kept: no flag
    r3 = V.variability_flags(offs, t, mag, sig, mag_lo=12.0, min_members=100)
    assert r3["flag"].sum() == 0
