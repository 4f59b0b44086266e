"""Pins of the f1 oracle functions (oracle/bls_oracle.c: oracle_sde, oracle_bin_shift, oracle_refine_spectrum,
oracle_refine_pick; readings S1-S4).  CPU only.  Hand-written spectra for the SDE; exact rational arithmetic
for the shifted bin rule; a noiseless injected box whose frequency lies BETWEEN coarse grid points and whose
edges lie a quarter bin off the bin grid, recovered to the fine step and the right shift with closed-form SR
and depth; brute force over boxes (explicit least squares on shifted member sets)."""
from fractions import Fraction

import numpy as np
import pytest

import oracle


def test_sde_hand_written_spectra():
    # mean 2, population sd sqrt(3): (5 - 2)/sqrt(3) = sqrt(3); (1 - 2)/sqrt(3)
    assert oracle.sde([1.0, 1.0, 1.0, 5.0], 3) == pytest.approx(np.sqrt(3.0), rel=1e-15)
    assert oracle.sde([1.0, 1.0, 1.0, 5.0], 0) == pytest.approx(-1.0 / np.sqrt(3.0), rel=1e-15)
    assert oracle.sde([2.0, 2.0, 2.0], 1) == 0.0                      # flat spectrum: sd = 0 -> 0
    sr = np.array([0.5, 4.0, 1.5, 2.0, 0.25, 3.75])
    for q in range(6):
        assert oracle.sde(sr, q) == pytest.approx((sr[q] - sr.mean()) / sr.std(), rel=1e-14)   # numpy: population std
    assert oracle.sde(10 * sr + 3, 1) == pytest.approx(oracle.sde(sr, 1), rel=1e-13)         # affine invariance


def _exact_bin(f, t, nb, shift):
    """The rule S3 in exact arithmetic on the ROUNDED intermediate values the rule prescribes."""
    p = float(Fraction(f) * Fraction(t))                  # RN(f t): Fraction -> float rounds to nearest even
    p2 = float(Fraction(p) - Fraction(shift))             # RN(p - shift)
    phi = Fraction(p2) - (Fraction(p2).numerator // Fraction(p2).denominator)
    xb = float(phi * nb)                                  # RN(phi nb)
    b = int(xb)
    return min(b, nb - 1)


def test_shifted_bin_rule_matches_exact_arithmetic():
    rng = np.random.default_rng(12)
    for nb, n_shift in ((64, 4), (200, 4), (400, 3), (100, 8)):
        for _ in range(3000):
            f = float(rng.uniform(0.03, 5.0))
            t = float(np.float32(rng.uniform(-5.0, 480.0)))
            h = int(rng.integers(0, n_shift))
            shift = h / (n_shift * nb)
            assert oracle.bin_index_shift(f, t, nb, shift) == _exact_bin(f, t, nb, shift)
    # shift 0 is the plain rule; edge cases: t = 0 with a shift lands in the LAST bin (phase -s wraps to 1 - s)
    assert oracle.bin_index_shift(1.7, 0.0, 50, 0.0) == oracle.bin_index(1.7, 0.0, 50) == 0
    assert oracle.bin_index_shift(1.7, 0.0, 50, 1.0 / 200) == 49
    assert oracle.bin_index_shift(2.0, 0.25, 10, 0.05) == 4            # phase 0.5 - 0.05 = 0.45 -> bin 4
    assert oracle.bin_index_shift(2.0, 0.25, 10, 0.0) == 5


def _noiseless(n, T, f_true, nb, a_true, k_true, frac_shift, delta):
    """n evenly spread epochs over T days; magnitude base + delta inside the box of true phases
    [(a + frac_shift)/nb, (a + frac_shift + k)/nb) at frequency f_true."""
    t = ((np.arange(n) + 0.5) * (T / n)).astype(np.float32)
    ph = (f_true * t.astype(np.float64)) % 1.0
    lo = (a_true + frac_shift) / nb
    inside = ((ph - lo) % 1.0) < k_true / nb
    mag = np.where(inside, 16.0 + delta, 16.0).astype(np.float32)
    return t, mag, np.full(n, 0.01, dtype=np.float32), inside


def test_noiseless_box_between_grid_points_is_recovered_to_the_fine_step_and_shift():
    nb, kmin, kmax = 50, 1, 8
    coarse = np.array([1.9, 2.0, 2.1])                    # df * T = 2 cycles: the coarse grid smears the box
    n_fine, n_shift = 101, 4
    f_lo, f_hi = oracle.refine_bounds(coarse, 1)
    assert (f_lo, f_hi) == (1.9, 2.1)
    step = (f_hi - f_lo) / (n_fine - 1)
    j_true, h_true, a_true, k_true, delta = 69, 1, 17, 5, 0.0625
    f_true = f_lo + j_true * step                         # 2.038: between the coarse points
    t, mag, sig, inside = _noiseless(4000, 20.0, f_true, nb, a_true, k_true, h_true / n_shift, delta)
    st, fr, sr, a, k, dp = oracle.refine_spectrum(t, mag, sig, f_lo, f_hi, n_fine, n_shift, nb, kmin, kmax)
    assert st == 0 and fr[j_true * n_shift] == f_true
    best = oracle.refine_pick(sr)
    assert best == j_true * n_shift + h_true              # recovered to the fine step AND the quarter-bin shift
    r = inside.mean()
    assert sr[best] == pytest.approx(r * (1 - r) * delta ** 2, rel=1e-9)      # closed form r(1-r) delta^2
    assert dp[best] == pytest.approx(delta, rel=1e-9)
    assert (a[best], k[best]) == (a_true, k_true)
    # without the shift the box straddles bin edges: strictly worse; the coarse frequencies are far worse
    assert sr[j_true * n_shift + 0] < sr[best] * (1 - 1e-3)
    _, c_sr, _, _, _ = oracle.spectrum(t, mag, sig, coarse, nb, kmin, kmax)
    assert c_sr.max() < 0.5 * sr[best]
    # epoch of the refined box (S4): mid-phase (a + k/2)/nb + s_h at f_true is the middle of the injected box
    mid = (a[best] + 0.5 * k[best]) / nb + h_true / (n_shift * nb)
    assert mid == pytest.approx((a_true + h_true / n_shift + 0.5 * k_true) / nb, abs=1e-15)


def test_refine_entries_match_bruteforce_over_boxes_on_shifted_member_sets():
    rng = np.random.default_rng(4)
    n, nb, kmin, kmax, n_fine, n_shift = 60, 12, 1, 4, 3, 3
    t = np.sort(rng.uniform(0, 9, n)).astype(np.float32)
    mag = (15 + rng.normal(0, 0.02, n)).astype(np.float32)
    sig = rng.uniform(0.01, 0.03, n).astype(np.float32)
    st, fr, sr, a, k, dp = oracle.refine_spectrum(t, mag, sig, 0.7, 0.9, n_fine, n_shift, nb, kmin, kmax)
    _, w, x = oracle.prepare(t, mag, sig)
    for q in range(n_fine * n_shift):
        j, h = divmod(q, n_shift)
        f = 0.7 + j * ((0.9 - 0.7) / (n_fine - 1))
        assert fr[q] == f
        bins = np.array([_exact_bin(f, float(ti), nb, h / (n_shift * nb)) for ti in t])
        best = (0.0, 0, kmin)
        for aa in range(nb):
            for kk in range(kmin, kmax + 1):
                inside = ((bins - aa) % nb) < kk
                if not inside.any() or inside.all():
                    continue
                # explicit weighted least squares of a two-level model: residual D; SR = sum w x^2 - D
                A = np.stack([inside.astype(float), (~inside).astype(float)], axis=1) * np.sqrt(w)[:, None]
                coef, res, _, _ = np.linalg.lstsq(A, x * np.sqrt(w), rcond=None)
                v = float(np.sum(w * x * x) - np.sum((A @ coef - x * np.sqrt(w)) ** 2))
                if v > best[0] * (1 + 1e-12):
                    best = (v, aa, kk)
        assert sr[q] == pytest.approx(best[0], rel=1e-9)
    assert oracle.refine_pick(sr) == int(np.argmax(sr))
    assert oracle.refine_pick(np.zeros(5)) == -1
    assert oracle.refine_pick(np.array([1.0, 3.0, 3.0, 2.0])) == 1       # ties: smallest index
