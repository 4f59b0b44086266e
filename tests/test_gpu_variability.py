"""-m gpu: bls_variability (f3, section 2.2.1) through the C ABI against oracle/variability.py on
the same seeded inputs: PTF-like ensembles of stars on several "chips" with planted variables, ragged
lengths, data faults, empty cells.  Flags, cells, kept counts and statuses must be identical; the fp64
statistics agree to rounding (different summation order)."""
import numpy as np
import pytest

import synth
from oracle import variability as V

pytestmark = pytest.mark.gpu


def _ensemble(n_stars, seed, n_groups):
    """C1-like cadence; per-star noise set by a magnitude-dependent floor (brighter = quieter)
    with chip-to-chip differences; 3 % of the stars vary with an extra 2-10 x RMS."""
    rng = np.random.default_rng(seed)
    cfg = dict(synth.config("C1"))
    curves, group = [], []
    for c in range(n_stars):
        t, mag, sig, _, _ = synth.make_curve(cfg, 5000 + c)
        n = int(rng.integers(60, 400))
        t, sig = t[:n], sig[:n]
        g = int(rng.integers(0, n_groups))
        m0 = rng.uniform(14.0, 17.0)
        floor = 0.004 * (1 + 0.5 * g) * 10 ** (0.25 * (m0 - 14.0))
        boost = rng.uniform(2, 10) if rng.uniform() < 0.03 else 1.0
        mag = m0 + rng.normal(0, floor * boost, n)
        curves.append((t, mag.astype(np.float32), np.full(n, floor, dtype=np.float32)))
        group.append(g)
    return curves, np.array(group, dtype=np.int32)


def _csr(curves):
    offs = np.zeros(len(curves) + 1, dtype=np.int64)
    for i, c in enumerate(curves):
        offs[i + 1] = offs[i] + len(c[0])
    cat = lambda j: np.concatenate([np.asarray(c[j], dtype=np.float32) for c in curves]) if curves else np.zeros(0, np.float32)
    return offs, cat(0), cat(1), cat(2)


def _run(offs, t, mag, sig, group, **kw):
    import torch
    import paper_1112_1701_b200 as bls
    dev = torch.device("cuda", 0)
    g = None if group is None else torch.from_numpy(group).to(dev)
    r = bls.variability(offs, torch.from_numpy(t).to(dev), torch.from_numpy(mag).to(dev), torch.from_numpy(sig).to(dev), g, **kw)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in r.items()}


def _compare(g, o):
    assert np.array_equal(g["status"], o["status"])
    assert np.array_equal(g["cell"], o["cell"])
    np.testing.assert_allclose(g["mean_mag"], o["mean_mag"], rtol=1e-13)
    np.testing.assert_allclose(g["rms"], o["rms"], rtol=1e-11, atol=1e-300)
    assert np.array_equal(g["kept"], o["kept"])
    np.testing.assert_allclose(g["expected"], o["expected"], rtol=1e-11)
    np.testing.assert_allclose(g["scatter"], o["scatter"], rtol=1e-9, atol=1e-18)
    # the flag is an integer decided by fp64 numbers that agree to ~1e-12: identical unless a star sits on the
    # threshold to that precision (none does in these seeded cases; such a star would be printed here)
    thr = o["expected"] + 2.0 * o["scatter"]
    knife = np.abs(o["rms"] - thr) <= 1e-9 * np.maximum(thr, 1e-300)
    diff = g["flag"] != o["flag"]
    assert not (diff & ~knife).any(), np.nonzero(diff & ~knife)[0]
    assert not diff.any()


def test_ensembles_on_four_chips_match_the_oracle():
    curves, group = _ensemble(1500, seed=3, n_groups=4)
    # data faults and an out-of-range star
    curves[10][1][3] = np.nan
    curves[20][2][0] = 0.0
    curves[30] = (np.zeros(1, np.float32), np.full(1, 15.0, np.float32), np.full(1, 0.01, np.float32))
    curves[40] = (curves[40][0], curves[40][1] + np.float32(9.0), curves[40][2])
    offs, t, mag, sig = _csr(curves)
    kw = dict(n_groups=4, mag_lo=13.5, mag_bin=0.1, n_mag_bins=40, clip=3.0, nsig=2.0, max_iter=5, min_members=5)
    o = V.variability_flags(offs, t, mag, sig, group, **{k: v for k, v in kw.items() if k != "n_groups"})
    g = _run(offs, t, mag, sig, group, **kw)
    _compare(g, o)
    assert list(g["status"][[10, 20, 30]]) == [2, 3, 1] and g["cell"][40] == -1
    assert 20 < g["flag"].sum() < 300 and (g["kept"] >= 5).any()
    print("\n[parity f3] %d stars, %d cells in use, %d flagged: flags, cells, kept counts identical; max rel diff rms %.2g, expected %.2g"
          % (len(group), len(set(o["cell"][o["cell"] >= 0])), int(g["flag"].sum()),
             np.max(np.abs(g["rms"] - o["rms"]) / np.maximum(o["rms"], 1e-300)),
             np.max(np.abs(g["expected"] - o["expected"]) / np.maximum(o["expected"], 1e-300))))


def test_one_group_default_and_bitwise_repeatable():
    curves, _ = _ensemble(700, seed=8, n_groups=1)
    offs, t, mag, sig = _csr(curves)
    kw = dict(mag_lo=13.0, mag_bin=0.1, n_mag_bins=50, clip=2.5, nsig=2.0, max_iter=3, min_members=8)
    o = V.variability_flags(offs, t, mag, sig, None, **kw)
    g1 = _run(offs, t, mag, sig, None, **kw)
    g2 = _run(offs, t, mag, sig, None, **kw)
    _compare(g1, o)
    for k in g1:
        assert np.array_equal(g1[k], g2[k]), k          # stable scatter + fixed-shape reductions


def test_many_stars_and_single_member_cells():
    rng = np.random.default_rng(2)
    n = 5000
    curves = []
    for c in range(n):
        m = int(rng.integers(2, 30))
        curves.append((np.sort(rng.uniform(0, 5, m)), 12.0 + 8.0 * rng.uniform() + rng.normal(0, 0.01 * (1 + 3 * (c % 50 == 0)), m),
                       rng.uniform(0.005, 0.02, m)))
    offs, t, mag, sig = _csr(curves)
    group = (np.arange(n) % 7).astype(np.int32)
    kw = dict(n_groups=7, mag_lo=12.0, mag_bin=0.1, n_mag_bins=80, clip=3.0, nsig=2.0, max_iter=5, min_members=3)
    o = V.variability_flags(offs, t, mag, sig, group, **{k: v for k, v in kw.items() if k != "n_groups"})
    g = _run(offs, t, mag, sig, group, **kw)
    _compare(g, o)


def test_empty_batch_and_bad_config():
    import torch
    import paper_1112_1701_b200 as bls
    z = torch.zeros(0, dtype=torch.float32, device="cuda")
    r = bls.variability(np.zeros(1, dtype=np.int64), z, z, z)
    assert r["flag"].numel() == 0
    with pytest.raises(bls.BlsError) as ei:
        bls.variability(np.zeros(1, dtype=np.int64), z, z, z, mag_bin=0.0)
    assert ei.value.code == bls.BLS_ERR_CONFIG
