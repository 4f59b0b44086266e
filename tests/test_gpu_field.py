"""-m gpu: bls_run_field (f2: field-shared cadence) through the C ABI.  A field is one epoch list and a dense
[stars][epochs] matrix with ABSENT entries (flagged measurements).  By definition each star's result is that of
the BLS search on its present epochs: checked element by element against the fp64 oracle run on exactly those
epochs, and against bls_run on the equivalent CSR batch."""
import numpy as np
import pytest

import oracle
import synth
from comparator import compare_spectrum
from gpu_common import run_gpu
from test_gpu_parity import check_curve_peaks

pytestmark = pytest.mark.gpu


def _field(n_stars, n_epochs, seed):
    rng = np.random.default_rng(seed)
    cfg = dict(synth.config("C1"))
    t = synth.make_curve(cfg, 77)[0][:n_epochs].astype(np.float32)           # one PTF-like cadence for the pointing
    mag = np.zeros((n_stars, n_epochs), dtype=np.float32)
    sig = np.zeros((n_stars, n_epochs), dtype=np.float32)
    for s in range(n_stars):
        star = 0.01 * 10 ** (0.5 * rng.normal())
        sg = star * (1 + 0.25 * np.abs(rng.normal(size=n_epochs)))
        m = rng.uniform(14, 18) + rng.normal(size=n_epochs) * sg
        if s % 3 == 0:                                                         # injected eclipses
            P, d, q = rng.uniform(0.3, 3), rng.uniform(0.03, 0.2), rng.uniform(0.02, 0.08)
            m = m + d * ((((t - rng.uniform(0, P)) / P) % 1.0) < q)
        mag[s], sig[s] = m, sg
    # 2 % of the entries absent, in the three ways the header allows
    drop = rng.uniform(size=mag.shape) < 0.02
    kind = rng.integers(0, 3, size=mag.shape)
    mag[drop & (kind == 0)] = np.nan
    sig[drop & (kind == 1)] = 0.0
    sig[drop & (kind == 2)] = np.inf
    sig[5, 1:] = -1.0                                                          # star 5: one present epoch -> TOO_FEW
    return t, mag, sig


def test_field_matches_the_oracle_on_present_epochs_and_the_csr_path():
    import torch
    import paper_1112_1701_b200 as bls
    n_stars, n_epochs, k = 24, 700, 5
    t, mag, sig = _field(n_stars, n_epochs, seed=17)
    grid = synth.Grid(3000, 0.1, 5.0, 200, 0.005, 0.15)
    freqs = synth.freq_grid(grid)
    dev = torch.device("cuda", 0)
    with bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k) as plan:
        sr = torch.full((n_stars, grid.nf), -1.0, dtype=torch.float32, device=dev)
        a = torch.full((n_stars, grid.nf), -1, dtype=torch.int16, device=dev)
        kk = torch.full((n_stars, grid.nf), -1, dtype=torch.int16, device=dev)
        dp = torch.full((n_stars, grid.nf), -1.0, dtype=torch.float32, device=dev)
        status = torch.full((n_stars,), -7, dtype=torch.int32, device=dev)
        plan.run_field(torch.from_numpy(t).to(dev), torch.from_numpy(mag).to(dev), torch.from_numpy(sig).to(dev), 2455000.5,
                       sr=sr, best_start=a, best_width=kk, depth=dp, status=status)
        peaks = plan.peaks_to_numpy(plan.topk(k), k)
        refined = plan.refine(k, 17, 2)
        kmin, kmax = plan.kmin, plan.kmax
        g_sr, g_dp, st = sr.cpu().numpy(), dp.cpu().numpy(), status.cpu().numpy()
        g_a = a.cpu().numpy().view(np.uint16).astype(np.int32)
        g_k = kk.cpu().numpy().view(np.uint16).astype(np.int32)
    assert st[5] == 1 and (g_sr[5] == 0).all() and (peaks[5]["freq_index"] == -1).all()
    present = np.isfinite(mag) & np.isfinite(sig) & (sig > 0)
    curves, offs = [], [0]
    worst = 0.0
    for s in range(n_stars):
        if s == 5:
            continue
        ok = present[s]
        assert st[s] == 0 and 0.95 * n_epochs < ok.sum() < n_epochs
        ts, ms, ss = t[ok], mag[s][ok], sig[s][ok]
        r = compare_spectrum(ts, ms, ss, freqs, grid.nb, kmin, kmax, g_sr[s], g_a[s], g_k[s], g_dp[s], label="field star %d" % s)
        check_curve_peaks(ts, freqs, grid.nb, r["oracle"], peaks[s], k, g_sr[s], "field star %d" % s)
        worst = max(worst, r["max_rel_err"])
        assert refined[s][0]["freq_index"] == peaks[s][0]["freq_index"] and refined[s][0]["sr"] >= peaks[s][0]["sr"] * (1 - 1e-6)
        assert peaks[s][0]["epoch"] > 2455000.5
        curves.append((ts, ms, ss))
        offs.append(offs[-1] + len(ts))
    # the same stars as a CSR batch through bls_run: same bins, so the same spectra up to the rounding of the prep sums
    cat = lambda j: np.concatenate([c[j] for c in curves]).astype(np.float32)
    b = synth.Batch(offsets=np.array(offs, dtype=np.int64), t=cat(0), mag=cat(1), sigma=cat(2),
                    t_origin=np.full(len(curves), 2455000.5), curve_ids=np.arange(len(curves)))
    g = run_gpu(b, grid, top_k=k, freqs=freqs)
    keep = [s for s in range(n_stars) if s != 5]
    np.testing.assert_allclose(g["sr"], g_sr[keep], rtol=1e-6, atol=0)
    assert (g["a"] == g_a[keep]).mean() > 0.999
    print("\n[parity f2] %d stars x %d shared epochs (2 %% absent), %d frequencies: max SR rel err vs the oracle %.3g; "
          "equal to the CSR path" % (n_stars, n_epochs, grid.nf, worst))


def test_field_faults():
    import torch
    import paper_1112_1701_b200 as bls
    dev = torch.device("cuda", 0)
    t = torch.linspace(0, 30, 50, device=dev)
    mag = 15 + 0.01 * torch.randn(3, 50, device=dev)
    sig = torch.full((3, 50), 0.01, device=dev)
    with bls.Plan(n_bins=32, q_min=0.05, q_max=0.2, freqs=np.linspace(0.2, 2.0, 40), max_top_k=2) as plan:
        status = torch.zeros(3, dtype=torch.int32, device=dev)
        t_bad = t.clone()
        t_bad[7] = float("nan")
        plan.run_field(t_bad, mag, sig, status=status)
        assert status.cpu().tolist() == [2, 2, 2]                 # a non-finite epoch time faults every star
        plan.run_field(t, mag, sig, status=status)
        assert status.cpu().tolist() == [0, 0, 0]
        assert plan.peaks_to_numpy(plan.topk(2), 2).shape == (3, 2)


def _run_field(t, mag, sig, grid, freqs, k, flags=0, scratch_bytes=0, origin=2455000.5):
    import torch
    import paper_1112_1701_b200 as bls
    B = bls.binding
    dev = torch.device("cuda", 0)
    n_stars = mag.shape[0]
    with bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k, flags=flags,
                  scratch_bytes=scratch_bytes) as plan:
        sr = torch.full((n_stars, grid.nf), -1.0, dtype=torch.float32, device=dev)
        a = torch.full((n_stars, grid.nf), -1, dtype=torch.int16, device=dev)
        kk = torch.full((n_stars, grid.nf), -1, dtype=torch.int16, device=dev)
        dp = torch.full((n_stars, grid.nf), -1.0, dtype=torch.float32, device=dev)
        status = torch.full((n_stars,), -7, dtype=torch.int32, device=dev)
        plan.run_field(torch.from_numpy(t).to(dev), torch.from_numpy(mag).to(dev), torch.from_numpy(sig).to(dev), origin,
                       sr=sr, best_start=a, best_width=kk, depth=dp, status=status)
        peaks = plan.peaks_to_numpy(plan.topk(k), k)
        torch.cuda.synchronize()
        return dict(sr=sr.cpu().numpy(), dp=dp.cpu().numpy(), st=status.cpu().numpy(), peaks=peaks,
                    a=a.cpu().numpy().view(np.uint16).astype(np.int32), k=kk.cpu().numpy().view(np.uint16).astype(np.int32),
                    kmin=plan.kmin, kmax=plan.kmax, kernel=plan.query(B.QUERY_SEARCH_KERNEL),
                    launches=plan.query(B.QUERY_LAST_SEARCH_LAUNCHES), n_canon=plan.query(B.QUERY_LAST_CANONICAL))


@pytest.mark.parametrize("n_epochs", [140, 300])
def test_field_kernel_at_the_papers_cadence_matches_the_oracle(n_epochs):
    """The field kernel (kernel 4: three stars per CTA share each epoch's phase and bin index) at the paper's shape:
    140 and 300 epochs per star, 64 bins.  31 stars = 10 groups of three and a last group of
    ONE; 2 % of the entries absent; star 5 has a single present epoch (TOO_FEW) inside a group of healthy stars; the
    cadence's first epoch is t = 0 (the zero-time path).  Every healthy star against the fp64 oracle on its present
    epochs at every frequency, spectra element by element and peak lists by R14; then the same field through the
    per-star kernels (BLS_FLAG_NO_FIELD_KERNEL), through the canonical phase rule, and in chunks that cut groups."""
    import paper_1112_1701_b200 as bls
    n_stars, k = 31, 5
    t, mag, sig = _field(n_stars, n_epochs, seed=100 + n_epochs)
    assert t[0] == 0.0
    grid = synth.Grid(2500, 0.1, 5.0, 64, 0.01, 0.15)
    freqs = synth.freq_grid(grid)
    g = _run_field(t, mag, sig, grid, freqs, k)
    assert g["kernel"] == 4 and g["launches"] == 1
    assert g["st"][5] == 1 and (g["sr"][5] == 0).all() and (g["peaks"][5]["freq_index"] == -1).all()
    present = np.isfinite(mag) & np.isfinite(sig) & (sig > 0)
    worst, near = 0.0, 0
    for s in range(n_stars):
        if s == 5:
            continue
        ok = present[s]
        assert g["st"][s] == 0
        ts, ms, ss = t[ok], mag[s][ok], sig[s][ok]
        r = compare_spectrum(ts, ms, ss, freqs, grid.nb, g["kmin"], g["kmax"], g["sr"][s], g["a"][s], g["k"][s], g["dp"][s],
                             label="field kernel star %d" % s)
        check_curve_peaks(ts, freqs, grid.nb, r["oracle"], g["peaks"][s], k, g["sr"][s], "field kernel star %d" % s)
        worst = max(worst, r["max_rel_err"])
        near += r["box_near_ties"]
    assert near <= max(3, 1e-4 * n_stars * grid.nf)
    # the per-star kernels on the same field: same integer bins, so the same spectra except at near-tied boxes
    h = _run_field(t, mag, sig, grid, freqs, k, flags=bls.BLS_FLAG_NO_FIELD_KERNEL)
    assert h["kernel"] != 4 and np.array_equal(h["st"], g["st"])
    np.testing.assert_allclose(g["sr"], h["sr"], rtol=2e-6, atol=0)
    assert (g["sr"] == h["sr"]).mean() > 0.999 and (g["a"] == h["a"]).mean() > 0.999
    # canonical phase rule for every point-fold: identical bins, identical everything
    c = _run_field(t, mag, sig, grid, freqs, k, flags=bls.BLS_FLAG_CANONICAL_PHASE)
    assert c["kernel"] == 4 and c["n_canon"] >= (n_epochs - 1) * grid.nf * 30
    for key in ("sr", "a", "k", "dp", "st"):
        assert np.array_equal(c[key], g[key]), key
    assert np.array_equal(c["peaks"], g["peaks"])
    # chunks of 7 stars: groups of 3 + 3 + 1 per launch, group borders differ from the one-launch run
    m = _run_field(t, mag, sig, grid, freqs, k, scratch_bytes=7 * grid.nf * 12)
    assert m["kernel"] == 4 and m["launches"] == 5
    for key in ("sr", "a", "k", "dp", "st"):
        assert np.array_equal(m[key], g[key]), key
    assert np.array_equal(m["peaks"], g["peaks"])
    print("\n[parity f2 field kernel] %d stars x %d shared epochs, %d frequencies, 64 bins: max SR rel err vs the oracle %.3g, "
          "%d box near-ties; per-star kernels, canonical rule and chunked launches agree" % (n_stars, n_epochs, grid.nf, worst, near))
