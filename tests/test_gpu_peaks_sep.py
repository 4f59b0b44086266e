"""-m gpu: bls_plan_set_peak_min_sep (reading R14 with the exact greedy minimum separation of SURVEY 8(c) reading 14)
through the C ABI against oracle.peaks_sep.  The selection is index work: for every curve the GPU's list must EQUAL
the oracle's greedy rule applied to the spectrum the GPU itself wrote (the a5 step in isolation, bit-exact), and it
must equal the rule applied to the oracle's own fp64 spectrum wherever the two spectra rank their peaks alike
(they differ only by fp32 rounding of near-equal values; the spectra themselves are compared in
test_gpu_parity.py)."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu


def _run(batch, grid, freqs, k, sep, refine=False):
    import torch
    import paper_1112_1701_b200 as bls
    dev = torch.device("cuda", 0)
    with bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k) as plan:
        plan.set_peak_min_sep(sep)
        nc, nf = batch.n_curves, len(freqs)
        sr = torch.empty((nc, nf), dtype=torch.float32, device=dev)
        plan.run(batch.offsets, torch.from_numpy(batch.t).to(dev), torch.from_numpy(batch.mag).to(dev),
                 torch.from_numpy(batch.sigma).to(dev), batch.t_origin, sr=sr)
        peaks = plan.peaks_to_numpy(plan.topk(k), k)
        ref = plan.refine(k, 9, 2) if refine else None
        return peaks, sr.cpu().numpy(), ref, (plan.kmin, plan.kmax)


@pytest.mark.parametrize("sep", [0, 1, 3, 25, 400])
def test_separated_lists_equal_the_oracles_greedy_rule(sep):
    cfg = synth.config("T0")
    batch, grid, k = synth.make_batch(cfg), cfg["grid"], 5
    freqs = synth.freq_grid(grid)
    peaks, g_sr, _, (kmin, kmax) = _run(batch, grid, freqs, k, sep)
    same_as_fp64 = 0
    for c in range(batch.n_curves):
        got = peaks[c]["freq_index"].astype(np.int64)
        assert np.array_equal(got, oracle.peaks_sep(g_sr[c].astype(np.float64), k, sep)), (c, sep)
        live = got[got >= 0]
        assert all(abs(int(a) - int(b)) > sep for i, a in enumerate(live) for b in live[i + 1:])
        assert np.array_equal(peaks[c]["sr"][got >= 0], g_sr[c][live])
        t, mag, sig = batch.curve(c)
        _, o_sr, _, _, _ = oracle.spectrum(t, mag, sig, freqs, grid.nb, kmin, kmax)
        same_as_fp64 += int(np.array_equal(got, oracle.peaks_sep(o_sr, k, sep)))
    assert same_as_fp64 >= batch.n_curves - 1
    if sep == 400:                                                   # wider than the grid: one peak per curve
        assert (peaks["freq_index"][:, 1:] == -1).all() and (peaks["freq_index"][:, 0] >= 0).all()


def test_c3_shaped_curve_the_five_slots_are_no_longer_sidelobes_of_one_signal():
    """configs[3]'s shape (5,000 epochs over two seasons, 400 bins, a grid so fine that one signal spans tens of
    samples) on a 20,000-frequency window around an injected eclipse: with separation 0 the five best local maxima
    crowd around the strongest signal (SURVEY 8(c) reading 14's probe: here within about 300 steps of a 20,000-step
    window); with a separation of 60 steps every slot is more than 60 steps from the others and the list reaches further, and bls_refine refines exactly that list."""
    cfg = dict(synth.config("C3"))
    truths = ((c, synth.make_curve(cfg, c)[4]) for c in range(3000))                # 1 % of C3's curves carry a signal
    cid = next(c for c, tr in truths if tr is not None and tr["depth"] > 0.04 and tr["P"] < 5.0)
    batch = synth.make_batch(cfg, [cid])
    tr = batch.truth[0]
    g3 = cfg["grid"]
    df = (g3.fmax - g3.fmin) / (g3.nf - 1)                          # C3's own frequency step
    f_sig = 1.0 / tr["P"]
    lo = max(g3.fmin, f_sig - 10000 * df)
    grid = synth.Grid(20000, lo, lo + 19999 * df, g3.nb, g3.qmin, g3.qmax)
    freqs = synth.freq_grid(grid)
    k = 5
    p0, g_sr, _, _ = _run(batch, grid, freqs, k, 0)
    p60, g_sr60, ref, _ = _run(batch, grid, freqs, k, 60, refine=True)
    assert np.array_equal(g_sr, g_sr60)                              # the spectrum does not depend on the setting
    i0 = p0[0]["freq_index"].astype(np.int64)
    i60 = p60[0]["freq_index"].astype(np.int64)
    assert np.array_equal(i0, oracle.peaks_sep(g_sr[0].astype(np.float64), k, 0))
    assert np.array_equal(i60, oracle.peaks_sep(g_sr[0].astype(np.float64), k, 60))
    assert i0[0] == i60[0]                                           # the best peak is the best peak
    span0 = int(i0.max() - i0.min())
    gaps60 = np.diff(np.sort(i60))
    assert (i60 >= 0).all() and gaps60.min() > 60
    # separation 0: all five slots sit on the one signal (a few hundred steps of a 20,000-step window)
    assert span0 <= 0.05 * grid.nf, "separation 0 was expected to crowd the slots around one signal (span %d)" % span0
    assert int(i60.max() - i60.min()) > span0
    assert np.array_equal(ref[0]["freq_index"].astype(np.int64), i60)
    print("\n[peak_min_sep] C3-shaped curve %d: separation 0 -> slots %s (span %d steps); separation 60 -> slots %s"
          % (cid, list(i0), span0, list(i60)))
