"""-m gpu: bls_refine (f1: SDE + fine re-search with shifted bin grids) through the C ABI against the oracle
(oracle.sde, oracle.refine_spectrum, oracle.refine_pick) on the same seeded inputs."""
import numpy as np
import pytest

import oracle
import synth
from gpu_common import run_gpu

pytestmark = pytest.mark.gpu

TIE_RTOL = 1e-6


def _refine(batch, grid, k, n_fine, n_shift, freqs=None, flags=0):
    import torch
    import paper_1112_1701_b200 as bls
    dev = torch.device("cuda", 0)
    if freqs is None:
        freqs = synth.freq_grid(grid)
    with bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k, flags=flags) as plan:
        nc, nf = batch.n_curves, len(freqs)
        sr = torch.empty((nc, nf), dtype=torch.float32, device=dev)
        plan.run(batch.offsets, torch.from_numpy(batch.t).to(dev), torch.from_numpy(batch.mag).to(dev),
                 torch.from_numpy(batch.sigma).to(dev), batch.t_origin, sr=sr)
        peaks = plan.peaks_to_numpy(plan.topk(k), k)
        ref = plan.refine(k, n_fine, n_shift)
        kmin, kmax = plan.kmin, plan.kmax
        return peaks, ref, sr.cpu().numpy(), freqs, kmin, kmax


def _members(t, f, nb, shift, a, k):
    """Point indices inside box (a, k) of the grid shifted by `shift` cycles, from the oracle's own rule S3."""
    b = np.array([oracle.bin_index_shift(f, float(ti), nb, shift) for ti in t])
    return np.nonzero(((b - int(a)) % nb) < int(k))[0]


def _check(batch, grid, k, n_fine, n_shift, freqs=None, label=""):
    peaks, ref, g_sr, freqs, kmin, kmax = _refine(batch, grid, k, n_fine, n_shift, freqs)
    near = 0
    exact = 0
    worst = 0.0
    for c in range(batch.n_curves):
        t, mag, sig = batch.curve(c)
        _, o_sr, _, _, _ = oracle.spectrum(t, mag, sig, freqs, grid.nb, kmin, kmax)
        for j in range(k):
            p, r = peaks[c][j], ref[c][j]
            assert r["freq_index"] == p["freq_index"]
            if p["freq_index"] < 0:
                assert r["fine_index"] == -1 and r["sr"] == 0
                continue
            q = int(p["freq_index"])
            # S1: SDE of the coarse peak from the coarse spectrum
            assert r["coarse_sr"] == p["sr"]
            assert r["sde"] == pytest.approx(oracle.sde(o_sr, q), rel=1e-4)
            f_lo, f_hi = oracle.refine_bounds(freqs, q)
            st, fr, fsr, fa, fk, fdp = oracle.refine_spectrum(t, mag, sig, f_lo, f_hi, n_fine, n_shift, grid.nb, kmin, kmax)
            best = oracle.refine_pick(fsr)
            gi = int(r["fine_index"]) * n_shift + int(r["shift_index"])
            assert r["freq"] == fr[gi]                                   # the fine frequency, bit for bit
            assert abs(r["sr"] - fsr[gi]) <= 1e-4 * fsr[gi]
            worst = max(worst, abs(r["sr"] - fsr[gi]) / fsr[gi])
            sh = lambda i: (i % n_shift) / (n_shift * grid.nb)
            if gi != best:
                # fine entries whose best boxes hold the SAME points are exact ties (the oracle's fp64 values differ
                # by rounding only): proven from the member sets; anything else must be a near-tie below 1e-6
                m_g = _members(t, fr[gi], grid.nb, sh(gi), fa[gi], fk[gi])
                m_b = _members(t, fr[best], grid.nb, sh(best), fa[best], fk[best])
                if np.array_equal(m_g, m_b):
                    exact += 1
                else:
                    assert (fsr[best] - fsr[gi]) <= TIE_RTOL * fsr[best], (label, c, j, gi, best, fsr[gi], fsr[best])
                    near += 1
            if (int(r["start_bin"]), int(r["width_bins"])) != (int(fa[gi]), int(fk[gi])):
                # another box at the same fine entry: score it from its member set (least-squares identity)
                _, w, x = oracle.prepare(t, mag, sig)
                m = _members(t, fr[gi], grid.nb, sh(gi), r["start_bin"], r["width_bins"])
                rr, ss = w[m].sum(), (w[m] * x[m]).sum()
                assert ss * ss / (rr * (1 - rr)) >= fsr[gi] * (1 - TIE_RTOL)
                near += 1
            else:
                assert r["depth"] == pytest.approx(fdp[gi], rel=1e-4)
            assert r["sr"] >= p["sr"] * (1 - 1e-6) or n_fine < 3      # the coarse frequency is on the fine grid (odd n_fine)
            assert r["period"] == pytest.approx(1.0 / r["freq"], rel=1e-15)
            mid = (r["start_bin"] + 0.5 * r["width_bins"]) / grid.nb + r["shift_index"] / (n_shift * grid.nb)
            assert r["epoch"] == pytest.approx(batch.t_origin[c] + mid / r["freq"], abs=1e-6)
            assert r["duration"] == pytest.approx(r["width_bins"] / grid.nb / r["freq"], rel=1e-12)
    print("\n[parity f1 %s] %d curves x %d peaks x %d fine x %d shifts: max SR rel err %.3g, %d picks explained by a proven "
          "exact tie, %d near-ties" % (label, batch.n_curves, k, n_fine, n_shift, worst, exact, near))
    assert near <= max(2, 0.02 * batch.n_curves * k)
    return peaks, ref


@pytest.mark.parametrize("name,n_fine,n_shift", [("T0", 33, 4), ("T1", 17, 3), ("T2", 9, 2)])
def test_refine_small_configs(name, n_fine, n_shift):
    cfg = synth.config(name)
    _check(synth.make_batch(cfg), cfg["grid"], cfg["top_k"], n_fine, n_shift, label=name)


def test_refine_c1_curves_with_injections():
    cfg = synth.config("C1")
    inj = [c for c in range(300) if synth.make_curve(cfg, c)[4] is not None][:3]
    ids = inj + [1, 2]
    batch = synth.make_batch(cfg, ids)
    peaks, ref = _check(batch, cfg["grid"], 5, 65, 4, label="C1")
    # a deep injected eclipse: the refined period is the injected one (or a harmonic) to the fine step
    for c, cid in enumerate(ids[:len(inj)]):
        tr = batch.truth[c]
        if tr["depth"] > 0.05:
            ratio = ref[c][0]["freq"] * tr["P"]
            assert min(abs(ratio * m - round(ratio * m)) for m in (1, 2, 3, 4)) < 0.01


def test_noiseless_box_between_grid_points_recovered():
    nb = 50
    coarse = np.array([1.9, 2.0, 2.1])
    n_fine, n_shift = 101, 4
    step = (2.1 - 1.9) / (n_fine - 1)
    f_true = 1.9 + 69 * step
    n = 4000
    t = ((np.arange(n) + 0.5) * (20.0 / n)).astype(np.float32)
    ph = (f_true * t.astype(np.float64)) % 1.0
    inside = ((ph - (17 + 0.25) / nb) % 1.0) < 5 / nb
    mag = np.where(inside, 16.0625, 16.0).astype(np.float32)
    b = synth.Batch(offsets=np.array([0, n]), t=t, mag=mag, sigma=np.full(n, 0.01, np.float32), t_origin=np.zeros(1),
                    curve_ids=np.zeros(1))
    grid = synth.Grid(3, 1.9, 2.1, nb, 0.02, 0.16)
    peaks, ref, _, _, _, _ = _refine(b, grid, 1, n_fine, n_shift, freqs=coarse)
    r = ref[0][0]
    assert (r["fine_index"], r["shift_index"], r["start_bin"], r["width_bins"]) == (69, 1, 17, 5)
    assert r["freq"] == f_true and r["depth"] == pytest.approx(0.0625, rel=1e-6)
    rr = inside.mean()
    assert r["sr"] == pytest.approx(rr * (1 - rr) * 0.0625 ** 2, rel=1e-6)
    assert r["sr"] > 2 * r["coarse_sr"]


def test_refine_argument_errors():
    import paper_1112_1701_b200 as bls
    cfg = synth.config("T1")
    batch = synth.make_batch(cfg)
    import torch
    dev = torch.device("cuda", 0)
    with bls.Plan(n_bins=64, q_min=0.02, q_max=0.15, freqs=synth.freq_grid(cfg["grid"]), max_top_k=3) as plan:
        with pytest.raises(bls.BlsError) as ei:
            plan.refine(2)                       # before any run
        assert ei.value.code == bls.BLS_ERR_ARG
        plan.run(batch.offsets, torch.from_numpy(batch.t).to(dev), torch.from_numpy(batch.mag).to(dev),
                 torch.from_numpy(batch.sigma).to(dev), batch.t_origin)
        for bad in (dict(k=4), dict(k=2, n_fine=300), dict(k=2, n_shift=9), dict(k=2, n_fine=0)):
            with pytest.raises(bls.BlsError):
                plan.refine(**bad)
        assert plan.refine(2, 8, 2).shape == (batch.n_curves, 2)


def test_refine_in_several_chunks_is_bitwise_identical_and_leaves_the_run_queries_alone():
    """bls_refine's fine spectrum reuses the plan's spectrum scratch in chunks of curves; with the default 2 GiB
    budget one chunk holds every tested batch, so the loop over chunks (chunk-local rows of the fine spectrum,
    global candidate / output indices) is forced here with a budget of two curves' fine spectra: 6 curves -> 3
    chunks.  Records must equal the one-chunk run bit for bit.  Also: BLS_QUERY_SEARCH_KERNEL / WS_SHAPE /
    TILE_FREQS describe the last bls_run, whatever bls_refine launched after it."""
    import torch
    import paper_1112_1701_b200 as bls
    B = bls.binding
    cfg = synth.config("T0")
    batch, grid = synth.make_batch(cfg), cfg["grid"]
    freqs = synth.freq_grid(grid)
    k, n_fine, n_shift = 3, 16, 2
    dev = torch.device("cuda", 0)
    d = [torch.from_numpy(x).to(dev) for x in (batch.t, batch.mag, batch.sigma)]
    recs, facts = [], []
    for scratch in (0, 2 * k * n_fine * n_shift * 12):
        with bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k, scratch_bytes=scratch) as plan:
            plan.run(batch.offsets, d[0], d[1], d[2], batch.t_origin)
            before = [plan.query(q) for q in (B.QUERY_SEARCH_KERNEL, B.QUERY_WS_SHAPE, B.QUERY_TILE_FREQS)]
            launches = plan.query(B.QUERY_LAST_LAUNCHES)
            recs.append(plan.refine(k, n_fine, n_shift))
            after = [plan.query(q) for q in (B.QUERY_SEARCH_KERNEL, B.QUERY_WS_SHAPE, B.QUERY_TILE_FREQS)]
            assert before == after
            facts.append(plan.query(B.QUERY_LAST_LAUNCHES) - launches)
    assert recs[0].tobytes() == recs[1].tobytes()
    assert (recs[0]["fine_index"] >= 0).sum() >= batch.n_curves            # something was refined
    # one grid kernel + (search + reduce) per chunk: 1 chunk vs 3 chunks
    assert facts == [3, 7], facts
