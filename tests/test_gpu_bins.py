"""-m gpu: the fold's bin rule against the oracle's on very many (f, t) pairs (the
"bin rule" pin: >= 1e9 pairs, zero mismatches).

The kernels take the bin from a fast fixed-point phase (one DFMA with a magic constant) and fall back to the
canonical rule (reading R8; S3 on a shifted grid) only when the fast position lies within G units of 2^-32 bin of
a bin edge: G = nb + 8 on the plain grid, 2 nb + 8 on the shifted grids of bls_refine.  Random pairs almost never
come that close (~1e-7 of them), so two kinds of input are used for each grid:
  * random pairs over the configurations' frequency and time ranges, drawn on the GPU (seeded) for speed;
  * ADVERSARIAL pairs constructed so that the true position is uniform within +-4 G units of a bin edge: a
    quarter to a third of them fall inside the guard band (the fast phase is quantised to 2^-32 cycle = nb units
    of position, so the band holds 3 of the ~9 reachable positions), the rest just outside, which is where a
    guard band too narrow for the fast phase's error shows up as a mismatch.
The oracle side (oracle_bin / oracle_bin_shift over arrays) is split over the host threads."""
from concurrent.futures import ThreadPoolExecutor
import os

import numpy as np
import pytest

import oracle

pytestmark = pytest.mark.gpu

THREADS = max(1, min(16, os.cpu_count() or 1))


def _oracle_bins(f, t, nb, shift=None):
    cuts = np.linspace(0, f.size, THREADS + 1).astype(np.int64)
    one = (lambda a, b: oracle.bins_many(f[a:b], t[a:b], nb)) if shift is None else \
          (lambda a, b: oracle.bins_shift_many(f[a:b], t[a:b], nb, shift))
    with ThreadPoolExecutor(THREADS) as ex:
        return np.concatenate(list(ex.map(lambda i: one(cuts[i], cuts[i + 1]), range(THREADS))))


def _random_pairs(gen, n):
    """f in [1/30, 5] cycles/day (fp64), t an fp32 value in [0, 490) days widened to fp64: the ranges of C1-C4."""
    import torch
    f = torch.rand(n, generator=gen, device="cuda", dtype=torch.float64) * (5.0 - 1.0 / 30.0) + 1.0 / 30.0
    t = (torch.rand(n, generator=gen, device="cuda", dtype=torch.float32) * 490.0).double()
    return f, t


def _adversarial_pairs(rng, n, nb, G, shift=0.0):
    """(f, t) whose phase f t - shift sits d bins from the edge of a random bin j, d uniform in +-4 G * 2^-32.
    f = (whole cycles + (j + d)/nb + shift) / t; the roundings of that expression move the position by about one
    unit of 2^-32 bin, far less than the +-4 G range, so the positions stay (near) uniform over it."""
    t = rng.uniform(1.0, 490.0, n).astype(np.float32).astype(np.float64)
    cycles = np.floor(rng.uniform(0.0, 5.0, n) * t) + 1.0
    j = rng.integers(0, nb, n).astype(np.float64)
    d = rng.uniform(-4.0 * G, 4.0 * G, n) * 2.0 ** -32
    f = (cycles + (j / nb + d / nb) + shift) / t
    return f, t


def test_plain_grid_1e9_random_and_1e7_adversarial_pairs():
    import torch
    import paper_1112_1701_b200 as bls
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1112_1701)
    nbs = (64, 100, 200, 400, 1000)
    batch, n_batches = 50_000_000, 20
    total = n_canon = 0
    for i in range(n_batches):
        nb = nbs[i % len(nbs)]
        f, t = _random_pairs(gen, batch)
        bins, nc = bls.debug_fold_bins(f, t, nb)
        fh, th = f.cpu().numpy(), t.cpu().numpy()
        bad = int((bins.cpu().numpy() != _oracle_bins(fh, th, nb)).sum())
        assert bad == 0, "nb=%d batch %d: %d mismatches" % (nb, i, bad)
        total += batch
        n_canon += nc
        del f, t, bins
    assert total >= 1_000_000_000
    rng = np.random.default_rng(77)
    adv = adv_canon = 0
    for nb in nbs:
        G = nb + 8
        f, t = _adversarial_pairs(rng, 2_000_000, nb, G)
        bins, nc = bls.debug_fold_bins(torch.from_numpy(f).cuda(), torch.from_numpy(t).cuda(), nb)
        bad = int((bins.cpu().numpy() != _oracle_bins(f, t, nb)).sum())
        assert bad == 0, "adversarial nb=%d: %d mismatches" % (nb, bad)
        # the construction does what it says: 3 of the 8 G / nb (about 9) reachable positions are in the guard band
        assert 0.2 < nc / f.size < 0.45, (nb, nc / f.size)
        adv += f.size
        adv_canon += nc
    print("\n[bins] plain grid: %d random pairs (%d in the guard band) + %d adversarial pairs within +-4G of an edge "
          "(%d in the guard band): 0 mismatches" % (total, n_canon, adv, adv_canon))


def test_shifted_grids_of_refine_random_and_adversarial_pairs():
    """The shifted fast path (additive constant kPhaseMagic - shift, G = 2 nb + 8) against oracle_bin_shift for
    n_shift in {2, 3, 4, 8} and every h: 1.7e8 random pairs and 1e7 adversarial ones in all."""
    import torch
    import paper_1112_1701_b200 as bls
    gen = torch.Generator(device="cuda")
    gen.manual_seed(1701_1112)
    rng = np.random.default_rng(78)
    nbs = (64, 100, 200, 400, 1000)
    total = n_canon = adv = adv_canon = 0
    combo = 0
    for n_shift in (2, 3, 4, 8):
        for h in range(n_shift):
            nb = nbs[combo % len(nbs)]
            combo += 1
            shift = h / (n_shift * nb)
            f, t = _random_pairs(gen, 10_000_000)
            bins, nc = bls.debug_fold_bins_shift(f, t, nb, h, n_shift)
            fh, th = f.cpu().numpy(), t.cpu().numpy()
            bad = int((bins.cpu().numpy() != _oracle_bins(fh, th, nb, shift)).sum())
            assert bad == 0, "nb=%d h=%d/%d: %d mismatches" % (nb, h, n_shift, bad)
            total += fh.size
            n_canon += nc
            G = 2 * nb + 8
            f, t = _adversarial_pairs(rng, 600_000, nb, G, shift)
            bins, nc = bls.debug_fold_bins_shift(torch.from_numpy(f).cuda(), torch.from_numpy(t).cuda(), nb, h, n_shift)
            bad = int((bins.cpu().numpy() != _oracle_bins(f, t, nb, shift)).sum())
            assert bad == 0, "adversarial nb=%d h=%d/%d: %d mismatches" % (nb, h, n_shift, bad)
            assert 0.2 < nc / f.size < 0.45, (nb, h, n_shift, nc / f.size)
            adv += f.size
            adv_canon += nc
    assert adv >= 10_000_000
    print("\n[bins] shifted grids: %d random pairs (%d in the guard band) + %d adversarial pairs (%d in the guard band): "
          "0 mismatches" % (total, n_canon, adv, adv_canon))
    # argument checks of the diagnostic
    z = torch.zeros(4, dtype=torch.float64, device="cuda")
    for h, ns in ((2, 2), (-1, 2), (0, 9), (0, 0)):
        with pytest.raises(bls.BlsError) as ei:
            bls.debug_fold_bins_shift(z, z, 100, h, ns)
        assert ei.value.code == bls.BLS_ERR_ARG
