"""-m gpu: bls_variability_noalloc, the variability pre-filter (f3, section 2.2.1) for programs that
may not allocate GPU memory at the point where they call it: a stage inside a process whose own pool already
holds all free device memory (a fresh cudaMalloc fails there), a per-exposure loop with a latency bound
(cudaMalloc / cudaFree can stall the whole device), or a plug-in that must leave its host application's memory
alone.  Its working memory is a fixed array built into libbls_b200.so, shared by every call on the GPU, so what
has to be shown is that (1) it gives what bls_variability gives, and (2) a second call is not disturbed by what
the first one left behind in that array.

The file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure and a
failure here must not hide the parity tests.  It passes alone in a fresh process (where its first call is the
one that looks up the array's address on the GPU) and after the rest of the suite."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

NAMES = ("status", "mean_mag", "rms", "cell", "expected", "scatter", "kept", "flag")


def _stars(n_stars, n_groups, seed, m_lo, m_hi):
    """Seeded ensemble in CSR form: ragged lengths, magnitude-dependent noise, a few planted variables, two data
    faults.  No BLS or filter arithmetic here: only inputs."""
    rng = np.random.default_rng(seed)
    n = rng.integers(20, 200, n_stars)
    offs = np.zeros(n_stars + 1, dtype=np.int64)
    offs[1:] = np.cumsum(n)
    t = np.concatenate([np.sort(rng.uniform(0.0, 90.0, k)) for k in n]).astype(np.float32)
    m0 = rng.uniform(m_lo, m_hi, n_stars)
    floor = 0.004 * 10 ** (0.25 * (m0 - 14.0))
    boost = np.where(rng.uniform(size=n_stars) < 0.04, rng.uniform(2, 10, n_stars), 1.0)
    mag = np.concatenate([m0[c] + rng.normal(0.0, floor[c] * boost[c], n[c]) for c in range(n_stars)]).astype(np.float32)
    sig = np.repeat(floor, n).astype(np.float32)
    mag[offs[7] + 2] = np.nan
    sig[offs[11]] = 0.0
    group = rng.integers(0, n_groups, n_stars).astype(np.int32)
    return offs, t, mag, sig, group


def _both(case, kw):
    """The allocating path and the no-allocation path on the same device inputs -> two dicts of numpy arrays."""
    import torch
    import paper_1112_1701_b200 as bls
    offs, t, mag, sig, group = case
    dev = torch.device("cuda", 0)
    d = [torch.from_numpy(x).to(dev) for x in (t, mag, sig, group)]
    ref = bls.variability(offs, d[0], d[1], d[2], d[3], **kw)
    torch.cuda.synchronize()
    got = bls.variability_noalloc(offs, d[0], d[1], d[2], d[3], **kw)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in ref.items()}, {k: v.cpu().numpy() for k, v in got.items()}


def _same(ref, got):
    # integer decisions identical; fp64 statistics within the tolerances tests/test_gpu_variability.py uses
    # against the oracle (the two paths run the same kernels, so in practice they are equal to the last bit)
    for k in ("status", "cell", "kept", "flag"):
        assert np.array_equal(ref[k], got[k]), k
    np.testing.assert_allclose(got["mean_mag"], ref["mean_mag"], rtol=1e-13)
    np.testing.assert_allclose(got["rms"], ref["rms"], rtol=1e-11, atol=1e-300)
    np.testing.assert_allclose(got["expected"], ref["expected"], rtol=1e-11)
    np.testing.assert_allclose(got["scatter"], ref["scatter"], rtol=1e-9, atol=1e-18)


def test_two_calls_in_a_row_match_the_allocating_path():
    # First call: many stars, many cells in use.  Second call: fewer stars in OTHER cells of a smaller table, so
    # member counts, cell offsets and clip marks left over from the first call would change its answer if the
    # entry point did not reset what it must.  Then the first case again, to catch the opposite direction.
    big = _stars(6000, n_groups=6, seed=41, m_lo=14.0, m_hi=18.0)
    kw_big = dict(n_groups=6, mag_lo=13.5, mag_bin=0.1, n_mag_bins=50, clip=3.0, nsig=2.0, max_iter=5, min_members=5)
    small = _stars(900, n_groups=2, seed=42, m_lo=15.0, m_hi=16.0)
    kw_small = dict(n_groups=2, mag_lo=14.8, mag_bin=0.1, n_mag_bins=14, clip=2.5, nsig=2.0, max_iter=3, min_members=4)
    ref1, got1 = _both(big, kw_big)
    ref2, got2 = _both(small, kw_small)
    ref3, got3 = _both(big, kw_big)
    _same(ref1, got1)
    _same(ref2, got2)
    _same(ref3, got3)
    for k in NAMES:
        assert np.array_equal(got1[k], got3[k]), k
    # the cases exercise what they claim to
    assert list(got1["status"][[7, 11]]) == [2, 3] and list(got2["status"][[7, 11]]) == [2, 3]
    assert got1["flag"].sum() > 20 and got2["flag"].sum() > 3
    assert len(set(got1["cell"][got1["cell"] >= 0])) > 150 and got2["cell"].max() < 28
    print("\n[no-alloc f3] 6000 / 900 / 6000 stars back to back: identical to bls_variability (%d, %d flagged)"
          % (int(got1["flag"].sum()), int(got2["flag"].sum())))


def test_results_land_in_caller_tensors_and_null_outputs_are_allowed():
    import torch
    import paper_1112_1701_b200 as bls
    case = _stars(500, n_groups=1, seed=43, m_lo=14.0, m_hi=15.0)
    kw = dict(n_groups=1, mag_lo=13.9, mag_bin=0.1, n_mag_bins=12, min_members=5)
    ref, got = _both(case, kw)
    _same(ref, got)
    # steady state: the caller's own output tensors are reused, nothing is made per call
    dev = torch.device("cuda", 0)
    offs, t, mag, sig, group = case
    d = [torch.from_numpy(x).to(dev) for x in (t, mag, sig, group)]
    out = bls.variability_noalloc(offs, d[0], d[1], d[2], d[3], **kw)
    ptrs = {k: v.data_ptr() for k, v in out.items()}
    for v in out.values():
        v.fill_(-3)
    again = bls.variability_noalloc(offs, d[0], d[1], d[2], d[3], out=out, **kw)
    torch.cuda.synchronize()
    assert {k: v.data_ptr() for k, v in again.items()} == ptrs
    _same(ref, {k: v.cpu().numpy() for k, v in again.items()})
    # only the flag wanted: status, cell, mean and rms then live in the built-in array
    import ctypes as C
    B = bls.binding
    flag = torch.full((500,), -3, dtype=torch.int32, device=dev)
    cfg = B.BlsVariabilityConfig(C.sizeof(B.BlsVariabilityConfig), 1, 13.9, 0.1, 12, 5, 3.0, 2.0, 5, 0)
    b = B.BlsBatch(500, offs.ctypes.data, d[0].data_ptr(), d[1].data_ptr(), d[2].data_ptr(), None)
    o = B.BlsVariabilityOutputs(None, None, None, None, None, None, None, flag.data_ptr())
    rc = bls.lib().bls_variability_noalloc(0, C.byref(cfg), C.byref(b), None, C.byref(o),
                                           C.c_void_p(torch.cuda.current_stream(dev).cuda_stream))
    torch.cuda.synchronize()
    assert rc == bls.BLS_OK
    ref1 = bls.variability(offs, d[0], d[1], d[2], None, **kw)
    torch.cuda.synchronize()
    assert np.array_equal(flag.cpu().numpy(), ref1["flag"].cpu().numpy())


def test_sizes_beyond_the_built_in_array_are_refused():
    import torch
    import paper_1112_1701_b200 as bls
    B = bls.binding
    z = torch.zeros(4, dtype=torch.float32, device="cuda")
    # too many stars (the offsets are not even walked: the check comes first)
    offs = np.zeros(B.NOALLOC_MAX_STARS + 2, dtype=np.int64)
    with pytest.raises(bls.BlsError) as ei:
        bls.variability_noalloc(offs, z, z, z, n_groups=1, n_mag_bins=10,
                                out={k: torch.zeros(offs.size, dtype=torch.float64 if k in ("mean_mag", "rms", "expected", "scatter")
                                                    else torch.int32, device="cuda") for k in NAMES})
    assert ei.value.code == bls.BLS_ERR_CAPACITY and "bls_variability" in str(ei.value)
    # too many cells
    with pytest.raises(bls.BlsError) as ei:
        bls.variability_noalloc(np.array([0, 2, 4], dtype=np.int64), z, z, z + 1, n_groups=B.NOALLOC_MAX_CELLS // 64 + 1, n_mag_bins=64)
    assert ei.value.code == bls.BLS_ERR_CAPACITY
    # exactly at both limits is accepted
    n = B.NOALLOC_MAX_STARS
    offs = np.arange(n + 1, dtype=np.int64) * 2
    rng = np.random.default_rng(5)
    t = torch.from_numpy(np.tile(np.array([0.0, 1.0], np.float32), n)).cuda()
    mag = torch.from_numpy((14.0 + 2.0 * np.repeat(rng.uniform(size=n), 2) + rng.normal(0, 0.01, 2 * n)).astype(np.float32)).cuda()
    sig = torch.full((2 * n,), 0.01, dtype=torch.float32, device="cuda")
    group = torch.from_numpy((np.arange(n) % 64).astype(np.int32)).cuda()
    kw = dict(n_groups=64, mag_lo=14.0, mag_bin=2.0 / 64, n_mag_bins=B.NOALLOC_MAX_CELLS // 64, min_members=2)
    got = bls.variability_noalloc(offs, t, mag, sig, group, **kw)
    ref = bls.variability(offs, t, mag, sig, group, **kw)
    torch.cuda.synchronize()
    _same({k: v.cpu().numpy() for k, v in ref.items()}, {k: v.cpu().numpy() for k, v in got.items()})
