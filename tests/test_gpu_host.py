"""-m gpu: bls_search_host -- the call bench.py's `e2e` figure times -- against the ORACLE (not against bls_run):
host buffers in pageable and in pinned memory, t_origin / status left NULL, an empty batch, curves with data
faults.  Peak lists are compared by reading R14 on the oracle's spectrum, ties proven from member sets
(tests/comparator.py); SR of each reported peak against the oracle's at that frequency within 1e-4."""
import ctypes as C

import numpy as np
import pytest

import oracle
import synth
from comparator import compare_peaks, exact_tie_runs

pytestmark = pytest.mark.gpu


def _plan(bls, grid, freqs, k):
    return bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k)


def _check_against_oracle(batch, grid, freqs, kmin, kmax, peaks, status, k, origin, faulty=()):
    orcs, _ = oracle.spectrum_batch(batch.offsets, batch.t, batch.mag, batch.sigma, freqs, grid.nb, kmin, kmax)
    for c in range(batch.n_curves):
        pk = peaks[c]
        if c in faulty:
            assert status[c] != 0 and (pk["freq_index"] == -1).all()
            continue
        assert status is None or status[c] == 0
        t, _, _ = batch.curve(c)
        _, o_sr, o_a, o_k, o_dp = orcs[c]
        if np.array_equal(oracle.peaks(o_sr, k), pk["freq_index"]):
            compare_peaks(o_sr, pk["freq_index"], pk["sr"], k, label="host curve %d" % c)
        else:
            ties, _ = exact_tie_runs(t, freqs, grid.nb, o_sr, o_a, o_k)
            compare_peaks(o_sr, pk["freq_index"], pk["sr"], k, label="host curve %d" % c, ties=ties)
        for p in pk:
            q = int(p["freq_index"])
            if q < 0:
                continue
            assert abs(p["sr"] - o_sr[q]) <= 1e-4 * o_sr[q] + 1e-12
            assert p["freq"] == freqs[q]
            mid = (p["start_bin"] + 0.5 * p["width_bins"]) / grid.nb
            assert p["epoch"] == pytest.approx((origin[c] if origin is not None else 0.0) + mid / freqs[q], abs=1e-6)


@pytest.mark.parametrize("pinned", [False, True])
def test_search_host_matches_the_oracle_from_pageable_and_pinned_buffers(pinned):
    import torch
    import paper_1112_1701_b200 as bls
    cfg = synth.config("T0")
    batch, grid, k = synth.make_batch(cfg), cfg["grid"], cfg["top_k"]
    freqs = synth.freq_grid(grid)
    arrs = [batch.offsets.astype(np.int64), batch.t, batch.mag, batch.sigma, np.asarray(batch.t_origin, dtype=np.float64)]
    if pinned:
        keep = [torch.from_numpy(np.ascontiguousarray(a)).pin_memory() for a in arrs]
        assert all(x.is_pinned() for x in keep)
        arrs = [x.numpy() for x in keep]
    with _plan(bls, grid, freqs, k) as plan:
        peaks, status = plan.search_host(arrs[0], arrs[1], arrs[2], arrs[3], arrs[4], k=k)
        again, _ = plan.search_host(arrs[0], arrs[1], arrs[2], arrs[3], arrs[4], k=k)      # staging buffers reused
        kmin, kmax = plan.kmin, plan.kmax
    assert peaks.tobytes() == again.tobytes()
    assert (status == 0).all() and (peaks["freq_index"][:, 0] >= 0).all()
    _check_against_oracle(batch, grid, freqs, kmin, kmax, peaks, status, k, batch.t_origin)


def test_search_host_with_null_origin_and_null_status_and_faulty_curves():
    import paper_1112_1701_b200 as bls
    B = bls.binding
    cfg = synth.config("T1")
    batch, grid, k = synth.make_batch(cfg), cfg["grid"], 3
    freqs = synth.freq_grid(grid)
    mag, sig = batch.mag.copy(), batch.sigma.copy()
    mag[batch.offsets[1] + 5] = np.inf           # curve 1: non-finite
    sig[batch.offsets[3] + 2] = -1.0             # curve 3: bad sigma
    batch.mag, batch.sigma = mag, sig
    nc = batch.n_curves
    with _plan(bls, grid, freqs, k) as plan:
        kmin, kmax = plan.kmin, plan.kmax
        peaks = np.zeros((nc, k), dtype=bls.PEAK_DTYPE)
        offs = np.ascontiguousarray(batch.offsets, dtype=np.int64)
        b = B.BlsBatch(nc, offs.ctypes.data, batch.t.ctypes.data, mag.ctypes.data, sig.ctypes.data, None)   # t_origin NULL
        rc = bls.lib().bls_search_host(plan._h, C.byref(b), k, C.c_void_p(peaks.ctypes.data), None)          # status NULL
        assert rc == bls.BLS_OK
        # with status: the faults are reported per curve, the call still succeeds
        p2, status = plan.search_host(offs, batch.t, mag, sig, None, k=k)
    assert peaks.tobytes() == p2.tobytes()
    assert list(status) == [0, 2, 0, 3, 0]
    _check_against_oracle(batch, grid, freqs, kmin, kmax, peaks, status, k, None, faulty=(1, 3))


def test_search_host_empty_batch_and_argument_errors():
    import paper_1112_1701_b200 as bls
    B = bls.binding
    cfg = synth.config("T0")
    grid = cfg["grid"]
    freqs = synth.freq_grid(grid)
    z = np.zeros(0, dtype=np.float32)
    with _plan(bls, grid, freqs, 5) as plan:
        peaks, status = plan.search_host(np.zeros(1, dtype=np.int64), z, z, z, None, k=5)
        assert peaks.shape == (0, 5) and status.shape == (0,)
        # a batch of curves that are all empty: every curve "too few points", no peaks
        peaks, status = plan.search_host(np.zeros(4, dtype=np.int64), z, z, z, None, k=2)
        assert list(status) == [1, 1, 1] and (peaks["freq_index"] == -1).all()
        out = np.zeros((1, 5), dtype=bls.PEAK_DTYPE)
        offs = np.array([0, 3], dtype=np.int64)
        t3 = np.array([0.0, 1.0, 2.0], dtype=np.float32)
        b = B.BlsBatch(1, offs.ctypes.data, t3.ctypes.data, t3.ctypes.data, None, None)                    # sigma NULL
        assert bls.lib().bls_search_host(plan._h, C.byref(b), 5, C.c_void_p(out.ctypes.data), None) == bls.BLS_ERR_NULL
        b = B.BlsBatch(1, offs.ctypes.data, t3.ctypes.data, t3.ctypes.data, t3.ctypes.data, None)
        assert bls.lib().bls_search_host(plan._h, C.byref(b), 6, C.c_void_p(out.ctypes.data), None) == bls.BLS_ERR_ARG
        assert bls.lib().bls_search_host(plan._h, C.byref(b), 5, None, None) == bls.BLS_ERR_NULL
        b = B.BlsBatch(-1, offs.ctypes.data, t3.ctypes.data, t3.ctypes.data, t3.ctypes.data, None)
        assert bls.lib().bls_search_host(plan._h, C.byref(b), 5, C.c_void_p(out.ctypes.data), None) == bls.BLS_ERR_BATCH
