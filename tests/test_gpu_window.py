"""-m gpu: bls_detection_efficiency (f4; Fig. 13) through the C ABI against oracle.detection_efficiency
on the same cadences: the synthetic survey cadences of configs C1 (PTF-like, weather gaps), C3 (two seasons) and C4
(nightly windows), ragged lengths incl. an empty and a one-epoch cadence.  The counts are integers decided by
identically rounded fp64 operations on both sides: they must be IDENTICAL."""
import numpy as np
import pytest

import oracle
import synth

pytestmark = pytest.mark.gpu


def _run(offs, t, freqs, d, n_phase, min_events=2):
    import torch
    import paper_1112_1701_b200 as bls
    cnt, eff = bls.detection_efficiency(offs, torch.from_numpy(t).cuda(), freqs, d, n_phase, min_events)
    torch.cuda.synchronize()
    return cnt.cpu().numpy(), eff.cpu().numpy()


def test_survey_cadences_match_the_oracle_exactly():
    curves = []
    for name, ids in (("C1", (0, 1, 2)), ("C3", (0,)), ("C4", (0, 1, 2, 3)), ("C2", (5, 6))):
        cfg = synth.config(name)
        for c in ids:
            curves.append(synth.make_curve(cfg, c)[0])
    curves.append(np.zeros(0, np.float32))
    curves.append(np.array([3.25], np.float32))
    offs = np.zeros(len(curves) + 1, dtype=np.int64)
    offs[1:] = np.cumsum([len(c) for c in curves])
    t = np.concatenate(curves).astype(np.float32)
    periods = np.concatenate([np.linspace(0.2, 3.0, 141), [0.5, 1.0, 1.5, 2.0, 5.0, 10.0]])
    freqs = 1.0 / periods
    for d, n_phase, me in ((0.02, 500, 2), (0.1, 333, 2), (0.05, 64, 3), (0.03, 1000, 1)):
        cnt, eff = _run(offs, t, freqs, d, n_phase, me)
        for c in range(len(curves)):
            oc, oe = oracle.detection_efficiency(curves[c], freqs, d, n_phase, me)
            assert np.array_equal(cnt[c], oc), (c, d, n_phase, np.nonzero(cnt[c] != oc)[0][:5])
            assert np.array_equal(eff[c], oe)
    # Fig. 13: fractional-day periods are detected nearly always, integer-day periods much less often
    cnt, eff = _run(offs, t, freqs, 0.02, 500)
    i1, i037 = len(periods) - 5, int(np.argmin(np.abs(periods - 0.38)))
    assert eff[0][i037] > 0.95 and eff[0][i1] < 0.6
    print("\n[parity f4] %d cadences x %d periods x 4 settings: detected-phase counts identical; C1 cadence: efficiency %.3f at "
          "P = %.2f d, %.3f at P = 1 d" % (len(curves), len(periods), eff[0][i037], periods[i037], eff[0][i1]))


def test_argument_errors():
    import torch
    import paper_1112_1701_b200 as bls
    t = torch.zeros(4, dtype=torch.float32, device="cuda")
    offs = np.array([0, 4], dtype=np.int64)
    for bad in (dict(duration=0.0), dict(duration=0.1, n_phase=0), dict(duration=0.1, min_events=0)):
        with pytest.raises(bls.BlsError) as ei:
            bls.detection_efficiency(offs, t, [1.0], **bad)
        assert ei.value.code == bls.BLS_ERR_ARG
    with pytest.raises(bls.BlsError):
        bls.detection_efficiency(offs, t, [-1.0], 0.1)


def test_either_output_may_be_left_out():
    """count / efficiency NULL = "do not write": the call then keeps that result in its own scratch (and takes no
    scratch for a result the caller does hold).  What is written must equal the both-outputs call."""
    import ctypes as C
    import torch
    import paper_1112_1701_b200 as bls
    B = bls.binding
    cfg = synth.config("C4")
    curves = [synth.make_curve(cfg, c)[0] for c in range(3)]
    offs = np.zeros(4, dtype=np.int64)
    offs[1:] = np.cumsum([len(c) for c in curves])
    t = torch.from_numpy(np.concatenate(curves).astype(np.float32)).cuda()
    freqs = np.ascontiguousarray(1.0 / np.linspace(0.3, 2.5, 37))
    cnt0, eff0 = bls.detection_efficiency(offs, t, freqs, 0.05, 200)
    torch.cuda.synchronize()
    b = B.BlsBatch(3, offs.ctypes.data, t.data_ptr(), None, None, None)
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    cnt = torch.full((3, 37), -1, dtype=torch.int32, device="cuda")
    eff = torch.full((3, 37), -1.0, dtype=torch.float64, device="cuda")
    L = bls.lib()
    assert L.bls_detection_efficiency(0, C.byref(b), 37, C.c_void_p(freqs.ctypes.data), 0.05, 200, 2, C.c_void_p(cnt.data_ptr()), None, st) == 0
    assert L.bls_detection_efficiency(0, C.byref(b), 37, C.c_void_p(freqs.ctypes.data), 0.05, 200, 2, None, C.c_void_p(eff.data_ptr()), st) == 0
    assert L.bls_detection_efficiency(0, C.byref(b), 37, C.c_void_p(freqs.ctypes.data), 0.05, 200, 2, None, None, st) == 0
    torch.cuda.synchronize()
    assert torch.equal(cnt, cnt0) and torch.equal(eff, eff0) and int(cnt0.sum()) > 0
