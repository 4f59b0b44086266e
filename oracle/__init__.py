"""ctypes loader for the fp64 CPU oracle (oracle/bls_oracle.c) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may
import this package.  Nothing under paper_1112_1701_b200/ imports it, and it imports nothing from
there.  All arithmetic lives in bls_oracle.c; this file only marshals numpy arrays and fans curves
out over host threads (ctypes releases the GIL during a foreign call).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bls_oracle.c")
_LIB = os.path.join(_HERE, "libbls_oracle.so")
_lib = None

_f32p = np.ctypeslib.ndpointer(dtype=np.float32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_i32p = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_i64p = np.ctypeslib.ndpointer(dtype=np.int64, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """Compile bls_oracle.c with gcc (-O2, no FMA contraction).  Returns the .so path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-std=c11", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.oracle_prepare.restype = C.c_int
        L.oracle_prepare.argtypes = [C.c_int64, _f32p, _f32p, _f32p, _f64p, _f64p]
        L.oracle_widths.restype = None
        L.oracle_widths.argtypes = [C.c_int, C.c_double, C.c_double,
                                    C.POINTER(C.c_int), C.POINTER(C.c_int)]
        L.oracle_bin.restype = C.c_int
        L.oracle_bin.argtypes = [C.c_double, C.c_double, C.c_int]
        L.oracle_spectrum.restype = C.c_int
        L.oracle_spectrum.argtypes = [C.c_int64, _f32p, _f32p, _f32p, C.c_int64, _f64p, C.c_int,
                                      C.c_int, C.c_int, _f64p, _i32p, _i32p, _f64p]
        L.oracle_sr_at.restype = C.c_double
        L.oracle_sr_at.argtypes = [C.c_int64, _f32p, _f32p, _f32p, C.c_double, C.c_int, C.c_int,
                                   C.c_int, C.POINTER(C.c_double)]
        L.oracle_fold_bins.restype = C.c_int
        L.oracle_fold_bins.argtypes = [C.c_int64, _f32p, _f32p, _f32p, C.c_double, C.c_int,
                                       _f64p, _f64p]
        L.oracle_peaks.restype = C.c_int
        L.oracle_peaks.argtypes = [C.c_int64, _f64p, C.c_int, _i64p]
        L.oracle_peaks_sep.restype = C.c_int
        L.oracle_peaks_sep.argtypes = [C.c_int64, _f64p, C.c_int, C.c_int64, _i64p]
        L.oracle_bins_many.restype = None
        L.oracle_bins_many.argtypes = [C.c_int64, _f64p, _f64p, C.c_int, _i32p]
        L.oracle_detection_efficiency.restype = None
        L.oracle_detection_efficiency.argtypes = [C.c_int64, _f32p, C.c_int64, _f64p, C.c_double, C.c_int, C.c_int,
                                                  _i32p, _f64p]
        L.oracle_sde.restype = C.c_double
        L.oracle_sde.argtypes = [C.c_int64, _f64p, C.c_int64]
        L.oracle_bin_shift.restype = C.c_int
        L.oracle_bin_shift.argtypes = [C.c_double, C.c_double, C.c_int, C.c_double]
        L.oracle_bins_shift_many.restype = None
        L.oracle_bins_shift_many.argtypes = [C.c_int64, _f64p, _f64p, C.c_int, C.c_double, _i32p]
        L.oracle_refine_spectrum.restype = C.c_int
        L.oracle_refine_spectrum.argtypes = [C.c_int64, _f32p, _f32p, _f32p, C.c_double, C.c_double, C.c_int, C.c_int,
                                             C.c_int, C.c_int, C.c_int, _f64p, _f64p, _i32p, _i32p, _f64p]
        L.oracle_refine_pick.restype = C.c_int64
        L.oracle_refine_pick.argtypes = [C.c_int64, _f64p]
        _lib = L
    return _lib


def _c32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def prepare(t, mag, sigma) -> Tuple[int, np.ndarray, np.ndarray]:
    t, mag, sigma = _c32(t), _c32(mag), _c32(sigma)
    w = np.zeros(max(t.size, 1)); x = np.zeros(max(t.size, 1))
    st = lib().oracle_prepare(t.size, t, mag, sigma, w, x)
    return st, w[:t.size], x[:t.size]


def widths(nb: int, q_min: float, q_max: float) -> Tuple[int, int]:
    lo, hi = C.c_int(), C.c_int()
    lib().oracle_widths(nb, q_min, q_max, C.byref(lo), C.byref(hi))
    return lo.value, hi.value


def bin_index(f: float, t: float, nb: int) -> int:
    return lib().oracle_bin(float(f), float(t), int(nb))


def bins_many(f, t, nb: int) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.float64); t = np.ascontiguousarray(t, dtype=np.float64)
    out = np.zeros(f.size, dtype=np.int32)
    lib().oracle_bins_many(f.size, f, t, int(nb), out)
    return out


def fold_bins(t, mag, sigma, f: float, nb: int):
    t, mag, sigma = _c32(t), _c32(mag), _c32(sigma)
    W = np.zeros(nb); Y = np.zeros(nb)
    st = lib().oracle_fold_bins(t.size, t, mag, sigma, float(f), nb, W, Y)
    return st, W, Y


def spectrum(t, mag, sigma, freqs, nb: int, kmin: int, kmax: int):
    """One curve -> (status, sr[nf] f64, a[nf] i32, k[nf] i32, depth[nf] f64)."""
    t, mag, sigma = _c32(t), _c32(mag), _c32(sigma)
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    nf = freqs.size
    sr = np.zeros(nf); dp = np.zeros(nf)
    a = np.zeros(nf, dtype=np.int32); k = np.zeros(nf, dtype=np.int32)
    st = lib().oracle_spectrum(t.size, t, mag, sigma, nf, freqs, nb, kmin, kmax, sr, a, k, dp)
    return st, sr, a, k, dp


def sr_at(t, mag, sigma, f: float, nb: int, a: int, k: int) -> Tuple[float, float]:
    t, mag, sigma = _c32(t), _c32(mag), _c32(sigma)
    d = C.c_double()
    v = lib().oracle_sr_at(t.size, t, mag, sigma, float(f), nb, int(a), int(k), C.byref(d))
    return v, d.value


def peaks(sr, kpk: int) -> np.ndarray:
    sr = np.ascontiguousarray(sr, dtype=np.float64)
    idx = np.full(kpk, -1, dtype=np.int64)
    lib().oracle_peaks(sr.size, sr, kpk, idx)
    return idx


def peaks_sep(sr, kpk: int, min_sep: int) -> np.ndarray:
    """Reading R14 with the exact greedy minimum separation (oracle_peaks_sep)."""
    sr = np.ascontiguousarray(sr, dtype=np.float64)
    idx = np.full(kpk, -1, dtype=np.int64)
    lib().oracle_peaks_sep(sr.size, sr, kpk, int(min_sep), idx)
    return idx


def sde(sr, q: int) -> float:
    sr = np.ascontiguousarray(sr, dtype=np.float64)
    return lib().oracle_sde(sr.size, sr, int(q))


def bin_index_shift(f: float, t: float, nb: int, shift: float) -> int:
    return lib().oracle_bin_shift(float(f), float(t), int(nb), float(shift))


def bins_shift_many(f, t, nb: int, shift: float) -> np.ndarray:
    f = np.ascontiguousarray(f, dtype=np.float64); t = np.ascontiguousarray(t, dtype=np.float64)
    out = np.zeros(f.size, dtype=np.int32)
    lib().oracle_bins_shift_many(f.size, f, t, int(nb), float(shift), out)
    return out


def refine_spectrum(t, mag, sigma, f_lo: float, f_hi: float, n_fine: int, n_shift: int, nb: int, kmin: int, kmax: int):
    """Fine spectrum around one peak -> (status, freq[m], sr[m], a[m], k[m], depth[m]), m = n_fine*n_shift,
    entry (j, h) at j*n_shift + h."""
    t, mag, sigma = _c32(t), _c32(mag), _c32(sigma)
    m = n_fine * n_shift
    fr = np.zeros(m); sr = np.zeros(m); dp = np.zeros(m)
    a = np.zeros(m, dtype=np.int32); k = np.zeros(m, dtype=np.int32)
    st = lib().oracle_refine_spectrum(t.size, t, mag, sigma, float(f_lo), float(f_hi), int(n_fine), int(n_shift),
                                      int(nb), int(kmin), int(kmax), fr, sr, a, k, dp)
    return st, fr, sr, a, k, dp


def refine_pick(sr) -> int:
    sr = np.ascontiguousarray(sr, dtype=np.float64)
    return int(lib().oracle_refine_pick(sr.size, sr))


def refine_bounds(freqs, q: int):
    """S2: the fine grid of coarse peak q spans its two neighbours on the coarse grid."""
    return float(freqs[max(q - 1, 0)]), float(freqs[min(q + 1, len(freqs) - 1)])


def detection_efficiency(t, freqs, duration: float, n_phase: int, min_events: int = 2):
    """f4 (W1-W4): (count[nf] int32, efficiency[nf] f64) of one cadence t (sorted ascending)."""
    t = _c32(t)
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    cnt = np.zeros(freqs.size, dtype=np.int32); eff = np.zeros(freqs.size)
    lib().oracle_detection_efficiency(t.size, t, freqs.size, freqs, float(duration), int(n_phase), int(min_events), cnt, eff)
    return cnt, eff


def host_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:  # pragma: no cover
        return os.cpu_count() or 1


def spectrum_batch(offsets, t, mag, sigma, freqs, nb, kmin, kmax,
                   curves: Optional[Sequence[int]] = None, threads: Optional[int] = None):
    """Run `spectrum` over curves of a CSR batch on `threads` host threads (default: all cores).
    Returns (list of per-curve result tuples in the order of `curves`, threads used)."""
    if curves is None:
        curves = range(len(offsets) - 1)
    curves = list(curves)
    threads = threads or host_cores()
    lib()

    def one(c):
        a, b = int(offsets[c]), int(offsets[c + 1])
        return spectrum(t[a:b], mag[a:b], sigma[a:b], freqs, nb, kmin, kmax)

    if threads <= 1 or len(curves) <= 1:
        return [one(c) for c in curves], 1
    used = min(threads, len(curves))
    with ThreadPoolExecutor(max_workers=used) as ex:
        return list(ex.map(one, curves)), used
