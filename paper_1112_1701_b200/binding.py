"""ctypes binding of libbls_b200.so (include/bls.h) -- argument marshalling only.

Same names as the C ABI: Plan wraps bls_plan_create / bls_run / bls_topk / bls_search_host /
bls_plan_query / bls_plan_destroy.  PyTorch is used for device memory and the current stream;
every arithmetic step runs in the CUDA kernels.  There is no CPU fallback: if the shared library
is missing or no CUDA device is present, this fails loudly.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbls_b200.so")

EXPORTS = ["bls_plan_create", "bls_run", "bls_topk", "bls_search_host", "bls_plan_destroy",
           "bls_plan_query", "bls_strerror", "bls_plan_last_cuda_error", "bls_debug_fold_bins",
           "bls_variability", "bls_refine", "bls_detection_efficiency", "bls_run_field", "bls_variability_noalloc",
           "bls_debug_fold_bins_shift", "bls_plan_set_peak_min_sep"]

BLS_OK = 0
BLS_ERR_NULL, BLS_ERR_CONFIG, BLS_ERR_BATCH, BLS_ERR_ARG, BLS_ERR_CUDA, BLS_ERR_UNSUPPORTED = -1, -2, -3, -4, -5, -6
BLS_ERR_CAPACITY = -7
NOALLOC_MAX_STARS, NOALLOC_MAX_CELLS = 16384, 4096      # include/bls.h BLS_NOALLOC_MAX_*
BLS_FLAG_NONE, BLS_FLAG_CANONICAL_PHASE, BLS_FLAG_SINGLE_BUFFER, BLS_FLAG_NO_SMALL_CTAS, BLS_FLAG_WARP_PER_TILE = 0, 1, 2, 4, 8
BLS_FLAG_NO_FIELD_KERNEL = 1 << 29


def BLS_FLAG_WARPS(n):
    return (int(n) & 0xff) << 8


def BLS_FLAG_FOLD_WARPS(n):
    return (int(n) & 0xff) << 16


def BLS_FLAG_FOLD_DEPTH(n):
    return (int(n) & 3) << 27


def BLS_FLAG_MERGE_WARPS(n):
    return (int(n) & 7) << 24


def BLS_FLAG_WS_SHAPE(n):
    return (int(n) & 7) << 4
(QUERY_KMIN, QUERY_KMAX, QUERY_NBINS, QUERY_NFREQ, QUERY_SCRATCH_BYTES, QUERY_LAST_LAUNCHES,
 QUERY_LAST_CANONICAL, QUERY_TILE_FREQS, QUERY_SEARCH_CTAS, QUERY_LAST_SEARCH_NS,
 QUERY_SEARCH_KERNEL, QUERY_LAST_SEARCH_LAUNCHES, QUERY_WS_SHAPE) = range(1, 14)


class BlsConfig(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("device", C.c_int32), ("n_freq", C.c_int64),
                ("freqs", C.POINTER(C.c_double)), ("f0", C.c_double), ("df", C.c_double),
                ("n_bins", C.c_int32), ("q_min", C.c_double), ("q_max", C.c_double),
                ("max_top_k", C.c_int32), ("scratch_bytes", C.c_int64), ("flags", C.c_uint32)]


class BlsBatch(C.Structure):
    _fields_ = [("n_curves", C.c_int64), ("offsets", C.c_void_p), ("t", C.c_void_p),
                ("mag", C.c_void_p), ("sigma", C.c_void_p), ("t_origin", C.c_void_p)]


class BlsFieldBatch(C.Structure):
    _fields_ = [("n_stars", C.c_int64), ("n_epochs", C.c_int64), ("t", C.c_void_p), ("mag", C.c_void_p),
                ("sigma", C.c_void_p), ("t_origin", C.c_void_p)]


class BlsOutputs(C.Structure):
    _fields_ = [("sr", C.c_void_p), ("best_start", C.c_void_p), ("best_width", C.c_void_p),
                ("depth", C.c_void_p), ("status", C.c_void_p)]


class BlsVariabilityConfig(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("n_groups", C.c_int32), ("mag_lo", C.c_double), ("mag_bin", C.c_double),
                ("n_mag_bins", C.c_int32), ("max_iter", C.c_int32), ("clip", C.c_double), ("nsig", C.c_double),
                ("min_members", C.c_int32), ("reserved", C.c_int32)]


class BlsVariabilityOutputs(C.Structure):
    _fields_ = [("status", C.c_void_p), ("mean_mag", C.c_void_p), ("rms", C.c_void_p), ("cell", C.c_void_p),
                ("expected", C.c_void_p), ("scatter", C.c_void_p), ("kept", C.c_void_p), ("flag", C.c_void_p)]


# numpy view of bls_peak (32 bytes, natural alignment)
PEAK_DTYPE = np.dtype([("freq_index", "<i4"), ("sr", "<f4"), ("depth", "<f4"), ("start_bin", "<u2"),
                       ("width_bins", "<u2"), ("freq", "<f8"), ("epoch", "<f8")], align=True)
assert PEAK_DTYPE.itemsize == 32

# numpy view of bls_refined_peak (64 bytes)
REFINED_DTYPE = np.dtype([("freq_index", "<i4"), ("fine_index", "<i4"), ("shift_index", "<i4"), ("start_bin", "<u2"),
                          ("width_bins", "<u2"), ("sr", "<f4"), ("depth", "<f4"), ("sde", "<f4"), ("coarse_sr", "<f4"),
                          ("freq", "<f8"), ("period", "<f8"), ("epoch", "<f8"), ("duration", "<f8")], align=True)
assert REFINED_DTYPE.itemsize == 64

_lib = None


class BlsError(RuntimeError):
    def __init__(self, code: int, detail: str = ""):
        self.code = code
        msg = lib().bls_strerror(code).decode() if _lib is not None else str(code)
        super().__init__("bls error %d: %s%s" % (code, msg, (" [" + detail + "]") if detail else ""))


def lib():
    """Load the shared library (built in-tree by paper_1112_1701_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libbls_b200.so is not built: run `python -m paper_1112_1701_b200.build` "
                              "(no CPU fallback exists)")
        L = C.CDLL(LIB_PATH)
        L.bls_plan_create.restype = C.c_int
        L.bls_plan_create.argtypes = [C.POINTER(BlsConfig), C.POINTER(C.c_void_p)]
        L.bls_run.restype = C.c_int
        L.bls_run.argtypes = [C.c_void_p, C.POINTER(BlsBatch), C.POINTER(BlsOutputs), C.c_void_p]
        L.bls_run_field.restype = C.c_int
        L.bls_run_field.argtypes = [C.c_void_p, C.POINTER(BlsFieldBatch), C.POINTER(BlsOutputs), C.c_void_p]
        L.bls_topk.restype = C.c_int
        L.bls_topk.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
        L.bls_search_host.restype = C.c_int
        L.bls_search_host.argtypes = [C.c_void_p, C.POINTER(BlsBatch), C.c_int32, C.c_void_p, C.c_void_p]
        L.bls_plan_destroy.restype = C.c_int
        L.bls_plan_destroy.argtypes = [C.c_void_p]
        L.bls_plan_query.restype = C.c_int
        L.bls_plan_query.argtypes = [C.c_void_p, C.c_int32, C.POINTER(C.c_int64)]
        L.bls_strerror.restype = C.c_char_p
        L.bls_strerror.argtypes = [C.c_int]
        L.bls_plan_last_cuda_error.restype = C.c_char_p
        L.bls_plan_last_cuda_error.argtypes = [C.c_void_p]
        L.bls_debug_fold_bins.restype = C.c_int
        L.bls_debug_fold_bins.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32,
                                          C.c_uint32, C.c_void_p, C.POINTER(C.c_int64)]
        L.bls_debug_fold_bins_shift.restype = C.c_int
        L.bls_debug_fold_bins_shift.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int64, C.c_int32, C.c_int32, C.c_int32,
                                                C.c_uint32, C.c_void_p, C.POINTER(C.c_int64)]
        L.bls_plan_set_peak_min_sep.restype = C.c_int
        L.bls_plan_set_peak_min_sep.argtypes = [C.c_void_p, C.c_int32]
        L.bls_refine.restype = C.c_int
        L.bls_refine.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]
        L.bls_detection_efficiency.restype = C.c_int
        L.bls_detection_efficiency.argtypes = [C.c_int32, C.POINTER(BlsBatch), C.c_int64, C.c_void_p, C.c_double, C.c_int32,
                                               C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.bls_variability.restype = C.c_int
        L.bls_variability.argtypes = [C.c_int32, C.POINTER(BlsVariabilityConfig), C.POINTER(BlsBatch), C.c_void_p,
                                      C.POINTER(BlsVariabilityOutputs), C.c_void_p]
        L.bls_variability_noalloc.restype = C.c_int
        L.bls_variability_noalloc.argtypes = [C.c_int32, C.POINTER(BlsVariabilityConfig), C.POINTER(BlsBatch), C.c_void_p,
                                      C.POINTER(BlsVariabilityOutputs), C.c_void_p]
        _lib = L
    return _lib


def detection_efficiency(offsets, t, freqs, duration: float, n_phase: int = 1000, min_events: int = 2, device: int = 0,
                         stream: Optional[int] = None):
    """bls_detection_efficiency: offsets host int64, t float32 CUDA tensor (each cadence sorted), freqs host float64.
    Returns (count int32 [n_curves, n_freq], efficiency float64 [n_curves, n_freq]) CUDA tensors."""
    import torch
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    n = offsets.size - 1
    dev = torch.device("cuda", device)
    cnt = torch.zeros((max(n, 1), freqs.size), dtype=torch.int32, device=dev)
    eff = torch.zeros((max(n, 1), freqs.size), dtype=torch.float64, device=dev)
    b = BlsBatch(n, offsets.ctypes.data, _ptr(t), None, None, None)
    if stream is None:
        stream = torch.cuda.current_stream(dev).cuda_stream
    rc = lib().bls_detection_efficiency(device, C.byref(b), freqs.size, C.c_void_p(freqs.ctypes.data), float(duration), int(n_phase),
                                        int(min_events), C.c_void_p(cnt.data_ptr()), C.c_void_p(eff.data_ptr()), C.c_void_p(stream))
    if rc != BLS_OK:
        raise BlsError(rc)
    return cnt[:n], eff[:n]


def variability(offsets, t, mag, sigma, group=None, *, n_groups: int = 1, mag_lo: float = 12.0, mag_bin: float = 0.1,
                n_mag_bins: int = 80, clip: float = 3.0, nsig: float = 2.0, max_iter: int = 5, min_members: int = 5,
                device: int = 0, stream: Optional[int] = None):
    """bls_variability: offsets host int64; t, mag, sigma float32 CUDA tensors; group int32 CUDA tensor or None.
    Returns a dict of CUDA tensors (status, mean_mag, rms, cell, expected, scatter, kept, flag)."""
    import torch
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n = offsets.size - 1
    dev = torch.device("cuda", device)
    i32 = lambda: torch.zeros(max(n, 1), dtype=torch.int32, device=dev)
    f64 = lambda: torch.zeros(max(n, 1), dtype=torch.float64, device=dev)
    out = dict(status=i32(), mean_mag=f64(), rms=f64(), cell=i32(), expected=f64(), scatter=f64(), kept=i32(), flag=i32())
    cfg = BlsVariabilityConfig(C.sizeof(BlsVariabilityConfig), int(n_groups), float(mag_lo), float(mag_bin), int(n_mag_bins),
                               int(max_iter), float(clip), float(nsig), int(min_members), 0)
    b = BlsBatch(n, offsets.ctypes.data, _ptr(t), _ptr(mag), _ptr(sigma), None)
    o = BlsVariabilityOutputs(*[_ptr(out[k]) for k in ("status", "mean_mag", "rms", "cell", "expected", "scatter", "kept", "flag")])
    if stream is None:
        stream = torch.cuda.current_stream(dev).cuda_stream
    rc = lib().bls_variability(device, C.byref(cfg), C.byref(b), C.c_void_p(_ptr(group)) if group is not None else None,
                               C.byref(o), C.c_void_p(stream))
    if rc != BLS_OK:
        raise BlsError(rc)
    return {k: v[:n] for k, v in out.items()}


def variability_noalloc(offsets, t, mag, sigma, group=None, *, out=None, n_groups: int = 1, mag_lo: float = 12.0,
                        mag_bin: float = 0.1, n_mag_bins: int = 80, clip: float = 3.0, nsig: float = 2.0, max_iter: int = 5,
                        min_members: int = 5, device: int = 0, stream: Optional[int] = None):
    """bls_variability_noalloc: the pre-filter of `variability` for callers that may not allocate GPU memory where
    they call it (all free memory already belongs to their own pool, a latency bound forbids cudaMalloc's stalls, or
    the host application owns every allocation).  The library call allocates nothing: its working memory is a fixed
    array inside the library, which limits it to NOALLOC_MAX_STARS stars and NOALLOC_MAX_CELLS cells
    (BlsError(BLS_ERR_CAPACITY) beyond that) and means calls that overlap on the GPU corrupt each other: issue them
    on one stream.  Make the first call on a GPU at start-up.

    `out`: the dict a previous call returned (or tensors of the same names and sizes): it is written in place, so
    a steady-state caller allocates nothing on the Python side either.  Without it the eight output tensors are made
    here with torch, as `variability` does.  Same arguments and same results as `variability` otherwise."""
    import torch
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n = offsets.size - 1
    dev = torch.device("cuda", device)
    names = ("status", "mean_mag", "rms", "cell", "expected", "scatter", "kept", "flag")
    if out is None:
        i32 = lambda: torch.zeros(max(n, 1), dtype=torch.int32, device=dev)
        f64 = lambda: torch.zeros(max(n, 1), dtype=torch.float64, device=dev)
        out = dict(status=i32(), mean_mag=f64(), rms=f64(), cell=i32(), expected=f64(), scatter=f64(), kept=i32(), flag=i32())
    else:
        for k in names:
            want = torch.float64 if k in ("mean_mag", "rms", "expected", "scatter") else torch.int32
            assert out[k].is_cuda and out[k].dtype == want and out[k].numel() >= n and out[k].is_contiguous(), k
    cfg = BlsVariabilityConfig(C.sizeof(BlsVariabilityConfig), int(n_groups), float(mag_lo), float(mag_bin), int(n_mag_bins),
                               int(max_iter), float(clip), float(nsig), int(min_members), 0)
    b = BlsBatch(n, offsets.ctypes.data, _ptr(t), _ptr(mag), _ptr(sigma), None)
    o = BlsVariabilityOutputs(*[_ptr(out[k]) for k in names])
    if stream is None:
        stream = torch.cuda.current_stream(dev).cuda_stream
    rc = lib().bls_variability_noalloc(device, C.byref(cfg), C.byref(b), C.c_void_p(_ptr(group)) if group is not None else None,
                                       C.byref(o), C.c_void_p(stream))
    if rc != BLS_OK:
        raise BlsError(rc)
    return {k: out[k][:n] for k in names}


def debug_fold_bins(f, t, n_bins: int, flags: int = 0, device: int = 0):
    """bls_debug_fold_bins: f, t float64 CUDA tensors -> (int32 CUDA tensor of bins, n_canonical)."""
    import torch
    assert f.is_cuda and t.is_cuda and f.dtype == torch.float64 and t.dtype == torch.float64
    bins = torch.empty(f.numel(), dtype=torch.int32, device=f.device)
    ncan = C.c_int64()
    rc = lib().bls_debug_fold_bins(device, C.c_void_p(f.data_ptr()), C.c_void_p(t.data_ptr()), f.numel(),
                                   int(n_bins), int(flags), C.c_void_p(bins.data_ptr()), C.byref(ncan))
    if rc != BLS_OK:
        raise BlsError(rc)
    return bins, ncan.value


def debug_fold_bins_shift(f, t, n_bins: int, h: int, n_shift: int, flags: int = 0, device: int = 0, bins=None):
    """bls_debug_fold_bins_shift: as debug_fold_bins on the bin grid shifted by h / (n_shift * n_bins) cycles.
    `bins`: optional int32 CUDA tensor to write into."""
    import torch
    assert f.is_cuda and t.is_cuda and f.dtype == torch.float64 and t.dtype == torch.float64
    if bins is None:
        bins = torch.empty(f.numel(), dtype=torch.int32, device=f.device)
    ncan = C.c_int64()
    rc = lib().bls_debug_fold_bins_shift(device, C.c_void_p(f.data_ptr()), C.c_void_p(t.data_ptr()), f.numel(), int(n_bins),
                                         int(h), int(n_shift), int(flags), C.c_void_p(bins.data_ptr()), C.byref(ncan))
    if rc != BLS_OK:
        raise BlsError(rc)
    return bins, ncan.value


def _ptr(x) -> Optional[int]:
    if x is None:
        return None
    if hasattr(x, "data_ptr"):
        return x.data_ptr() if x.numel() else None
    if isinstance(x, np.ndarray):
        return x.ctypes.data if x.size else None
    return int(x)


class Plan:
    """bls_plan: trial grid + device scratch.  freqs=None uses the uniform grid f0 + k*df."""

    def __init__(self, *, n_bins: int, q_min: float, q_max: float, freqs=None, n_freq: Optional[int] = None,
                 f0: float = 0.0, df: float = 0.0, max_top_k: int = 5, device: int = 0,
                 scratch_bytes: int = 0, flags: int = 0):
        L = lib()
        cfg = BlsConfig()
        cfg.struct_size = C.sizeof(BlsConfig)
        cfg.device = device
        self._freqs = None
        if freqs is not None:
            self._freqs = np.ascontiguousarray(freqs, dtype=np.float64)
            cfg.n_freq = self._freqs.size
            cfg.freqs = self._freqs.ctypes.data_as(C.POINTER(C.c_double))
        else:
            cfg.n_freq = int(n_freq)
            cfg.freqs = None
            cfg.f0, cfg.df = float(f0), float(df)
        cfg.n_bins, cfg.q_min, cfg.q_max = int(n_bins), float(q_min), float(q_max)
        cfg.max_top_k, cfg.scratch_bytes, cfg.flags = int(max_top_k), int(scratch_bytes), int(flags)
        handle = C.c_void_p()
        rc = L.bls_plan_create(C.byref(cfg), C.byref(handle))
        if rc != BLS_OK:
            raise BlsError(rc)
        self._h = handle
        self.device = device
        self.n_freq = int(cfg.n_freq)
        self.n_bins = int(n_bins)
        self.max_top_k = int(max_top_k)
        self._n_curves = 0
        self._keep = None

    # -- lifetime ---------------------------------------------------------------------------------
    def destroy(self):
        if getattr(self, "_h", None):
            lib().bls_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def _check(self, rc: int):
        if rc != BLS_OK:
            raise BlsError(rc, lib().bls_plan_last_cuda_error(self._h).decode())

    def query(self, what: int) -> int:
        v = C.c_int64()
        self._check(lib().bls_plan_query(self._h, what, C.byref(v)))
        return v.value

    @property
    def kmin(self) -> int:
        return self.query(QUERY_KMIN)

    @property
    def kmax(self) -> int:
        return self.query(QUERY_KMAX)

    # -- bls_run ----------------------------------------------------------------------------------
    def run(self, offsets, t, mag, sigma, t_origin=None, *, sr=None, best_start=None, best_width=None,
            depth=None, status=None, stream: Optional[int] = None):
        """offsets / t_origin: host numpy (int64 / float64).  t, mag, sigma and the optional outputs:
        CUDA torch tensors (float32; best_* int16/uint16 storage).  Enqueues on `stream`
        (default: torch's current stream)."""
        import torch
        offsets = np.ascontiguousarray(offsets, dtype=np.int64)
        n_curves = offsets.size - 1
        for name, x in (("t", t), ("mag", mag), ("sigma", sigma)):
            if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
                raise TypeError("%s must be a contiguous float32 CUDA tensor" % name)
        origin = None if t_origin is None else np.ascontiguousarray(t_origin, dtype=np.float64)
        b = BlsBatch(n_curves, offsets.ctypes.data, _ptr(t), _ptr(mag), _ptr(sigma),
                     None if origin is None else origin.ctypes.data)
        outs = None
        if any(x is not None for x in (sr, best_start, best_width, depth, status)):
            outs = BlsOutputs(_ptr(sr), _ptr(best_start), _ptr(best_width), _ptr(depth), _ptr(status))
        if stream is None:
            stream = torch.cuda.current_stream(t.device).cuda_stream
        self._keep = (offsets, origin, t, mag, sigma)
        rc = lib().bls_run(self._h, C.byref(b), C.byref(outs) if outs is not None else None,
                           C.c_void_p(stream))
        self._check(rc)
        self._n_curves = n_curves

    # -- bls_run_field ----------------------------------------------------------------------------
    def run_field(self, t, mag, sigma, t_origin: Optional[float] = None, *, sr=None, best_start=None, best_width=None,
                  depth=None, status=None, stream: Optional[int] = None):
        """t: float32 CUDA [n_epochs]; mag, sigma: float32 CUDA [n_stars, n_epochs] (non-finite / sigma <= 0 = absent)."""
        import torch
        assert mag.dim() == 2 and mag.shape == sigma.shape and mag.shape[1] == t.numel()
        for name, x in (("t", t), ("mag", mag), ("sigma", sigma)):
            if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
                raise TypeError("%s must be a contiguous float32 CUDA tensor" % name)
        origin = None if t_origin is None else np.array([float(t_origin)], dtype=np.float64)
        fb = BlsFieldBatch(mag.shape[0], mag.shape[1], _ptr(t), _ptr(mag), _ptr(sigma),
                           None if origin is None else origin.ctypes.data)
        outs = None
        if any(x is not None for x in (sr, best_start, best_width, depth, status)):
            outs = BlsOutputs(_ptr(sr), _ptr(best_start), _ptr(best_width), _ptr(depth), _ptr(status))
        if stream is None:
            stream = torch.cuda.current_stream(t.device).cuda_stream
        self._keep = (origin, t, mag, sigma)
        self._check(lib().bls_run_field(self._h, C.byref(fb), C.byref(outs) if outs is not None else None, C.c_void_p(stream)))
        self._n_curves = int(mag.shape[0])

    # -- bls_topk ---------------------------------------------------------------------------------
    def topk(self, k: int, stream: Optional[int] = None):
        """Returns a CUDA uint8 tensor [n_curves*k*32] holding bls_peak records (see peaks_to_numpy)."""
        import torch
        dev = torch.device("cuda", self.device)
        out = torch.empty(max(self._n_curves * k, 1) * PEAK_DTYPE.itemsize, dtype=torch.uint8, device=dev)
        if stream is None:
            stream = torch.cuda.current_stream(dev).cuda_stream
        self._check(lib().bls_topk(self._h, int(k), C.c_void_p(out.data_ptr()), C.c_void_p(stream)))
        return out[: self._n_curves * k * PEAK_DTYPE.itemsize]

    def set_peak_min_sep(self, steps: int) -> None:
        """bls_plan_set_peak_min_sep: greedy minimum separation (grid steps) between a curve's reported peaks, from the
        next run on; 0 = plain top-k local maxima."""
        self._check(lib().bls_plan_set_peak_min_sep(self._h, int(steps)))

    # -- bls_refine --------------------------------------------------------------------------------
    def refine(self, k: int, n_fine: int = 64, n_shift: int = 4, stream: Optional[int] = None) -> np.ndarray:
        """bls_refine on the last run; returns host records [n_curves, k] of REFINED_DTYPE (synchronises)."""
        import torch
        dev = torch.device("cuda", self.device)
        out = torch.zeros(max(self._n_curves * k, 1) * REFINED_DTYPE.itemsize, dtype=torch.uint8, device=dev)
        if stream is None:
            stream = torch.cuda.current_stream(dev).cuda_stream
        self._check(lib().bls_refine(self._h, int(k), int(n_fine), int(n_shift), C.c_void_p(out.data_ptr()), C.c_void_p(stream)))
        return out[: self._n_curves * k * REFINED_DTYPE.itemsize].cpu().numpy().view(REFINED_DTYPE).reshape(-1, k)

    def peaks_to_numpy(self, raw, k: int) -> np.ndarray:
        return raw.cpu().numpy().view(PEAK_DTYPE).reshape(-1, k)

    # -- bls_search_host ----------------------------------------------------------------------------
    def search_host(self, offsets, t, mag, sigma, t_origin=None, k: int = 5):
        """Everything from HOST numpy arrays: H2D, bls_run, bls_topk, D2H, synchronise."""
        offsets = np.ascontiguousarray(offsets, dtype=np.int64)
        t = np.ascontiguousarray(t, dtype=np.float32)
        mag = np.ascontiguousarray(mag, dtype=np.float32)
        sigma = np.ascontiguousarray(sigma, dtype=np.float32)
        n_curves = offsets.size - 1
        origin = None if t_origin is None else np.ascontiguousarray(t_origin, dtype=np.float64)
        peaks = np.zeros((max(n_curves, 1), k), dtype=PEAK_DTYPE)
        status = np.zeros(max(n_curves, 1), dtype=np.int32)
        b = BlsBatch(n_curves, offsets.ctypes.data, _ptr(t), _ptr(mag), _ptr(sigma),
                     None if origin is None else origin.ctypes.data)
        rc = lib().bls_search_host(self._h, C.byref(b), int(k), C.c_void_p(peaks.ctypes.data),
                                   C.c_void_p(status.ctypes.data))
        self._check(rc)
        self._n_curves = n_curves
        return peaks[:n_curves], status[:n_curves]
