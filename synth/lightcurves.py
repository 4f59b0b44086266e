"""Seeded, per-curve addressable synthetic PTF-like light curves.

These stand in for the PTF/M-dwarfs photometry the paper searched (PAPER.md L53-57 cadence,
L97/L117 noise floor, L151 + Table 3 L290-299 eclipse depths and periods), which is not public.
The five workloads are the ones BASELINE.json `configs[0..4]` describe (C0..C4); the recipe is
restated in DESIGN.md "Input recipe".

This module only *generates inputs* (times, magnitudes, errors, frequency grids).  It holds none
of the BLS arithmetic: no weights, no folding, no statistic.  Both the CPU oracle's tests and the
CUDA path's tests / bench draw their inputs from here so that they see identical arrays.

Every curve is generated from its own counter-based stream
`Philox(key=seed_cfg, counter=[0, curve_id, 0, 0])`, so any subset of a configuration can be
regenerated without the rest.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence

import numpy as np

SEED_BASE = 11121701


@dataclass(frozen=True)
class Grid:
    """Trial grid: nf frequencies uniform in [fmin, fmax] (cycles/day), nb phase bins, q range."""
    nf: int
    fmin: float
    fmax: float
    nb: int
    qmin: float
    qmax: float


@dataclass
class Batch:
    """Ragged CSR batch of light curves (host numpy arrays)."""
    offsets: np.ndarray      # int64 [n_curves+1]
    t: np.ndarray            # float32 [n_points] days since the curve's first epoch
    mag: np.ndarray          # float32 [n_points]
    sigma: np.ndarray        # float32 [n_points]
    t_origin: np.ndarray     # float64 [n_curves] HJD of the curve's first epoch
    curve_ids: np.ndarray    # int64 [n_curves]
    truth: List[Optional[dict]] = field(default_factory=list)  # injected (P, depth, q, T0) or None

    @property
    def n_curves(self) -> int:
        return len(self.offsets) - 1

    @property
    def n_points(self) -> int:
        return int(self.offsets[-1])

    def curve(self, c: int):
        a, b = int(self.offsets[c]), int(self.offsets[c + 1])
        return self.t[a:b], self.mag[a:b], self.sigma[a:b]


# ----------------------------------------------------------------------------------------------
# Configurations (BASELINE.json configs[0..4]) plus two small ones used by the parity tests.
# ----------------------------------------------------------------------------------------------
CONFIGS: Dict[str, dict] = {
    # configs[0]: single curve, 500 epochs in 60 nightly 6-hour windows, fixed injected eclipse.
    "C0": dict(index=0, n_curves=1, n_min=500, n_max=500, cadence="nightly", nights=60,
               noise="const", sigma0=0.01, inject_frac=1.0,
               inject=dict(P=(0.40, 0.40), depth=(0.05, 0.05), q=(0.10, 0.10)),
               grid=Grid(2000, 0.1, 5.0, 100, 0.01, 0.10), top_k=5),
    # configs[1]: 1,000 x 1,500 epochs, PTF-like cadence, lognormal per-star noise.
    "C1": dict(index=1, n_curves=1000, n_min=1500, n_max=1500, cadence="ptf", seasons=1,
               noise="lognormal", sigma0=0.01, inject_frac=0.01,
               inject=dict(P=(0.3, 5.0), depth=(0.01, 0.2), q=(0.01, 0.08)),
               grid=Grid(20000, 0.1, 5.0, 200, 0.005, 0.15), top_k=5),
    # configs[2]: 100,000 ragged curves, N ~ U{500..4000}, top-5 only.
    "C2": dict(index=2, n_curves=100000, n_min=500, n_max=4000, cadence="ptf", seasons=1,
               noise="lognormal", sigma0=0.01, inject_frac=0.005,
               inject=dict(P=(0.3, 5.0), depth=(0.01, 0.2), q=(0.01, 0.08)),
               grid=Grid(50000, 0.1, 5.0, 200, 0.005, 0.15), top_k=5),
    # configs[3]: 10,000 x 5,000 epochs, two seasons one year apart, fine grid.
    "C3": dict(index=3, n_curves=10000, n_min=5000, n_max=5000, cadence="ptf", seasons=2,
               noise="lognormal", sigma0=0.01, inject_frac=0.01,
               inject=dict(P=(0.2, 30.0), depth=(0.01, 0.2), q=(0.01, 0.08)),
               grid=Grid(500000, 1.0 / 30.0, 5.0, 400, 0.002, 0.10), top_k=5),
    # configs[4]: 1,000,000 x 200 epochs over 30 days of random nightly sampling.
    "C4": dict(index=4, n_curves=1000000, n_min=200, n_max=200, cadence="nightly", nights=30,
               noise="const", sigma0=0.02, inject_frac=0.01,
               inject=dict(P=(0.3, 3.0), depth=(0.01, 0.2), q=(0.02, 0.08)),
               grid=Grid(5000, 0.3, 5.0, 64, 0.02, 0.15), top_k=5),
    # Small cases for element-by-element parity: several frequency tiles plus a ragged tail,
    # ragged lengths, both cadences.  Not in BASELINE.json.
    "T0": dict(index=10, n_curves=6, n_min=60, n_max=700, cadence="ptf", seasons=1,
               noise="lognormal", sigma0=0.01, inject_frac=0.5,
               inject=dict(P=(0.3, 5.0), depth=(0.02, 0.2), q=(0.02, 0.08)),
               grid=Grid(300, 0.1, 5.0, 100, 0.01, 0.12), top_k=5),
    "T1": dict(index=11, n_curves=5, n_min=150, n_max=260, cadence="nightly", nights=30,
               noise="const", sigma0=0.02, inject_frac=0.5,
               inject=dict(P=(0.3, 3.0), depth=(0.02, 0.2), q=(0.02, 0.08)),
               grid=Grid(173, 0.3, 5.0, 64, 0.02, 0.15), top_k=4),
    "T2": dict(index=12, n_curves=3, n_min=900, n_max=1300, cadence="ptf", seasons=2,
               noise="lognormal", sigma0=0.01, inject_frac=0.5,
               inject=dict(P=(0.2, 30.0), depth=(0.02, 0.2), q=(0.01, 0.08)),
               grid=Grid(421, 1.0 / 30.0, 5.0, 400, 0.002, 0.10), top_k=5),
}


def config(name: str) -> dict:
    return CONFIGS[name]


def freq_grid(g: Grid) -> np.ndarray:
    """f_k = fmin + k*df, df = (fmax-fmin)/(nf-1), each evaluated in fp64 (no running sum)."""
    if g.nf == 1:
        return np.array([g.fmin], dtype=np.float64)
    df = (g.fmax - g.fmin) / (g.nf - 1)
    return g.fmin + np.arange(g.nf, dtype=np.float64) * df


def _rng(cfg: dict, curve_id: int) -> np.random.Generator:
    key = SEED_BASE + int(cfg["index"])
    return np.random.Generator(np.random.Philox(key=key, counter=[0, int(curve_id), 0, 0]))


def curve_lengths(cfg: dict, curve_ids: Sequence[int]) -> np.ndarray:
    """Number of epochs of each curve (needs the curve's own stream only)."""
    out = np.empty(len(curve_ids), dtype=np.int64)
    for j, cid in enumerate(curve_ids):
        out[j] = _length(cfg, _rng(cfg, cid))
    return out


def _length(cfg: dict, rng: np.random.Generator) -> int:
    # first draw of every stream, so curve_lengths() and make_curve() agree
    return int(rng.integers(cfg["n_min"], cfg["n_max"] + 1))


def _times_nightly(rng, n, nights):
    """C0 / C4: night ~ U{0..nights-1}, time in night ~ U[0, 0.25 d); sorted."""
    night = rng.integers(0, nights, size=n).astype(np.float64)
    t = night + rng.uniform(0.0, 0.25, size=n)
    t.sort()
    return t


def _times_ptf(rng, n, seasons):
    """C1-C3: `seasons` seasons of 120 days one year apart; each night kept w.p. 0.7; night length
    U[4,8] h starting at night + U[0,0.05) d; slots every 10 min with N(0, 20 s) jitter; exactly n
    slots chosen at random; sorted.  If the kept nights offer fewer than n slots the season is
    lengthened night by night (needed for the longest C2 curves)."""
    slot = 10.0 / 1440.0
    season_len = 120
    while True:
        times = []
        for s in range(seasons):
            base = 365.0 * s
            keep = rng.uniform(size=season_len) < 0.7
            length = rng.uniform(4.0, 8.0, size=season_len) / 24.0
            start = rng.uniform(0.0, 0.05, size=season_len)
            for d in np.nonzero(keep)[0]:
                k = int(np.floor(length[d] / slot))
                times.append(base + d + start[d] + slot * np.arange(k))
        allt = np.concatenate(times) if times else np.empty(0)
        if allt.size >= n:
            break
        season_len += 30
    pick = rng.choice(allt.size, size=n, replace=False)
    t = allt[pick] + rng.normal(0.0, 20.0 / 86400.0, size=n)
    t.sort()
    return t


def make_curve(cfg: dict, curve_id: int):
    """One light curve -> (t32, mag32, sigma32, t_origin, truth)."""
    rng = _rng(cfg, curve_id)
    n = _length(cfg, rng)
    if cfg["cadence"] == "nightly":
        t = _times_nightly(rng, n, cfg["nights"])
    else:
        t = _times_ptf(rng, n, cfg["seasons"])
    if cfg["noise"] == "const":
        sig = np.full(n, cfg["sigma0"], dtype=np.float64)
    else:
        star = cfg["sigma0"] * 10.0 ** (0.5 * rng.normal())
        sig = star * (1.0 + 0.25 * np.abs(rng.normal(size=n)))
    m0 = rng.uniform(14.0, 18.0)
    mag = m0 + rng.normal(size=n) * sig
    truth = None
    inj = cfg["inject"]
    u = rng.uniform()
    P = rng.uniform(*inj["P"])
    depth = rng.uniform(*inj["depth"])
    q = rng.uniform(*inj["q"])
    T0 = rng.uniform(0.0, P)
    if u < cfg["inject_frac"]:
        ph = (t - T0) / P
        ph -= np.floor(ph)
        mag = mag + depth * (ph < q)
        truth = dict(P=P, depth=depth, q=q, T0=T0)
    hjd0 = 2455000.0 + rng.uniform(0.0, 365.0)
    t_origin = hjd0 + t[0]
    t_rel = (t - t[0]).astype(np.float32)
    if truth is not None:
        truth["T0_rel"] = T0 - t[0]          # epoch of ingress in the stored time system
    return t_rel, mag.astype(np.float32), sig.astype(np.float32), t_origin, truth


def _make_chunk(args):
    """Curves `ids` of `cfg` as one packed piece: (lengths, t, mag, sigma, origins, truths)."""
    cfg, ids = args
    curves = [make_curve(cfg, int(c)) for c in ids]
    cat = (lambda j: np.concatenate([cv[j] for cv in curves]) if curves else np.empty(0, np.float32))
    return (np.asarray([cv[0].size for cv in curves], dtype=np.int64), cat(0), cat(1), cat(2),
            np.asarray([cv[3] for cv in curves], dtype=np.float64), [cv[4] for cv in curves])


def make_batch(cfg: dict, curve_ids: Optional[Sequence[int]] = None, workers: int = 1) -> Batch:
    """CSR batch of the requested curves (all curves of the configuration by default).  Every curve
    has its own counter-based stream, so the result does not depend on `workers` (processes used to
    generate large batches; 1 = in this process)."""
    if curve_ids is None:
        curve_ids = range(cfg["n_curves"])
    curve_ids = np.asarray(list(curve_ids), dtype=np.int64)
    if workers > 1 and len(curve_ids) >= 64 * workers:
        import multiprocessing as mp
        chunks = np.array_split(curve_ids, workers * 8)
        with mp.get_context("spawn").Pool(workers) as pool:     # spawn: safe after CUDA has been initialised
            parts = pool.map(_make_chunk, [(cfg, ch) for ch in chunks])
    else:
        parts = [_make_chunk((cfg, curve_ids))]
    lengths = np.concatenate([p[0] for p in parts]) if parts else np.zeros(0, np.int64)
    offsets = np.zeros(len(curve_ids) + 1, dtype=np.int64)
    np.cumsum(lengths, out=offsets[1:])
    cat = (lambda j, dt: np.concatenate([p[j] for p in parts]).astype(dt, copy=False))
    return Batch(offsets=offsets, t=cat(1, np.float32), mag=cat(2, np.float32), sigma=cat(3, np.float32),
                 t_origin=cat(4, np.float64), curve_ids=curve_ids, truth=[tr for p in parts for tr in p[5]])


def make_field(n_stars: int, n_epochs: int, seed: int = 0, absent_frac: float = 0.02):
    """One pointing in the field layout of bls_run_field (row f2): every star is measured on the same exposures
    (about 3,000 M-dwarfs per pointing; L115: 0-2 % of the epochs rejected; L121: 140 epochs in the
    figure's example, 300-epoch sets).  Returns (t [n_epochs] float32 days from the first epoch, mag and sigma
    [n_stars, n_epochs] float32 with absent entries marked by NaN magnitudes).  The cadence is the first n_epochs
    of a C1 curve's PTF-like cadence; per-star noise floors are log-normal around 10 mmag; every third star carries
    box eclipses (P 0.3-3 d, depth 0.03-0.2 mag, q 0.02-0.08).  Inputs only: none of the BLS arithmetic."""
    rng = np.random.Generator(np.random.Philox(key=SEED_BASE + 977, counter=[0, int(seed), 0, 0]))
    t = make_curve(CONFIGS["C1"], 77)[0][:n_epochs].astype(np.float32)
    assert t.size == n_epochs, "C1 cadences have 1,500 epochs"
    star = 0.01 * 10.0 ** (0.5 * rng.normal(size=(n_stars, 1)))
    sig = (star * (1.0 + 0.25 * np.abs(rng.normal(size=(n_stars, n_epochs))))).astype(np.float32)
    mag = rng.uniform(14.0, 18.0, size=(n_stars, 1)) + rng.normal(size=(n_stars, n_epochs)) * sig
    inj = np.arange(n_stars) % 3 == 0
    P = rng.uniform(0.3, 3.0, size=(n_stars, 1))
    depth = rng.uniform(0.03, 0.2, size=(n_stars, 1))
    q = rng.uniform(0.02, 0.08, size=(n_stars, 1))
    T0 = rng.uniform(0.0, 1.0, size=(n_stars, 1)) * P
    in_box = (((t[None, :].astype(np.float64) - T0) / P) % 1.0) < q
    mag = np.where(inj[:, None] & in_box, mag + depth, mag).astype(np.float32)
    mag[rng.uniform(size=mag.shape) < absent_frac] = np.nan
    return t, mag, sig
