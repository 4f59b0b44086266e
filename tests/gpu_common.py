"""Helpers for the -m gpu parity tests: run a synthetic configuration through the C ABI (Python
binding) and fetch spectra + peaks as numpy arrays."""
from __future__ import annotations

import numpy as np

import synth


def run_gpu(batch, grid, top_k=5, flags=0, scratch_bytes=0, want_spectrum=True, freqs=None):
    import torch
    import paper_1112_1701_b200 as bls
    dev = torch.device("cuda", 0)
    if freqs is None:
        freqs = synth.freq_grid(grid)
    plan = bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=max(top_k, 1),
                    flags=flags, scratch_bytes=scratch_bytes)
    nc, nf = batch.n_curves, len(freqs)
    t = torch.from_numpy(batch.t).to(dev)
    mag = torch.from_numpy(batch.mag).to(dev)
    sig = torch.from_numpy(batch.sigma).to(dev)
    out = {}
    kw = {}
    if want_spectrum:
        kw = dict(sr=torch.full((nc, nf), -1.0, dtype=torch.float32, device=dev),
                  best_start=torch.full((nc, nf), -1, dtype=torch.int16, device=dev),
                  best_width=torch.full((nc, nf), -1, dtype=torch.int16, device=dev),
                  depth=torch.full((nc, nf), -1.0, dtype=torch.float32, device=dev))
    status = torch.full((max(nc, 1),), -7, dtype=torch.int32, device=dev)
    plan.run(batch.offsets, t, mag, sig, batch.t_origin, status=status, **kw)
    raw = plan.topk(top_k)
    torch.cuda.synchronize()
    out["peaks"] = plan.peaks_to_numpy(raw, top_k) if nc else np.zeros((0, top_k), dtype=bls.PEAK_DTYPE)
    out["status"] = status.cpu().numpy()[:nc]
    if want_spectrum:
        out["sr"] = kw["sr"].cpu().numpy()
        out["a"] = kw["best_start"].cpu().numpy().view(np.uint16).astype(np.int32)
        out["k"] = kw["best_width"].cpu().numpy().view(np.uint16).astype(np.int32)
        out["depth"] = kw["depth"].cpu().numpy()
    out["kmin"], out["kmax"] = plan.kmin, plan.kmax
    out["n_canonical"] = plan.query(bls.binding.QUERY_LAST_CANONICAL) if nc else 0
    out["launches"] = plan.query(bls.binding.QUERY_LAST_LAUNCHES)
    out["kernel"] = plan.query(bls.binding.QUERY_SEARCH_KERNEL)
    out["freqs"] = freqs
    plan.destroy()
    return out
