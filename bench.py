#!/usr/bin/env python
"""bench.py -- throughput of the BLS hot path on B200 (BASELINE.json metric: point-folds/s, curves/s,
fraction of the stated roofline), with the fp64 oracle timed beside it and compared with it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (prep -> fold/search/merge -> peaks -> top-k) over one batch
of synthetic light curves of the chosen configuration.  The default is C2 = BASELINE.json configs[2]
at FULL size (100,000 curves of 500-4,000 epochs, 50,000 frequencies, 200 bins, top-5): the largest
configuration whose 20 timed steps fit the driver's bench arm.  Prints ONE JSON line (rank 0).

  value        whole-job point-folds/s, inputs resident in HBM (CUDA events around bls_run + bls_topk)
  e2e          the same metric through bls_search_host with pinned HOST buffers (H2D + D2H inside)
  roofline     the search kernel against the issue-rate roofline stated in DESIGN.md section 7
  cpu_baseline the oracle as it stands on the host cores, bounded sample, and the parity of the timed
               step's peaks against it
  per_config   C0, C1, C3 (full) and C4 (full): one timed step each (after warm-up), same fields in short;
               F2: bls_run_field at the paper's cadence, field kernel against the per-star kernels
With --impl reference the oracle itself is the timed arm (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import synth  # noqa: E402

METRIC = "bls_point_folds_per_sec"
UNIT = "point-folds/s"

# Roofline constants, measured on B200 by microbench/issue_rates.cu
# (profiles/r02b_microbench.md): lane-operations per clock per SM.
LSU_LANE_OPS_PER_CLK_SM = 32.0       # shared wavefront pipe: conflict-free ATOMS.ADD 31.97
XU_LANE_OPS_PER_CLK_SM = 16.0        # MUFU.RSQ 16.00: one per box
ISSUE_LANE_INSTR_PER_CLK_SM = 128.0  # 4 schedulers x 32 lanes
# fewest instructions the method needs: fold = point load, DFMA, IMAD.WIDE, 2 ATOMS; box = 1/2 (FFMA2 + FADD2 +
# FFMA2 + FMUL2 + FMNMX3) + MUFU with packed f32x2 arithmetic
FOLD_MIN_INSTR, BOX_MIN_INSTR = 5.0, 3.5


def pair_clocks(n_mean, nb, kmax, nk):
    """Lower bounds, in SM clocks, for one (curve, frequency) pair on one SM."""
    t_lsu = (2.0 * n_mean + 2.0 * (nb + kmax)) / LSU_LANE_OPS_PER_CLK_SM
    t_xu = nb * nk / XU_LANE_OPS_PER_CLK_SM
    t_issue = (FOLD_MIN_INSTR * n_mean + BOX_MIN_INSTR * nb * nk) / ISSUE_LANE_INSTR_PER_CLK_SM
    t_sum = 2.0 * n_mean / LSU_LANE_OPS_PER_CLK_SM + nb * nk / XU_LANE_OPS_PER_CLK_SM   # SURVEY 8(d) sum form
    return {"lsu": t_lsu, "xu": t_xu, "issue": t_issue, "min": max(t_lsu, t_xu, t_issue),
            "method": max(t_lsu, t_issue), "sum_form": t_sum}


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML in-process)."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            # CUDA_VISIBLE_DEVICES may remap ordinals: go through the UUID torch reports
            import torch
            uuid = str(torch.cuda.get_device_properties(index).uuid)
            h = None
            for cand in ("GPU-" + uuid, uuid):
                try:
                    h = pynvml.nvmlDeviceGetHandleByUUID(cand.encode() if isinstance(cand, str) else cand)
                    break
                except Exception:
                    h = None
            self.h = h if h is not None else pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # pragma: no cover
            self.nv = None
            self.err = repr(e)

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40,
                 "sw_thermal_slowdown": 0x20, "hw_power_brake": 0x80, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(0.02)

    def start(self):
        if self.nv:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()

    def stop(self):
        if self._thr:
            self._stop.set()
            self._thr.join()
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def oracle_rate(cfg, batch, freqs, kmin, kmax, curves, threads=None):
    """Time the oracle as it stands on `curves` of the batch at all frequencies; returns the spectra too."""
    import oracle
    oracle.lib()
    t0 = time.perf_counter()
    res, used = oracle.spectrum_batch(batch.offsets, batch.t, batch.mag, batch.sigma, freqs,
                                      cfg["grid"].nb, kmin, kmax, curves=curves, threads=threads)
    dt = time.perf_counter() - t0
    pts = sum(int(batch.offsets[c + 1] - batch.offsets[c]) for c in curves)
    return pts * len(freqs) / dt, len(curves) / dt, used, dt, res


def run_reference(args, cfg, rank, world):
    """--impl reference: the fp64 oracle on the host cores, same metric/config.  Rank 0 only."""
    if rank != 0:
        return
    import oracle
    grid = cfg["grid"]
    freqs = synth.freq_grid(grid)
    kmin, kmax = oracle.widths(grid.nb, grid.qmin, grid.qmax)
    cores = oracle.host_cores()
    n_sample = max(cores, 8)           # curves per step: about 0.5 s/curve/core at C1, 1.2 at C2
    batch = synth.make_batch(cfg, range(min(n_sample, cfg["n_curves"])))
    curves = list(range(batch.n_curves))
    for _ in range(min(args.warmup, 1)):
        oracle_rate(cfg, batch, freqs, kmin, kmax, curves[:cores])
    tot_pf, tot_t, used = 0.0, 0.0, cores
    for _ in range(args.steps):
        pf_s, _, used, dt, _ = oracle_rate(cfg, batch, freqs, kmin, kmax, curves)
        tot_pf += pf_s * dt
        tot_t += dt
    value = tot_pf / tot_t
    sample = "%d curves x %d frequencies of %s per step (of %d curves)" % (len(curves), grid.nf, args.config, cfg["n_curves"])
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": workload_name(args.config, cfg)},
            "curves_per_sec": value / (grid.nf * batch.n_points / batch.n_curves),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def rank_curve_ids(n_curves_per_rank, rank):
    """Replicas only: rank r searches curve ids [r*n, (r+1)*n) of the configuration's
    per-curve addressable generator -- disjoint across ranks, no data-path collective."""
    return range(rank * n_curves_per_rank, (rank + 1) * n_curves_per_rank)


def max_over_ranks(value, dist, device):
    """Timing rule: the step time of a multi-rank run is the maximum over ranks."""
    if dist is None:
        return float(value)
    import torch
    tt = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def workload_name(name, cfg):
    g = cfg["grid"]
    return "%s: %d curves x %s epochs, %d freqs in [%.4g,%.4g]/d, %d bins, q in [%g,%g], top-%d" % (
        name, cfg["n_curves"], (str(cfg["n_min"]) if cfg["n_min"] == cfg["n_max"] else "%d-%d" % (cfg["n_min"], cfg["n_max"])),
        g.nf, g.fmin, g.fmax, g.nb, g.qmin, g.qmax, cfg["top_k"])


def profile_facts(name):
    """Per-launch DRAM bytes and shared wavefronts per (curve, frequency) pair of the search kernel from the
    committed `ncu --set full` captures (profiles/search_kernel_ncu_facts.json); None where not captured."""
    p = os.path.join(ROOT, "profiles", "search_kernel_ncu_facts.json")
    try:
        return json.load(open(p)).get(name) or {}
    except Exception:
        return {}


def parity_of_sample(batch, grid, freqs, kmin, kmax, k, curves, spectra, peaks):
    """The timed step's peak lists (and their SR values) against the oracle spectra of the cpu_baseline
    sample: tests/comparator.py, the same checks `pytest -m gpu` runs (peaks-only: the timed step writes no
    spectrum, so SR is compared at the reported peaks)."""
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle
    from comparator import SR_RTOL, compare_peaks, exact_tie_runs
    rep = {"curves": len(curves), "peak_slots": 0, "max_rel_err_at_peaks": 0.0, "exact_tie_slots": 0,
           "near_tie_slots": 0, "unexplained": 0, "tolerance": "SR 1e-4 rel; peak lists = R14 on the tie-collapsed "
           "oracle spectrum, near-ties inside 2e-6 counted (tests/comparator.py)"}
    for c, orc in zip(curves, spectra):
        st, o_sr, o_a, o_k, _ = orc
        pk = peaks[c]
        t = batch.curve(c)[0]
        try:
            if np.array_equal(oracle.peaks(o_sr, k), pk["freq_index"]):
                r = compare_peaks(o_sr, pk["freq_index"], pk["sr"], k)
            else:
                ties, _ = exact_tie_runs(t, freqs, grid.nb, o_sr, o_a, o_k)
                r = compare_peaks(o_sr, pk["freq_index"], pk["sr"], k, ties=ties)
            rep["exact_tie_slots"] += r["exact_tie_slots"]
            rep["near_tie_slots"] += r["near_tie_slots"]
            idx = pk["freq_index"][pk["freq_index"] >= 0]
            if idx.size:
                rel = np.abs(pk["sr"][:idx.size].astype(np.float64) - o_sr[idx]) / o_sr[idx]
                rep["max_rel_err_at_peaks"] = max(rep["max_rel_err_at_peaks"], float(rel.max()))
                if rel.max() > SR_RTOL:
                    rep["unexplained"] += 1
        except AssertionError as e:
            rep["unexplained"] += 1
            rep.setdefault("first_failure", str(e)[:200])
        rep["peak_slots"] += k
    return rep


def time_config(name, cfg, steps, warmup, *, rank=0, world=1, dist=None, local_rank=0, flags=0, do_e2e=True,
                do_cpu=True, workers=1, prefix_warmup=0, do_refine=False):
    """Time `steps` passes of the hot path over the configuration (this rank's replica).  Returns the
    fields of the bench line for it.  prefix_warmup > 0: the warm-up runs on that many curves, then one
    full untimed step grows the plan's scratch (long configurations in per_config)."""
    import torch
    import paper_1112_1701_b200 as bls
    from paper_1112_1701_b200 import binding as B

    dev = torch.device("cuda", local_rank)
    props = torch.cuda.get_device_properties(dev)
    n_sm = props.multi_processor_count
    grid = cfg["grid"]
    freqs = synth.freq_grid(grid)
    t_gen = time.perf_counter()
    batch = synth.make_batch(cfg, rank_curve_ids(cfg["n_curves"], rank), workers=workers)
    t_gen = time.perf_counter() - t_gen
    k = cfg["top_k"]
    n_pts, n_curves = batch.n_points, batch.n_curves
    pf_per_step = float(n_pts) * grid.nf

    plan = bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k, device=local_rank, flags=flags)
    kmin, kmax = plan.kmin, plan.kmax
    t_d = torch.from_numpy(batch.t).to(dev)
    m_d = torch.from_numpy(batch.mag).to(dev)
    s_d = torch.from_numpy(batch.sigma).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def step():
        plan.run(batch.offsets, t_d, m_d, s_d, batch.t_origin)
        return plan.topk(k)

    if prefix_warmup and prefix_warmup < n_curves:
        npre = int(batch.offsets[prefix_warmup])
        for _ in range(max(warmup, 3)):
            plan.run(batch.offsets[:prefix_warmup + 1], t_d[:npre], m_d[:npre], s_d[:npre], batch.t_origin[:prefix_warmup])
            plan.topk(k)
        step()
    else:
        for _ in range(max(warmup, 3)):
            step()
    torch.cuda.synchronize()
    launches_per_step = plan.query(B.QUERY_LAST_LAUNCHES)

    sampler = ClockSampler(local_rank)
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    search_ns, search_launches = 0, 0
    wall0 = time.perf_counter()
    for i in range(steps):
        flush.zero_()                       # L2 flush between timed iterations (outside the events)
        ev[i][0].record()
        raw = step()
        ev[i][1].record()
        search_ns += plan.query(B.QUERY_LAST_SEARCH_NS)   # synchronises; outside the event pair
        search_launches += plan.query(B.QUERY_LAST_SEARCH_LAUNCHES)
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    t_ms = max_over_ranks(t_ms, dist, dev)
    if dist:
        dist.barrier()
    ms_per_step = t_ms / steps
    value = world * pf_per_step / (ms_per_step * 1e-3)
    curves_s = world * n_curves / (ms_per_step * 1e-3)
    peaks = plan.peaks_to_numpy(raw, k)
    del flush

    # ---- f1: cost of refining the top-k peaks of the timed step (64 fine frequencies x 4 bin shifts each) ----
    refine = None
    if do_refine:
        plan.refine(k, 64, 4)                                 # warm-up (grows nothing: reuses the spectrum scratch)
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        r0.record()
        refined = plan.refine(k, 64, 4)
        r1.record()
        torch.cuda.synchronize()
        rms_ = r0.elapsed_time(r1)
        ok = refined["freq_index"] >= 0
        refine = {"api": "bls_refine(k=%d, n_fine=64, n_shift=4)" % k, "ms": rms_, "share_of_step": rms_ / ms_per_step,
                  "point_folds": float(n_pts) * k * 64 * 4,
                  "median_sr_gain": float(np.median(refined["sr"][ok] / refined["coarse_sr"][ok])) if ok.any() else None,
                  "median_sde": float(np.median(refined["sde"][ok])) if ok.any() else None}

    # ---- end to end: host buffers in, peaks out, through bls_search_host -------------------------
    e2e = None
    if do_e2e:
        pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
        ht, hm, hs = pin(batch.t), pin(batch.mag), pin(batch.sigma)
        long_step = ms_per_step > 1000.0
        for _ in range(1 if long_step else 2):
            plan.search_host(batch.offsets, ht, hm, hs, batch.t_origin, k)
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        n_e2e = 3 if long_step else max(3, min(steps, 10))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            hp, hst = plan.search_host(batch.offsets, ht, hm, hs, batch.t_origin, k)
        e2e_s = (time.perf_counter() - t0) / n_e2e
        e2e_s = max_over_ranks(e2e_s, dist, dev)
        assert np.array_equal(hp["freq_index"], peaks["freq_index"])
        e2e = {"value": world * pf_per_step / e2e_s, "unit": UNIT,
               "h2d_bytes_per_step": int(3 * 4 * n_pts + 8 * (n_curves + 1) + 8 * n_curves),
               "d2h_bytes_per_step": int(n_curves * k * B.PEAK_DTYPE.itemsize + 4 * n_curves),
               "ms_per_step": 1e3 * e2e_s, "steps": n_e2e, "api": "bls_search_host (pinned host buffers)"}
        del ht, hm, hs

    out = {"value": value, "ms_per_step": ms_per_step, "curves_per_sec": curves_s, "e2e": e2e, "clocks": clocks,
           "gpu_launches": int(launches_per_step * steps), "wall_s_timed_region": wall, "steps": steps, "refine": refine,
           "config": {"workload": workload_name(name, cfg), "curves_per_gpu": n_curves, "points_per_gpu": n_pts,
                      "l2": "flushed between timed iterations (256 MB memset)",
                      "timing": "CUDA events per step on the launching stream, max over ranks",
                      "generation_s": round(t_gen, 1)},
           "canonical_rule_point_folds_per_step": plan.query(B.QUERY_LAST_CANONICAL)}
    if rank != 0:
        plan.destroy()
        return out

    # ---- roofline of the dominant kernel (search) -----------------------------------------------
    nk = kmax - kmin + 1
    n_mean = n_pts / n_curves
    kernel_name = {1: "search_kernel", 2: "search_ws_kernel", 3: "search_wt_kernel"}.get(plan.query(B.QUERY_SEARCH_KERNEL), "?")
    search_s = search_ns * 1e-9 / steps
    achieved = pf_per_step / search_s
    max_hz = (clocks.get("sm_max_mhz") or props.clock_rate / 1e3) * 1e6
    pc = pair_clocks(n_mean, grid.nb, kmax, nk)
    clk_per_pair = n_sm * max_hz * search_s / (n_curves * grid.nf)
    peak = n_sm * max_hz * n_mean / pc["min"]
    facts = profile_facts(name)
    # per launch (one launch = one chunk of curves): pairs, algorithmic point-folds, average duration, DRAM bytes
    pairs_per_launch = n_curves * grid.nf * steps / max(search_launches, 1)
    bpp = facts.get("dram_bytes_per_pair")
    out["roofline"] = {
        "bound": "alu", "kernel": kernel_name, "achieved": achieved, "peak": peak, "unit": UNIT, "frac": achieved / peak,
        "traffic": (bpp * pairs_per_launch) if bpp else None,
        "per_launch": {"launches_per_step": search_launches / steps, "avg_launch_ms": 1e3 * search_s * steps / max(search_launches, 1),
                       "point_folds": pf_per_step * steps / max(search_launches, 1),
                       "traffic_is_from_committed_ncu_capture_not_this_run": "dram__bytes_read.sum + dram__bytes_write.sum per (curve, frequency) pair of the "
                                         "ncu --set full capture (%s) x pairs per launch" % facts.get("source")},
        "peak_def": "n_SM*f_max*N/t_min per (curve,frequency) pair, t_min = max(LSU (2N+2(nb+kmax))/32, XU nb*nk/16, "
                    "issue (5N+3.5 nb nk)/128) clk = max(%.0f, %.0f, %.0f); rates measured by microbench/issue_rates.cu "
                    "(profiles/r02b_microbench.md); f_max=%d MHz, n_SM=%d (DESIGN.md section 7)" % (
                        pc["lsu"], pc["xu"], pc["issue"], max_hz / 1e6, n_sm),
        "clk_per_pair": clk_per_pair,
        "frac_method_floor": pc["method"] / clk_per_pair,
        "method_floor_def": "max(LSU, issue) only: the XU term (one MUFU.RSQ per box) is a property of the instruction mix "
                            "chosen for the division, not of the method; the >= 50 %% target is claimed against `frac`",
        "frac_sum_form": pc["sum_form"] / clk_per_pair,
        "fold_stage_peak": n_sm * max_hz * LSU_LANE_OPS_PER_CLK_SM / 2.0,
        "frac_of_fold_stage_peak": achieved / (n_sm * max_hz * LSU_LANE_OPS_PER_CLK_SM / 2.0),
        "lsu_wavefronts_per_pair": {"measured": facts.get("shared_wavefronts_per_pair"),
                                    "algorithmic": (2.0 * n_mean + 2.0 * (grid.nb + kmax)) / 32.0},
        "kernel_ms": 1e3 * search_s, "kernel_share_of_step": search_s / (ms_per_step * 1e-3),
        "box_evals_per_s": n_curves * grid.nf * grid.nb * nk / search_s,
        "peak_source": "derived from measured issue rates (no HBM/tensor bound applies); "
                       "MEASURED_PEAKS.json hbm_gbs is not the bound of this kernel"}

    # ---- the oracle beside it (bounded sample) and the parity of the timed step against it -------
    if do_cpu and world == 1:                              # rank 0 at N = 1 only
        import oracle
        cores = oracle.host_cores()
        # bounded sample: a short probe sizes the sample to about 15 s of wall time on this box's cores
        probe = list(range(min(n_curves, cores)))
        _, cv_probe, _, _, _ = oracle_rate(cfg, batch, freqs, kmin, kmax, probe)
        n_s = int(min(n_curves, max(len(probe), 15.0 * cv_probe)))
        curves = list(range(n_s))
        pf_s, cv_s, used, dt, spectra = oracle_rate(cfg, batch, freqs, kmin, kmax, curves)
        out["cpu_baseline"] = {"value": pf_s, "unit": UNIT, "cores": used, "kind": "oracle", "curves_per_sec": cv_s,
                               "sample": "first %d curves x all %d frequencies of %s, %.1f s wall" % (n_s, grid.nf, name, dt),
                               "parity": parity_of_sample(batch, grid, freqs, kmin, kmax, k, curves, spectra, peaks)}
    plan.destroy()
    return out


def time_field(local_rank=0, n_stars=30000, nf=5000, nb=64, steps=3):
    """per_config["F2"]: bls_run_field on one synthetic pointing at the paper's cadence (140 and 300 shared epochs,
    2 % absent, 64 bins, widths 1..10), through the field kernel (three stars per CTA share each epoch's bin index)
    and through the per-star kernels on the same inputs: search-kernel time from the library's own CUDA events."""
    import torch
    import paper_1112_1701_b200 as bls
    from paper_1112_1701_b200 import binding as B
    dev = torch.device("cuda", local_rank)
    props = torch.cuda.get_device_properties(dev)
    clk = props.clock_rate * 1e3                     # max SM clock, Hz (as the roofline block uses)
    grid = synth.Grid(nf, 0.1, 5.0, nb, 0.01, 0.15)
    freqs = synth.freq_grid(grid)
    out = {"workload": "F2: one pointing, %d stars x {140, 300} shared epochs (2 %% absent), %d freqs in [0.1,5]/d, %d bins, "
                       "q in [0.01,0.15], top-5" % (n_stars, nf, nb), "steps": steps}
    for n_epochs in (140, 300):
        t, mag, sig = synth.make_field(n_stars, n_epochs, seed=n_epochs)
        td, md, sd = (torch.from_numpy(x).to(dev) for x in (t, mag, sig))
        n_present = int(np.isfinite(mag).sum())
        row = {}
        for name, flags in (("field_kernel", 0), ("per_star_kernels", B.BLS_FLAG_NO_FIELD_KERNEL)):
            with bls.Plan(n_bins=nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=5, device=local_rank, flags=flags) as plan:
                for _ in range(3):
                    plan.run_field(td, md, sd, 0.0)
                    plan.topk(5)
                ns = []
                for _ in range(steps):
                    plan.run_field(td, md, sd, 0.0)
                    plan.topk(5)
                    ns.append(plan.query(B.QUERY_LAST_SEARCH_NS))
                sec = float(np.mean(ns)) * 1e-9
                row[name] = {"kernel": int(plan.query(B.QUERY_SEARCH_KERNEL)), "search_ms": sec * 1e3,
                             "clk_per_pair": props.multi_processor_count * clk * sec / (n_stars * nf),
                             "point_folds_per_sec": n_present * nf / sec, "stars_per_sec": n_stars / sec}
        row["speedup"] = row["per_star_kernels"]["search_ms"] / row["field_kernel"]["search_ms"]
        out["E%d" % n_epochs] = row
    return out


PER_CONFIG = [("C0", 0), ("C1", 0), ("C3", 100), ("C4", 20000)]     # (name, curves of the warm-up prefix; 0 = whole batch)


def short(r):
    """The per_config entry of one configuration."""
    rf = r.get("roofline") or {}
    return {"workload": r["config"]["workload"], "steps": r["steps"], "ms_per_step": r["ms_per_step"],
            "point_folds_per_sec": r["value"], "curves_per_sec": r["curves_per_sec"], "kernel": rf.get("kernel"),
            "clk_per_pair": rf.get("clk_per_pair"), "roofline_frac": rf.get("frac"),
            "frac_method_floor": rf.get("frac_method_floor"), "frac_of_fold_stage_peak": rf.get("frac_of_fold_stage_peak"),
            "kernel_share_of_step": rf.get("kernel_share_of_step"),
            "clocks": r["clocks"], "generation_s": r["config"]["generation_s"], "refine_top_k": r.get("refine")}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--max-curves", type=int, default=0, help="run only a prefix of the configuration")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (C0, C1, C3, C4)")
    ap.add_argument("--flags", type=lambda v: int(v, 0), default=0, help="bls_config.flags (tuning only)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = dict(synth.config(args.config))
    if args.max_curves:
        cfg["n_curves"] = min(cfg["n_curves"], args.max_curves)

    if args.impl == "reference":
        run_reference(args, cfg, rank, world)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the BLS library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    try:
        workers = max(1, len(os.sched_getaffinity(0)) // max(world, 1))
    except AttributeError:  # pragma: no cover
        workers = os.cpu_count() or 1

    # weak scaling: every rank searches its own n_curves curves (curve ids offset by rank)
    r = time_config(args.config, cfg, args.steps, args.warmup, rank=rank, world=world, dist=dist, local_rank=local_rank,
                    flags=args.flags, do_e2e=not args.no_e2e, do_cpu=not args.no_cpu_baseline, workers=workers,
                    do_refine=(world == 1))
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    per_config = None
    if not args.no_per_config and world == 1 and not args.max_curves:
        per_config = {}
        for name, prefix in PER_CONFIG:
            if name == args.config:
                continue
            try:
                rc = time_config(name, dict(synth.config(name)), 3 if prefix == 0 else 1, 3, local_rank=local_rank, flags=args.flags,
                                 do_e2e=False, do_cpu=False, workers=workers, prefix_warmup=prefix)
                per_config[name] = short(rc)
            except Exception as e:  # a secondary line must not sink the headline
                per_config[name] = {"error": repr(e)[:300]}
        per_config[args.config] = short(r)
        try:
            per_config["F2"] = time_field(local_rank)
        except Exception as e:
            per_config["F2"] = {"error": repr(e)[:300]}

    line = {"metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32 fixed-point bins, fp64 phase, fp32 box ranking, fp64 SR from integer box sums",
            "data": "synthetic", "curves_per_sec": r["curves_per_sec"], "config": r["config"],
            "e2e": r["e2e"], "gpu_launches": r["gpu_launches"], "clocks": r["clocks"],
            "roofline": r.get("roofline"), "cpu_baseline": r.get("cpu_baseline"), "refine_top_k": r.get("refine"),
            "per_config": per_config,
            "wall_s_timed_region": r["wall_s_timed_region"],
            "canonical_rule_point_folds_per_step": r["canonical_rule_point_folds_per_step"]}
    print(json.dumps(line), flush=True)
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
