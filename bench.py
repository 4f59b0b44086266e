#!/usr/bin/env python
"""bench.py -- throughput of the BLS hot path on B200 (BASELINE.json metric: point-folds/s, curves/s,
fraction of the stated roofline), with the fp64 oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C1] [--impl ours|reference]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

A "step" is one pass of the whole hot path (prep -> fold/search -> peaks -> top-k) over one batch of
synthetic light curves of the chosen configuration (default C1 = BASELINE.json configs[1]: 1,000
curves x 1,500 epochs, 20,000 frequencies, 200 bins).  Prints ONE JSON line (rank 0).

  value      whole-job point-folds/s, inputs resident in HBM (CUDA events around bls_run + bls_topk)
  e2e        the same metric through bls_search_host with pinned HOST buffers (H2D + D2H inside)
  roofline   the search kernel against the issue-rate roofline stated in DESIGN.md
  cpu_baseline  the oracle as it stands on the host cores, bounded sample
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

# Roofline constants, measured on B200 by paper_1112_1701_b200/microbench/issue_rates.cu
# (profiles/r01a_microbench.md): lane-operations per clock per SM.
LSU_LANE_OPS_PER_CLK_SM = 32.0       # shared wavefront pipe: conflict-free ATOMS.ADD 31.96
XU_LANE_OPS_PER_CLK_SM = 16.0        # MUFU.RSQ 16.00: one per box
ISSUE_LANE_INSTR_PER_CLK_SM = 128.0  # 4 schedulers x 32 lanes
FOLD_MIN_INSTR, BOX_MIN_INSTR = 5.0, 4.5
N_SM = 148


def pair_clocks(n_mean, nb, kmax, nk):
    """Lower bounds, in SM clocks, for one (curve, frequency) pair on one SM."""
    t_lsu = (2.0 * n_mean + 2.0 * (nb + kmax)) / LSU_LANE_OPS_PER_CLK_SM
    t_xu = nb * nk / XU_LANE_OPS_PER_CLK_SM
    t_issue = (FOLD_MIN_INSTR * n_mean + BOX_MIN_INSTR * nb * nk) / ISSUE_LANE_INSTR_PER_CLK_SM
    t_sum = 2.0 * n_mean / LSU_LANE_OPS_PER_CLK_SM + nb * nk / XU_LANE_OPS_PER_CLK_SM   # SURVEY 8(d) sum form
    return {"lsu": t_lsu, "xu": t_xu, "issue": t_issue, "min": max(t_lsu, t_xu, t_issue), "sum_form": t_sum}


def stated_peak_pf_per_s(n_mean, nb, kmax, nk, clk_hz, n_sm=N_SM, which="min"):
    """Whole-path ceiling n_SM * f * N / t_min, t_min = max over pipes."""
    return n_sm * clk_hz * n_mean / pair_clocks(n_mean, nb, kmax, nk)[which]


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
    """Time the oracle as it stands on `curves` of the batch at all frequencies."""
    import oracle
    oracle.lib()
    t0 = time.perf_counter()
    _, used = oracle.spectrum_batch(batch.offsets, batch.t, batch.mag, batch.sigma, freqs,
                                    cfg["grid"].nb, kmin, kmax, curves=curves, threads=threads)
    dt = time.perf_counter() - t0
    pts = sum(int(batch.offsets[c + 1] - batch.offsets[c]) for c in curves)
    return pts * len(freqs) / dt, len(curves) / dt, used, dt


def run_reference(args, cfg, rank, world):
    """--impl reference: the fp64 oracle on the host cores, same metric/config.  Rank 0 only."""
    if rank != 0:
        return
    import oracle
    grid = cfg["grid"]
    freqs = synth.freq_grid(grid)
    kmin, kmax = oracle.widths(grid.nb, grid.qmin, grid.qmax)
    cores = oracle.host_cores()
    n_sample = max(cores, 8)           # curves per step: about 0.5 s/curve/core at C1
    batch = synth.make_batch(cfg, range(min(n_sample, cfg["n_curves"])))
    curves = list(range(batch.n_curves))
    for _ in range(min(args.warmup, 1)):
        oracle_rate(cfg, batch, freqs, kmin, kmax, curves[:cores])
    tot_pf, tot_t, used = 0.0, 0.0, cores
    for _ in range(args.steps):
        pf_s, _, used, dt = oracle_rate(cfg, batch, freqs, kmin, kmax, curves)
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C1")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--max-curves", type=int, default=0, help="run only a prefix of the configuration")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
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
    import paper_1112_1701_b200 as bls
    from paper_1112_1701_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the BLS library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    # weak scaling: every rank searches its own n_curves curves (curve ids offset by rank)
    grid = cfg["grid"]
    freqs = synth.freq_grid(grid)
    ids = rank_curve_ids(cfg["n_curves"], rank)
    batch = synth.make_batch(cfg, ids)
    k = cfg["top_k"]
    n_pts, n_curves = batch.n_points, batch.n_curves
    pf_per_step = float(n_pts) * grid.nf

    plan = bls.Plan(n_bins=grid.nb, q_min=grid.qmin, q_max=grid.qmax, freqs=freqs, max_top_k=k, device=local_rank, flags=args.flags)
    kmin, kmax = plan.kmin, plan.kmax
    t_d = torch.from_numpy(batch.t).to(dev)
    m_d = torch.from_numpy(batch.mag).to(dev)
    s_d = torch.from_numpy(batch.sigma).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def step():
        plan.run(batch.offsets, t_d, m_d, s_d, batch.t_origin)
        return plan.topk(k)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    launches_per_step = plan.query(B.QUERY_LAST_LAUNCHES)

    sampler = ClockSampler(local_rank)
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    search_ns = 0
    wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.zero_()                       # L2 flush between timed iterations (outside the events)
        ev[i][0].record()
        raw = step()
        ev[i][1].record()
        search_ns += plan.query(B.QUERY_LAST_SEARCH_NS)   # synchronises; outside the event pair
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    t_ms = max_over_ranks(t_ms, dist, dev)
    if dist:
        dist.barrier()
    ms_per_step = t_ms / args.steps
    value = world * pf_per_step / (ms_per_step * 1e-3)
    curves_s = world * n_curves / (ms_per_step * 1e-3)
    peaks = plan.peaks_to_numpy(raw, k)

    # ---- end to end: host buffers in, peaks out, through bls_search_host -------------------------
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
        ht, hm, hs = pin(batch.t), pin(batch.mag), pin(batch.sigma)
        for _ in range(2):
            plan.search_host(batch.offsets, ht, hm, hs, batch.t_origin, k)
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        n_e2e = max(3, min(args.steps, 10))
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            hp, hst = plan.search_host(batch.offsets, ht, hm, hs, batch.t_origin, k)
        e2e_s = (time.perf_counter() - t0) / n_e2e
        e2e_s = max_over_ranks(e2e_s, dist, dev)
        assert np.array_equal(hp["freq_index"], peaks["freq_index"])
        e2e = {"value": world * pf_per_step / e2e_s, "unit": UNIT,
               "h2d_bytes_per_step": int(3 * 4 * n_pts + 8 * (n_curves + 1) + 8 * n_curves),
               "d2h_bytes_per_step": int(n_curves * k * B.PEAK_DTYPE.itemsize + 4 * n_curves),
               "ms_per_step": 1e3 * e2e_s, "api": "bls_search_host (pinned host buffers)"}

    if rank != 0:
        plan.destroy()
        if dist:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (search) -----------------------------------------------
    nk = kmax - kmin + 1
    n_mean = n_pts / n_curves
    plan_kernel_name = {1: "search_kernel", 2: "search_ws_kernel", 3: "search_wt_kernel"}.get(plan.query(B.QUERY_SEARCH_KERNEL), "?")
    search_s = search_ns * 1e-9 / args.steps
    achieved = pf_per_step / search_s
    max_hz = (clocks.get("sm_max_mhz") or 1965) * 1e6
    peak = stated_peak_pf_per_s(n_mean, grid.nb, kmax, nk, max_hz)
    peak_sum = stated_peak_pf_per_s(n_mean, grid.nb, kmax, nk, max_hz, which="sum_form")
    pc = pair_clocks(n_mean, grid.nb, kmax, nk)
    traffic = None
    tp = os.path.join(ROOT, "profiles", "search_kernel_dram_bytes.json")
    if os.path.exists(tp):
        try:
            traffic = json.load(open(tp)).get(args.config)
        except Exception:
            traffic = None
    roofline = {"bound": "alu", "kernel": plan_kernel_name, "achieved": achieved, "peak": peak,
                "unit": UNIT, "frac": achieved / peak, "traffic": traffic,
                "peak_def": "n_SM*f_max*N/t_min per (curve,frequency) pair, t_min = max(LSU (2N+2(nb+kmax))/32, XU nb*nk/16, "
                            "issue (5N+4.5 nb nk)/128) clk = max(%.0f, %.0f, %.0f); rates measured by microbench/issue_rates.cu "
                            "(profiles/r01a_microbench.md); f_max=%d MHz, n_SM=%d (DESIGN.md section 7)" % (
                                pc["lsu"], pc["xu"], pc["issue"], max_hz / 1e6, N_SM),
                "clk_per_pair": N_SM * max_hz * search_s / (n_curves * grid.nf),
                "frac_sum_form": achieved / peak_sum,
                "fold_stage_peak": N_SM * max_hz * LSU_LANE_OPS_PER_CLK_SM / 2.0,
                "frac_of_fold_stage_peak": achieved / (N_SM * max_hz * LSU_LANE_OPS_PER_CLK_SM / 2.0),
                "kernel_ms": 1e3 * search_s, "kernel_share_of_step": search_s / (ms_per_step * 1e-3),
                "box_evals_per_s": n_curves * grid.nf * grid.nb * nk / search_s,
                "peak_source": "derived from measured issue rates (no HBM/tensor bound applies); "
                               "MEASURED_PEAKS.json hbm_gbs is not the bound of this kernel"}

    # ---- the oracle beside it (bounded sample; also a parity spot check of the timed result) -----
    cpu = None
    if not args.no_cpu_baseline and world == 1:           # rank 0 at N = 1 only
        import oracle
        cores = oracle.host_cores()
        # bounded sample: a short probe sizes the sample to about 15 s of wall time on this box's cores
        probe = list(range(min(n_curves, cores)))
        _, cv_probe, _, _ = oracle_rate(cfg, batch, freqs, kmin, kmax, probe)
        n_s = int(min(n_curves, max(len(probe), 15.0 * cv_probe)))
        curves = list(range(n_s))
        pf_s, cv_s, used, dt = oracle_rate(cfg, batch, freqs, kmin, kmax, curves)
        cpu = {"value": pf_s, "unit": UNIT, "cores": used, "kind": "oracle", "curves_per_sec": cv_s,
               "sample": "first %d curves x all %d frequencies of %s, %.1f s wall" % (n_s, grid.nf, args.config, dt)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32 fixed-point bins, fp64 phase, fp32 box statistic",
            "data": "synthetic", "curves_per_sec": curves_s,
            "config": {"workload": workload_name(args.config, cfg), "curves_per_gpu": n_curves,
                       "points_per_gpu": n_pts, "l2": "flushed between timed iterations (256 MB memset)",
                       "timing": "CUDA events per step on the launching stream, max over ranks"},
            "e2e": e2e, "gpu_launches": int(launches_per_step * args.steps), "clocks": clocks,
            "roofline": roofline, "cpu_baseline": cpu, "wall_s_timed_region": wall,
            "canonical_rule_point_folds_per_step": plan.query(B.QUERY_LAST_CANONICAL)}
    print(json.dumps(line), flush=True)
    plan.destroy()
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
