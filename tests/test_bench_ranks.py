"""N > 1 path of bench.py on CPU (gloo, world_size 2): replicas only -- each rank generates its own
disjoint curves from the per-curve addressable generator, and the step time is the max over ranks."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    import synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = dict(synth.config("T1"))
    cfg["n_curves"] = 3
    ids = list(bench.rank_curve_ids(cfg["n_curves"], rank))
    batch = synth.make_batch(cfg, ids)
    t_ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))
    gathered = [None] * world
    dist.all_gather_object(gathered, (ids, batch.n_points, float(batch.t.sum()), t_ms))
    if rank == 0:
        out.put(gathered)
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_take_disjoint_curves_and_max_time():
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get()
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (ids0, n0, s0, t0), (ids1, n1, s1, t1) = res
    assert ids0 == [0, 1, 2] and ids1 == [3, 4, 5]
    assert (n0, s0) != (n1, s1)                     # different curves, not copies
    assert t0 == t1 == 15.0                          # max over ranks, same on every rank
    # the rank's batch is exactly the corresponding slice of the whole configuration
    sys.path.insert(0, ROOT)
    import synth
    cfg = dict(synth.config("T1"))
    whole = synth.make_batch(cfg, range(6))
    assert n0 + n1 == whole.n_points
    assert np.isclose(s0 + s1, float(whole.t.sum()), rtol=1e-6)
