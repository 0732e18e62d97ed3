"""The N>1 path of bench.py on CPU: two gloo ranks, as torchrun would start them.

The hot path does not shard ("replicas only"): the only exchange between ranks is the
MAX of the timed region, and the whole-job value is world x per-replica units / that time.  These
tests run bench.py's own helpers under a real world_size-2 gloo group (rendezvous on 127.0.0.1).
"""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    import tracegen
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # each rank "measured" a different time; every rank must see the maximum
        ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))
        dist.barrier()
        # every rank draws its own traces: same config, different seeds
        cfg = tracegen.scaled(tracegen.get_config(2), N=512, N_eval=512, L=1)
        params = tracegen.make_params(cfg)
        idx, _ = tracegen.gen_trace(cfg, params, seed=bench.rank_seed(cfg.seed, 0, rank))
        sums = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
        dist.all_gather(sums, idx.to(torch.int64).sum().reshape(1))
        out.put((rank, ms, [int(x) for x in sums], bench.whole_job_value(1000, 4, world, ms)))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_max_time_and_independent_traces():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, sums, value in res:
        assert ms == 15.0                                   # MAX over ranks, seen by every rank
        assert sums[0] != sums[1]                           # the replicas' traces differ
        assert value == 2 * 1000 * 4 / 15e-3                # whole-job aggregate over both replicas


def test_single_rank_needs_no_group():
    import bench
    assert bench.max_over_ranks(3.5, None, torch.device("cpu")) == 3.5
    assert bench.rank_seed(2000, 1, 3) == 2000 + 17 + 3027
