"""N > 1 path of bench.py on CPU: world_size-2 gloo.  The hot path does not shard (replicas only):
what N > 1 adds is the aggregation — step time = MAX over ranks, work units = SUM over ranks."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import synth
    assert bench.dist_env() == (rank, world, rank)
    w = synth.wan13b_batch()                         # every replica draws the same structure (weak scaling)
    flops = synth.attention_flops(w.shape, w.sessions)
    ms_local = 5.0 + rank                            # rank 1 is the slow one
    ms, units = bench.aggregate(ms_local, float(flops), world, torch.device("cpu"))
    ret[rank] = (ms, units, flops, [s.prior_frames for s in w.sessions])
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_max_time_sum_units():
    world = 2
    port = _free_port()
    ctx = mp.get_context("spawn")
    ret = ctx.Manager().dict()
    procs = [ctx.Process(target=_worker, args=(r, world, port, ret)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    (ms0, u0, f0, pr0), (ms1, u1, f1, pr1) = ret[0], ret[1]
    assert ms0 == ms1 == 6.0                         # max over ranks
    assert u0 == u1 == float(f0 + f1)                # whole-job units
    assert pr0 == pr1 == [15, 3, 0, 6, 6, 15, 9, 0]


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate(3.5, 7.0, 1, torch.device("cpu")) == (3.5, 7.0)
