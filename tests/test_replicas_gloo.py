"""N > 1 path on CPU: world_size-2 gloo processes exercise the replica logic bench.py uses under torchrun (which
events and seeds a rank owns, max-over-ranks time, summed work).  No GPU and no product kernel is involved: the
data path has no collective (replicas only)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import workloads
    from paper_2203_11043_b200 import replicas
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # one independent event per rank: different seeds give different clouds
        w = workloads.make(0, seed=replicas.rank_seed(workloads.SEED, rank), n=64)
        # a batch of independent events sharded over the ranks
        we = workloads.make_events([5, 0, 7, 3, 11])
        lo, hi, loc = replicas.shard_offsets(we["offsets"], rank, world)
        ms_local = 10.0 + 5.0 * rank                       # rank 1 is the slower one
        units_local = float(len(w["xyz"]) ** 2 + (hi - lo))
        dist.barrier()
        rate, ms, units = replicas.whole_job_rate(ms_local, units_local)
        q.put((rank, float(w["xyz"].sum()), lo, hi, loc.tolist(), rate, ms, units))
    finally:
        dist.destroy_process_group()


def test_two_rank_replicas_aggregate_max_time_and_summed_work():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, lo0, hi0, loc0, rate0, ms0, u0), (r1, s1, lo1, hi1, loc1, rate1, ms1, u1) = out
    assert s0 != s1                                         # independent events
    assert (lo0, hi0, lo1, hi1) == (0, 12, 12, 26)          # events [0,3) and [3,5) of sizes 5,0,7 | 3,11
    assert loc0 == [0, 5, 5, 12] and loc1 == [0, 3, 14]
    assert ms0 == ms1 == 15.0                               # max over ranks
    assert u0 == u1 == 2 * 64 * 64 + 26                     # sum over ranks
    assert rate0 == rate1 == pytest.approx(u0 / 15e-3)


def test_shard_events_is_a_balanced_partition():
    sys.path.insert(0, ROOT)
    from paper_2203_11043_b200 import replicas
    for n in (0, 1, 7, 8, 1000):
        for world in (1, 2, 3, 8):
            cuts = [replicas.shard_events(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        replicas.shard_events(4, 2, 2)
    assert replicas.aggregate(3.0, 4.0) == (3.0, 4.0)       # no process group: identity
