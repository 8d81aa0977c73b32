"""Target sharding, N > 1 path on CPU: world_size-2 (and 3) gloo processes run the PRODUCT's
host orchestration (paper_2203_11043_b200/sharded.py: message sizing, all-gather of the shares, commit, integer
reductions of image and counters) around an oracle-backed engine (tests/shard_oracle_engine.py), and the result must
equal the unsharded oracle bit for bit: same FP64 arithmetic per target, same stable order."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
N_HOLES, STEPS = 700, 12


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _workload():
    import workloads
    w = workloads.make(3, n=N_HOLES)               # a track: holes retire from the first step on, shares move
    return w


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from paper_2203_11043_b200 import sharded
    from shard_oracle_engine import OracleShardEngine
    from util import oracle_params
    from oracle import goracle as g
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = _workload()
        eng = OracleShardEngine(oracle_params(w, flags=g.FP32_STATE), w["params"])
        ev = sharded.ShardedEvent(eng, rank, world,
                                  lambda mb: sharded.DistExchange(torch, "cpu", mb, world),
                                  lambda nb: torch.zeros(nb, dtype=torch.uint8))
        ev.load_carriers(w["xyz"])
        sizes = [ev.nbytes]
        ev.step(STEPS)
        st = ev.refresh()
        sizes.append(ev.nbytes)
        red = sharded.dist_reduce_sum(torch, "cpu")
        tot = ev.totals(red)
        img = ev.image(red)
        xyz, ids = eng.read_carriers()
        # a second leg through run_to_collection with a step cap
        done, left = ev.run_to_collection(max_steps=5)
        q.put((rank, st, tot, img, xyz, ids, sizes, done, left, eng.state()["step"]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_event_over_gloo_equals_the_unsharded_oracle(world):
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from util import oracle_sim
    from oracle import goracle as g
    port = _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted((q.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0

    w = _workload()
    o = oracle_sim(w, flags=g.FP32_STATE)
    o.load(w["xyz"])
    o.step(STEPS)
    oxyz, oids = o.carriers()
    ost = o.state()
    oimg = o.image()
    for rank, st, tot, img, xyz, ids, sizes, done, left, step_after in out:
        assert st["step"] == ost["step"] == STEPS and st["n_active"] == ost["n_active"]
        assert np.array_equal(ids, oids)
        assert np.array_equal(xyz.astype(np.float64), oxyz)              # bit-exact: same arithmetic, same order
        assert tot["n_collected"] == ost["n_collected"] and tot["n_out_of_window"] == ost["n_out_of_window"]
        assert tot["pair_interactions"] == ost["pair_interactions"]
        assert tot["n_active"] + tot["n_collected"] == N_HOLES
        assert np.array_equal(img, oimg)
        assert sizes[1] <= sizes[0] and (sizes[0] - 256) % (16 * 256) == 0
        assert done == 5 and step_after == STEPS + 5 and left > 0
    assert len({o_[8] for o_ in out}) == 1                               # every rank sees the same n_active
    # the holes retired between loads are split over the ranks: no rank saw all of them
    assert ost["n_collected"] > 0


def test_share_of_is_a_contiguous_tile_partition():
    sys.path.insert(0, ROOT)
    from paper_2203_11043_b200 import sharded
    for n in (0, 1, 255, 256, 257, 5000, 131072, 1048575):
        for world in (1, 2, 3, 8, 64):
            cuts = [sharded.share_of(n, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and sum(c[1] for c in cuts) == n
            pos = 0
            for t0, nt in cuts:
                assert t0 == pos or nt == 0
                assert t0 % 256 == 0 or nt == 0
                pos += nt
            tiles = [(nt + 255) // 256 for _, nt in cuts]
            assert max(tiles) - min(tiles) <= 1
