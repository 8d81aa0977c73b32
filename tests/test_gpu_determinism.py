"""Race evidence without compute-sanitizer (closed on this pool, profiles/r2_sanitizer.md): every kernel family that
exchanges data through shared memory, DSMEM, look-back words or grid barriers is run TWICE from the same input and must
give bit-identical state, image, counters and collection records.  A data race (a missing barrier around the
double-buffered source tiles, a look-back that reads a stale count, an in-place compaction that overwrites an unread
slot) shows up as a difference between two runs or as a broken conservation law; it cannot hide behind a tolerance."""
import numpy as np
import pytest

import workloads
from paper_2203_11043_b200 import binding
from util import gpu_sim

pytestmark = pytest.mark.gpu


def _snapshot(sim, n):
    xyz, ids = sim.read_carriers()
    img, over = sim.read_image()
    st = sim.state()
    fin, fst = sim.read_collected()
    assert int(img.sum()) + over + st["n_active"] == n
    return xyz, ids, img, over, st, fin, fst


def _same(a, b):
    assert np.array_equal(a[1], b[1]) and np.array_equal(a[0], b[0])
    assert np.array_equal(a[2], b[2]) and a[3] == b[3] and a[4] == b[4]
    assert np.array_equal(a[6], b[6]) and np.array_equal(a[5], b[5], equal_nan=True)


@pytest.mark.parametrize("n,persist", [(700, False), (3500, False), (13000, False), (40000, False),
                                       (300, True), (2500, True), (5000, True), (12500, True), (24000, True),
                                       (300, 2), (2500, 2), (5000, 2)])
def test_all_pairs_steps_are_bit_reproducible(n, persist):
    w = workloads.make(3, n=n)                                                 # a track: retirements every step
    runs = []
    for _ in range(2):
        s = gpu_sim(w)
        s.set_persistent(persist)
        s.load_carriers(w["xyz"])
        s.step(21)
        runs.append(_snapshot(s, n))
        s.close()
    _same(*runs)
    assert runs[0][4]["n_active"] < n                                          # the compaction really ran on a shrinking set


def test_events_treecode_and_sharded_paths_are_bit_reproducible():
    import torch
    from paper_2203_11043_b200 import binding, sharded
    sizes = [5, 26, 40, 100, 200, 400, 700, 1500, 0, 3000, 4096]
    we = workloads.make_events(sizes)
    runs = []
    for _ in range(2):
        s = gpu_sim(we, max_carriers=len(we["xyz"]))
        s.load_events(we["xyz"], we["offsets"])
        s.run_events(15)
        img, over = s.read_image()
        act, stp = s.events()
        per = [s.read_event_carriers(e) for e in range(len(sizes))]
        runs.append((img, over, act, stp, per, s.state()))
        s.close()
    a, b = runs
    assert np.array_equal(a[0], b[0]) and a[1] == b[1] and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3]) and a[5] == b[5]
    for (xa, ia), (xb, ib) in zip(a[4], b[4]):
        assert np.array_equal(ia, ib) and np.array_equal(xa, xb)
    w = workloads.make(3, n=30000)
    runs = []
    for _ in range(2):
        s = gpu_sim(w)
        s.set_farfield(0.5, min_active=20000)
        s.load_carriers(w["xyz"])
        s.step(13)
        runs.append(_snapshot(s, 30000))
        s.close()
    _same(*runs)
    w = workloads.make(1, n=8 * 700)
    runs = []
    for _ in range(2):
        stream = torch.cuda.Stream()                          # virtual ranks are ordered by ONE stream
        es = [binding.from_workload(w, stream=stream) for _ in range(3)]
        vr = sharded.VirtualRanks(es, lambda nb: torch.empty(nb, dtype=torch.uint8, device="cuda"))
        vr.load_carriers(w["xyz"])
        vr.step(9)
        torch.cuda.synchronize()
        runs.append((es[0].read_carriers(), vr.image(), vr.totals()))
        for e in es:
            e.close()
    assert np.array_equal(runs[0][0][1], runs[1][0][1]) and np.array_equal(runs[0][0][0], runs[1][0][0])
    assert np.array_equal(runs[0][1], runs[1][1]) and runs[0][2] == runs[1][2]
