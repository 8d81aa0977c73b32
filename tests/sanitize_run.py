"""Small cases that reach every kernel family of the library, for compute-sanitizer (SURVEY.md section 4 T6, section 5
"Race detection"):

    compute-sanitizer --tool racecheck|memcheck|initcheck|synccheck python tests/sanitize_run.py

One tool per run (B200_PROFILING.md).  Not a pytest file: the sanitizer slows kernels 10-100x, so the sizes are the
smallest that still take every code path (several tiles, ragged tails, decaying populations).  Exits non-zero if a
result is inconsistent; the sanitizer reports its own findings."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import torch  # noqa: E402
import workloads  # noqa: E402
from paper_2203_11043_b200 import binding, sharded  # noqa: E402


def conserved(sim, n):
    st = sim.state()
    img, over = sim.read_image()
    assert int(img.sum()) + over + st["n_active"] == n, (int(img.sum()), over, st, n)


def main():
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)
    done = []
    # all-pairs: one-step kernels k_field<1|2|4> + k_advance (persistent path off), shared-memory double buffering
    for n in (700, 3500, 13000):
        w = workloads.make(3, n=n)
        s = binding.from_workload(w, stream=stream)
        s.set_persistent(False)
        s.load_carriers(w["xyz"])
        s.eval_field()
        s.step(9)                    # 8 through the CUDA graph + 1 direct
        conserved(s, n)
        s.close()
        done.append("k_field/k_advance n=%d" % n)
    # persistent multi-step kernels: k_steps_warp<1|2> (a warp owns its targets: shuffle butterfly, one grid barrier per
    # step, normals drawn in the barrier wait) and k_steps<1|2|4> (grid barriers, two-level scans, ping-pong state)
    for n, mode in ((300, 1), (2500, 1), (5000, 1), (12500, 1), (300, 2), (2500, 2)):
        w = workloads.make(3, n=n)
        s = binding.from_workload(w, stream=stream)
        s.set_persistent(mode)
        s.load_carriers(w["xyz"])
        s.step(7)
        conserved(s, n)
        s.run_to_collection(40)
        conserved(s, n)
        s.close()
        done.append("k_steps n=%d" % n)
    # Coulomb off: k_drift_multi + k_compact
    w = workloads.make(0, n=900)
    s = binding.from_workload(w, flags=binding.COULOMB_OFF, stream=stream)
    s.load_carriers(w["xyz"])
    s.step(30)
    conserved(s, 900)
    s.close()
    done.append("k_drift_multi")
    # batched events: warp-per-event, CTA-per-event tiers, cluster-per-event (DSMEM)
    sizes = [5, 26, 40, 100, 200, 400, 700, 1500, 0, 3000]
    we = workloads.make_events(sizes)
    s = binding.from_workload(we, max_carriers=len(we["xyz"]), stream=stream)
    s.load_events(we["xyz"], we["offsets"])
    s.run_events(12)
    conserved(s, len(we["xyz"]))
    s.close()
    done.append("k_events / k_events_warp / k_events_cluster")
    # treecode: Hilbert keys, radix sort, nodes, walk, evaluate; then the switch back to all-pairs as the track decays
    w = workloads.make(3, n=30000)
    s = binding.from_workload(w, stream=stream)
    s.set_farfield(0.5, min_active=20000)
    s.load_carriers(w["xyz"])
    s.step(10)
    conserved(s, 30000)
    s.close()
    done.append("k_tree_* / k_radix_*")
    # target sharding: k_shard_compact / k_shard_commit over 3 virtual ranks
    w = workloads.make(1, n=8 * 300)
    alloc = lambda nb: torch.empty(nb, dtype=torch.uint8, device="cuda")
    es = [binding.from_workload(w, stream=stream) for _ in range(3)]
    vr = sharded.VirtualRanks(es, alloc)
    vr.load_carriers(w["xyz"])
    vr.step(6)
    tot = vr.totals()
    assert int(vr.image().sum()) + tot["n_out_of_window"] + tot["n_active"] == 8 * 300
    for e in es:
        e.close()
    done.append("k_shard_*")
    # front end: k_gen_cloud / k_gen_events
    s = binding.Gcoreccd(4096, stream=stream)
    s.generate_cloud(1000, (0.0, 0.0, 100.0), 0.5, 7)
    s.step(3)
    conserved(s, 1000)
    s.reset()
    s.generate_xray_events([100.0, 1000.0, 5000.0], [(0, 0, 50.0), (30.0, 0, 300.0), (0, 40.0, 600.0)], [0.1, 0.3, 0.5], 9)
    s.run_events(5)
    s.close()
    done.append("k_gen_*")
    torch.cuda.synchronize()
    print("sanitize_run: ok —", "; ".join(done))
    return 0


if __name__ == "__main__":
    sys.exit(main())
