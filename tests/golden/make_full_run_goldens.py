"""Writes tests/golden/full_run_cfg{1,2}.txt: whole events on the ORACLE, load -> full collection.

    python tests/golden/make_full_run_goldens.py 1      # cfg1, 16,384 holes: ~4e11 pairs, minutes
    python tests/golden/make_full_run_goldens.py 2      # cfg2, 131,072 holes: ~1e13 pairs, 1-2 h on 8 cores

Imports only oracle/ and the seeded input generator (workloads.py, which holds none of the method's
arithmetic); nothing here ever touches the CUDA path, so every stored value is the oracle's.

What is stored and why (BASELINE.json:north_star: "the collected image exactly conserving the hole count,
with per-pixel charge and cloud second moments within 1%"; Fig. 5 caption: the image is the
"2D histogram of the output positions", bin = pixel width; the loop runs until every charge has
arrived):
  * the run's step count, sum over steps of N_a^2, out-of-window count;
  * n_active after every 25th step (the decay of the population, PAPER.md:68 exit test);
  * per group (cloud) of the workload: count, centroid, second moments of the collected (x, y) and the mean
    collection step, from the oracle's per-id collection records;
  * the image, sparse (iy ix count).
The oracle runs in FP32-state mode (Pos is 3N floats; R19) from the same FP32 input the
GPU gets.  The system is chaotic (R16): the GPU tests compare these statistically, never bit for bit.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
sys.path.insert(0, ROOT)

import workloads                      # noqa: E402  (seeded inputs only)
from oracle import goracle as g       # noqa: E402

EVERY = 25


def run(cfg, n=None, out=None, log=sys.stderr):
    w = workloads.make(cfg, n=n)
    P = w["params"]
    prm = g.make_params(T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"],
                        z_well_um=P["z_well_um"], pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"],
                        softening_um=P["softening_um"], eps_si=P["eps_si"], seed=P["seed"],
                        img_nx=P["img_nx"], img_ny=P["img_ny"], img_x0_um=P["img_x0_um"],
                        img_y0_um=P["img_y0_um"], flags=g.FP32_STATE)
    sim = g.Sim(prm)
    sim.load(w["xyz"])
    n0 = len(w["xyz"])
    decay = [(0, sim.state()["n_active"])]
    t0 = time.time()
    while sim.state()["n_active"] > 0:
        sim.step(EVERY)
        st = sim.state()
        decay.append((st["step"], st["n_active"]))
        print("cfg%d step %d n_active %d pairs %.4g  %.0f s" % (cfg, st["step"], st["n_active"],
                                                               st["pair_interactions"], time.time() - t0),
              file=log, flush=True)
    st = sim.state()
    img = sim.image()
    fin, fstep = sim.collected()
    assert int(img.sum()) + st["n_out_of_window"] == n0 and st["n_collected"] == n0
    lines = []
    A = lines.append
    A("# Oracle full run, load -> full collection.  Written by tests/golden/make_full_run_goldens.py %d%s"
      % (cfg, "" if n is None else " %d" % n))
    A("# (oracle/goracle.c in FP32-state mode on workloads.make(%d%s); PAPER.md:68 loop, PAPER.md:122 image)."
      % (cfg, "" if n is None else ", n=%d" % n))
    A("# %s" % w["name"])
    A("# oracle threads %d, wall %.0f s" % (g.num_threads(), time.time() - t0))
    A("n_loaded %d" % n0)
    A("steps %d" % st["step"])
    A("pair_interactions %d" % st["pair_interactions"])
    A("out_of_window %d" % st["n_out_of_window"])
    A("image_shape %d %d" % img.shape)
    A("# n_active after step s (every %d steps; the last entry is the final step)" % EVERY)
    for s, na in decay:
        A("decay %d %d" % (s, na))
    A("# group name id_lo id_hi  mean_x mean_y  var_x var_y cov_xy  mean_collection_step   (um, um^2; collected x,y)")
    for name, lo, hi in w["groups"]:
        x, y = fin[lo:hi, 0], fin[lo:hi, 1]
        mx, my = x.mean(), y.mean()
        A("group %s %d %d  %.9f %.9f  %.9f %.9f %.9f  %.6f" % (name, lo, hi, mx, my, ((x - mx) ** 2).mean(),
                                                             ((y - my) ** 2).mean(), ((x - mx) * (y - my)).mean(),
                                                             fstep[lo:hi].astype(np.float64).mean()))
    A("# px iy ix count   (non-zero pixels, row-major [iy][ix])")
    iy, ix = np.nonzero(img)
    for a, b in zip(iy, ix):
        A("px %d %d %d" % (a, b, img[a, b]))
    out = out or os.path.join(HERE, "full_run_cfg%d.txt" % cfg)
    with open(out + ".tmp", "w") as f:
        f.write("\n".join(lines) + "\n")
    os.replace(out + ".tmp", out)
    sim.close()
    return out


if __name__ == "__main__":
    cfg = int(sys.argv[1])
    n = int(sys.argv[2]) if len(sys.argv) > 2 else None
    print(run(cfg, n))
