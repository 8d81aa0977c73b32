"""Writes tests/golden/full_run_cfg{1,2,3}.txt and full_run_cfg4_n131072.txt: whole events on the ORACLE, load -> full collection.

    python tests/golden/make_full_run_goldens.py 1      # cfg1, 16,384 holes: ~4e11 pairs, minutes
    python tests/golden/make_full_run_goldens.py 2      # cfg2, 131,072 holes: ~1e13 pairs, 3 h on 8 cores / 31 min on 16 fast ones
    python tests/golden/make_full_run_goldens.py 3      # cfg3, 262,144-hole track: 1.1e13 pairs
    python tests/golden/make_full_run_goldens.py 4 131072   # cfg4's mix of 4 tracks + 64 clouds at 1/8 of its holes
    python tests/golden/make_full_run_goldens.py 4 524288   # ... at 1/2: 4.4e13 pairs, 2.3 h on 16 fast cores
                                                            # (full_run_cfg4_n<N>.txt; full size is 1.8e14 pairs)

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
SUB = 5


def run(cfg, n=None, out=None, log=sys.stderr):
    w = workloads.make(cfg, n=n)
    P = w["params"]
    prm = g.make_params(T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"],
                        z_well_um=P["z_well_um"], pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"],
                        softening_um=P["softening_um"], eps_si=P["eps_si"], seed=P["seed"],
                        img_nx=P["img_nx"], img_ny=P["img_ny"], img_x0_um=P["img_x0_um"],
                        img_y0_um=P["img_y0_um"], flags=g.FP32_STATE)
    n0 = len(w["xyz"])
    # A run of hours is checkpointed every EVERY steps (carriers, ids, step and what has been collected so far) and
    # resumes from the checkpoint if one is there: the oracle's restart is bit-exact (tests/test_oracle_step.py,
    # "restart equivalence"), a resumed run equals an uninterrupted one.  Everything collected before the
    # checkpoint is carried in `base`; the segment after it adds its own image, records and counters.
    out = out or os.path.join(HERE, "full_run_cfg%d%s.txt" % (cfg, "" if n is None else "_n%d" % n))
    ckpt = out + ".ckpt.npz"
    sim = g.Sim(prm)
    base = dict(img=np.zeros((P["img_ny"], P["img_nx"]), dtype=np.uint64), fin=np.full((n0, 3), np.nan),
                fstep=np.full(n0, np.iinfo(np.uint64).max, dtype=np.uint64), pairs=0, oow=0, wall=0.0)
    if os.path.exists(ckpt):
        c = np.load(ckpt)
        assert int(c["n0"]) == n0 and int(c["cfg"]) == cfg
        sim.load_state(c["xyz"].astype(np.float64), c["ids"], int(c["step"]))
        base.update(img=c["img"], fin=c["fin"], fstep=c["fstep"], pairs=int(c["pairs"]), oow=int(c["oow"]),
                    wall=float(c["wall"]))
        decay = [tuple(int(v) for v in r) for r in c["decay"]]
        print("resumed from %s at step %d, n_active %d" % (ckpt, int(c["step"]), len(c["ids"])), file=log, flush=True)
    else:
        sim.load(w["xyz"])
        decay = [(0, sim.state()["n_active"])]

    def merged():
        st = sim.state()
        img = base["img"] + sim.image().astype(np.uint64)
        f, fs = sim.collected()
        fin, fstep = base["fin"].copy(), base["fstep"].copy()
        m = fs[:n0] != np.iinfo(np.uint64).max
        fin[:len(m)][m] = f[:n0][m]
        fstep[:len(m)][m] = fs[:n0][m]
        return st, img, fin, fstep, base["pairs"] + st["pair_interactions"], base["oow"] + st["n_out_of_window"]

    t0 = time.time()
    last_save = t0
    while sim.state()["n_active"] > 0:
        # (in sub-chunks, so that a checkpoint can be taken between the recorded decay points of a slow run)
        sim.step(min(SUB, EVERY - sim.state()["step"] % EVERY))
        st = sim.state()
        if st["step"] % EVERY == 0 or st["n_active"] == 0:
            decay.append((st["step"], st["n_active"]))
        print("cfg%d step %d n_active %d pairs %.4g  %.0f s" % (cfg, st["step"], st["n_active"],
                                                               base["pairs"] + st["pair_interactions"],
                                                               base["wall"] + time.time() - t0),
              file=log, flush=True)
        if time.time() - last_save > float(os.environ.get("GOLDEN_CKPT_S", "600")) and st["n_active"] > 0:
            _, img, fin, fstep, pairs, oow = merged()
            xyz, ids = sim.carriers()
            assert np.array_equal(xyz, xyz.astype(np.float32).astype(np.float64))   # FP32-state mode
            np.savez_compressed(ckpt + ".tmp.npz", cfg=cfg, n0=n0, xyz=xyz.astype(np.float32), ids=ids, step=st["step"],
                                img=img, fin=fin, fstep=fstep, pairs=pairs, oow=oow,
                                wall=base["wall"] + time.time() - t0, decay=np.array(decay, dtype=np.int64))
            os.replace(ckpt + ".tmp.npz", ckpt)
            last_save = time.time()
    st, img, fin, fstep, pairs, oow = merged()
    assert int(img.sum()) + oow == n0 and not np.isnan(fin).any()
    st = dict(st, pair_interactions=pairs, n_out_of_window=oow)
    t0 -= base["wall"]
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
    with open(out + ".tmp", "w") as f:
        f.write("\n".join(lines) + "\n")
    os.replace(out + ".tmp", out)
    if os.path.exists(ckpt):
        os.remove(ckpt)
    sim.close()
    return out


if __name__ == "__main__":
    cfg = int(sys.argv[1])
    n = int(sys.argv[2]) if len(sys.argv) > 2 else None
    print(run(cfg, n))
