"""Writes tests/golden/traj10_cfg{2,3,4}.txt: the first 10 steps of a FULL-SIZE config on the ORACLE, sampled.

    python tests/golden/make_trajectory_goldens.py 3       # cfg3, 262,144 holes: 10 x 6.9e10 pairs, ~5 min on 8 cores
    python tests/golden/make_trajectory_goldens.py 2       # cfg2, 131,072 holes: ~1 min
    python tests/golden/make_trajectory_goldens.py 4       # cfg4, 1,048,576 holes: 10 x 1.1e12 pairs, > 1 h

Imports only oracle/ and the seeded input generator (workloads.py); nothing here touches the CUDA path.

BASELINE.json:north_star: "trajectories within 1e-3 um after 10 steps".  The oracle (FP32-state mode, PAPER.md:84;
the step of PAPER.md:68) advances ALL holes of the config 10 steps; for M sampled holes (seeded choice among the holes
still drifting after 10 steps) the file keeps the id, the position after step 10, and the smallest distance to any
other drifting hole seen at the start of each of the 10 steps (R21: a hole may leave the 1e-3 um band only
after an oracle-side encounter closer than 0.1 um).  Also kept: n_active after each step, and the ids among the
sampled range that were collected inside the window (retire decisions).
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

STEPS = 10
M = 1024


def nearest_other(xyz, rows):
    """Distance from each hole in `rows` to its nearest OTHER hole of xyz (float64, chunked)."""
    out = np.empty(len(rows))
    c = max(1, int(2e7 // max(1, len(xyz))))
    for a in range(0, len(rows), c):
        r = rows[a:a + c]
        d2 = ((xyz[None, :, :] - xyz[r][:, None, :]) ** 2).sum(axis=2)
        d2[np.arange(len(r)), r] = np.inf
        out[a:a + c] = np.sqrt(d2.min(axis=1))
    return out


def run(cfg, log=sys.stderr):
    w = workloads.make(cfg)
    P = w["params"]
    prm = g.make_params(T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"],
                        z_well_um=P["z_well_um"], pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"],
                        softening_um=P["softening_um"], eps_si=P["eps_si"], seed=P["seed"],
                        img_nx=P["img_nx"], img_ny=P["img_ny"], img_x0_um=P["img_x0_um"],
                        img_y0_um=P["img_y0_um"], flags=g.FP32_STATE)
    sim = g.Sim(prm)
    n0 = len(w["xyz"])
    rng = np.random.default_rng(1000 + cfg)
    # cfg4 is ten steps of 1.1e12 pairs each: the run is checkpointed after every step and resumes from the checkpoint
    # (the oracle's restart is bit-exact: tests/test_oracle_step.py "restart equivalence"; FP32-state mode)
    ckpt = os.path.join(HERE, "traj10_cfg%d.txt.ckpt.npz" % cfg)
    if os.path.exists(ckpt):
        c = np.load(ckpt)
        assert int(c["n0"]) == n0
        sim.load_state(c["xyz"].astype(np.float64), c["ids"], int(c["step"]))
        pick, n_act, s_done, wall = c["pick"], [int(v) for v in c["n_act"]], int(c["step"]), float(c["wall"])
        closest = {int(i): float(v) for i, v in zip(pick, c["closest"])}
        print("resumed from %s at step %d" % (ckpt, s_done), file=log, flush=True)
    else:
        sim.load(w["xyz"])
        _, ids0 = sim.carriers()
        pick = np.sort(rng.choice(ids0, size=min(2 * M, len(ids0)), replace=False))     # candidates; survivors are cut to M
        closest = {int(i): np.inf for i in pick}
        n_act = [sim.state()["n_active"]]
        s_done, wall = 0, 0.0
    t0 = time.time() - wall
    for s in range(s_done, STEPS):
        xyz, ids = sim.carriers()
        rows = np.searchsorted(ids, pick)
        ok = (rows < len(ids))
        ok[ok] &= ids[rows[ok]] == pick[ok]
        d = nearest_other(xyz, rows[ok])
        for i, v in zip(pick[ok], d):
            closest[int(i)] = min(closest[int(i)], float(v))
        sim.step(1)
        n_act.append(sim.state()["n_active"])
        print("cfg%d step %d n_active %d  %.0f s" % (cfg, s + 1, n_act[-1], time.time() - t0), file=log, flush=True)
        if s + 1 < STEPS and time.time() - t0 > float(os.environ.get("GOLDEN_CKPT_S", "300")):
            xyz, ids = sim.carriers()
            assert np.array_equal(xyz, xyz.astype(np.float32).astype(np.float64))
            np.savez_compressed(ckpt + ".tmp.npz", n0=n0, xyz=xyz.astype(np.float32), ids=ids, step=s + 1, pick=pick,
                                closest=np.array([closest[int(i)] for i in pick]), n_act=np.array(n_act),
                                wall=time.time() - t0)
            os.replace(ckpt + ".tmp.npz", ckpt)
    xyz, ids = sim.carriers()
    alive = pick[np.isin(pick, ids)]
    retired = pick[~np.isin(pick, ids)]
    keep = alive[:M] if len(alive) > M else alive
    lines = []
    A = lines.append
    A("# Oracle, first %d steps of the full-size config, sampled holes.  Written by" % STEPS)
    A("# tests/golden/make_trajectory_goldens.py %d (oracle/goracle.c, FP32-state mode, on workloads.make(%d))." % (cfg, cfg))
    A("# %s" % w["name"])
    A("# north_star: trajectories within 1e-3 um after 10 steps (PAPER.md:68 step, PAPER.md:84 FP32 state)")
    A("n_loaded %d" % n0)
    A("steps %d" % STEPS)
    A("n_active " + " ".join(str(v) for v in n_act))
    A("# ids of sampled candidates collected inside the window")
    A("retired " + " ".join(str(int(v)) for v in retired))
    A("# hole id  x y z after step %d (um, FP32 values)  smallest distance to another drifting hole in the window (um)" % STEPS)
    rows = np.searchsorted(ids, keep)
    for i, r in zip(keep, rows):
        A("hole %d %.9g %.9g %.9g %.6g" % (int(i), xyz[r, 0], xyz[r, 1], xyz[r, 2], closest[int(i)]))
    out = os.path.join(HERE, "traj10_cfg%d.txt" % cfg)
    with open(out + ".tmp", "w") as f:
        f.write("\n".join(lines) + "\n")
    os.replace(out + ".tmp", out)
    if os.path.exists(ckpt):
        os.remove(ckpt)
    sim.close()
    return out


if __name__ == "__main__":
    print(run(int(sys.argv[1])))
