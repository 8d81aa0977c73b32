"""GPU parity at BASELINE.json's full sizes (configs 2-4), in the launch configuration bench.py times.
The oracle cannot run these in full, so it computes sampled outputs one by one: the field at sampled targets
against all sources, and one whole step of sampled carriers restarted from an exported GPU snapshot
(snapshot-restart).  Invariants hold at any size."""
import numpy as np
import pytest

from oracle import goracle as g
import workloads
from util import field_rel_err, gpu_sim, oracle_params

pytestmark = pytest.mark.gpu

M_SAMPLE = {2: 2048, 3: 1024, 4: 512}


def _sampled_field_check(sim, P, rng, m):
    xyz, ids = sim.read_carriers()
    E = sim.eval_field()
    t = np.sort(rng.choice(len(xyz), size=min(m, len(xyz)), replace=False)).astype(np.uint64)
    Eref = g.coulomb_field(xyz.astype(np.float64), eps_um=P["softening_um"], Kp=g.coulomb_constant(P["eps_si"]), targets=t)
    unfl, fl = field_rel_err(E[t.astype(np.int64)], Eref)
    assert unfl <= 1e-4, (unfl, fl)
    return xyz, ids, t, Eref


def _snapshot_restart_check(sim, w, xyz, ids, t, Eref):
    """Oracle advances the sampled carriers one step from the GPU snapshot; compare with the GPU's next step."""
    step = sim.state()["step"]
    op = oracle_params(w, flags=g.FP32_STATE)
    sim.step(1)
    xyz1, ids1 = sim.read_carriers()
    pos_of = {int(i): k for k, i in enumerate(ids1)}
    worst, flag_mismatch = 0.0, 0
    for k, j in enumerate(t.astype(np.int64)):
        r_new, collected = g.advance(op, step, int(ids[j]), xyz[j].astype(np.float64), Eref[k])
        if int(ids[j]) in pos_of:
            if collected:
                flag_mismatch += 1
                assert abs(r_new[2]) < 1e-3
                continue
            worst = max(worst, float(np.abs(xyz1[pos_of[int(ids[j])]].astype(np.float64) - r_new).max()))
        else:
            if not collected:
                flag_mismatch += 1
                assert abs(r_new[2]) < 1e-3
    assert worst <= 2e-4, worst           # one step: FP32 field error x drift + one FP32 rounding of the position
    assert flag_mismatch <= 1


@pytest.mark.parametrize("cfg", [2, 3, 4])
def test_full_size_sampled_field_and_snapshot_restart(cfg):
    w = workloads.make(cfg)
    P = w["params"]
    n0 = len(w["xyz"])
    rng = np.random.default_rng(cfg)
    sim = gpu_sim(w)
    sim.load_carriers(w["xyz"])
    st = sim.state()
    assert st["n_loaded"] == n0 and st["n_active"] + st["n_collected"] == n0
    xyz, ids, t, Eref = _sampled_field_check(sim, P, rng, M_SAMPLE[cfg])
    _snapshot_restart_check(sim, w, xyz, ids, t, Eref)
    # a few more steps, then again on the evolved (and, for tracks, compacted) state
    sim.step(9 if cfg < 4 else 3)
    st = sim.state()
    img, over = sim.read_image()
    assert int(img.sum()) + over + st["n_active"] == n0
    xyz, ids, t, Eref = _sampled_field_check(sim, P, rng, M_SAMPLE[cfg])
    assert np.all(np.diff(ids.astype(np.int64)) > 0)
    assert np.all(xyz[:, 2] > 0) and np.all(xyz[:, 2] <= 675.0) and np.isfinite(xyz).all()
    if cfg < 4:
        _snapshot_restart_check(sim, w, xyz, ids, t, Eref)
    sim.close()


def test_cfg2_ten_step_trajectories_on_sampled_carriers():
    # 10 GPU steps at N = 131,072; the oracle follows 256 sampled carriers with fields from the GPU's own
    # exported snapshots (each snapshot is an independent one-step check; errors do not compound through chaos)
    w = workloads.make(2)
    P = w["params"]
    sim = gpu_sim(w)
    sim.load_carriers(w["xyz"])
    rng = np.random.default_rng(42)
    t = np.sort(rng.choice(len(w["xyz"]), size=256, replace=False)).astype(np.uint64)
    op = oracle_params(w, flags=g.FP32_STATE)
    worst = 0.0
    for s in range(10):
        xyz, ids = sim.read_carriers()
        assert len(ids) == len(w["xyz"])                   # nobody arrives in the first 10 steps from 600 um
        Eref = g.coulomb_field(xyz.astype(np.float64), eps_um=P["softening_um"], Kp=g.coulomb_constant(P["eps_si"]), targets=t)
        sim.step(1)
        xyz1, _ = sim.read_carriers()
        for k, j in enumerate(t.astype(np.int64)):
            r_new, _c = g.advance(op, s, int(ids[j]), xyz[j].astype(np.float64), Eref[k])
            worst = max(worst, float(np.abs(xyz1[j].astype(np.float64) - r_new).max()))
    assert worst <= 2e-4, worst
    assert sim.state()["pair_interactions"] == 10 * 131072 ** 2
    sim.close()
