"""Pins of the oracle's time step: drift against closed forms and golden Euler runs,
two-carrier repulsion against r^3 = r0^3 + 6 mu0 K' t, diffusion against the lateral-spread closed
form, invariants (conservation, ordering, restart) and the FP32-state mode."""
import math

import numpy as np
import pytest

from oracle import goracle as g
import workloads


def _sim(**kw):
    return g.Sim(g.make_params(**kw))


# ------------------------------------------------------------------ drift only
def test_euler_drift_golden(golden):
    for z0, steps, zf in golden("euler_drift.txt"):
        s = _sim(flags=g.COULOMB_OFF | g.DIFFUSION_OFF)
        s.load(np.array([[0.0, 0.0, float(z0)]], dtype=np.float32))
        done = s.run(100000)
        assert done == int(steps)
        xyz, st = s.collected()
        assert xyz[0, 2] == pytest.approx(float(zf), abs=1e-5)
        assert xyz[0, 0] == 0.0 and xyz[0, 1] == 0.0                     # the depletion field is z-directed
        assert int(st[0]) == int(steps) - 1


def test_drift_time_low_field_closed_form():
    # For |E| << E_c eq. 2 gives mu -> mu0 and dz/dt = 1e-5 mu0 (a1 z 1e-4 - a2) integrates to
    # t = ln(a2/(a2 - a1 z0 1e-4)) / (1e-9 a1 mu0)  [ns].  Fields of a few V/cm: (E/E_c)^beta < 1e-3.
    a1, a2, z0 = 28.1, 2.0, 600.0
    mu0 = g.mobility(0.0, 140.0)
    t_exact = math.log(a2 / (a2 - a1 * z0 * 1e-4)) / (1e-9 * a1 * mu0)
    errs = []
    for dt in (40.0, 20.0, 10.0):
        s = _sim(a1=a1, a2=a2, dt_ns=dt, flags=g.COULOMB_OFF | g.DIFFUSION_OFF)
        s.load(np.array([[0.0, 0.0, z0]], dtype=np.float32))
        steps = s.run(10 ** 7)
        # interpolate the crossing inside the last step for a sub-step estimate
        xyz, _ = s.collected()
        v_end = 1e-5 * mu0 * a2                                           # speed at z ~ 0
        t_num = steps * dt - (0.0 - xyz[0, 2]) / v_end
        errs.append(t_num - t_exact)
    assert abs(errs[-1]) / t_exact < 2e-3                                 # mobility correction + O(dt)
    # first-order convergence of explicit Euler: the error halves with dt (after removing the dt-independent part)
    d1, d2 = errs[0] - errs[1], errs[1] - errs[2]
    assert d1 / d2 == pytest.approx(2.0, rel=0.15)


def test_drift_time_converges_to_quadrature_of_eq2():
    # t(z0) = int_0^z0 dz / (1e-5 mu(|E(z)|) |E(z)|), by Simpson on the oracle's own mu (this pins the
    # integrator, not eq. 2).  SURVEY App. A quotes 6.1134 ns (200 um) and 30.548 ns (600 um).
    a1, a2 = 2.81e4, 2.0e3
    for z0, t_survey in [(200.0, 6.1134), (600.0, 30.548)]:
        zs = np.linspace(0.0, z0, 20001)
        Es = np.abs(a1 * zs * 1e-4 - a2)
        f = 1.0 / (1e-5 * np.array([g.mobility(E, 140.0) for E in Es]) * Es)
        h = zs[1] - zs[0]
        t_quad = h / 3 * (f[0] + f[-1] + 4 * f[1:-1:2].sum() + 2 * f[2:-1:2].sum())
        assert t_quad == pytest.approx(t_survey, rel=2e-5)
        errs = []
        for dt in (0.05, 0.025):
            s = _sim(dt_ns=dt, flags=g.COULOMB_OFF | g.DIFFUSION_OFF)
            s.load(np.array([[0.0, 0.0, z0]], dtype=np.float32))
            steps = s.run(10 ** 6)
            xyz, _ = s.collected()
            v_end = 1e-5 * g.mobility(a2, 140.0) * a2
            errs.append(steps * dt + xyz[0, 2] / v_end - t_quad)
        assert abs(errs[0]) < 0.05 and abs(errs[1]) < abs(errs[0])        # O(dt)
        assert errs[0] / errs[1] == pytest.approx(2.0, rel=0.2)


def test_drift_step_bounded_by_saturation_velocity():
    w = workloads.make(0)
    s = g.Sim(g.make_params(**{**_kw(w), "flags": g.DIFFUSION_OFF}))
    s.load(w["xyz"])
    vsat_dt = 1.31e8 * 1.24 * 140.0 ** -0.52 * 1e-5 * 0.05                 # 6.218 um
    assert vsat_dt == pytest.approx(6.218, abs=1e-3)
    for _ in range(5):
        before, ids0 = s.carriers()
        s.step(1)
        after, ids1 = s.carriers()
        keep = np.isin(ids0, ids1)
        assert np.linalg.norm(after - before[keep], axis=1).max() <= vsat_dt


def _kw(w):
    P = w["params"]
    return dict(T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"], z_well_um=P["z_well_um"],
                pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"], softening_um=P["softening_um"],
                eps_si=P["eps_si"], seed=P["seed"], img_nx=P["img_nx"], img_ny=P["img_ny"],
                img_x0_um=P["img_x0_um"], img_y0_um=P["img_y0_um"])


# ------------------------------------------------------------------ two carriers, Coulomb only
def _separation(r0, t, dt, eps=1e-3):
    s = _sim(dt_ns=dt, softening_um=eps, thickness_um=1e6, flags=g.DEPLETION_OFF | g.DIFFUSION_OFF)
    s.load(np.array([[-r0 / 2, 0.0, 500.0], [r0 / 2, 0.0, 500.0]], dtype=np.float64).astype(np.float32))
    s.step(int(round(t / dt)))
    xyz, _ = s.carriers()
    assert abs(xyz[0, 1]) + abs(xyz[1, 1]) == 0.0 and xyz[0, 2] == xyz[1, 2] == 500.0   # motion stays on the axis
    assert xyz[0, 0] == pytest.approx(-xyz[1, 0], rel=1e-14)                             # symmetric
    return xyz[1, 0] - xyz[0, 0]


def test_two_carrier_separation_golden_and_closed_form(golden):
    for r0, t, closed, euler in golden("two_carrier.txt"):
        r0, t, closed, euler = float(r0), float(t), float(closed), float(euler)
        # the closed form itself, from the golden constant mu0 K'
        assert (r0 ** 3 + 6 * 0.030616501 * t) ** (1 / 3) == pytest.approx(closed, rel=1e-8)
        assert _separation(r0, t, 0.05) == pytest.approx(euler, abs=1e-6)


def test_two_carrier_separation_converges_to_closed_form():
    # r^3 = r0^3 + 6 mu0 K' 1e-5 t for constant mobility; at 1 um the field is 1.2 V/cm << E_c so eq. 2
    # deviates by (E/E_c)^beta/beta ~ 1e-4 relative in mu, i.e. ~2e-5 um in r.
    r0, t = 1.0, 10.0
    closed = (r0 ** 3 + 6 * 1e-5 * g.mobility(0.0, 140.0) * g.coulomb_constant(11.7) * t) ** (1 / 3)
    seps = [_separation(r0, t, dt) for dt in (0.1, 0.05, 0.025, 0.0125)]
    assert all(s > closed for s in seps)                                  # Euler overshoots a decelerating expansion
    d = np.diff(seps)                                                     # first order: successive differences halve
    assert d[0] / d[1] == pytest.approx(2.0, rel=0.05) and d[1] / d[2] == pytest.approx(2.0, rel=0.05)
    # Richardson extrapolation lands on the eq.-2 + softening ODE value the survey quotes (1.41561185)
    rich = 2 * seps[3] - seps[2]
    assert rich == pytest.approx(1.41561185, abs=2e-6)
    assert rich == pytest.approx(closed, abs=5e-5)


# ------------------------------------------------------------------ diffusion, Coulomb off
@pytest.mark.parametrize("z0", [200.0, 600.0])
def test_lateral_spread_closed_form(golden, z0):
    sig = {float(r[0]): float(r[1]) for r in golden("lateral_sigma.txt")}
    # closed form from golden constants: 2 (kT/q)/a1 ln(a2/(a2-a1 z0)), a1 per cm -> um^2 needs 1e8/1e4... done in um:
    kT = 0.0120642666
    var = 2 * kT / (2.81e4 * 1e-8) * math.log(2e3 / (2e3 - 2.81e4 * z0 * 1e-4))
    assert math.sqrt(var) == pytest.approx(sig[z0], rel=1e-5)
    n = 200000
    s = _sim(flags=g.COULOMB_OFF, img_nx=8, img_ny=8)
    s.load(np.tile(np.array([[0.0, 0.0, z0]], dtype=np.float32), (n, 1)))
    s.run(100000)
    xyz, st = s.collected()
    assert s.state()["n_active"] == 0 and not np.isnan(xyz).any()
    vx, vy = xyz[:, 0].var(), xyz[:, 1].var()
    assert vx == pytest.approx(var, rel=0.012) and vy == pytest.approx(var, rel=0.012)   # 1 % + sampling sqrt(2/N)=0.3 %
    assert abs(xyz[:, 0].mean()) < 4 * math.sqrt(var / n) and abs(xyz[:, 1].mean()) < 4 * math.sqrt(var / n)
    assert abs(np.corrcoef(xyz[:, 0], xyz[:, 1])[0, 1]) < 0.01
    # arrival-step window quoted in SURVEY App. D for dt = 0.05 ns
    lo, hi = (109, 138) if z0 == 200.0 else (544, 708)
    assert lo - 15 <= st.min() and st.max() <= hi + 25


def test_lateral_spread_tightens_with_dt():
    z0, n = 10.0, 100000
    var = 1.10226 ** 2
    r = []
    for dt in (0.05, 0.0125):
        s = _sim(flags=g.COULOMB_OFF, dt_ns=dt, img_nx=8, img_ny=8)
        s.load(np.tile(np.array([[0.0, 0.0, z0]], dtype=np.float32), (n, 1)))
        s.run(100000)
        xyz, _ = s.collected()
        r.append(0.5 * (xyz[:, 0].var() + xyz[:, 1].var()) / var)
    assert abs(r[1] - 1.0) < abs(r[0] - 1.0) + 0.01 and abs(r[1] - 1.0) < 0.03


# ------------------------------------------------------------------ whole-step invariants
def test_conservation_ordering_and_slab_invariants_every_step():
    w = workloads.make(0, n=256)
    s = g.Sim(g.make_params(**_kw(w)))
    s.load(w["xyz"])
    n0 = 256
    prev_ids = s.carriers()[1]
    assert np.array_equal(prev_ids, np.arange(n0))                        # ids = load order
    pairs = 0
    while s.state()["n_active"] > 0:
        na = s.state()["n_active"]
        s.step(1)
        pairs += na * na
        st = s.state()
        xyz, ids = s.carriers()
        assert int(s.image().sum()) + st["n_out_of_window"] + st["n_active"] == n0
        assert st["n_collected"] == n0 - st["n_active"]
        assert np.all(np.diff(ids.astype(np.int64)) > 0) and np.all(np.isin(ids, prev_ids))   # stable compaction
        assert np.all(xyz[:, 2] > 0.0) and np.all(xyz[:, 2] <= 675.0)
        assert st["pair_interactions"] == pairs
        prev_ids = ids
    assert 110 <= s.state()["step"] <= 170                                # 136 steps for cfg 0
    assert s.step(5) == 0 and s.state()["step"] <= 170                    # no-op once empty


def test_restart_equivalence_counter_based_rng():
    w = workloads.make(1, n=8 * 16)
    a = g.Sim(g.make_params(**_kw(w)))
    a.load(w["xyz"])
    a.step(20)
    b = g.Sim(g.make_params(**_kw(w)))
    b.load(w["xyz"])
    b.step(10)
    xyz, ids = b.carriers()
    c = g.Sim(g.make_params(**_kw(w)))
    c.load_state(xyz, ids, b.state()["step"])
    c.step(10)
    xa, ia = a.carriers()
    xc, ic = c.carriers()
    assert np.array_equal(ia, ic) and np.array_equal(xa, xc)


def test_load_rules():
    s = _sim()
    with pytest.raises(ValueError):
        s.load(np.array([[0, 0, 676.0]], dtype=np.float32))               # above the back surface
    with pytest.raises(ValueError):
        s.load(np.array([[0, np.nan, 1.0]], dtype=np.float32))
    s.load(np.array([[7.0, -8.0, 0.0], [0.0, 0.0, 5.0], [1e5, 0.0, -1.0]], dtype=np.float32))
    st = s.state()
    assert st["n_active"] == 1 and st["n_collected"] == 2 and st["n_out_of_window"] == 1
    img = s.image()
    assert img.sum() == 1 and img[(int((-8.0 + 480) // 15)), int((7.0 + 480) // 15)] == 1
    assert s.carriers()[1].tolist() == [1]


def test_reflection_at_back_surface():
    # Coulomb and depletion off, diffusion on: a carrier just below the back surface must stay inside the slab
    s = _sim(flags=g.COULOMB_OFF | g.DEPLETION_OFF, img_nx=4, img_ny=4)
    s.load(np.tile(np.array([[0, 0, 674.9]], dtype=np.float32), (4096, 1)))
    s.step(1)
    xyz, ids = s.carriers()
    assert xyz[:, 2].max() <= 675.0 and (xyz[:, 2] > 674.9).sum() > 0
    # mirrored population: without reflection half would be above 675; z-distribution is folded
    sig = g.diffusion_sigma(g.mobility(0.0, 140.0), 140.0, 0.05)
    frac_far = (xyz[:, 2] < 674.9 - sig).mean()
    assert frac_far == pytest.approx(0.1587 + (1 - 0.5 * (1 + math.erf((sig + 0.2) / sig / math.sqrt(2)))), abs=0.03)


def test_fp32_state_mode_rounds_state_only():
    w = workloads.make(0, n=64)
    p64 = g.make_params(**_kw(w))
    p32 = g.make_params(**{**_kw(w), "flags": g.FP32_STATE})
    a, b = g.Sim(p64), g.Sim(p32)
    a.load(w["xyz"])
    b.load(w["xyz"])
    a.step(1)
    b.step(1)
    xa, xb = a.carriers()[0], b.carriers()[0]
    assert np.array_equal(xb, xa.astype(np.float32).astype(np.float64))   # one step: identical up to the final rounding
    b.step(9)
    xb = b.carriers()[0]
    assert np.array_equal(xb, xb.astype(np.float32).astype(np.float64))


def test_coulomb_widens_the_collected_cloud():
    # PAPER.md:56 "larger as the number of charges is increased": sigma_final(Coulomb on) > Coulomb off, grows with N
    res = {}
    for n in (128, 1024):
        w = workloads.make(0, n=n)
        for fl in (0, g.COULOMB_OFF):
            s = g.Sim(g.make_params(**{**_kw(w), "flags": fl}))
            s.load(w["xyz"])
            s.run(10000)
            xyz, _ = s.collected()
            res[(n, fl)] = math.sqrt(0.5 * (xyz[:, 0].var() + xyz[:, 1].var()))
    assert res[(1024, 0)] > res[(1024, g.COULOMB_OFF)] * 1.05
    assert res[(1024, 0)] > res[(128, 0)]
    assert res[(1024, g.COULOMB_OFF)] == pytest.approx(math.sqrt(28.3269 + 1.0), rel=0.06)   # 5.415 um
