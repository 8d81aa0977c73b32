"""Helpers shared by the GPU parity tests: the same workload handed to the oracle and to the CUDA path."""
import os

import numpy as np

from oracle import goracle as g


def oracle_params(w, flags=0, **over):
    P = dict(w["params"])
    P.update(over)
    return g.make_params(T_K=P["T_K"], a1=P["a1"], a2=P["a2"], thickness_um=P["thickness_um"], z_well_um=P["z_well_um"],
                         pixel_pitch_um=P["pixel_pitch_um"], dt_ns=P["dt_ns"], softening_um=P["softening_um"],
                         eps_si=P["eps_si"], seed=P["seed"], img_nx=P["img_nx"], img_ny=P["img_ny"],
                         img_x0_um=P["img_x0_um"], img_y0_um=P["img_y0_um"], flags=flags)


def oracle_sim(w, flags=0, **over):
    s = g.Sim(oracle_params(w, flags, **over))
    return s


def gpu_sim(w, flags=0, max_carriers=None, **over):
    from paper_2203_11043_b200 import binding
    w2 = dict(w)
    w2["params"] = dict(w["params"])
    w2["params"].update(over)
    return binding.from_workload(w2, flags=flags, max_carriers=max_carriers)


def field_rel_err(E, Eref):
    """max_j |dE_j| / |E_j| (unfloored, the judged number) and the floored variant of DESIGN.md R20."""
    d = np.linalg.norm(E.astype(np.float64) - Eref, axis=1)
    nrm = np.linalg.norm(Eref, axis=1)
    rms = np.sqrt((nrm ** 2).mean())
    with np.errstate(divide="ignore", invalid="ignore"):
        unfloored = np.where(nrm > 0, d / nrm, 0.0)
    floored = d / np.maximum(nrm, 1e-3 * rms)
    return unfloored.max(), floored.max()


def image_moments(img, x0, y0, pitch):
    img = img.astype(np.float64)
    ny, nx = img.shape
    xs = x0 + (np.arange(nx) + 0.5) * pitch
    ys = y0 + (np.arange(ny) + 0.5) * pitch
    tot = img.sum()
    mx = (img.sum(axis=0) * xs).sum() / tot
    my = (img.sum(axis=1) * ys).sum() / tot
    vx = (img.sum(axis=0) * (xs - mx) ** 2).sum() / tot
    vy = (img.sum(axis=1) * (ys - my) ** 2).sum() / tot
    return mx, my, vx, vy


R_ENC = 0.1          # um: DESIGN.md R21 excuse radius (an ORACLE-side encounter closer than this inside the window)
EXCUSED = []         # (label, n_carriers, n_suspects) of every trajectory check of the session; printed by conftest


def closest_encounters(history, suspects):
    """Smallest distance to any other drifting hole that each suspect id saw at the start of a step of the oracle's
    window.  history = [(xyz, ids) before each step]."""
    closest = {int(i): np.inf for i in suspects}
    for hx, hid in history:
        for i in closest:
            k = np.searchsorted(hid, i)
            if k < len(hid) and hid[k] == i:
                r = np.linalg.norm(hx - hx[k], axis=1)
                r[k] = np.inf
                closest[i] = min(closest[i], float(r.min()))
    return closest


def traj_assert(xyz, ids, oxyz, oids, history, n_total, tol, r_enc=R_ENC, max_frac=0.02, label="",
                r_ext=None, max_ext=0, r_knock=None, max_knock=0):
    """GPU (xyz, ids) vs FP32-state oracle (oxyz, oids) after some steps; `history` = the oracle's (xyz, ids) before
    each of those steps.  DESIGN.md R21: a carrier may exceed `tol` (or differ in its retire flag) only if the ORACLE's
    trajectory shows a neighbour closer than r_enc = 0.1 um inside the window, and at most max_frac = 2 % (+2) may do
    so.  The number of excused carriers is recorded (EXCUSED) and bounded here, so the clause cannot silently absorb a
    regression.  DESIGN.md R21b (dense batched events only; the single-event tests leave these at 0): at most max_ext
    carriers per check may instead show an encounter inside r_ext (several steps of amplification at 0.1-0.2 um), and
    at most max_knock may be the knock-on of an excused carrier (closer than r_knock to one inside the window).
    Returns the per-carrier max-coordinate error."""
    common = np.intersect1d(ids, oids)
    xyz_c, oxyz_c = xyz[np.isin(ids, common)], oxyz[np.isin(oids, common)]
    d = np.abs(xyz_c.astype(np.float64) - oxyz_c).max(axis=1) if len(common) else np.zeros(0)
    suspects = sorted(set(common[d > tol].tolist()) | set(np.setxor1d(ids, oids).tolist()))   # incl. retire-flag mismatches
    closest = closest_encounters(history, suspects) if suspects else {}
    primary = [i for i, r in closest.items() if r < r_enc]
    ext = [i for i, r in closest.items() if not r < r_enc and r_ext is not None and r < r_ext]
    rest = [i for i in closest if i not in primary and i not in ext]
    knock = []
    if rest and r_knock is not None and (primary or ext):
        for i in rest:
            near = np.inf
            for hx, hid in history:
                k = np.searchsorted(hid, i)
                kp = np.searchsorted(hid, primary + ext)
                kp = kp[(kp < len(hid))]
                kp = kp[np.isin(hid[kp], primary + ext)]
                if k < len(hid) and hid[k] == i and len(kp):
                    near = min(near, float(np.linalg.norm(hx[kp] - hx[k], axis=1).min()))
            if near < r_knock:
                knock.append(i)
    EXCUSED.append((label, int(n_total), len(suspects), sorted(round(r, 4) for r in closest.values()), len(ext), len(knock)))
    if os.environ.get("GCORECCD_TRAJ_DIAG"):                 # survey mode: record every suspect, assert nothing
        return d
    assert len(suspects) <= max_frac * n_total + 2, (label, len(suspects), n_total)
    bad = {i: closest[i] for i in rest if i not in knock}
    assert not bad, (label, bad, "exceeds %g um without an oracle-side encounter inside %g um" % (tol, r_enc))
    assert len(ext) <= max_ext and len(knock) <= max_knock, (label, len(ext), len(knock), [closest[i] for i in ext + knock])
    return d
