"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the CUDA path and the oracle (tests, bench.py) and therefore holds
none of the method's arithmetic: it only draws initial hole positions (float32, um) and
names the device constants of BASELINE.json:configs[0].  The X-ray clouds stand in for the
paper's Gaussian initial clouds and the straight tracks for its GEANT4
muon hole list, neither of which is available.
"""
import math

import numpy as np

SEED = 20220322

# BASELINE.json:configs[0] device constants (the paper prints only 675 um, 15 um and 140 K)
COMMON = dict(T_K=140.0, a1=2.81e4, a2=2.0e3, thickness_um=675.0, z_well_um=0.0,
              pixel_pitch_um=15.0, dt_ns=0.05, softening_um=1e-3, eps_si=11.7, seed=SEED)

CONFIG_N = {0: 1024, 1: 16384, 2: 131072, 3: 262144, 4: 1048576}


def _rng(seed, tag):
    return np.random.Generator(np.random.Philox(key=[int(seed) & (2 ** 64 - 1), int(tag)]))


def gaussian_cloud(rng, n, sigma_um, centre):
    return rng.standard_normal((n, 3)) * sigma_um + np.asarray(centre, dtype=np.float64)


def _reflect_into_slab(p, thickness):
    z = p[:, 2]
    over = z > thickness
    z[over] = 2.0 * thickness - z[over]
    return p


def straight_track(rng, n, entry_xy, zenith_rad, azimuth_rad, thickness, sigma_perp_um):
    """n holes uniform along the segment from (entry, z=thickness) to z=0, Gaussian offsets in the
    plane perpendicular to the track; z>thickness is mirrored back, z<=0 is left (collected at load)."""
    d = np.array([math.sin(zenith_rad) * math.cos(azimuth_rad), math.sin(zenith_rad) * math.sin(azimuth_rad),
                  -math.cos(zenith_rad)])
    length = thickness / math.cos(zenith_rad)
    start = np.array([entry_xy[0], entry_xy[1], thickness])
    # orthonormal basis of the transverse plane
    a = np.array([0.0, 0.0, 1.0]) if abs(d[2]) < 0.9 else np.array([1.0, 0.0, 0.0])
    e1 = np.cross(d, a)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(d, e1)
    s = rng.random(n) * length
    o = rng.standard_normal((n, 2)) * sigma_perp_um
    p = start + s[:, None] * d + o[:, :1] * e1 + o[:, 1:] * e2
    return _reflect_into_slab(p, thickness), start + 0.5 * length * d


def make(config, seed=SEED, n=None):
    """Return dict(xyz float32 (N,3), params dict, groups list of (name, id_lo, id_hi), name)."""
    P = dict(COMMON)
    P["seed"] = seed
    th, pitch = P["thickness_um"], P["pixel_pitch_um"]
    rng = _rng(seed, 0x494E4954 + config)
    groups = []
    if config == 0:
        N = n or CONFIG_N[0]
        xyz = gaussian_cloud(rng, N, 1.0, (0.0, 0.0, 200.0))
        P.update(img_nx=64, img_ny=64, img_x0_um=-480.0, img_y0_um=-480.0)
        groups.append(("cloud0", 0, N))
        name = "cfg0: point X-ray cloud, %d holes, sigma 1 um at depth 200 um" % N
    elif config == 1:
        per = 2048 if n is None else max(1, n // 8)
        parts = []
        for k in range(8):
            c = (rng.uniform(-480.0, 480.0), rng.uniform(-480.0, 480.0), rng.uniform(10.0, 665.0))
            parts.append(gaussian_cloud(rng, per, 0.5, c))
            groups.append(("cloud%d" % k, k * per, (k + 1) * per))
        xyz = np.concatenate(parts)
        P.update(img_nx=64, img_ny=64, img_x0_um=-480.0, img_y0_um=-480.0)
        name = "cfg1: 8 X-ray clouds x %d holes, sigma 0.5 um, depth U[10,665] um" % per
    elif config == 2:
        N = n or CONFIG_N[2]
        xyz = gaussian_cloud(rng, N, 2.0, (0.0, 0.0, 600.0))
        P.update(img_nx=64, img_ny=64, img_x0_um=-480.0, img_y0_um=-480.0)
        groups.append(("cloud0", 0, N))
        name = "cfg2: single cloud, %d holes, sigma 2 um at depth 600 um" % N
    elif config == 3:
        N = n or CONFIG_N[3]
        phi = 2.0 * math.pi * rng.random()
        xyz, mid = straight_track(rng, N, (0.0, 0.0), math.radians(60.0), phi, th, 0.1)
        P.update(img_nx=128, img_ny=128, img_x0_um=float(np.floor(mid[0] / pitch) * pitch - 64 * pitch),
                 img_y0_um=float(np.floor(mid[1] / pitch) * pitch - 64 * pitch))
        groups.append(("track0", 0, N))
        name = "cfg3: inclined muon track, %d holes, zenith 60 deg, sigma_perp 0.1 um" % N
    elif config == 4:
        N = n or CONFIG_N[4]
        n_cloud = 64
        per_cloud = 2048 if n is None else max(1, N // 512)
        per_track = (N - n_cloud * per_cloud) // 4
        parts, lo = [], 0
        half = 64 * pitch
        for k in range(4):
            entry = (rng.uniform(-half, half), rng.uniform(-half, half))
            zen, azi = math.radians(rng.uniform(0.0, 70.0)), 2.0 * math.pi * rng.random()
            cnt = per_track if k < 3 else N - n_cloud * per_cloud - 3 * per_track
            p, _ = straight_track(rng, cnt, entry, zen, azi, th, 0.1)
            parts.append(p)
            groups.append(("track%d" % k, lo, lo + cnt))
            lo += cnt
        for k in range(n_cloud):
            c = (rng.uniform(-half, half), rng.uniform(-half, half), rng.uniform(10.0, 665.0))
            parts.append(gaussian_cloud(rng, per_cloud, 0.5, c))
            groups.append(("cloud%d" % k, lo, lo + per_cloud))
            lo += per_cloud
        xyz = np.concatenate(parts)
        P.update(img_nx=256, img_ny=256, img_x0_um=-1920.0, img_y0_um=-1920.0)
        name = "cfg4: 4 muon tracks + 64 X-ray clouds, %d holes" % N
    else:
        raise ValueError("config must be 0..4")
    xyz = np.ascontiguousarray(xyz.astype(np.float32))
    # keep the float32 state inside the slab (rounding can land exactly on the back surface; that is allowed)
    xyz[:, 2] = np.minimum(xyz[:, 2], np.float32(th))
    return dict(xyz=xyz, params=P, groups=groups, name=name, config=config)


def make_events(sizes, seed=SEED, sigma_um=0.5, depth_range=(10.0, 665.0), half_window_um=400.0):
    """A batch of INDEPENDENT X-ray events: event k is a Gaussian cloud of
    sizes[k] holes (sigma_um) at a depth uniform in depth_range and a lateral centre uniform over the central
    +-half_window_um of the 64x64-pixel window.  Holes of different events never interact.  Returns
    dict(xyz float32 (N,3), offsets uint64 (n_events+1), params, name)."""
    P = dict(COMMON)
    P["seed"] = seed
    P.update(img_nx=64, img_ny=64, img_x0_um=-480.0, img_y0_um=-480.0)
    rng = _rng(seed, 0x45564E54)
    parts, off = [], [0]
    for s in sizes:
        c = (rng.uniform(-half_window_um, half_window_um), rng.uniform(-half_window_um, half_window_um),
             rng.uniform(depth_range[0], depth_range[1]))
        parts.append(gaussian_cloud(rng, int(s), sigma_um, c))
        off.append(off[-1] + int(s))
    xyz = np.concatenate(parts) if parts else np.zeros((0, 3))
    xyz = np.ascontiguousarray(xyz.astype(np.float32))
    xyz[:, 2] = np.minimum(xyz[:, 2], np.float32(P["thickness_um"]))
    return dict(xyz=xyz, offsets=np.asarray(off, dtype=np.uint64), params=P,
                name="%d independent X-ray events, %d holes in total (sigma %.2g um)" % (len(sizes), off[-1], sigma_um))
