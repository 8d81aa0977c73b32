"""Pins for the oracle's X-ray front end: hole count N = E_e / w and the seeded Gaussian cloud.
The generator is pinned by (a) the Philox known-answer path it shares with the pinned normal stream, re-derived
here from the raw Philox words with the counter layout stated in DESIGN.md, (b) sample moments against N(c, sigma^2),
(c) structural properties: index-addressed (chunked generation = one call), mirrored at the back surface."""
import math

import numpy as np

from oracle import goracle as g


def test_hole_count_paper_values():
    # w = 3.77 eV at 140 K
    assert g.xray_hole_count(100.0) == 26          # 26.5 pairs -> 26 carriers (PAPER.md:106 example energy)
    assert g.xray_hole_count(3.77) == 1
    assert g.xray_hole_count(3.76) == 0
    assert g.xray_hole_count(7500.0, 3.64) == 2060  # BASELINE.json configs[1]: "approx. a 7.5 keV deposit at 3.64 eV/pair"
    assert g.xray_hole_count(-1.0) == 0 and g.xray_hole_count(10.0, 0.0) == 0


def test_cloud_matches_box_muller_of_raw_words():
    seed, c, s = 0x1234567890ABCDEF, (3.0, -7.0, 200.0), 0.8
    xyz = g.xray_cloud(seed, 5, c, s, first_index=(1 << 32) + 9)
    for i in range(5):
        k = (1 << 32) + 9 + i
        w = g.philox4x32_10([k & 0xffffffff, 0x58524159, k >> 32, 0], [seed & 0xffffffff, seed >> 32])
        ua = ((int(w[0]) >> 9) + 0.5) / 2 ** 23
        fa = (int(w[1]) >> 8) / 2 ** 24
        ub = ((int(w[2]) >> 9) + 0.5) / 2 ** 23
        fb = (int(w[3]) >> 8) / 2 ** 24
        Ra, Rb = math.sqrt(-2 * math.log(ua)), math.sqrt(-2 * math.log(ub))
        ref = np.array([c[0] + s * Ra * math.cos(2 * math.pi * fa), c[1] + s * Ra * math.sin(2 * math.pi * fa),
                        c[2] + s * Rb * math.cos(2 * math.pi * fb)]).astype(np.float32)
        assert np.array_equal(xyz[i], ref)


def test_cloud_moments():
    n, c, s = 400000, np.array([10.0, -20.0, 300.0]), 2.0
    xyz = g.xray_cloud(20220322, n, c, s).astype(np.float64)
    assert np.all(np.abs(xyz.mean(0) - c) < 5 * s / math.sqrt(n))
    assert np.all(np.abs(xyz.var(0) / s ** 2 - 1) < 5 * math.sqrt(2.0 / n))
    cc = np.corrcoef(xyz.T)
    assert abs(cc[0, 1]) < 0.01 and abs(cc[0, 2]) < 0.01 and abs(cc[1, 2]) < 0.01
    z = (xyz - c) / s
    assert abs((z ** 4).mean() - 3.0) < 0.05


def test_cloud_is_index_addressed_and_seeded():
    a = g.xray_cloud(7, 1000, (0, 0, 100), 1.0)
    b = np.concatenate([g.xray_cloud(7, 400, (0, 0, 100), 1.0), g.xray_cloud(7, 600, (0, 0, 100), 1.0, first_index=400)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, g.xray_cloud(8, 1000, (0, 0, 100), 1.0))


def test_cloud_mirrored_at_back_surface():
    xyz = g.xray_cloud(3, 20000, (0, 0, 675.0), 1.0, thickness_um=675.0)
    assert xyz[:, 2].max() <= 675.0
    free = g.xray_cloud(3, 20000, (0, 0, 675.0), 1.0, thickness_um=1e9)
    over = free[:, 2] > 675.0
    assert over.sum() > 9000
    assert np.allclose(xyz[over, 2], (2 * 675.0 - free[over, 2].astype(np.float64)).astype(np.float32), atol=1e-4)
    assert np.array_equal(xyz[~over], free[~over])
