"""Pins for the oracle's X-ray front end: hole count N = E_e / w and the seeded Gaussian cloud.
The generator is pinned by (a) three holes computed without any oracle code (tests/golden/xray_cloud.txt, written by a
pure-Python restatement of the definition whose Philox is pinned by the published vectors), (b) sample moments against
N(c, sigma^2),
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


def test_cloud_matches_three_holes_computed_without_the_oracle(golden):
    # tests/golden/xray_cloud.txt: written by tests/golden/make_xray_cloud_golden.py, a pure-Python restatement of the
    # definition (its Philox round function is itself pinned by the published known-answer vectors)
    rows = golden("xray_cloud.txt")
    assert len(rows) == 3
    for r in rows:
        seed, k, c, s = int(r[0]), int(r[1]), [float(v) for v in r[2:5]], float(r[5])
        words, ref = [int(v, 16) for v in r[6:10]], np.array([float(v) for v in r[10:13]], dtype=np.float32)
        assert g.philox4x32_10([k & 0xffffffff, 0x58524159, k >> 32, 0], [seed & 0xffffffff, seed >> 32]) == words
        got = g.xray_cloud(seed, 1, c, s, first_index=k)[0]
        # libm's log / cos may differ from Python's in the last FP64 bit: at most one FP32 ulp after rounding
        assert np.all(np.abs(got.astype(np.float64) - ref) <= np.spacing(np.abs(ref)).astype(np.float64)), (got, ref)


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
