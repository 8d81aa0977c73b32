"""Pins of the oracle's eq. 6 double loop: closed forms, conservation law, symmetries,
shell theorem, and an independently written brute force (pair-symmetric, long double)."""
import math

import numpy as np
import pytest

from oracle import goracle as g

KP = 1.2307389297799718


def test_two_carriers_closed_form_with_and_without_softening():
    for d, eps in [(1.0, 0.0), (1.0, 1e-3), (0.01, 1e-3), (5.0, 0.5), (1e-3, 1e-3)]:
        xyz = np.array([[0.0, 0.0, 10.0], [d, 0.0, 10.0]])
        E = g.coulomb_field(xyz, eps_um=eps, Kp=KP)
        mag = KP * d / (d * d + eps * eps) ** 1.5
        assert E[0] == pytest.approx([-mag, 0.0, 0.0], rel=1e-14, abs=1e-300)   # pushed away from the other hole
        assert E[1] == pytest.approx([+mag, 0.0, 0.0], rel=1e-14, abs=1e-300)
    # one hole at 1 um in vacuum-free silicon: 1.2307 V/cm (SURVEY §8 header)
    E = g.coulomb_field(np.array([[0, 0, 0], [0, 0, 1.0]]), eps_um=0.0, Kp=g.coulomb_constant(11.7))
    assert E[1, 2] == pytest.approx(1.23073893, rel=1e-8) and E[0, 2] == pytest.approx(-1.23073893, rel=1e-8)


def test_self_term_is_zero_and_single_carrier_feels_nothing():
    E = g.coulomb_field(np.array([[3.0, -2.0, 100.0]]), eps_um=1e-3)
    assert np.all(E == 0.0)
    # coincident carriers with eps>0: finite and zero
    E = g.coulomb_field(np.array([[1.0, 1.0, 1.0]] * 3), eps_um=1e-3)
    assert np.all(E == 0.0)


def test_direction_is_along_axis_for_oblique_pair():
    a, b = np.array([1.0, 2.0, 3.0]), np.array([-2.0, 0.5, 7.0])
    E = g.coulomb_field(np.stack([a, b]), eps_um=0.0, Kp=KP)
    r = b - a
    d = np.linalg.norm(r)
    assert E[1] == pytest.approx(KP * r / d ** 3, rel=1e-14)
    assert E[0] == pytest.approx(-KP * r / d ** 3, rel=1e-14)


def test_newtons_third_law_zero_net_field():
    rng = np.random.default_rng(1)
    for n, sig in [(2, 1.0), (17, 0.1), (500, 2.0), (2048, 0.5)]:
        xyz = rng.standard_normal((n, 3)) * sig + [0, 0, 300.0]
        E = g.coulomb_field(xyz, eps_um=1e-3)
        net = np.linalg.norm(E.sum(axis=0))
        assert net <= 1e-12 * np.linalg.norm(E, axis=1).sum()


def test_translation_rotation_permutation():
    rng = np.random.default_rng(2)
    xyz = rng.standard_normal((300, 3))
    E = g.coulomb_field(xyz, eps_um=1e-2)
    scale = np.abs(E).max()
    # translation (exactly representable shift keeps differences identical up to rounding of the sums)
    Et = g.coulomb_field(xyz + np.array([8.0, -16.0, 512.0]), eps_um=1e-2)
    assert np.abs(Et - E).max() <= 1e-11 * scale
    # rotation: E(R x) = R E(x)
    q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    Er = g.coulomb_field(xyz @ q.T, eps_um=1e-2)
    assert np.abs(Er - E @ q.T).max() <= 1e-12 * scale
    # permutation of the carriers permutes the result
    p = rng.permutation(300)
    Ep = g.coulomb_field(xyz[p], eps_um=1e-2)
    assert np.abs(Ep - E[p]).max() <= 1e-12 * scale
    # mirror: x -> -x flips E_x only
    m = np.array([-1.0, 1.0, 1.0])
    Em = g.coulomb_field(xyz * m, eps_um=1e-2)
    assert np.abs(Em - E * m).max() <= 1e-12 * scale


def test_inverse_square_scaling():
    rng = np.random.default_rng(3)
    xyz = rng.standard_normal((64, 3))
    E1 = g.coulomb_field(xyz, eps_um=0.0)
    E2 = g.coulomb_field(2.0 * xyz, eps_um=0.0)
    assert np.abs(E2 * 4.0 - E1).max() <= 1e-13 * np.abs(E1).max()
    # linear in K
    assert g.coulomb_field(xyz, eps_um=0.0, Kp=3.0) == pytest.approx(3.0 * g.coulomb_field(xyz, eps_um=0.0, Kp=1.0), rel=1e-15)


def _brute_force_longdouble(xyz, eps, Kp):
    """Independent second implementation: pair-symmetric i<j loop in long double, power via **1.5."""
    n = xyz.shape[0]
    p = xyz.astype(np.longdouble)
    E = np.zeros((n, 3), dtype=np.longdouble)
    for i in range(n):
        for j in range(i + 1, n):
            r = p[j] - p[i]
            f = r / (r.dot(r) + np.longdouble(eps) ** 2) ** np.longdouble(1.5)
            E[j] += f
            E[i] -= f
    return (E * np.longdouble(Kp)).astype(np.float64)


def test_brute_force_tiny_n():
    rng = np.random.default_rng(4)
    for n, sig, eps in [(2, 1.0, 1e-3), (7, 0.05, 1e-3), (33, 1.0, 0.0), (64, 0.5, 1e-2)]:
        xyz = rng.standard_normal((n, 3)) * sig + [10.0, -5.0, 200.0]
        E = g.coulomb_field(xyz, eps_um=eps, Kp=KP)
        ref = _brute_force_longdouble(xyz, eps, KP)
        assert np.abs(E - ref).max() <= 1e-13 * np.abs(ref).max()


def test_target_subset_matches_full():
    rng = np.random.default_rng(5)
    xyz = rng.standard_normal((257, 3))
    E = g.coulomb_field(xyz, eps_um=1e-3)
    t = np.array([256, 0, 13, 13, 100], dtype=np.uint64)
    Es = g.coulomb_field(xyz, eps_um=1e-3, targets=t)
    assert np.array_equal(Es, E[t.astype(int)])


def test_shell_theorem_outside_and_inside():
    # M carriers uniformly on a sphere of radius a; a test carrier far lighter than the shell is emulated by
    # reading the field AT extra probe carriers and subtracting the probes' mutual fields analytically (eps=0).
    rng = np.random.default_rng(6)
    M, a = 20000, 1.0
    v = rng.standard_normal((M, 3))
    shell = a * v / np.linalg.norm(v, axis=1, keepdims=True)
    for r_probe, expect in [(3.0, M * KP / 9.0), (0.3, 0.0)]:
        pts = np.concatenate([shell, [[r_probe, 0.0, 0.0]]])
        E = g.coulomb_field(pts, eps_um=0.0, Kp=KP, targets=[M])[0]
        # shot noise of a random shell is ~ K' sqrt(M) / d^2 with d the distance to the surface
        tol = 4.0 * KP * math.sqrt(M) / (r_probe - a) ** 2 if r_probe > a else 0.02 * M * KP / a ** 2
        assert abs(E[0] - expect) <= tol and abs(E[1]) <= tol and abs(E[2]) <= tol
        if expect:
            assert abs(E[0] - expect) <= 0.01 * expect


def test_gaussian_cloud_enclosed_charge():
    # field at radius r of an isotropic Gaussian cloud: N K' [erf(r/(sqrt2 s)) - sqrt(2/pi)(r/s) exp(-r^2/2s^2)]/r^2
    rng = np.random.default_rng(7)
    N, s = 40000, 1.0
    cloud = rng.standard_normal((N, 3)) * s
    for r in (0.5, 1.5, 4.0):
        frac = math.erf(r / (math.sqrt(2) * s)) - math.sqrt(2 / math.pi) * (r / s) * math.exp(-r * r / (2 * s * s))
        expect = N * KP * frac / r ** 2
        # average over probe directions to beat shot noise
        dirs = rng.standard_normal((32, 3))
        dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
        radial = []
        for d in dirs:
            pts = np.concatenate([cloud, [r * d]])
            E = g.coulomb_field(pts, eps_um=1e-3, Kp=KP, targets=[N])[0]
            radial.append(E.dot(d))
        assert np.mean(radial) == pytest.approx(expect, rel=0.05)


def test_softening_limit_recovers_eq5():
    rng = np.random.default_rng(8)
    xyz = rng.standard_normal((50, 3))
    E0 = g.coulomb_field(xyz, eps_um=0.0)
    prev = None
    for eps in (1e-1, 1e-2, 1e-3):
        err = np.abs(g.coulomb_field(xyz, eps_um=eps) - E0).max()
        if prev is not None:
            assert err < prev / 50                                        # O(eps^2) convergence
        prev = err
