"""The far-field variant's STATED bound (include/gcoreccd.h, gc_tree.cuh), checked on the CPU with the oracle's exact
eq. 6 and no product code: for m unit charges inside a ball of radius a about their centre of charge c, seen from a
point at distance d = a / t (t < 1) from c,
    | E_exact - m K' (x - c)/d^3 |  <=  B(t) m K'/d^2 ,   B(t) = t^2 (3 - 2 t)/(1 - t)^2 .
Random clusters (uniform in the ball, on its surface, two antipodal clumps = the worst case for the quadrupole), random
directions.  Also the sharper statement the GPU tests use: summed over members at distances r_i <= (1 + t) d."""
import numpy as np
import pytest

from oracle import goracle as g


def B(t):
    return t * t * (3.0 - 2.0 * t) / (1.0 - t) ** 2


def _clusters(rng, m, a):
    u = rng.standard_normal((m, 3))
    u /= np.linalg.norm(u, axis=1)[:, None]
    yield "ball", u * (a * rng.random(m) ** (1.0 / 3.0))[:, None]
    yield "shell", u * a
    axis = rng.standard_normal(3)
    axis /= np.linalg.norm(axis)
    yield "dumbbell", np.where((np.arange(m) % 2 == 0)[:, None], axis * a, -axis * a) * (1.0 - 1e-9 * rng.random((m, 1)))


@pytest.mark.parametrize("t", [0.05, 0.2, 0.3, 0.5, 0.7, 0.9])
def test_monopole_about_the_centre_of_charge_obeys_the_stated_bound(t):
    rng = np.random.default_rng(int(t * 1000))
    Kp = g.coulomb_constant(11.7)
    worst = 0.0
    for m in (2, 8, 64, 513):
        for a in (0.01, 1.0, 40.0):
            for name, pts in _clusters(rng, m, a):
                c = pts.mean(axis=0)
                rel = pts - c
                a_eff = np.linalg.norm(rel, axis=1).max()                  # radius about the centre of charge
                d = a_eff / t
                for _ in range(6):
                    n = rng.standard_normal(3)
                    n /= np.linalg.norm(n)
                    x = c + d * n
                    # exact field at x from the m charges: eq. 6 with eps = 0, target appended as a chargeless probe:
                    # the oracle sums over ALL points, so subtract nothing — the probe's own term is exactly 0
                    allp = np.vstack([pts, x[None, :]]) + np.array([0.0, 0.0, 300.0])
                    E = g.coulomb_field(allp, eps_um=0.0, Kp=Kp, targets=np.array([m], dtype=np.uint64))[0]
                    E_mono = m * Kp * (x - c) / d ** 3
                    err = np.linalg.norm(E - E_mono)
                    bound = B(t) * m * Kp / d ** 2
                    assert err <= bound * (1.0 + 1e-9) + 1e-12 * m * Kp / d ** 2, (name, m, a, t, err / bound)
                    worst = max(worst, err / bound)
                    # the form the GPU tests use: B (1+t)^2 sum_i K'/r_i^2 >= B m K'/d^2
                    r2 = ((x - pts) ** 2).sum(axis=1)
                    assert (1.0 + t) ** 2 * (Kp / r2).sum() >= m * Kp / d ** 2 * (1.0 - 1e-12)
    assert worst > 0.05                                                      # the bound is not vacuous: the dumbbell gets close


def test_bound_function_values():
    assert B(0.0) == 0.0
    assert B(0.3) == pytest.approx(0.4408163265306122, rel=1e-12)
    assert B(0.5) == pytest.approx(2.0, rel=1e-12)
    # it is the tail of the gradient's multipole series: sum_{k>=2} (k+1) t^k
    for t in (0.1, 0.4, 0.8):
        assert B(t) == pytest.approx(sum((k + 1) * t ** k for k in range(2, 4000)), rel=1e-9)
