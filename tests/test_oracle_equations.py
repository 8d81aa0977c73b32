"""Pins of the oracle's model equations (eqs. 1-4, K of eq. 6) and its Philox normal stream.

None of these re-types the oracle's formula: they use special cases, limits, identities, golden values
produced independently (tests/golden/*.txt, each with its citation) and statistical moments.
"""
import math

import numpy as np
import pytest

from oracle import goracle as g


# ------------------------------------------------------------------ eq. 1
def test_eq1_depletion_field_zero_crossing_and_endpoints():
    a1, a2 = 2.81e4, 2.0e3
    assert g.depletion_field(0.0, a1, a2) == -2000.0                      # E(0) = -a2
    assert abs(g.depletion_field(675.0, a1, a2) - (-103.25)) < 1e-9
    assert abs(g.depletion_field(600.0, a1, a2) - (-314.0)) < 1e-9
    assert abs(g.depletion_field(200.0, a1, a2) - (-1438.0)) < 1e-9
    zstar = a2 / a1 * 1e4                                                 # um, field reverses here
    assert abs(zstar - 711.744) < 1e-3
    assert abs(g.depletion_field(zstar, a1, a2)) < 1e-9
    # linear: second difference vanishes
    e = [g.depletion_field(z, a1, a2) for z in (100.0, 300.0, 500.0)]
    assert abs(e[0] - 2 * e[1] + e[2]) < 1e-9


# ------------------------------------------------------------------ eq. 2
def test_eq2_golden_values(golden):
    for E, T, mu in golden("eq2_mobility.txt"):
        assert g.mobility(float(E), float(T)) == pytest.approx(float(mu), rel=1e-8)


def test_eq2_low_field_and_half_field_identities(golden):
    c = {r[0]: float(r[1]) for r in golden("constants.txt")}
    for T in (77.0, 140.0, 300.0):
        mu0 = g.mobility(0.0, T)
        # E -> 0 leaves the numerator alone: mu(0,T) T^2.2 = 1.31e8
        assert mu0 * T ** 2.2 == pytest.approx(1.31e8, rel=1e-12)
    # at E = E_c the bracket is exactly 2: mu/mu0 = 2^(-1/beta)
    Ec, beta = c["E_c"], c["beta"]
    assert g.mobility(Ec, 140.0) / g.mobility(0.0, 140.0) == pytest.approx(c["half_field_ratio"], rel=1e-8)
    assert 2.0 ** (-1.0 / beta) == pytest.approx(c["half_field_ratio"], rel=1e-8)


def test_eq2_saturation_velocity_and_monotonicity(golden):
    c = {r[0]: float(r[1]) for r in golden("constants.txt")}
    # mu E -> v_sat = 1.31e8 * 1.24 * T^-0.52 as E -> infinity (the bracket -> (E/Ec)^beta)
    v7 = g.mobility(1e7, 140.0) * 1e7
    v9 = g.mobility(1e9, 140.0) * 1e9
    assert v7 == pytest.approx(1.24332e7, rel=1e-5)
    assert v9 == pytest.approx(c["v_sat"], rel=1e-4)
    assert v7 < v9 < c["v_sat"] * (1 + 1e-12)
    Es = np.logspace(-2, 7, 200)
    mus = np.array([g.mobility(E, 140.0) for E in Es])
    assert np.all(np.diff(mus) < 0)                                        # strictly decreasing in E
    assert np.all(np.diff(mus * Es) > 0)                                   # drift velocity increasing
    # textbook check of the units reading R1: silicon hole mobility at 300 K is about 450-480 cm^2/Vs
    assert 440.0 < g.mobility(0.0, 300.0) < 490.0


# ------------------------------------------------------------------ eqs. 3-4, eq. 6 constant
def test_constants_golden(golden):
    c = {r[0]: (float(r[1]), float(r[2])) for r in golden("constants.txt")}
    assert g.coulomb_constant(11.7) == pytest.approx(c["K_prime"][0], rel=c["K_prime"][1])
    assert g.coulomb_constant(0.0) == g.coulomb_constant(11.7)            # 0 => default 11.7
    assert g.thermal_voltage(140.0) == pytest.approx(c["kT_over_q"][0], rel=c["kT_over_q"][1])
    mu0 = g.mobility(0.0, 140.0)
    s = g.diffusion_sigma(mu0, 140.0, 0.05)
    assert s == pytest.approx(c["sigma_step"][0], rel=c["sigma_step"][1])
    assert s * s / (2 * 0.05) == pytest.approx(c["D_low_field"][0], rel=c["D_low_field"][1])
    assert 1e-5 * mu0 * g.coulomb_constant(11.7) == pytest.approx(c["mu0_K_prime"][0], rel=c["mu0_K_prime"][1])


def test_coulomb_constant_against_si_definition():
    # vacuum: q/(4 pi eps0) = 1.43996e-9 V m (the textbook 14.4 eV Angstrom) -> 14.3996 (V/cm) um^2
    assert g.coulomb_constant(1.0) == pytest.approx(14.39964548, rel=1e-8)
    assert g.coulomb_constant(11.7) * 11.7 == pytest.approx(g.coulomb_constant(1.0), rel=1e-14)


def test_diffusion_sigma_scaling_laws():
    # sigma^2 linear in mu, T and dt (eqs. 3-4)
    s = g.diffusion_sigma(1000.0, 100.0, 0.1)
    assert g.diffusion_sigma(4000.0, 100.0, 0.1) == pytest.approx(2 * s, rel=1e-14)
    assert g.diffusion_sigma(1000.0, 400.0, 0.1) == pytest.approx(2 * s, rel=1e-14)
    assert g.diffusion_sigma(1000.0, 100.0, 0.4) == pytest.approx(2 * s, rel=1e-14)
    # k_B/q = 8.617333262e-5 V/K (exact SI ratio)
    assert g.thermal_voltage(1.0) == pytest.approx(8.617333262e-5, rel=1e-9)


# ------------------------------------------------------------------ Philox4x32-10
def test_philox_known_answers(golden):
    for row in golden("philox_kat.txt"):
        v = [int(t, 16) for t in row]
        assert g.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_philox_is_a_bijection_of_the_counter_on_a_small_slice():
    # distinct counters -> distinct outputs (a dropped round input would collide massively)
    outs = {tuple(g.philox4x32_10([i, 0, s, 0], [7, 9])) for i in range(64) for s in range(64)}
    assert len(outs) == 64 * 64


def test_normal_stream_golden(golden):
    for row in golden("normal_stream.txt"):
        seed, cid, step = int(row[0]), int(row[1]), int(row[2])
        words = [int(t, 16) for t in row[3:7]]
        n, w = g.normals(seed, cid, step)
        assert w == words
        assert np.allclose(n, [float(t) for t in row[7:10]], rtol=0, atol=1e-11)


def test_normal_stream_keying_is_seed_id_step():
    n0, w0 = g.normals(1, 2, 3)
    assert g.normals(1, 2, 3)[1] == w0                                    # pure function
    assert g.normals(2, 2, 3)[1] != w0 and g.normals(1, 3, 3)[1] != w0 and g.normals(1, 2, 4)[1] != w0
    # 64-bit seed and step: high halves matter
    assert g.normals(1 + (1 << 32), 2, 3)[1] != w0
    assert g.normals(1, 2, 3 + (1 << 32))[1] != w0
    # the words are Philox(ctr=(id,0,step_lo,step_hi), key=(seed_lo,seed_hi))
    assert g.normals(0x1111111122222222, 5, 0x3333333344444444)[1] == \
        g.philox4x32_10([5, 0, 0x44444444, 0x33333333], [0x22222222, 0x11111111])


def test_normal_stream_moments():
    ids = np.arange(200000)
    n = np.array([g.normals(20220322, int(i), 3)[0] for i in ids[:100000]] +
                 [g.normals(20220322, 17, int(s))[0] for s in ids[:100000]])
    assert n.shape == (200000, 3)
    flat = n.reshape(-1)                                                  # 6e5 draws
    assert abs(flat.mean()) < 0.01
    assert abs(flat.var() - 1.0) < 0.01
    assert abs((flat ** 4).mean() / flat.var() ** 2 - 3.0) < 0.05
    # the three components are uncorrelated
    cc = np.corrcoef(n.T)
    assert np.all(np.abs(cc - np.eye(3)) < 0.01)
    # Box-Muller radius truncation: |n| <= sqrt(-2 ln 2^-24) = 5.768
    assert np.abs(flat).max() <= math.sqrt(-2.0 * math.log(2.0 ** -24)) + 1e-12
