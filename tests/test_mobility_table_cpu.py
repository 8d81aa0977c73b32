"""eq. 2 as the kernels evaluate it: piecewise degree-8 interpolants of (1 + (E/Ec)^beta)^(-1/beta) on every
sixteenth of a binade of E/Ec, tabulated in long double at gcoreccd_create (gc_integrate.cuh mobility).
gcoreccd_mobility_table_host builds and evaluates the SAME table on the host, so its accuracy is checked here without a
GPU against the oracle's direct evaluation of eq. 2 (itself pinned in tests/test_oracle_equations.py); the GPU suite then
checks that the device evaluates the table to the same bits (tests/test_gpu_parity.py)."""
import numpy as np
import pytest

from oracle import goracle as g
from paper_2203_11043_b200 import binding


@pytest.mark.parametrize("T", [140.0, 77.0, 300.0])
def test_table_reproduces_eq2_to_double_rounding(T):
    rng = np.random.default_rng(int(T))
    E = np.concatenate([np.logspace(-1, 8, 40001), rng.uniform(50.0, 5000.0, 40000)])      # 0.1 V/cm .. 1e8 V/cm
    mu = binding.mobility_table_host(T, E)
    ref = np.array([g.mobility(e, T) for e in E])
    rel = np.abs(mu - ref) / ref
    assert rel.max() <= 2e-15, (rel.max(), E[np.argmax(rel)])          # both within ~2 ulp of the exact value
    assert np.median(rel) <= 2.3e-16


def test_table_is_continuous_across_rows_and_falls_back_outside():
    T = 140.0
    Ec = 1.24 * T ** 1.68
    # row boundaries: r = 2^e (1 + j/16); the two doubles either side must give the same value up to rounding
    edges = np.array([2.0 ** e * (1.0 + j / 16.0) for e in range(-16, 16) for j in range(16)]) * Ec
    lo, hi = np.nextafter(edges, 0.0), edges
    a, b = binding.mobility_table_host(T, lo), binding.mobility_table_host(T, hi)
    assert np.all(np.abs(a - b) <= 1e-15 * a)                      # each side within ~2 ulp of the exact value
    # outside the table (r < 2^-16, r >= 2^16, r = 0): the direct form
    out = binding.mobility_table_host(T, np.array([0.0, 1e-9, Ec * 2.0 ** -17, Ec * 2.0 ** 16, 1e12]))
    ref = np.array([g.mobility(e, T) for e in (0.0, 1e-9, Ec * 2.0 ** -17, Ec * 2.0 ** 16, 1e12)])
    assert np.all(np.abs(out - ref) <= 4e-15 * ref) and out[0] == pytest.approx(1.31e8 * T ** -2.2, rel=1e-15)
    # monotone decreasing in E (saturation), as eq. 2 is
    E = np.logspace(0, 7, 20001)
    assert np.all(np.diff(binding.mobility_table_host(T, E)) <= 0.0)
