"""Pins of the oracle's volume spectrum (O7, the paper's ParticlesVolumeSpectrum product,
PAPER.md:68-76) against things other than itself: a hand case with values exactly on the edges, numpy's histogram
on random data, totals, and the closed-form bin masses of the paper's exponential spectrum on the paper's bins."""
import math
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import sdm_workloads as W  # noqa: E402


def test_hand_case_with_values_on_the_edges():
    edges = np.array([1.0, 2.0, 4.0, 8.0])
    #             below  =e0   inside  =e1   inside  =e2  inside  =e3(out)  above   nan
    v = np.array([0.5,   1.0,  1.5,    2.0,  3.0,    4.0, 7.9,    8.0,      9.0,    np.nan])
    xi = np.array([100,  1,    2,      3,    4,      5,   6,      700,      800,    900], np.int64)
    count, sum_xi, sum_xi_v = oracle.volume_spectrum(xi, v, edges)
    assert count.tolist() == [2, 2, 2]                      # [1,2): 1.0, 1.5   [2,4): 2.0, 3.0   [4,8): 4.0, 7.9
    assert sum_xi.tolist() == [1 + 2, 3 + 4, 5 + 6]
    assert sum_xi_v.tolist() == [1 * 1.0 + 2 * 1.5, 3 * 2.0 + 4 * 3.0, 5 * 4.0 + 6 * 7.9]


def test_zero_multiplicity_entries_count_as_entries_only():
    count, sum_xi, sum_xi_v = oracle.volume_spectrum(np.array([0, 0, 3], np.int64), np.array([1.5, 1.6, 1.7]),
                                                     np.array([1.0, 2.0]))
    assert count.tolist() == [3] and sum_xi.tolist() == [3] and sum_xi_v.tolist() == [3 * 1.7]


def test_invalid_edges_are_refused():
    xi, v = np.ones(3, np.int64), np.ones(3)
    for bad in ([1.0], [2.0, 1.0], [1.0, 1.0, 2.0], [1.0, np.inf], [np.nan, 1.0]):
        with pytest.raises(ValueError):
            oracle.volume_spectrum(xi, v, np.array(bad))


def test_against_numpy_histogram_and_totals():
    rng = np.random.default_rng(7)
    n = 200_000
    v = np.exp(rng.uniform(np.log(1e-16), np.log(1e-7), n))
    xi = rng.integers(0, 10 ** 9, n).astype(np.int64)
    edges = 4.0 / 3.0 * math.pi * np.logspace(np.log10(10e-6), np.log10(5e-3), 32) ** 3
    assert not np.isin(v, edges).any()                      # numpy closes the last bin on the right; avoid the edge
    count, sum_xi, sum_xi_v = oracle.volume_spectrum(xi, v, edges)
    assert np.array_equal(count, np.histogram(v, bins=edges)[0])
    exact = [int(xi[(v >= edges[b]) & (v < edges[b + 1])].sum()) for b in range(31)]
    assert sum_xi.tolist() == exact
    want = np.histogram(v, bins=edges, weights=xi.astype(np.float64) * v)[0]
    assert np.allclose(sum_xi_v, want, rtol=1e-12, atol=0.0)
    inside = (v >= edges[0]) & (v < edges[-1])
    assert count.sum() == inside.sum() and sum_xi.sum() == int(xi[inside].sum())


def test_paper_bins_on_the_exponential_spectrum_closed_form():
    """configs[0] / PAPER.md:48-53: n(v) = (n0/v0) exp(-v/v0), sampled deterministically with equal multiplicities
    (R28).  Mass in [v1, v2) = n0 v0 [(1 + x) e^-x] from x2 = v2/v0 to x1 = v1/v0; number = n0 [e^-x]."""
    w = W.cfg0(n_sd=2 ** 13)
    edges_r = np.logspace(np.log10(10e-6), np.log10(5e-3), 32)
    edges = 4.0 / 3.0 * math.pi * edges_r ** 3
    count, sum_xi, sum_xi_v = oracle.volume_spectrum(w.xi, w.v, edges)
    n0, v0 = W.N0_PER_M3 * w.dV, W.V0
    x = edges / v0
    number = n0 * (np.exp(-x[:-1]) - np.exp(-x[1:]))
    mass = n0 * v0 * ((1 + x[:-1]) * np.exp(-x[:-1]) - (1 + x[1:]) * np.exp(-x[1:]))
    # each SD stands for n0 / n_sd droplets: the bin sums are the analytic integrals to within one SD per edge
    assert np.all(np.abs(sum_xi - number) <= 1.01 * w.xi[0])
    # ... and the bin masses to within one SD's mass at each edge (plus 0.5 % for the sampling inside the bin)
    assert np.all(np.abs(sum_xi_v - mass) <= w.xi[0] * (edges[:-1] + edges[1:]) + 5e-3 * mass)
    big = mass > 1e-2 * mass.sum()
    assert big.sum() >= 6 and np.all(np.abs(sum_xi_v[big] / mass[big] - 1.0) < 0.01)
    assert abs(sum_xi_v.sum() / mass.sum() - 1.0) < 1e-3
    assert count.sum() == np.count_nonzero((w.v >= edges[0]) & (w.v < edges[-1]))
