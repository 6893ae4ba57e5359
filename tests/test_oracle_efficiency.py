"""Pins of the oracle's tabulated collision efficiency (reading R39), -m "not gpu".

PAPER.md:96 only names "more sophisticated collision kernels representing such phenomena as the geometric sweep-out
and the influence of electric field on the collision probability" (the Berry 1966 example); the tables themselves
are not in the container.  What is built is the MECHANISM -- a caller-supplied table E(r_big, r_small / r_big),
interpolated in a fixed order -- and it is pinned by what the mathematics fixes: a constant table is the geometric
kernel bit for bit, a 2 x 2 table is checked by hand, random tables against scipy's bilinear interpolator, and the
values outside the grid are those on its edge."""
import numpy as np
import pytest

import oracle
import sdm_workloads as W


def _vol(r):
    return 4.0 / 3.0 * np.pi * r ** 3


def test_constant_table_is_the_geometric_kernel_bit_for_bit():
    rng = np.random.default_rng(2)
    radius = np.array([1e-6, 5e-6, 2e-5, 1e-4, 1e-3])
    for E in (1.0, 0.37, 0.0):
        kt = oracle.geometric_table(radius, np.full((5, 7), E))
        kg = oracle.geometric(E)
        for _ in range(2000):
            vj, vk = np.exp(rng.uniform(np.log(1e-22), np.log(1e-6), 2))
            assert oracle.kernel(kt, vj, vk) == oracle.kernel(kg, vj, vk)
    # and a whole run: the same bits after every step
    w = W.small("cfg3")
    a, b = w.copy(), w.copy()
    kt = oracle.geometric_table(radius, np.full((5, 3), 1.0))
    for s in range(3):
        oracle.coalescence_step(a.xi, a.v, a.cell_id, w.n_cell, w.dt, 0.4, oracle.geometric(1.0), 42, s)
        oracle.coalescence_step(b.xi, b.v, b.cell_id, w.n_cell, w.dt, 0.4, kt, 42, s)
    assert np.array_equal(a.xi, b.xi) and np.array_equal(a.v.view(np.int64), b.v.view(np.int64))
    assert not np.array_equal(a.xi, w.xi)


def test_two_by_two_table_by_hand():
    kp = oracle.geometric_table([10e-6, 30e-6], [[0.0, 1.0], [2.0, 3.0]])   # rows: radius, columns: ratio 0 and 1
    E = lambda r, p: oracle.efficiency(kp, r, p)
    assert E(10e-6, 0.0) == 0.0 and E(10e-6, 1.0) == 1.0 and E(30e-6, 0.0) == 2.0 and E(30e-6, 1.0) == 3.0
    assert E(20e-6, 0.0) == pytest.approx(1.0, rel=1e-15) and E(20e-6, 1.0) == pytest.approx(2.0, rel=1e-15)
    assert E(10e-6, 0.5) == 0.5 and E(30e-6, 0.25) == 2.25
    assert E(20e-6, 0.5) == pytest.approx(1.5, rel=1e-15)
    assert E(15e-6, 0.5) == pytest.approx(0.5 + 0.25 * 2.0, rel=1e-15)    # e0 = 0.5, e1 = 2.5, t_r = 1/4
    # outside the grid: the value on its edge
    assert E(1e-6, 0.5) == 0.5 and E(1.0, 0.5) == 2.5 and E(0.0, 0.0) == 0.0
    # the kernel itself: K = E pi (r_j + r_k)^2 |vt_j - vt_k| with r = 10 and 20 um -> r_big = 20 um, p = 1/2
    K = oracle.kernel(kp, _vol(10e-6), _vol(20e-6))
    want = 1.5 * np.pi * (30e-6) ** 2 * abs(1.19e8 * (4e-10 - 1e-10))
    assert K == pytest.approx(want, rel=1e-9)
    assert oracle.kernel(kp, _vol(20e-6), _vol(10e-6)) == K               # symmetric: (r_big, p) ignores the order


def test_random_tables_against_scipy():
    scipy_interp = pytest.importorskip("scipy.interpolate")
    rng = np.random.default_rng(8)
    radius = np.sort(np.exp(rng.uniform(np.log(1e-6), np.log(1e-3), 9)))
    table = rng.random((9, 6))
    kp = oracle.geometric_table(radius, table)
    ref = scipy_interp.RegularGridInterpolator((radius, np.linspace(0.0, 1.0, 6)), table, method="linear")
    r = np.exp(rng.uniform(np.log(radius[0]), np.log(radius[-1]), 4000))
    p = rng.random(4000)
    got = np.array([oracle.efficiency(kp, a, b) for a, b in zip(r, p)])
    assert np.allclose(got, ref(np.stack([r, p], 1)), rtol=1e-12, atol=1e-15)
    # on the grid nodes: the entries themselves
    for i in range(9):
        for j in range(6):
            assert oracle.efficiency(kp, radius[i], j / 5.0) == pytest.approx(table[i, j], rel=1e-14, abs=1e-16)


def test_efficiency_changes_the_run_and_keeps_the_invariants():
    """an efficiency below one thins the collisions; sum xi v exact with integer volumes (R22)"""
    w = W.small("cfg4s")
    w.v = np.rint(w.v / w.v.min()).clip(1, 2 ** 20)          # integer-valued volumes
    radius = np.array([0.1, 1.0, 10.0, 100.0])               # metres: these "droplets" are huge, only the sums matter
    kt = oracle.geometric_table(radius, np.linspace(0.1, 0.9, 12).reshape(4, 3))
    total0 = oracle.total_xi_v_exact(w.xi, w.v)
    xi0 = w.xi.sum()
    for s in range(3):
        oracle.coalescence_step(w.xi, w.v, w.cell_id, w.n_cell, w.dt, 1e30, kt, 42, s)
        assert oracle.total_xi_v_exact(w.xi, w.v) == total0
        assert w.xi.sum() <= xi0


def test_bad_tables_are_rejected():
    for radius, table in (([1.0], [[1.0, 1.0]]), ([1.0, 1.0], [[0, 1], [0, 1]]), ([1.0, 2.0], [[0.0], [1.0]]),
                          ([1.0, 2.0], [[0, -1], [0, 1]]), ([1.0, 2.0], [[0, np.inf], [0, 1]])):
        with pytest.raises(ValueError):
            oracle.geometric_table(radius, table)
