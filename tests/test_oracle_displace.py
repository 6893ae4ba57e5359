"""Pins of the oracle's displacement step (O8, readings R36-R38), -m "not gpu".

The paper states no scheme (PAPER.md:80 names the dynamic, PAPER.md:112-118 the grid and the flow), so the pins are
what the reading and the mathematics fix: hand cases on cell edges and at the periodic seam, numpy's own floor / mod
on random data, and a divergence-free shear flow with whole-cell Courant numbers whose result has a closed form
(every row shifts by its own number of cells: occupancy permutes, positions move by exact integers)."""
import numpy as np
import pytest

import oracle
import sdm_workloads as W


def test_cell_index_hand_cases_on_edges():
    nx, nz = 4, 3
    # (x, z) -> cell: a position ON an edge belongs to the upper cell (floor); row-major, x fastest
    cases = [((0.0, 0.0), 0), ((0.999, 0.0), 0), ((1.0, 0.0), 1), ((3.999, 0.0), 3), ((0.0, 1.0), 4),
             ((2.5, 1.5), 6), ((3.0, 2.0), 11), ((np.nextafter(4.0, 0), np.nextafter(3.0, 0)), 11), ((1.0, 2.999), 9)]
    for (x, z), want in cases:
        assert oracle.cell_of(x, z, nx, nz) == want, (x, z)
    x = np.array([c[0][0] for c in cases])
    z = np.array([c[0][1] for c in cases])
    assert oracle.cell_id_from_positions(x, z, nx, nz).tolist() == [c[1] for c in cases]


def test_cell_index_against_numpy_floor():
    rng = np.random.default_rng(3)
    nx, nz = 37, 29
    x, z = rng.random(100_000) * nx, rng.random(100_000) * nz
    x[:50] = np.arange(50) % nx          # exactly on the edges
    z[:50] = np.arange(50) % nz
    want = (np.floor(z).astype(np.int64) * nx + np.floor(x).astype(np.int64)).astype(np.int32)
    assert np.array_equal(oracle.cell_id_from_positions(x, z, nx, nz), want)


def test_wrap_hand_cases_and_numpy_mod():
    n = 128
    assert oracle.wrap_periodic(127.75 + 0.5, n) == 0.25          # through the seam upwards
    assert oracle.wrap_periodic(0.25 - 0.5, n) == 127.75          # and downwards
    assert oracle.wrap_periodic(128.0, n) == 0.0                  # exactly one period
    assert oracle.wrap_periodic(0.0, n) == 0.0 and oracle.wrap_periodic(127.5, n) == 127.5
    assert oracle.wrap_periodic(-1e-300, n) == 0.0                # -tiny + n rounds to n: folded to 0 (stated reading)
    assert oracle.wrap_periodic(-128.0, n) == 0.0 and oracle.wrap_periodic(255.5, n) == 127.5
    rng = np.random.default_rng(4)
    q = rng.uniform(-n, 2 * n, 50_000)
    got = np.array([oracle.wrap_periodic(float(v), n) for v in q])
    want = np.mod(q, n)                                            # the same single rounding on either side
    assert np.array_equal(got[want < n], want[want < n])
    assert np.all((got >= 0) & (got < n))


@pytest.mark.parametrize("dt", [1.0, 0.5])
def test_shear_flow_with_whole_cell_courant_numbers_has_a_closed_form(dt):
    """u depends on the row only (du/dx = 0, w = 0: divergence-free) and u dt is a whole number of cells: every
    super-droplet of row j moves by exactly k_j cells, so cell occupancy is a permutation of the old one."""
    rng = np.random.default_rng(11)
    nx, nz, n = 16, 8, 20_000
    k = rng.integers(-nx + 1, nx, nz)                               # cells per step, per row
    u = np.repeat(k.astype(np.float64) / dt, nx)                    # per cell, row-major
    w = np.zeros(nx * nz)
    x = rng.integers(0, nx * 8, n) / 8.0                            # multiples of 1/8: every sum is exact
    z = rng.integers(0, nz * 8, n) / 8.0
    cell0 = oracle.cell_id_from_positions(x, z, nx, nz)
    x1, z1, cell1 = x.copy(), z.copy(), np.zeros(n, np.int32)
    oracle.displace(x1, z1, cell1, nx, nz, u, w, dt)
    row, col = cell0 // nx, cell0 % nx
    assert np.array_equal(z1, z)
    assert np.array_equal(x1, np.mod(x + k[row], nx))
    assert np.array_equal(cell1, row * nx + np.mod(col + k[row], nx))
    occ0 = np.bincount(cell0, minlength=nx * nz).reshape(nz, nx)
    occ1 = np.bincount(cell1, minlength=nx * nz).reshape(nz, nx)
    for j in range(nz):
        assert np.array_equal(occ1[j], np.roll(occ0[j], k[j]))


def test_single_eddy_keeps_positions_inside_and_follows_the_definition():
    """The paper's single-eddy flow as input: every step of the oracle equals the definition written
    out with numpy (velocity of the cell before the move, one product, one sum, the wrap), positions stay inside."""
    w = W.small("cfg3")
    nx, nz = 19, 17
    u, wv = W.single_eddy(nx, nz, courant_max=0.9)
    x, z = W.positions_in_cells(w.cell_id, nx, nz)
    cell = w.cell_id.copy()
    assert np.array_equal(oracle.cell_id_from_positions(x, z, nx, nz), cell)
    for step in range(5):
        c = (np.floor(z).astype(np.int64) * nx + np.floor(x).astype(np.int64))
        xn = np.mod(x + u[c] * 1.0, nx)
        zn = np.mod(z + wv[c] * 1.0, nz)
        xn[xn >= nx] = 0.0
        zn[zn >= nz] = 0.0
        oracle.displace(x, z, cell, nx, nz, u, wv, 1.0)
        assert np.array_equal(x, xn) and np.array_equal(z, zn)
        assert np.all((x >= 0) & (x < nx) & (z >= 0) & (z < nz))
        assert np.array_equal(cell, (np.floor(zn).astype(np.int64) * nx + np.floor(xn).astype(np.int64)).astype(np.int32))
    assert np.any(np.diff(cell) < 0)                    # the order is no longer cell-major: what NEXT-4 is for
    # updraft on the left, downdraft on the right
    W2 = wv.reshape(nz, nx)
    assert W2[:, : nx // 2].mean() > 0 > W2[:, nx // 2 + 1:].mean()


def test_bad_arguments():
    x = np.zeros(4)
    with pytest.raises(ValueError):
        oracle.cell_id_from_positions(x, x, 0, 4)
    with pytest.raises(ValueError):
        oracle.displace(x.copy(), x.copy(), np.zeros(4, np.int32), 2, 2, np.zeros(4), np.zeros(4), 0.0)
