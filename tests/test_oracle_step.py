"""Pins P3-P6, P9, P10, P12 for the oracle's coalescence step: the shuffle,
the pair set and scale factor, the probability formula and gamma draw (brute force on 2- and 3-SD
cells), the update / clamp / split rules (hand cases), exact conservation, compaction, resume.
None of these re-use the oracle's own formulas: expectations are hand-computed numbers, Fractions,
or statistical frequencies."""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import oracle

HERE = os.path.dirname(os.path.abspath(__file__))
GOLDEN = os.path.join(HERE, "golden")


def _arrs(xi, v, cell):
    return (np.array(xi, np.int64), np.array(v, np.float64), np.array(cell, np.int32))


# ----------------------------------------------------------------------------- P12 worked step
def test_worked_step_from_survey():
    g = json.load(open(os.path.join(GOLDEN, "survey_p12_vectors.json")))["worked_step"]
    xi, v, cell = _arrs(g["xi"], g["v"], g["cell_id"])
    kp = oracle.golovin(g["golovin_b"])
    for step, want in enumerate(g["steps"]):
        d = oracle.coalescence_step(xi, v, cell, g["n_cell"], g["dt"], g["dV"], kp, 42, step, debug=True)
        assert d["perm"].tolist() == want["perm"]
        assert xi.tolist() == want["xi_after"]
        assert v.tolist() == [float(x) for x in want["v_after"]]
        for pr in want["pairs"]:
            assert d["gamma"][pr["j0"]] == pr["gamma"]
            assert d["gamma_clamped"][pr["j0"]] == pr["gamma_clamped"]
            if "u" in pr:
                assert oracle.sd_random(42, step, pr["j0"])[1] == pr["u"]
        assert int((xi * v).sum()) == g["sum_xi_v"]
        assert oracle.total_xi_v_exact(xi, v) == g["sum_xi_v"]


# ----------------------------------------------------------------------------- P3 shuffle
def test_shuffle_invariants_multi_cell():
    rng = np.random.default_rng(0)
    n, n_cell = 5000, 37
    cell = rng.integers(0, n_cell, n).astype(np.int32)
    xi = np.ones(n, np.int64)
    v = np.ones(n, np.float64)
    kp = oracle.golovin(0.0)  # K = 0: no collisions, state unchanged
    d = oracle.coalescence_step(xi, v, cell, n_cell, 1.0, 1.0, kp, 42, 5, debug=True)
    perm = d["perm"]
    assert sorted(perm.tolist()) == list(range(n))                      # a permutation
    keys, _ = oracle.sd_random_batch(42, 5, 0, n)
    sk = (cell[perm].astype(np.uint64) << np.uint64(32)) | keys[perm].astype(np.uint64)
    assert np.all(sk[1:] >= sk[:-1])                                      # sort key non-decreasing
    ties = np.nonzero(sk[1:] == sk[:-1])[0]
    assert np.all(perm[ties + 1] > perm[ties])                            # ties in index order
    assert np.array_equal(d["cell_start"], np.concatenate(([0], np.cumsum(np.bincount(cell, minlength=n_cell)))))
    assert np.all(xi == 1) and np.all(v == 1.0)


def test_shuffle_stability_on_forced_ties():
    """Key collisions are certain at N = 2^20 (R4); force them here by brute-force search of equal
    low-entropy situation: same cell, and check order against a (key, index) lexicographic sort."""
    n = 3000
    cell = np.zeros(n, np.int32)
    keys, _ = oracle.sd_random_batch(42, 0, 0, n)
    d = oracle.coalescence_step(np.ones(n, np.int64), np.ones(n), cell, 1, 1.0, 1.0, oracle.golovin(0.0), 42, 0,
                                debug=True)
    want = np.lexsort((np.arange(n), keys))  # primary: key, secondary: index
    assert np.array_equal(d["perm"], want.astype(np.int32))


def test_three_sd_cell_orders_uniform():
    """3-SD cell: each of the 6 orders with frequency 1/6, each SD left unpaired 1/3 of the time."""
    n_steps = 60_000
    counts = {}
    unpaired = np.zeros(3)
    for s in range(n_steps):
        keys, _ = oracle.sd_random_batch(42, s, 0, 3)
        order = tuple(np.lexsort((np.arange(3), keys)).tolist())
        counts[order] = counts.get(order, 0) + 1
        unpaired[order[2]] += 1
    assert len(counts) == 6
    exp = n_steps / 6
    chi2 = sum((c - exp) ** 2 / exp for c in counts.values())
    assert chi2 < 5 + 6 * math.sqrt(10)          # 5 dof: mean 5, sd sqrt(10)
    assert np.all(np.abs(unpaired / n_steps - 1 / 3) < 5 * math.sqrt((1 / 3) * (2 / 3) / n_steps))
    # ... and the oracle's own step uses exactly that order
    for s in (0, 1, 2, 17):
        keys, _ = oracle.sd_random_batch(42, s, 0, 3)
        d = oracle.coalescence_step(np.ones(3, np.int64), np.ones(3), np.zeros(3, np.int32), 1, 1.0, 1.0,
                                    oracle.golovin(0.0), 42, s, debug=True)
        assert d["perm"].tolist() == np.lexsort((np.arange(3), keys)).tolist()


# ----------------------------------------------------------------------------- P4 pair set and scale
@pytest.mark.parametrize("n_c", list(range(0, 10)) + [31, 32, 33, 200])
def test_pair_count_and_scale_brute_force(n_c):
    """All SDs identical, K xi dt/dV = 4 exactly, so p = 4 * scale is an integer and gamma = p exactly.
    Expected scale from the definition (n(n-1)/2)/floor(n/2) with Fractions."""
    n_cell = 3
    cell = np.concatenate((np.zeros(1, np.int32), np.full(n_c, 1, np.int32), np.full(1, 2, np.int32)))
    n = len(cell)
    xi = np.full(n, 2 ** 40, np.int64)
    v = np.full(n, 1.0)
    # Golovin b = 2^-39: K = b (v+v) = 2^-38 ; K * xi = 4 ; dt/dV = 1
    kp = oracle.golovin(2.0 ** -39)
    d = oracle.coalescence_step(xi, v, cell, n_cell, 1.0, 1.0, kp, 42, 0, debug=True)
    n_pairs = n_c // 2
    g = d["gamma"]
    assert np.count_nonzero(g) == n_pairs
    if n_pairs:
        scale = Fraction(n_c * (n_c - 1), 2) / n_pairs
        assert scale.denominator == 1
        assert set(g[g != 0].tolist()) == {4 * int(scale)}
        # closed form used by the CUDA side (R9)
        assert int(scale) == (n_c if n_c % 2 else n_c - 1)
        # gamma is recorded at the first-sorted member of each pair: even offsets in the cell
        start = d["cell_start"][1]
        firsts = d["perm"][start:start + 2 * n_pairs:2]
        assert np.all(g[firsts] != 0)
    # cells 0 and 2 hold a single SD: untouched
    assert g[0] == 0 and g[-1] == 0


# ----------------------------------------------------------------------------- P5 probability and gamma
def _two_sd_gamma(xi_pair, v_pair, b, dt, dV, step):
    xi, v, cell = _arrs(xi_pair, v_pair, [0, 0])
    d = oracle.coalescence_step(xi, v, cell, 1, dt, dV, oracle.golovin(b), 42, step, debug=True)
    j0 = d["perm"][0]
    return int(d["gamma"][j0]), int(d["gamma_clamped"][j0]), j0, xi, v


def test_two_sd_probability_by_hand_and_frequency():
    # p = b (v1+v2) max(xi) dt/dV * 1 = 0.5 * (1+3) * 8 * (1/128) = 0.125 (all dyadic => exact)
    hits = 0
    n_steps = 40_000
    for s in range(n_steps):
        g, gt, j0, _, _ = _two_sd_gamma([8, 5], [1.0, 3.0], 0.5, 1.0, 128.0, s)
        u = oracle.sd_random(42, s, j0)[1]
        assert g == (1 if u < 0.125 else 0)          # gamma = floor(p) + [u < frac p] with p = 0.125
        assert gt == g                                 # floor(8/5) = 1 >= gamma
        hits += g
    f = hits / n_steps
    assert abs(f - 0.125) < 4 * math.sqrt(0.125 * 0.875 / n_steps)


def test_two_sd_gamma_2_or_3_with_frequencies():
    # p = 2.3 is not dyadic; build it as b (v1+v2) xi dt/dV with b=2.3/8, v=1+3, xi=2, dt/dV=1
    # independent arithmetic: ((b*(v1+v2))*xi)*1*1 evaluated in Python floats the same left-to-right way
    b = 2.3 / 8.0
    p = ((b * (1.0 + 3.0)) * 2.0) * 1.0 * 1.0
    assert abs(p - 2.3) < 1e-15
    n_steps = 40_000
    c3 = 0
    for s in range(n_steps):
        g, gt, j0, xi, v = _two_sd_gamma([2, 1], [1.0, 3.0], b, 1.0, 1.0, s)
        u = oracle.sd_random(42, s, j0)[1]
        assert g == 2 + (1 if u < p - 2.0 else 0)
        assert gt == 2                                 # clamp floor(2/1) = 2
        c3 += g == 3
    assert abs(c3 / n_steps - 0.3) < 4 * math.sqrt(0.3 * 0.7 / n_steps)


def test_three_sd_scale_is_three_and_max_xi_is_used():
    # 3 SDs in one cell: one pair, scale = 3.  K xi_max dt/dV = 2^-4  ->  p = 3/16
    n_steps = 30_000
    hits = 0
    for s in range(n_steps):
        xi, v, cell = _arrs([4, 16, 16], [1.0, 1.0, 1.0], [0, 0, 0])
        d = oracle.coalescence_step(xi, v, cell, 1, 1.0, 1.0, oracle.golovin(2.0 ** -9), 42, s, debug=True)
        j0, k0 = d["perm"][0], d["perm"][1]
        pair_max = max([4, 16, 16][j0], [4, 16, 16][k0])
        p = 2.0 ** -8 * pair_max * 3
        u = oracle.sd_random(42, s, j0)[1]
        assert d["gamma"][j0] == (1 if u < p else 0)
        hits += int(d["gamma"][j0])
    # pairs: (4,16) x2 orders..: all three unordered pairs equally likely; every pair contains a 16
    assert abs(hits / n_steps - 3 / 16) < 4 * math.sqrt((3 / 16) * (13 / 16) / n_steps)


def test_expected_multiplicity_loss_matches_kernel_rate():
    """E[decrease of sum xi] per step = K xi_j xi_k dt/dV for a 2-SD cell (gamma * xi_k is removed
    from xi_j when no clamp/split intervenes)."""
    n_steps = 40_000
    loss = 0
    K_dtdV = (0.25 * (1.0 + 1.0)) * (1.0 / 1024.0)      # b (v+v) dt/dV
    for s in range(n_steps):
        xi, v, cell = _arrs([1000, 10], [1.0, 1.0], [0, 0])
        oracle.coalescence_step(xi, v, cell, 1, 1.0, 1024.0, oracle.golovin(0.25), 42, s)
        loss += 1010 - int(xi.sum())
    expect = K_dtdV * 1000 * 10                          # = 4.8828 per step; p = 0.488
    p = K_dtdV * 1000
    sd = 10 * math.sqrt(p * (1 - p) / n_steps)
    assert abs(loss / n_steps - expect) < 4 * sd


def test_gamma_from_p_special_values():
    assert oracle.gamma_from_p(0.0, 0.0) == 0
    assert oracle.gamma_from_p(0.5, 0.49) == 1
    assert oracle.gamma_from_p(0.5, 0.5) == 0            # strict <
    assert oracle.gamma_from_p(7.0, 0.0) == 7            # integer p: fraction 0, never +1
    assert oracle.gamma_from_p(7.25, 0.2) == 8
    assert oracle.gamma_from_p(2.0 ** 63, 0.1) == 2 ** 63 - 1   # R11 saturation
    assert oracle.gamma_from_p(1e300, 0.1) == 2 ** 63 - 1
    assert oracle.gamma_from_p(float("nan"), 0.1) == 0
    assert oracle.gamma_from_p(2.0 ** 62, 0.999) == 2 ** 62


# ----------------------------------------------------------------------------- P6 update / clamp / split
@pytest.mark.parametrize("xi_j,xi_k,g,want_gt,want_xi", [
    (10, 3, 2, 2, (4, 3)),      # plain
    (10, 3, 7, 3, (1, 3)),      # clamp to floor(10/3) = 3, remainder 1
    (9, 3, 5, 3, (1, 2)),       # clamp 3, remainder 0 -> split floor(3/2)=1 and 2
    (5, 5, 1, 1, (2, 3)),       # equal multiplicities -> split
    (1, 1, 1, 1, (0, 1)),       # split producing a zero (R14)
    (7, 2, 0, 0, (7, 2)),       # no collision
    (7, 0, 3, 0, (7, 0)),       # dead partner: no-op (R7)
])
def test_pair_update_hand_cases(xi_j, xi_k, g, want_gt, want_xi):
    vj, vk = 2.0, 5.0
    gt, a, b, c, d = oracle.pair_update(xi_j, xi_k, vj, vk, g)
    assert gt == want_gt
    assert (a, b) == want_xi
    if want_gt == 0:
        assert (c, d) == (vj, vk)
    else:
        vnew = want_gt * vj + vk
        rem = xi_j - want_gt * xi_k
        if rem > 0:
            assert (c, d) == (vj, vnew)          # only the k droplet grows
        else:
            assert (c, d) == (vnew, vnew)        # split: both carry the merged volume
        # mass conservation of the rule itself (integers): xi_j vj + xi_k vk is unchanged
        assert a * c + b * d == xi_j * vj + xi_k * vk


def test_exact_conservation_with_integer_volumes_and_monotone_multiplicity():
    """R22: integer-valued volumes stay integers < 2^53, so sum xi*v is conserved EXACTLY (128-bit
    integer accumulation), sum xi never increases, the number of SDs is constant."""
    rng = np.random.default_rng(3)
    n_cell, n = 50, 4000
    cell = rng.integers(0, n_cell, n).astype(np.int32)
    xi = rng.integers(1, 40, n).astype(np.int64)
    xi[rng.random(n) < 0.1] = 7            # plenty of equal pairs
    v = rng.integers(1, 6, n).astype(np.float64)
    total0 = oracle.total_xi_v_exact(xi, v)
    assert total0 == int(sum(int(a) * int(b) for a, b in zip(xi, v)))
    kp = oracle.golovin(0.05)
    last = int(xi.sum())
    n_split_zero = 0
    for s in range(60):
        d = oracle.coalescence_step(xi, v, cell, n_cell, 1.0, 1.0, kp, 42, s, debug=True)
        assert oracle.total_xi_v_exact(xi, v) == total0
        now = int(xi.sum())
        assert now <= last
        last = now
        assert np.all(xi >= 0) and np.all(v == np.rint(v)) and v.max() < 2.0 ** 53
        assert np.all(d["gamma_clamped"] <= d["gamma"])
        n_split_zero += int(np.count_nonzero(xi == 0))
    assert last < 0.8 * int(total0)        # something did happen
    assert n_split_zero > 0                # the xi=1,1 -> (0,1) branch was exercised
    assert len(xi) == n


def test_physical_volumes_conserved_to_rounding():
    import sdm_workloads as W
    w = W.cfg0(n_sd=2 ** 10, n_steps=300)
    kp = oracle.golovin(w.b)
    m0 = float(np.sum(w.xi.astype(np.float64) * w.v))
    oracle.run(w.xi, w.v, w.cell_id, 1, w.dt, w.dV, kp, 42, 0, 300)
    m1 = float(np.sum(w.xi.astype(np.float64) * w.v))
    assert abs(m1 - m0) / m0 < 1e-12


# ----------------------------------------------------------------------------- P9 compaction, stats
def test_remove_zero_multiplicity_definition():
    rng = np.random.default_rng(5)
    n = 1000
    xi = rng.integers(0, 3, n).astype(np.int64)
    v = rng.random(n)
    cell = rng.integers(0, 9, n).astype(np.int32)
    keep = xi != 0
    want = (xi[keep].copy(), v[keep].copy(), cell[keep].copy())
    m = oracle.remove_zero_multiplicity(xi, v, cell)
    assert m == int(keep.sum())
    assert np.array_equal(xi[:m], want[0]) and np.array_equal(v[:m], want[1]) and np.array_equal(cell[:m], want[2])
    # idempotent
    assert oracle.remove_zero_multiplicity(xi, v, cell, n_sd=m) == m
    assert np.array_equal(xi[:m], want[0])
    # degenerate: empty, all zero, none zero
    assert oracle.remove_zero_multiplicity(xi, v, cell, n_sd=0) == 0
    z = np.zeros(5, np.int64)
    assert oracle.remove_zero_multiplicity(z, np.ones(5), np.zeros(5, np.int32)) == 0


def test_cell_stats_against_numpy():
    rng = np.random.default_rng(6)
    n, n_cell = 3000, 17
    xi = rng.integers(0, 1000, n).astype(np.int64)
    v = rng.random(n)
    cell = rng.integers(0, n_cell, n).astype(np.int32)
    cnt, sx, sxv, sxv2 = oracle.cell_stats(xi, v, cell, n_cell)
    assert np.array_equal(cnt, np.bincount(cell, minlength=n_cell))
    assert np.array_equal(sx, np.bincount(cell, weights=xi, minlength=n_cell).astype(np.int64))
    assert np.allclose(sxv, np.bincount(cell, weights=xi * v, minlength=n_cell), rtol=1e-13)
    assert np.allclose(sxv2, np.bincount(cell, weights=xi * v * v, minlength=n_cell), rtol=1e-13)


# ----------------------------------------------------------------------------- P10 resume
def test_resume_is_exact():
    import sdm_workloads as W
    w = W.small("cfg4")
    kp = oracle.golovin(w.b)
    a = w.copy()
    oracle.run(a.xi, a.v, a.cell_id, a.n_cell, a.dt, a.dV, kp, 42, 0, 6)
    b = w.copy()
    oracle.run(b.xi, b.v, b.cell_id, b.n_cell, b.dt, b.dV, kp, 42, 0, 3)
    xi2, v2 = b.xi.copy(), b.v.copy()            # "dump / reload"
    oracle.run(xi2, v2, b.cell_id, b.n_cell, b.dt, b.dV, kp, 42, 3, 3)
    assert np.array_equal(a.xi, xi2) and np.array_equal(a.v.view(np.int64), v2.view(np.int64))


def test_degenerate_inputs():
    kp = oracle.golovin(1.0)
    e = (np.zeros(0, np.int64), np.zeros(0), np.zeros(0, np.int32))
    assert oracle.coalescence_step(*e, 4, 1.0, 1.0, kp, 42, 0, debug=True)["cell_start"].tolist() == [0] * 5
    xi, v, cell = _arrs([5], [1.0], [2])
    oracle.coalescence_step(xi, v, cell, 4, 1.0, 1.0, kp, 42, 0)
    assert xi.tolist() == [5]
    with pytest.raises(ValueError):
        oracle.coalescence_step(xi, v, np.array([4], np.int32), 4, 1.0, 1.0, kp, 42, 0)
    with pytest.raises(ValueError):
        oracle.coalescence_step(xi, v, cell, 4, 0.0, 1.0, kp, 42, 0)
