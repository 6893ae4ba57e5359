"""GPU parity tests proper (-m gpu): the CUDA path, called through the C ABI, against the oracle,
element by element on identically seeded inputs.

Bar (BASELINE.json north_star): multiplicities, every gamma, the permutation and cell_start
bit-exact; volumes within 1e-12 relative in fp64 (the kernels are written to be bit-exact: same
operation order, no FMA; test_volumes_bit_exact asserts that stronger property separately)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import sdm_workloads as W  # noqa: E402

VOL_RTOL = 1e-12


def _sdm():
    import paper_2103_17238_b200 as sdm
    return sdm


@pytest.fixture(scope="module")
def dev():
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device; the SDM step has no CPU fallback")
    return torch.device("cuda", 0)


def _okp(w):
    return oracle.golovin(w.b) if w.kernel_kind == W.GOLOVIN else oracle.geometric(w.E)


def _gkp(w):
    sdm = _sdm()
    return sdm.golovin(w.b) if w.kernel_kind == W.GOLOVIN else sdm.geometric(w.E)


def _to_dev(w, dev):
    return (torch.from_numpy(w.xi.copy()).to(dev), torch.from_numpy(w.v.copy()).to(dev),
            torch.from_numpy(w.cell_id.copy()).to(dev))


def _assert_vol_close(got, want, what=""):
    got = np.asarray(got)
    want = np.asarray(want)
    denom = np.maximum(np.abs(want), 1e-300)
    rel = np.abs(got - want) / denom
    assert rel.max(initial=0.0) <= VOL_RTOL, f"{what}: max rel volume error {rel.max()}"


def _run_parity(w, dev, path=None, check_debug=True, bit_exact=False, narrow_key_bits=None, expect_last_path=None,
                track_zeros=False, skip_key_digits=None):
    """Steps the oracle and the GPU side by side over w.n_steps steps, comparing after every step."""
    sdm = _sdm()
    ow = w.copy()
    n = w.n_sd
    with sdm.SDMContext(max(n, 1), w.n_cell, device=dev) as ctx:
        if path is not None:
            ctx.set_path(path)
        if narrow_key_bits is not None:
            ctx.set_option(sdm.OPT_NARROW_KEY_BITS, narrow_key_bits)
        if track_zeros:
            ctx.set_option(sdm.OPT_TRACK_ZEROS, 1)
        if skip_key_digits is not None:
            ctx.set_option(sdm.OPT_SKIP_KEY_DIGITS, skip_key_digits)
        xi, v, cell = _to_dev(w, dev)
        dbg = ctx.debug_outputs(n, w.n_cell) if check_debug else None
        okp, gkp = _okp(w), _gkp(w)
        stats = dict(gamma_nonzero=0, clamped=0, splits_to_zero=0, compactions=0, removed=0)
        for s in range(w.n_steps):
            od = oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, w.seed, s, n_sd=n,
                                         debug=True)
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, gkp, w.seed, s, n_sd=n)
            assert ctx.poll_error() == 0
            if check_debug:
                assert np.array_equal(dbg["cell_start"].cpu().numpy(), od["cell_start"]), f"cell_start step {s}"
                assert np.array_equal(dbg["perm"][:n].cpu().numpy(), od["perm"]), f"perm step {s}"
                assert np.array_equal(dbg["gamma"][:n].cpu().numpy(), od["gamma"]), f"gamma step {s}"
                assert np.array_equal(dbg["gamma_clamped"][:n].cpu().numpy(), od["gamma_clamped"]), f"gamma~ step {s}"
            gx = xi[:n].cpu().numpy()
            gv = v[:n].cpu().numpy()
            assert np.array_equal(gx, ow.xi[:n]), f"multiplicity step {s}"
            _assert_vol_close(gv, ow.v[:n], f"step {s}")
            if bit_exact:
                assert np.array_equal(gv.view(np.int64), ow.v[:n].view(np.int64)), f"volume bits step {s}"
            stats["gamma_nonzero"] += int(np.count_nonzero(od["gamma"]))
            stats["clamped"] += int(np.count_nonzero(od["gamma_clamped"] < od["gamma"]))
            stats["splits_to_zero"] += int(np.count_nonzero(ow.xi[:n] == 0))
            if w.compact_every and (s + 1) % w.compact_every == 0:
                n_o = oracle.remove_zero_multiplicity(ow.xi, ow.v, ow.cell_id, n_sd=n)
                n_g = ctx.remove_zero_multiplicity(xi, v, cell, n_sd=n)
                assert n_g == n_o, f"compaction count step {s}"
                stats["compactions"] += 1
                stats["removed"] += n - n_o
                n = n_o
                assert np.array_equal(xi[:n].cpu().numpy(), ow.xi[:n])
                assert np.array_equal(cell[:n].cpu().numpy(), ow.cell_id[:n])
                _assert_vol_close(v[:n].cpu().numpy(), ow.v[:n], f"after compaction {s}")
        if expect_last_path is not None:
            assert ctx.last_path() == expect_last_path
        return stats


# ------------------------------------------------------------------------------------------- a1
def test_philox_keys_and_uniforms_bit_exact(dev):
    sdm = _sdm()
    with sdm.SDMContext(1024, 1, device=dev) as ctx:
        for seed, step, i0, n in [(42, 0, 0, 100_003), (42, 7, 2 ** 32 - 50, 1000), (2 ** 40 + 17, 2 ** 32 + 7, 5, 999),
                                  (0, 0, 0, 1), (2 ** 64 - 1, 2 ** 64 - 1, 2 ** 40, 33)]:
            key, u = ctx.philox_fill(seed, step, i0, n)
            ok, ou = oracle.sd_random_batch(seed, step, i0, n)
            assert np.array_equal(key.cpu().numpy().view(np.uint32), ok)
            assert np.array_equal(u.cpu().numpy().view(np.int64), ou.view(np.int64))


# ------------------------------------------------------------------------------------------- kernels
@pytest.mark.parametrize("kind", ["golovin", "geometric"])
def test_kernel_function_bit_exact(dev, kind):
    sdm = _sdm()
    rng = np.random.default_rng(21)
    n = 200_000
    vj = np.exp(rng.uniform(np.log(1e-24), np.log(1e-4), n))
    vk = np.exp(rng.uniform(np.log(1e-24), np.log(1e-4), n))
    # regime boundaries of the fall-speed law, equal volumes, zero volume
    r_edge = np.array([40e-6, 600e-6, np.nextafter(40e-6, 0), np.nextafter(600e-6, 1)])
    v_edge = 4.0 / 3.0 * np.pi * r_edge ** 3
    vj[:4], vk[:4] = v_edge, v_edge[::-1]
    vj[4], vk[4] = 1e-15, 1e-15
    vj[5], vk[5] = 0.0, 1e-15
    okp = oracle.golovin(1500.0) if kind == "golovin" else oracle.geometric(1.0)
    gkp = sdm.golovin(1500.0) if kind == "golovin" else sdm.geometric(1.0)
    want = np.array([oracle.kernel(okp, float(a), float(b)) for a, b in zip(vj[:20_000], vk[:20_000])])
    with sdm.SDMContext(1024, 1, device=dev) as ctx:
        got = ctx.kernel_eval(gkp, torch.from_numpy(vj).to(dev), torch.from_numpy(vk).to(dev)).cpu().numpy()
    assert np.array_equal(got[:20_000].view(np.int64), want.view(np.int64))
    # symmetry on the device
    with sdm.SDMContext(1024, 1, device=dev) as ctx:
        got2 = ctx.kernel_eval(gkp, torch.from_numpy(vk).to(dev), torch.from_numpy(vj).to(dev)).cpu().numpy()
    assert np.array_equal(got.view(np.int64), got2.view(np.int64))


# ------------------------------------------------------------------------------------------- whole step
@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
def test_small_configs_general_path(dev, name):
    sdm = _sdm()
    st = _run_parity(W.small(name), dev, path=sdm.PATH_GENERAL, bit_exact=True)
    if name in ("cfg0", "cfg4s"):
        assert st["gamma_nonzero"] > 0
    if name == "cfg4s":
        assert st["clamped"] > 0 and st["removed"] > 0       # large gamma, clamp, split->0, compaction
    if name == "cfg3z":
        assert st["removed"] > 0


@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg3", "cfg4s"])
@pytest.mark.parametrize("skip", [0, 1, 3])
def test_general_path_skipped_key_digits_are_repaired_exactly(dev, name, skip):
    """SDM_OPT_SKIP_KEY_DIGITS: the LSD passes sort only the top (4 - skip) key digits and k_tie_repair orders the
    tied runs by (key, index); the permutation, every gamma and the state stay those of the oracle.  skip = 3 leaves
    8 sorted key bits: in the single-cell configs every super-droplet sits in a long tied run."""
    sdm = _sdm()
    w = W.small(name, interleave=(name in ("cfg3", "cfg4s")))
    if name in ("cfg0", "cfg1"):
        w = W.cfg0(n_sd=3001, n_steps=4) if name == "cfg0" else W.cfg1(n_sd=5003, n_steps=3)
    _run_parity(w, dev, path=sdm.PATH_GENERAL, bit_exact=True, skip_key_digits=skip)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
def test_small_configs_interleaved_order(dev, name):
    """R30: the same super-droplets in a random memory order (the general, unsorted-cell_id case)."""
    sdm = _sdm()
    _run_parity(W.small(name, interleave=True), dev, path=sdm.PATH_GENERAL, bit_exact=True)


@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
def test_small_configs_auto_path(dev, name):
    _run_parity(W.small(name), dev, path=None, bit_exact=True)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
def test_small_configs_cell_sorted_path(dev, name):
    """per-cell register sort fused with the pair kernel; same bits as the oracle."""
    sdm = _sdm()
    st = _run_parity(W.small(name), dev, path=sdm.PATH_CELL_SORTED, bit_exact=True)
    if name == "cfg4s":
        assert st["clamped"] > 0 and st["removed"] > 0


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
@pytest.mark.parametrize("interleave", [True, False])
def test_small_configs_hybrid_path(dev, name, interleave):
    """cell-digit LSD passes + fused per-cell sort/pair kernel: any order of cell_id, same bits as the oracle."""
    sdm = _sdm()
    st = _run_parity(W.small(name, interleave=interleave), dev, path=sdm.PATH_HYBRID, bit_exact=True,
                     expect_last_path=sdm.PATH_HYBRID)
    if name == "cfg4s":
        assert st["clamped"] > 0 and st["removed"] > 0


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
@pytest.mark.parametrize("path", ["general", "cell_sorted", "hybrid"])
def test_small_configs_without_debug_outputs(dev, name, path):
    """The launch configuration bench.py times: debug outputs off, so the conservative early-out
    (pair_may_collide) decides which pairs run the full rule, and the fused kernels count the zeros for
    the compaction call (SDM_OPT_TRACK_ZEROS).  Same bits as the oracle after every step."""
    sdm = _sdm()
    if name == "cfg1" and path != "general":
        pytest.skip("single cell: general path only")
    p = {"general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED, "hybrid": sdm.PATH_HYBRID}[path]
    st = _run_parity(W.small(name, interleave=(path == "hybrid")), dev, path=p, check_debug=False, bit_exact=True,
                     track_zeros=True)
    if name in ("cfg3z", "cfg4s"):
        assert st["removed"] > 0


@pytest.mark.parametrize("dV", [400.0, 4.0, 0.04, 4e-4])
@pytest.mark.parametrize("path", ["general", "cell_sorted"])
def test_geometric_early_out_is_exact(dev, dV, path):
    """The fp32 interval bound of the geometric kernel must never hide a collision: cfg3's spectrum with
    the cell volume scaled so that p runs from << 1 to >> 1, debug outputs off, against the oracle."""
    sdm = _sdm()
    w = W.small("cfg3")
    w.dV = dV
    p = {"general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED}[path]
    _run_parity(w, dev, path=p, check_debug=False, bit_exact=True, track_zeros=True)


@pytest.mark.parametrize("path", ["cell_sorted", "hybrid"])
@pytest.mark.parametrize("bits", [1, 5, 12])
def test_fused_kernel_wide_redo(dev, path, bits):
    """With only a few key bits in the 32-bit sort word nearly every cell has neighbours whose truncated keys
    tie, so the exact 64-bit redo runs all the time; the result must not change."""
    sdm = _sdm()
    if path == "cell_sorted":
        _run_parity(W.small("cfg4"), dev, path=sdm.PATH_CELL_SORTED, bit_exact=True, narrow_key_bits=bits)
    else:
        _run_parity(W.small("cfg3", interleave=True), dev, path=sdm.PATH_HYBRID, bit_exact=True, narrow_key_bits=bits)


@pytest.mark.parametrize("n,n_cell", [(5000, 257), (9000, 70_000), (4096, 4096), (300, 1_000_000), (3000, 2)])
def test_hybrid_cell_count_extremes(dev, n, n_cell):
    """one more than a digit, more cells than SDs, 17+ and 20 cell bits (8-byte words), one cell digit"""
    sdm = _sdm()
    rng = np.random.default_rng(n_cell + 1)
    cell = rng.integers(0, n_cell, n).astype(np.int32)
    if n_cell == 2:                                   # 200 + 256 SDs: the largest legal cell, one cell digit
        cell = np.concatenate([np.zeros(200, np.int32), np.ones(256, np.int32)])
        rng.shuffle(cell)
        n = len(cell)
    xi = rng.integers(1, 1000, n).astype(np.int64)
    xi[rng.random(n) < 0.2] = 77
    v = rng.integers(1, 9, n).astype(np.float64)
    w = W.Workload("edge", xi, v, cell, n_cell, 1.0, 1.0, W.GOLOVIN, 2.0 ** -10, 0.0, 3, 2)
    _run_parity(w, dev, path=sdm.PATH_HYBRID, bit_exact=True, expect_last_path=sdm.PATH_HYBRID)


def test_hybrid_path_refuses_large_cells(dev):
    """a cell of more than 256 SDs: the device check skips the whole step and reports it"""
    sdm = _sdm()
    w = W.cfg3(n_cell=8, per_cell=300, n_steps=1, interleave=True)
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        before = xi.clone(), v.clone()
        ctx.set_path(sdm.PATH_HYBRID)
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, 0)
        assert ctx.poll_error() == -4
        assert torch.equal(xi, before[0]) and torch.equal(v, before[1])


@pytest.mark.parametrize("per_cell", [1, 2, 3, 31, 32, 33, 63, 64, 65, 127, 129, 255, 256])
def test_cell_sorted_path_cell_sizes(dev, per_cell):
    """every register-tile width of the per-cell sort, at and around its boundaries, plus empty cells"""
    sdm = _sdm()
    rng = np.random.default_rng(per_cell)
    n_cell = 41
    counts = np.full(n_cell, per_cell)
    counts[[3, 4, 17, 40]] = 0                      # empty cells, including the last one
    counts[5] = max(per_cell - 1, 0)
    cell = np.repeat(np.arange(n_cell, dtype=np.int32), counts)
    n = len(cell)
    xi = rng.integers(1, 60, n).astype(np.int64)
    xi[rng.random(n) < 0.2] = 9
    v = rng.integers(1, 9, n).astype(np.float64)
    w = W.Workload("edge", xi, v, cell, n_cell, 1.0, 1.0, W.GOLOVIN, 2.0 ** -9, 0.0, 4, 2)
    _run_parity(w, dev, path=sdm.PATH_CELL_SORTED, bit_exact=True)


def test_auto_path_switches_to_cell_sorted(dev):
    sdm = _sdm()
    w = W.small("cfg3")
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        kp = _gkp(w)
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 0)
        assert ctx.last_path() == sdm.PATH_GENERAL          # first sight of this cell_id array
        torch.cuda.synchronize()
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 1)
        assert ctx.last_path() == sdm.PATH_CELL_SORTED      # verdict: sorted, cells <= 256
        # an interleaved array with small cells: general once, then the hybrid path
        wi = W.small("cfg3", interleave=True)
        xi2, v2, cell2 = _to_dev(wi, dev)
        for s in range(3):
            ctx.coalescence_step(xi2, v2, cell2, wi.n_cell, wi.dt, wi.dV, kp, 42, s)
            torch.cuda.synchronize()
            assert ctx.last_path() == (sdm.PATH_GENERAL if s == 0 else sdm.PATH_HYBRID)
        # cells larger than the fast path's limit: general path
        big = W.cfg3(n_cell=8, per_cell=300, n_steps=3)
        xb, vb, cb = _to_dev(big, dev)
        for s in range(3):
            ctx.coalescence_step(xb, vb, cb, big.n_cell, big.dt, big.dV, kp, 42, s)
            torch.cuda.synchronize()
            assert ctx.last_path() == sdm.PATH_GENERAL
        assert ctx.poll_error() == 0


def test_cell_sorted_path_refuses_unsorted_input(dev):
    """explicit CELL_SORTED on an unsorted array, and AUTO with a verdict that went stale because
    cell_id was modified in place: the step is not applied and SDM_ERR_BAD_DATA is reported."""
    sdm = _sdm()
    w = W.small("cfg3")
    kp = _gkp(w)
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        cell[100], cell[5000] = cell[5000].item(), cell[100].item()      # break the order
        ctx.set_path(sdm.PATH_CELL_SORTED)
        before = xi.clone(), v.clone()
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 0)
        assert ctx.poll_error() == -4
        assert torch.equal(xi, before[0]) and torch.equal(v, before[1])
        # AUTO: learn "sorted", then break the array in place
        ctx.set_path(sdm.PATH_AUTO)
        xi, v, cell = _to_dev(w, dev)
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 0)
        torch.cuda.synchronize()
        cell[100], cell[5000] = cell[5000].item(), cell[100].item()
        before = xi.clone(), v.clone()
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 1)
        assert ctx.last_path() == sdm.PATH_CELL_SORTED
        assert ctx.poll_error() == -4                                     # caught on the device
        assert torch.equal(xi, before[0]) and torch.equal(v, before[1])
        # the verdict was reset: the next step takes the general path and matches the oracle
        ow = w.copy()
        oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), 42, 0)
        ow.cell_id[100], ow.cell_id[5000] = ow.cell_id[5000], ow.cell_id[100]
        oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), 42, 1)
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 1)
        assert ctx.last_path() == sdm.PATH_GENERAL and ctx.poll_error() == 0
        assert np.array_equal(xi.cpu().numpy(), ow.xi)


def test_worked_step_on_device(dev):
    """The SURVEY P12 worked example straight through the C ABI."""
    sdm = _sdm()
    xi = torch.tensor([10, 3, 5, 5, 7, 1], dtype=torch.int64, device=dev)
    v = torch.tensor([1, 2, 3, 4, 5, 6], dtype=torch.float64, device=dev)
    cell = torch.tensor([0, 0, 0, 0, 0, 1], dtype=torch.int32, device=dev)
    want = [([3, 3, 3, 2, 7, 1], [1, 2, 7, 7, 6, 6], [4, 0, 3, 2, 1, 5]),
            ([1, 1, 2, 2, 7, 1], [1, 9, 9, 8, 6, 6], [0, 3, 1, 2, 4, 5]),
            ([0, 1, 2, 2, 1, 1], [10, 10, 9, 26, 6, 6], [3, 4, 0, 1, 2, 5])]
    with sdm.SDMContext(16, 2, device=dev) as ctx:
        dbg = ctx.debug_outputs(6, 2)
        for s, (wxi, wv, wperm) in enumerate(want):
            ctx.coalescence_step(xi, v, cell, 2, 1.0, 8.0, sdm.golovin(1.0), 42, s)
            assert xi.tolist() == wxi and v.tolist() == [float(x) for x in wv]
            assert dbg["perm"][:6].tolist() == wperm
        n = ctx.remove_zero_multiplicity(xi, v, cell)
        assert n == 5 and xi[:5].tolist() == [1, 2, 2, 1, 1] and cell[:5].tolist() == [0, 0, 0, 0, 1]


# ------------------------------------------------------------------------------------------- edges
@pytest.mark.parametrize("n", [0, 1, 2, 3, 31, 32, 33, 4095, 4096, 4097, 8191, 12289])
def test_ragged_sizes_single_cell(dev, n):
    rng = np.random.default_rng(n)
    xi = rng.integers(1, 50, n).astype(np.int64)
    v = rng.integers(1, 9, n).astype(np.float64)
    w = W.Workload("edge", xi, v, np.zeros(n, np.int32), 1, 1.0, 1.0, W.GOLOVIN, 2.0 ** -8, 0.0, 3, 1)
    _run_parity(w, dev, bit_exact=True)


@pytest.mark.parametrize("n,n_cell", [(5000, 3), (5000, 257), (9000, 70_000), (4096, 4096), (300, 1_000_000)])
def test_cell_count_extremes(dev, n, n_cell):
    """few big cells, one more than a digit, more cells than SDs (mostly empty), 17+ cell bits."""
    rng = np.random.default_rng(n_cell)
    cell = rng.integers(0, n_cell, n).astype(np.int32)
    xi = rng.integers(1, 1000, n).astype(np.int64)
    xi[rng.random(n) < 0.2] = 77
    v = rng.integers(1, 9, n).astype(np.float64)
    w = W.Workload("edge", xi, v, cell, n_cell, 1.0, 1.0, W.GOLOVIN, 2.0 ** -10, 0.0, 3, 2)
    _run_parity(w, dev, bit_exact=True)


def test_all_zero_and_no_zero_compaction(dev):
    sdm = _sdm()
    n = 10_000
    with sdm.SDMContext(n, 4, device=dev) as ctx:
        xi = torch.zeros(n, dtype=torch.int64, device=dev)
        v = torch.ones(n, dtype=torch.float64, device=dev)
        cell = torch.zeros(n, dtype=torch.int32, device=dev)
        assert ctx.remove_zero_multiplicity(xi, v, cell) == 0
        xi = torch.arange(1, n + 1, dtype=torch.int64, device=dev)
        assert ctx.remove_zero_multiplicity(xi, v, cell) == n
        assert torch.equal(xi, torch.arange(1, n + 1, dtype=torch.int64, device=dev))
        assert ctx.remove_zero_multiplicity(xi, v, cell, n_sd=0) == 0
        # single zero at the very front / very end
        xi[0] = 0
        assert ctx.remove_zero_multiplicity(xi, v, cell) == n - 1
        assert xi[0].item() == 2 and xi[n - 2].item() == n
        xi2 = torch.arange(1, n + 1, dtype=torch.int64, device=dev)
        xi2[n - 1] = 0
        assert ctx.remove_zero_multiplicity(xi2, v, cell) == n - 1


def test_compaction_random_against_oracle(dev):
    sdm = _sdm()
    rng = np.random.default_rng(9)
    for n, pz in [(100_003, 0.5), (50_000, 0.01), (70_001, 0.99), (2049, 0.3)]:
        xi = rng.integers(1, 10, n).astype(np.int64)
        xi[rng.random(n) < pz] = 0
        v = rng.random(n)
        cell = rng.integers(0, 100, n).astype(np.int32)
        with sdm.SDMContext(n, 100, device=dev) as ctx:
            gx, gv, gc = (torch.from_numpy(a.copy()).to(dev) for a in (xi, v, cell))
            m = ctx.remove_zero_multiplicity(gx, gv, gc)
        mo = oracle.remove_zero_multiplicity(xi, v, cell)
        assert m == mo
        assert np.array_equal(gx[:m].cpu().numpy(), xi[:m])
        assert np.array_equal(gv[:m].cpu().numpy(), v[:m])
        assert np.array_equal(gc[:m].cpu().numpy(), cell[:m])


def test_cell_stats_against_oracle(dev):
    sdm = _sdm()
    for name in ("cfg1", "cfg3", "cfg4"):
        w = W.small(name, interleave=(name == "cfg4"))
        with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
            xi, v, cell = _to_dev(w, dev)
            cnt, sx, sxv, sxv2 = ctx.cell_stats(xi, v, cell, w.n_cell)
        ocnt, osx, osxv, osxv2 = oracle.cell_stats(w.xi, w.v, w.cell_id, w.n_cell)
        assert np.array_equal(cnt.cpu().numpy(), ocnt)
        assert np.array_equal(sx.cpu().numpy(), osx)
        assert np.allclose(sxv.cpu().numpy(), osxv, rtol=1e-12, atol=0.0)
        assert np.allclose(sxv2.cpu().numpy(), osxv2, rtol=1e-12, atol=0.0)


def test_resume_bit_exact(dev):
    """P10: 2k steps == k steps + dump/reload + k steps (counter-based RNG)."""
    sdm = _sdm()
    w = W.small("cfg4")
    kp = _gkp(w)
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        a = _to_dev(w, dev)
        for s in range(6):
            ctx.coalescence_step(*a, w.n_cell, w.dt, w.dV, kp, 42, s)
        b = _to_dev(w, dev)
        for s in range(3):
            ctx.coalescence_step(*b, w.n_cell, w.dt, w.dV, kp, 42, s)
    host = [t.cpu().clone() for t in b]
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx2:
        c = [t.to(dev) for t in host]
        for s in range(3, 6):
            ctx2.coalescence_step(*c, w.n_cell, w.dt, w.dV, kp, 42, s)
    assert torch.equal(a[0], c[0]) and torch.equal(a[1].view(torch.int64), c[1].view(torch.int64))


def test_host_buffer_entry_point(dev):
    sdm = _sdm()
    w = W.small("cfg3")
    ow = w.copy()
    oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), 42, 0)
    xi = torch.from_numpy(w.xi.copy()).pin_memory()
    v = torch.from_numpy(w.v.copy()).pin_memory()
    cell = torch.from_numpy(w.cell_id.copy()).pin_memory()
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev, host_staging=True) as ctx:
        ctx.coalescence_step_host(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, 0)
    assert np.array_equal(xi.numpy(), ow.xi)
    _assert_vol_close(v.numpy(), ow.v)


def test_errors_and_bad_data(dev):
    sdm = _sdm()
    n = 1000
    with sdm.SDMContext(n, 8, device=dev) as ctx:
        xi = torch.ones(n, dtype=torch.int64, device=dev)
        v = torch.ones(n, dtype=torch.float64, device=dev)
        cell = torch.zeros(n, dtype=torch.int32, device=dev)
        kp = sdm.golovin(1.0)
        for bad in [dict(dt=0.0), dict(dV=-1.0), dict(dt=float("nan")), dict(n_cell=0)]:
            args = dict(n_cell=8, dt=1.0, dV=1.0)
            args.update(bad)
            with pytest.raises(sdm.SDMError) as e:
                ctx.coalescence_step(xi, v, cell, args["n_cell"], args["dt"], args["dV"], kp, 42, 0)
            assert e.value.status == -1
        with pytest.raises(sdm.SDMError) as e:
            ctx.coalescence_step(xi, v, cell, 9, 1.0, 1.0, kp, 42, 0)
        assert e.value.status == -2                               # n_cell > max_n_cell
        with pytest.raises(sdm.SDMError) as e:
            ctx.coalescence_step(xi, v, cell, 8, 1.0, 1.0, sdm.KernelParams(kind=7, _pad=0, b=1.0, E=1.0), 42, 0)
        assert e.value.status == -1
        with pytest.raises(sdm.SDMError) as e:
            ctx.coalescence_step(xi, v, cell, 8, 1.0, 1.0, sdm.golovin(-1.0), 42, 0)
        assert e.value.status == -1
        # device-side bad data: cell_id out of range -> sticky flag, memory-safe
        cell[17] = 8
        ctx.coalescence_step(xi, v, cell, 8, 1.0, 1.0, kp, 42, 0)
        assert ctx.poll_error() == -4
        assert ctx.poll_error() == 0                              # cleared
        cell[17] = -3
        ctx.coalescence_step(xi, v, cell, 8, 1.0, 1.0, kp, 42, 1)
        assert ctx.poll_error() == -4
        assert ctx.launch_count() > 0


# ------------------------------------------------------------------------------------------- full size
FULL = {
    "cfg0": lambda: W.cfg0(),
    "cfg1": lambda: W.cfg1(),
    "cfg2": lambda: W.cfg2(),
    "cfg3": lambda: W.cfg3(),
    "cfg4": lambda: W.cfg4(),
}


@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
def test_full_size_configs_two_steps(dev, name):
    """BASELINE.json sizes, in the launch configuration bench.py times (auto path, debug outputs off):
    two consecutive steps (+ the per-step compaction of configs[3]) against the oracle, every element."""
    sdm = _sdm()
    w = FULL[name]()
    ow = w.copy()
    okp, gkp = _okp(w), _gkp(w)
    n = w.n_sd
    with sdm.SDMContext(n, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        for s in range(2):
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, w.seed, s, n_sd=n)
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, gkp, w.seed, s, n_sd=n)
            if w.compact_every:
                n_o = oracle.remove_zero_multiplicity(ow.xi, ow.v, ow.cell_id, n_sd=n)
                assert ctx.remove_zero_multiplicity(xi, v, cell, n_sd=n) == n_o
                n = n_o
            assert ctx.poll_error() == 0
            assert np.array_equal(xi[:n].cpu().numpy(), ow.xi[:n]), f"{name} multiplicity step {s}"
            gv = v[:n].cpu().numpy()
            _assert_vol_close(gv, ow.v[:n], f"{name} step {s}")
            assert np.array_equal(gv.view(np.int64), ow.v[:n].view(np.int64))


def test_cfg0_long_run_matches_oracle(dev):
    """configs[0] for 600 steps (thousands of splits, p up to ~10): state identical at the end."""
    sdm = _sdm()
    w = W.cfg0(n_steps=600)
    ow = w.copy()
    oracle.run(ow.xi, ow.v, ow.cell_id, 1, w.dt, w.dV, _okp(w), 42, 0, 600)
    with sdm.SDMContext(w.n_sd, 1, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        kp = _gkp(w)
        for s in range(600):
            ctx.coalescence_step(xi, v, cell, 1, w.dt, w.dV, kp, 42, s)
        assert ctx.poll_error() == 0
    assert np.array_equal(xi.cpu().numpy(), ow.xi)
    assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v.view(np.int64))


# ------------------------------------------------------------------------------------------- multi-GPU plan
@pytest.mark.parametrize("name", ["cfg3", "cfg4s"])
@pytest.mark.parametrize("path", ["general", "cell_sorted"])
def test_shards_with_index_base_reproduce_the_unsharded_step(dev, name, path):
    """contiguous cell ranges stepped separately with SDM_OPT_INDEX_BASE = first array entry of the
    shard give exactly the bits of the unsharded step (here: two shards one after the other on one GPU, each
    against the unsharded ORACLE result)."""
    sdm = _sdm()
    w = W.small(name)
    ow = w.copy()
    okp = _okp(w)
    n_steps = 3
    for s in range(n_steps):
        oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, w.seed, s)
    p = {"general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED}[path]
    for rank in range(2):
        sh = W.shard(w, rank, 2)
        sw = sh.work
        with sdm.SDMContext(sw.n_sd, sw.n_cell, device=dev) as ctx:
            ctx.set_path(p)
            ctx.set_option(sdm.OPT_INDEX_BASE, sh.index_base)
            xi, v, cell = _to_dev(sw, dev)
            for s in range(n_steps):
                ctx.coalescence_step(xi, v, cell, sw.n_cell, sw.dt, sw.dV, _gkp(sw), sw.seed, s)
            assert ctx.poll_error() == 0
            lo, n = sh.index_base, sw.n_sd
            assert np.array_equal(xi.cpu().numpy(), ow.xi[lo:lo + n])
            assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v[lo:lo + n].view(np.int64))


# ------------------------------------------------------------------------------------------- NEXT-2: spectrum
def _paper_volume_edges():
    return 4.0 / 3.0 * np.pi * np.logspace(np.log10(10e-6), np.log10(5e-3), 32) ** 3


@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg3", "cfg4"])
def test_volume_spectrum_against_oracle(dev, name):
    """sdm_volume_spectrum on the paper's 31 bins: counts and sum xi exact, sum xi v within 1e-12 relative."""
    sdm = _sdm()
    w = W.small(name)
    edges = _paper_volume_edges()
    if name in ("cfg3", "cfg4"):                     # their spectra sit below 10 um: bins that actually fill
        edges = np.exp(np.linspace(np.log(w.v[w.v > 0].min() * 0.5), np.log(w.v.max() * 0.9), 40))
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        kp = _gkp(w)
        for s in range(3):
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, w.seed, s)
        got = [t.cpu().numpy() for t in ctx.volume_spectrum(xi, v, edges)]
        hx, hv = xi.cpu().numpy(), v.cpu().numpy()
    want = oracle.volume_spectrum(hx, hv, edges)
    assert want[0].sum() > 0.5 * w.n_sd
    assert np.array_equal(got[0], want[0])
    assert np.array_equal(got[1], want[1])
    assert np.allclose(got[2], want[2], rtol=VOL_RTOL, atol=0.0)


def test_volume_spectrum_edges_and_degenerate_inputs(dev):
    sdm = _sdm()
    edges = np.array([1.0, 2.0, 4.0, 8.0])
    v = np.array([0.5, 1.0, 1.5, 2.0, 3.0, 4.0, 7.9, 8.0, 9.0, np.nan])
    xi = np.array([100, 1, 2, 3, 4, 5, 6, 700, 800, 900], np.int64)
    with sdm.SDMContext(1024, 1, device=dev) as ctx:
        got = [t.cpu().numpy() for t in ctx.volume_spectrum(torch.from_numpy(xi).to(dev), torch.from_numpy(v).to(dev), edges)]
        assert got[0].tolist() == [2, 2, 2] and got[1].tolist() == [3, 7, 11]
        assert got[2].tolist() == [1 * 1.0 + 2 * 1.5, 3 * 2.0 + 4 * 3.0, 5 * 4.0 + 6 * 7.9]
        # all in one bin (one 32-lane group per warp), ragged length, two edges only
        n = 1000 + 7
        xi1 = torch.full((n,), 3, dtype=torch.int64, device=dev)
        v1 = torch.full((n,), 1.25, dtype=torch.float64, device=dev)
        c, sx, sv = ctx.volume_spectrum(xi1, v1, [1.0, 2.0])
        assert c.item() == n and sx.item() == 3 * n and sv.item() == 3 * n * 1.25
        # empty input, and bad edges
        c, sx, sv = ctx.volume_spectrum(xi1, v1, edges, n_sd=0)
        assert c.sum().item() == 0
        for bad in ([1.0], [2.0, 1.0], [1.0, float("inf")], list(range(1, 1028))):
            with pytest.raises(sdm.SDMError):
                ctx.volume_spectrum(xi1, v1, bad)


# ------------------------------------------------------------------------------------------- races / path equality
@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_full_size_paths_agree_and_repeat(dev, name):
    """BASELINE.json sizes: the three paths give the same bits, and running a path twice from the same state
    gives the same bits again (a race in the look-back, the rank tables, the tie repair or the fused kernel's
    staging would show up as a difference between runs or paths).  The oracle comparison at these sizes is
    test_full_size_configs_two_steps; this one needs no CPU time, so it runs more steps."""
    sdm = _sdm()
    w = FULL[name]()
    n, n_steps = w.n_sd, 4
    kp = _gkp(w)
    results = []
    with sdm.SDMContext(n, w.n_cell, device=dev) as ctx:
        ctx.set_option(sdm.OPT_TRACK_ZEROS, 1)
        for path in (sdm.PATH_GENERAL, sdm.PATH_CELL_SORTED, sdm.PATH_HYBRID, sdm.PATH_GENERAL, sdm.PATH_CELL_SORTED):
            ctx.set_path(path)
            xi, v, cell = _to_dev(w, dev)
            m = n
            for s in range(n_steps):
                ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, w.seed, s, n_sd=m)
                if w.compact_every:
                    m = ctx.remove_zero_multiplicity(xi, v, cell, n_sd=m)
            assert ctx.poll_error() == 0
            results.append((m, xi[:m].clone(), v[:m].clone()))
    m0, xi0, v0 = results[0]
    assert int((xi0 != torch.from_numpy(w.xi[:m0]).to(dev)).sum()) > 0        # something did collide
    for m, xi, v in results[1:]:
        assert m == m0
        assert torch.equal(xi, xi0)
        assert torch.equal(v.view(torch.int64), v0.view(torch.int64))
