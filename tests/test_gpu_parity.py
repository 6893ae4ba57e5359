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
                track_zeros=False, skip_key_digits=None, fused_r=None, bucket_bits=None, box_cluster=None):
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
        if fused_r is not None:
            ctx.set_option(sdm.OPT_FUSED_WORDS_PER_LANE, fused_r)
        if bucket_bits is not None:
            ctx.set_option(sdm.OPT_BUCKET_BITS, bucket_bits)
        if box_cluster is not None:
            ctx.set_option(sdm.OPT_BOX_CLUSTER, box_cluster)
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
@pytest.mark.parametrize("fused_r", [4, 8])
def test_fused_kernel_tie_repair(dev, path, bits, fused_r):
    """With only a few key bits in the 32-bit sort word nearly every cell has neighbours whose truncated keys
    tie (with 1 bit: runs of half a cell), so the exact repair by the regenerated full key runs all the time, inside
    the lanes and across their boundaries; the result must not change."""
    sdm = _sdm()
    if path == "cell_sorted":
        _run_parity(W.small("cfg4"), dev, path=sdm.PATH_CELL_SORTED, bit_exact=True, narrow_key_bits=bits, fused_r=fused_r)
    else:
        _run_parity(W.small("cfg3", interleave=True), dev, path=sdm.PATH_HYBRID, bit_exact=True, narrow_key_bits=bits,
                    fused_r=fused_r)


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
@pytest.mark.parametrize("path", ["cell_sorted", "hybrid"])
@pytest.mark.parametrize("fused_r", [4, 8])
def test_fused_kernel_words_per_lane(dev, name, path, fused_r):
    """Every group shape of the fused kernel (classes of 32 / 64 / 128 / 256 slots on P / R lanes of R words, classes of
    48 / 96 / 192 slots on P / 6 lanes of 6 words; uniform cell
    sizes served as one class, mixed sizes through the class lists) gives the oracle's bits."""
    sdm = _sdm()
    p = {"cell_sorted": sdm.PATH_CELL_SORTED, "hybrid": sdm.PATH_HYBRID}[path]
    _run_parity(W.small(name, interleave=(path == "hybrid")), dev, path=p, bit_exact=True, fused_r=fused_r)
    _run_parity(W.small(name, interleave=(path == "hybrid")), dev, path=p, check_debug=False, bit_exact=True,
                track_zeros=True, fused_r=fused_r)


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


@pytest.mark.parametrize("per_cell", [1, 2, 3, 15, 16, 17, 31, 32, 33, 47, 48, 49, 63, 64, 65, 95, 96, 97, 127, 128, 129,
                                      191, 192, 193, 255, 256])
@pytest.mark.parametrize("fused_r", [None, 4, 8])
def test_cell_sorted_path_cell_sizes(dev, per_cell, fused_r):
    """every size class of the per-cell sort, at and around its boundaries, plus empty cells"""
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
    _run_parity(w, dev, path=sdm.PATH_CELL_SORTED, bit_exact=True, fused_r=fused_r)


def test_auto_path_picks_the_path_that_fits(dev):
    sdm = _sdm()
    w = W.small("cfg3")
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        kp = _gkp(w)
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 0)
        assert ctx.last_path() == sdm.PATH_CELL_SORTED      # analysed on the device: sorted, cells <= 256
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 1)
        assert ctx.last_path() == sdm.PATH_CELL_SORTED
        # an interleaved array with small cells: general once (which sees the cell sizes), then the hybrid path
        wi = W.small("cfg3", interleave=True)
        xi2, v2, cell2 = _to_dev(wi, dev)
        for s in range(3):
            ctx.coalescence_step(xi2, v2, cell2, wi.n_cell, wi.dt, wi.dV, kp, 42, s)
            assert ctx.last_path() == (sdm.PATH_GENERAL if s == 0 else sdm.PATH_HYBRID)
        # cells larger than the fast path's limit: general path
        big = W.cfg3(n_cell=8, per_cell=300, n_steps=3)
        xb, vb, cb = _to_dev(big, dev)
        for s in range(3):
            ctx.coalescence_step(xb, vb, cb, big.n_cell, big.dt, big.dV, kp, 42, s)
            assert ctx.last_path() == sdm.PATH_GENERAL
        assert ctx.poll_error() == 0


def test_explicit_cell_sorted_path_refuses_unsorted_input(dev):
    """explicit CELL_SORTED on an unsorted array is the caller's error: the step is not applied and
    SDM_ERR_BAD_DATA is reported."""
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
        with pytest.raises(sdm.SDMError) as e:                            # the multi-step entry reports it at once
            ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, 0, 3)
        assert e.value.status == -4
        assert torch.equal(xi, before[0]) and torch.equal(v, before[1])
        assert ctx.poll_error() == 0


def test_auto_falls_back_when_cell_id_is_rewritten_in_place(dev):
    """AUTO never refuses valid input: cell_id rewritten in place between steps (what a displacement step does) makes
    the next step take the path that fits -- oracle-identical output, status 0 (What's weak 8)."""
    sdm = _sdm()
    w = W.small("cfg3")
    ow = w.copy()
    okp, kp = _okp(w), _gkp(w)
    rng = np.random.default_rng(5)
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        expect = [sdm.PATH_CELL_SORTED, sdm.PATH_GENERAL, sdm.PATH_HYBRID, sdm.PATH_HYBRID, sdm.PATH_HYBRID]
        for s in range(5):
            if s == 1:      # a few super-droplets move to neighbouring cells: no longer sorted
                moved = rng.choice(w.n_sd, 200, replace=False)
                ow.cell_id[moved] = np.clip(ow.cell_id[moved] + rng.integers(-1, 2, 200), 0, w.n_cell - 1).astype(np.int32)
                cell.copy_(torch.from_numpy(ow.cell_id))
            if s == 4:      # and the caller sorts everything again, in place
                order = np.argsort(ow.cell_id, kind="stable")
                ow.xi, ow.v, ow.cell_id = ow.xi[order].copy(), ow.v[order].copy(), ow.cell_id[order].copy()
                xi.copy_(torch.from_numpy(ow.xi)); v.copy_(torch.from_numpy(ow.v)); cell.copy_(torch.from_numpy(ow.cell_id))
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, 42, s)
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, s)
            assert ctx.last_path() == expect[s], f"step {s}"
            assert ctx.poll_error() == 0
            assert np.array_equal(xi.cpu().numpy(), ow.xi), f"step {s}"
            assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v.view(np.int64)), f"step {s}"


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_back_to_back_auto_steps_without_host_sync(dev, name):
    """Several AUTO steps enqueued with nothing but the library's own calls in between (no poll, no synchronize,
    no compaction): every call returns 0 and the result is the oracle's (a not-ready event query must not
    poison the context)."""
    sdm = _sdm()
    for interleave in (False, True):
        w = W.small(name, interleave=interleave)
        ow = w.copy()
        okp, kp = _okp(w), _gkp(w)
        with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
            xi, v, cell = _to_dev(w, dev)
            for s in range(5):
                ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, s)   # raises on rc != 0
            assert ctx.poll_error() == 0
            for s in range(5):
                oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, 42, s)
            assert np.array_equal(xi.cpu().numpy(), ow.xi)
            assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v.view(np.int64))


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


@pytest.mark.parametrize("n", [1, 2, 3, 33, 127, 128, 129, 1000, 1024, 1025, 2049, 4097, 8191, 8192])
@pytest.mark.parametrize("kind", ["golovin", "geometric"])
@pytest.mark.parametrize("box_cluster", [1, 0])
def test_box_step_one_block(dev, n, kind, box_cluster):
    """SURVEY 8(f) NEXT-1, tiny N: the whole step of a one-cell box in one launch (counting placement of the keys
    instead of radix passes), on a cluster of eight blocks with the state in distributed shared memory and on one
    block.  Permutation, every gamma and the state equal the oracle's, with and without debug outputs, for ragged
    sizes around the per-block share of 1024."""
    sdm = _sdm()
    rng = np.random.default_rng(7 * n + len(kind))
    if kind == "golovin":
        xi = rng.integers(1, 50, n).astype(np.int64)
        xi[rng.random(n) < 0.3] = 7
        v = rng.integers(1, 9, n).astype(np.float64)
        w = W.Workload("box", xi, v, np.zeros(n, np.int32), 1, 1.0, 1.0, W.GOLOVIN, 2.0 ** -8 / max(n, 1) * 64, 0.0, 4, 2)
    else:
        w0 = W.cfg1(n_sd=n, n_steps=4)
        w = W.Workload("box", w0.xi, w0.v, w0.cell_id, 1, 1.0, w0.dV / 50.0, W.GEOMETRIC, 0.0, 1.0, 4, 0)
    st = _run_parity(w, dev, path=sdm.PATH_BOX, bit_exact=True, expect_last_path=sdm.PATH_BOX, box_cluster=box_cluster)
    _run_parity(w, dev, path=None, check_debug=False, bit_exact=True, expect_last_path=sdm.PATH_BOX, box_cluster=box_cluster)
    if n >= 1000:
        assert st["gamma_nonzero"] > 0


@pytest.mark.parametrize("n", [1, 2, 3, 5, 64, 129, 1000, 4097, 8193, 40_123, 300_001])
@pytest.mark.parametrize("kind", ["golovin", "geometric"])
@pytest.mark.parametrize("bits", [0, 1, 3])
def test_bucket_path_single_cell(dev, n, kind, bits):
    """One cell in key buckets (two-level counting placement + the pair kernel): the permutation, every gamma and the
    state equal the oracle's for every coarse bucket count (bits: 0 = automatic, else that many more key bits than
    automatic: few entries in many buckets, empty buckets), ragged sizes and both kernels."""
    sdm = _sdm()
    rng = np.random.default_rng(11 * n + len(kind))
    if kind == "golovin":
        xi = rng.integers(1, 50, n).astype(np.int64)
        xi[rng.random(n) < 0.3] = 7
        v = rng.integers(1, 9, n).astype(np.float64)
        w = W.Workload("box", xi, v, np.zeros(n, np.int32), 1, 1.0, 1.0, W.GOLOVIN, 2.0 ** -8 / max(n, 1) * 64, 0.0, 4, 2)
    else:
        w0 = W.cfg1(n_sd=n, n_steps=4)
        w = W.Workload("box", w0.xi, w0.v, w0.cell_id, 1, 1.0, w0.dV / 50.0, W.GEOMETRIC, 0.0, 1.0, 4, 0)
    auto_bits = 1
    while auto_bits < 12 and (2048 << auto_bits) < n:
        auto_bits += 1
    opts = {} if bits == 0 else {"bucket_bits": min(auto_bits + 3 * bits, 12)}
    st = _run_parity(w, dev, path=sdm.PATH_BUCKET, bit_exact=True, expect_last_path=sdm.PATH_BUCKET, **opts)
    _run_parity(w, dev, path=sdm.PATH_BUCKET, check_debug=False, bit_exact=True, track_zeros=True, **opts)
    if n >= 1000:
        assert st["gamma_nonzero"] > 0


def test_auto_takes_the_bucket_path_for_a_large_single_cell(dev):
    sdm = _sdm()
    _run_parity(W.small("cfg1"), dev, path=None, bit_exact=True, expect_last_path=sdm.PATH_BUCKET)
    _run_parity(W.small("cfg3"), dev, path=sdm.PATH_BUCKET, bit_exact=True, expect_last_path=sdm.PATH_GENERAL)


def test_bucket_overflow_is_reported(dev):
    """A coarse bucket of more than 4096 entries cannot happen with the automatic bucket count (twice the largest
    average); forced with two key bits on 20 000 super-droplets it is reported, not silently mishandled."""
    sdm = _sdm()
    n = 20_000
    with sdm.SDMContext(n, 1, device=dev) as ctx:
        ctx.set_path(sdm.PATH_BUCKET)
        ctx.set_option(sdm.OPT_BUCKET_BITS, 2)
        xi = torch.full((n,), 5, dtype=torch.int64, device=dev)
        v = torch.ones(n, dtype=torch.float64, device=dev)
        cell = torch.zeros(n, dtype=torch.int32, device=dev)
        ctx.coalescence_step(xi, v, cell, 1, 1.0, 1.0, sdm.golovin(1e-3), 42, 0)
        assert ctx.poll_error() == -4


def test_box_path_falls_back_to_general_when_it_does_not_fit(dev):
    sdm = _sdm()
    w = W.small("cfg1")          # 40 123 super-droplets in one cell: more than one block takes
    _run_parity(w, dev, path=sdm.PATH_BOX, bit_exact=True, expect_last_path=sdm.PATH_GENERAL)
    w = W.small("cfg3")          # many cells
    _run_parity(w, dev, path=sdm.PATH_BOX, bit_exact=True, expect_last_path=sdm.PATH_GENERAL)


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


# ------------------------------------------------------------------------------------------- the time loop
def _run_multi(w, dev, path, n_steps, compact_every, chunks=(None,)):
    """sdm_coalescence_steps against oracle.run, in one call or split into several calls (resume)."""
    sdm = _sdm()
    ow = w.copy()
    n_o = oracle.run(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), w.seed, 0, n_steps, compact_every)
    with sdm.SDMContext(max(w.n_sd, 1), w.n_cell, device=dev) as ctx:
        if path is not None:
            ctx.set_path(path)
        xi, v, cell = _to_dev(w, dev)
        n, s = w.n_sd, 0
        parts = [n_steps] if chunks == (None,) else list(chunks)
        assert sum(parts) == n_steps
        for k in parts:
            # a call's compaction schedule counts from ITS first step: split only at multiples of compact_every
            assert compact_every == 0 or s % compact_every == 0
            n = ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), w.seed, s, k, compact_every, n_sd=n)
            s += k
        assert ctx.poll_error() == 0
        last = ctx.last_path()
    assert n == n_o
    assert np.array_equal(xi[:n].cpu().numpy(), ow.xi[:n])
    assert np.array_equal(cell[:n].cpu().numpy(), ow.cell_id[:n])
    assert np.array_equal(v[:n].cpu().numpy().view(np.int64), ow.v[:n].view(np.int64))
    return n, last


@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg3z", "cfg4", "cfg4s"])
@pytest.mark.parametrize("path", ["auto", "general", "cell_sorted", "hybrid"])
def test_multi_step_entry_matches_oracle_run(dev, name, path):
    """sdm_coalescence_steps == oracle_run: n steps with the config's compaction schedule in ONE call,
    on every path; cfg3z starts with 2 % zeros (halt at the first due step), cfg4s produces zeros all the time."""
    sdm = _sdm()
    if name in ("cfg0", "cfg1") and path in ("cell_sorted", "hybrid"):
        pytest.skip("single cell: general path only")
    w = W.small(name, interleave=(path == "hybrid"))
    p = {"auto": None, "general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED, "hybrid": sdm.PATH_HYBRID}[path]
    n_steps = {"cfg0": 40, "cfg4s": 30}.get(name, 7)
    n, last = _run_multi(w, dev, p, n_steps, w.compact_every)
    if name in ("cfg3z", "cfg4s"):
        assert n < w.n_sd
    if path == "auto" and name not in ("cfg0", "cfg1"):
        assert last == sdm.PATH_CELL_SORTED


@pytest.mark.parametrize("name,compact_every", [("cfg4s", 1), ("cfg4s", 3), ("cfg3z", 2), ("cfg4s", 0), ("cfg4s", 20)])
def test_multi_step_entry_compaction_schedules(dev, name, compact_every):
    """every step / every third step / never / every 20th; more steps than one chunk of the run loop (64) so that a
    halt is noticed while later chunks are already enqueued.  Small inputs take up to 64 steps inside one launch of the
    fused kernel when no compaction is due in between: 0 gives launches of 64, 20 launches of 20, 3 launches of 3."""
    w = W.small(name)
    _run_multi(w, dev, None, 150 if name == "cfg4s" else 9, compact_every)


@pytest.mark.parametrize("name,compact_every,n_steps", [("cfg2", 0, 20), ("cfg3", 1, 12), ("cfg3z", 5, 20), ("cfg4", 0, 24),
                                                        ("cfg4s", 0, 40), ("cfg4s", 10, 40), ("cfg4s", 1, 12)])
@pytest.mark.parametrize("path", ["hybrid", "auto"])
def test_multi_step_entry_resident_hybrid_run(dev, name, compact_every, n_steps, path):
    """HYBRID runs of eight steps or more work on cell-grouped copies of the attributes (gathered once per run,
    scattered back when it ends or halts for a compaction): same bits as the step-by-step loop on interleaved input,
    with no compaction, with compactions that find nothing, with a halt in the first steps (cfg3z) and with halts all
    the time (cfg4s, every step: the runs fall back to gathering in every step)."""
    sdm = _sdm()
    w = W.small(name, interleave=True)
    _, last = _run_multi(w, dev, sdm.PATH_HYBRID if path == "hybrid" else None, n_steps, compact_every)
    assert last == sdm.PATH_HYBRID


def test_multi_step_entry_interleaved_auto_and_resume(dev):
    """AUTO on an interleaved array: one GENERAL step, then HYBRID for the rest of the call; and a run split into
    three calls equals the run in one call (counter-based RNG: step0 carries the position)."""
    sdm = _sdm()
    _, last = _run_multi(W.small("cfg4s", interleave=True), dev, None, 30, 10)
    assert last == sdm.PATH_HYBRID
    _run_multi(W.small("cfg4s"), dev, None, 30, 10, chunks=(10, 0, 20))
    _run_multi(W.small("cfg0"), dev, None, 40, 0, chunks=(1, 39))


@pytest.mark.parametrize("n,path", [(3000, "box"), (8192, "box"), (20_000, "bucket"), (20_000, "general")])
@pytest.mark.parametrize("compact_every", [0, 1, 4])
def test_single_cell_time_loop_with_zeros(dev, n, path, compact_every):
    """One cell whose multiplicities are small (1 .. 3): equal-multiplicity splits produce zeros all the time.  The
    time loop on the BOX path (many steps inside one launch, cut at every due compaction), the BUCKET path and the
    GENERAL path equals oracle.run for every compaction schedule, and the array really shrinks."""
    sdm = _sdm()
    rng = np.random.default_rng(n + compact_every)
    xi = rng.integers(1, 4, n).astype(np.int64)
    v = rng.integers(1, 9, n).astype(np.float64)
    w = W.Workload("box", xi, v, np.zeros(n, np.int32), 1, 1.0, 1.0, W.GOLOVIN, 0.5 / n, 0.0, 12, compact_every)
    p = {"box": sdm.PATH_BOX, "bucket": sdm.PATH_BUCKET, "general": sdm.PATH_GENERAL}[path]
    n_out, last = _run_multi(w, dev, p, 12, compact_every)
    assert last == p
    if compact_every:
        assert n_out < n
    _run_multi(w, dev, None, 12, compact_every, chunks=(4, 8))      # AUTO, resumed


@pytest.mark.parametrize("compact_every", [0, 7])
def test_bucket_time_loop_with_the_next_placement_ahead(dev, compact_every):
    """Inside sdm_coalescence_steps the BUCKET path starts level 1 of the NEXT step's placement on a side stream beside
    this step's pair kernel (not across a due compaction).  60 steps of 2^19 super-droplets in one call equal the same
    steps taken one call at a time -- which never runs anything ahead -- bit for bit, and the first three equal the
    oracle; twice, so that a placement left over from the first run cannot leak into the second."""
    sdm = _sdm()
    w = W.cfg1(n_sd=1 << 19, n_steps=3)
    kp = _gkp(w)
    ow = w.copy()
    n_o = oracle.run(ow.xi, ow.v, ow.cell_id, 1, w.dt, w.dV, _okp(w), w.seed, 0, 3, 0)
    with sdm.SDMContext(w.n_sd, 1, device=dev) as ctx:
        ctx.set_path(sdm.PATH_BUCKET)
        for rep in range(2):
            xi, v, cell = _to_dev(w, dev)
            n = ctx.coalescence_steps(xi, v, cell, 1, w.dt, w.dV, kp, w.seed, 0, 3, 0)
            assert n == n_o and ctx.last_path() == sdm.PATH_BUCKET
            assert np.array_equal(xi[:n].cpu().numpy(), ow.xi[:n])
            assert np.array_equal(v[:n].cpu().numpy().view(np.int64), ow.v[:n].view(np.int64))
            n = ctx.coalescence_steps(xi, v, cell, 1, w.dt, w.dV, kp, w.seed, 3, 57, compact_every, n_sd=n)
            xs, vs, cs = _to_dev(w, dev)
            m = w.n_sd
            for s in range(60):
                ctx.coalescence_step(xs, vs, cs, 1, w.dt, w.dV, kp, w.seed, s, n_sd=m)
                if compact_every and s >= 3 and (s - 3 + 1) % compact_every == 0:   # the second call's schedule
                    m = ctx.remove_zero_multiplicity(xs, vs, cs, n_sd=m)
            assert ctx.poll_error() == 0
            assert n == m
            assert torch.equal(xi[:n], xs[:n]) and torch.equal(v[:n].view(torch.int64), vs[:n].view(torch.int64))


@pytest.mark.parametrize("n,path", [(5000, "box"), (30_000, "bucket")])
def test_single_cell_paths_honour_index_base_and_the_table_kernel(dev, n, path):
    """SDM_OPT_INDEX_BASE (R34) and SDM_KERNEL_GEOMETRIC_TABLE (R39) on the single-cell paths: the same bits as the
    oracle with the same counter offset / table."""
    sdm = _sdm()
    p = {"box": sdm.PATH_BOX, "bucket": sdm.PATH_BUCKET}[path]
    w0 = W.cfg1(n_sd=n, n_steps=3)
    radius = np.array([1e-6, 2e-5, 1e-4, 2e-3])
    table = np.array([[0.1, 0.3, 0.2], [0.5, 0.9, 0.7], [1.0, 0.8, 1.2], [0.6, 1.1, 0.4]])
    base = 7_000_000_123
    with sdm.SDMContext(n, 1, device=dev) as ctx:
        ctx.set_path(p)
        ctx.set_option(sdm.OPT_INDEX_BASE, base)
        ctx.set_collision_efficiency(radius, table)
        xi, v, cell = _to_dev(w0, dev)
        ow = w0.copy()
        okp = oracle.geometric_table(radius, table)
        for s in range(3):
            ctx.coalescence_step(xi, v, cell, 1, 1.0, w0.dV / 200.0, sdm.geometric_table(), 42, s)
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, 1, 1.0, w0.dV / 200.0, okp, 42, s, index_base=base)
        assert ctx.poll_error() == 0 and ctx.last_path() == p
        assert np.array_equal(xi.cpu().numpy(), ow.xi)
        assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v.view(np.int64))
        assert np.count_nonzero(ow.xi != w0.xi) > 0


def test_multi_step_entry_edge_cases(dev):
    sdm = _sdm()
    w = W.small("cfg3")
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        before = xi.clone()
        assert ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, 0, 0, 1) == w.n_sd
        assert torch.equal(xi, before)
        assert ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, 0, 5, 1, n_sd=0) == 0
        for bad in (dict(n_steps=-1), dict(compact_every=-1)):
            args = dict(n_steps=1, compact_every=0)
            args.update(bad)
            with pytest.raises(sdm.SDMError) as e:
                ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, 0, args["n_steps"], args["compact_every"])
            assert e.value.status == -1
        # everything zero: the first due compaction empties the array and the run ends
        xi.zero_()
        assert ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, 0, 4, 1) == 0
        assert ctx.poll_error() == 0


def test_host_entry_with_a_different_cell_layout_per_call(dev):
    """sdm_coalescence_step_host re-uploads cell_id into the same staging address every call; what AUTO
    learned about the previous contents must not leak into the next call."""
    sdm = _sdm()
    wa, wb = W.small("cfg3"), W.small("cfg3", interleave=True)
    wc = W.cfg3(n_cell=16, per_cell=300, n_steps=1)           # cells too large for the fused kernel
    with sdm.SDMContext(max(wa.n_sd, wc.n_sd), max(wa.n_cell, wc.n_cell), device=dev, host_staging=True) as ctx:
        for s, w in enumerate([wa, wb, wa, wc, wb, wa]):
            ow = w.copy()
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), 42, s)
            xi, v, cell = (torch.from_numpy(a.copy()).pin_memory() for a in (w.xi, w.v, w.cell_id))
            ctx.coalescence_step_host(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, s)
            assert np.array_equal(xi.numpy(), ow.xi), f"call {s}"
            assert np.array_equal(v.numpy().view(np.int64), ow.v.view(np.int64)), f"call {s}"
        assert ctx.poll_error() == 0


@pytest.mark.parametrize("case", ["sorted", "sorted_zeros", "interleaved", "mixed_sizes", "ragged"])
def test_host_entry_pipeline(dev, case):
    """sdm_coalescence_step_host on arrays large enough for its pipeline (uploads in pieces cut at cell boundaries, the
    step on every piece as it arrives, downloads on a third stream): cell-major cells of one size take it; input zeros
    with compaction make it fetch the compacted arrays; interleaved order and mixed cell sizes fall back to the plain
    sequence; a piece count that does not divide the cells.  Two calls each, against the oracle."""
    sdm = _sdm()
    if case == "mixed_sizes":
        w = W.cfg4(n_cell=5003, n_steps=2)
    else:
        w = W.cfg3(n_cell=2311 if case == "ragged" else 2400, per_cell=128, n_steps=2, interleave=(case == "interleaved"),
                   zero_fraction=0.02 if case == "sorted_zeros" else 0.0)
    assert w.n_sd >= 1 << 18
    ow = w.copy()
    xi, v, cell = (torch.from_numpy(a.copy()).pin_memory() for a in (w.xi, w.v, w.cell_id))
    n = n_o = w.n_sd
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev, host_staging=True) as ctx:
        for s in range(2):
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), 42, s, n_sd=n_o)
            n_o = oracle.remove_zero_multiplicity(ow.xi, ow.v, ow.cell_id, n_sd=n_o)
            n = ctx.coalescence_step_host(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), 42, s, n_sd=n, compact=True)
            assert n == n_o, f"call {s}"
            assert np.array_equal(xi.numpy()[:n], ow.xi[:n]), f"call {s}"
            assert np.array_equal(cell.numpy()[:n], ow.cell_id[:n]), f"call {s}"
            assert np.array_equal(v.numpy()[:n].view(np.int64), ow.v[:n].view(np.int64)), f"call {s}"
        assert ctx.poll_error() == 0
        if case in ("sorted", "sorted_zeros", "ragged"):
            assert ctx.last_path() == sdm.PATH_CELL_SORTED
    if case == "sorted_zeros":
        assert n < w.n_sd


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


def _compare_state(xi, v, cell, ow, n, what):
    assert np.array_equal(xi[:n].cpu().numpy(), ow.xi[:n]), f"{what}: multiplicity"
    assert np.array_equal(cell[:n].cpu().numpy(), ow.cell_id[:n]), f"{what}: cell_id"
    assert np.array_equal(v[:n].cpu().numpy().view(np.int64), ow.v[:n].view(np.int64)), f"{what}: volume bits"


@pytest.mark.parametrize("path", ["general", "cell_sorted", "hybrid"])
def test_full_size_cfg3z_compaction_moves_data(dev, path):
    """configs[3] at full size with 2 % of the input multiplicities 0 (R32 "3z"): the in-place k_compact runs over
    4096 ticketed tiles in several waves and really moves data; two steps, a compaction after each, every element
    against the oracle, on each path."""
    sdm = _sdm()
    w = W.cfg3(zero_fraction=0.02)
    ow = w.copy()
    okp, gkp = _okp(w), _gkp(w)
    p = {"general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED, "hybrid": sdm.PATH_HYBRID}[path]
    n = w.n_sd
    with sdm.SDMContext(n, w.n_cell, device=dev) as ctx:
        ctx.set_path(p)
        ctx.set_option(sdm.OPT_TRACK_ZEROS, 1)
        xi, v, cell = _to_dev(w, dev)
        for s in range(2):
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, w.seed, s, n_sd=n)
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, gkp, w.seed, s, n_sd=n)
            n_o = oracle.remove_zero_multiplicity(ow.xi, ow.v, ow.cell_id, n_sd=n)
            n_g = ctx.remove_zero_multiplicity(xi, v, cell, n_sd=n)
            assert n_g == n_o and (s > 0 or n_o < n - 100_000)
            n = n_o
            assert ctx.poll_error() == 0
            _compare_state(xi, v, cell, ow, n, f"{path} step {s}")


def test_full_size_cfg4_stress_crosses_a_compaction(dev):
    """configs[4] at full size with dV = 1 m^3 (R32 "4s"): large gamma, the clamp, splits to zero (the first zeros
    appear at step 12); 22 steps in ONE sdm_coalescence_steps call with compactions due after steps 10 (nothing to
    remove) and 20 (the run halts on the device, the host compacts ~4.5e5 entries out of 6.5e6 over 3200 tiles and
    resumes), every element against oracle_run."""
    sdm = _sdm()
    w = W.cfg4(stress=True)
    ow = w.copy()
    n_o = oracle.run(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), w.seed, 0, 22, 10)
    assert n_o < w.n_sd - 100_000
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        n = ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), w.seed, 0, 22, 10)
        assert ctx.poll_error() == 0 and ctx.last_path() == sdm.PATH_CELL_SORTED
    assert n == n_o
    _compare_state(xi, v, cell, ow, n, "cfg4s 22 steps")


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
@pytest.mark.parametrize("path", ["general", "hybrid"])
def test_full_size_interleaved_order(dev, name, path):
    """R30: the full-size configs in a random memory order -- the input the GENERAL and HYBRID paths exist for --
    one step (+ configs[3]'s compaction call) against the oracle, every element."""
    sdm = _sdm()
    w = W.cfg3(interleave=True) if name == "cfg3" else W.cfg4(interleave=True)
    ow = w.copy()
    p = {"general": sdm.PATH_GENERAL, "hybrid": sdm.PATH_HYBRID}[path]
    n = w.n_sd
    with sdm.SDMContext(n, w.n_cell, device=dev) as ctx:
        ctx.set_path(p)
        xi, v, cell = _to_dev(w, dev)
        oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), w.seed, 0)
        ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), w.seed, 0)
        if w.compact_every:
            assert ctx.remove_zero_multiplicity(xi, v, cell) == oracle.remove_zero_multiplicity(ow.xi, ow.v, ow.cell_id)
        assert ctx.poll_error() == 0 and ctx.last_path() == p
    _compare_state(xi, v, cell, ow, n, f"{name} interleaved {path}")


@pytest.mark.parametrize("name", ["cfg3", "cfg4"])
def test_full_size_multi_step_entry(dev, name):
    """The launch configuration bench.py times: sdm_coalescence_steps on the full-size config (AUTO, debug outputs
    off), three steps with the config's compaction schedule, every element against oracle_run."""
    sdm = _sdm()
    w = FULL[name]()
    ow = w.copy()
    n_o = oracle.run(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), w.seed, 0, 3, w.compact_every)
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        n = ctx.coalescence_steps(xi, v, cell, w.n_cell, w.dt, w.dV, _gkp(w), w.seed, 0, 3, w.compact_every)
        assert ctx.poll_error() == 0 and ctx.last_path() == sdm.PATH_CELL_SORTED
    assert n == n_o
    _compare_state(xi, v, cell, ow, n, f"{name} multi-step")


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


@pytest.mark.parametrize("name", ["cfg3z", "cfg4s"])
def test_shards_cross_a_compaction_with_rebased_index_base(dev, name):
    """after a compaction the Philox counter of a shard's first entry is the number of survivors on the
    ranks before it.  Two shards (one after the other on one GPU), each advanced with sdm_coalescence_steps from
    compaction to compaction, index_base re-based by sdm_workloads.rebase() from the surviving counts -- the 8-byte
    all_gather of a multi-GPU run -- against the UNSHARDED oracle run, bit for bit."""
    sdm = _sdm()
    w = W.small(name)
    every = w.compact_every
    n_rounds = 3
    ow = w.copy()
    n_o = oracle.run(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, _okp(w), w.seed, 0, n_rounds * every, every)
    assert n_o < w.n_sd
    shards = [W.shard(w, r, 2) for r in range(2)]
    ctxs = [sdm.SDMContext(sh.work.n_sd, sh.work.n_cell, device=dev) for sh in shards]
    try:
        state = [_to_dev(sh.work, dev) for sh in shards]
        counts = [sh.work.n_sd for sh in shards]
        for rnd in range(n_rounds):
            bases = W.rebase(counts)
            if rnd == 0:
                assert bases == [sh.index_base for sh in shards]
            for r, sh in enumerate(shards):
                sw = sh.work
                ctxs[r].set_option(sdm.OPT_INDEX_BASE, bases[r])
                counts[r] = ctxs[r].coalescence_steps(*state[r], sw.n_cell, sw.dt, sw.dV, _gkp(sw), sw.seed, rnd * every,
                                                      every, every, n_sd=counts[r])
                assert ctxs[r].poll_error() == 0
        assert sum(counts) == n_o
        lo = 0
        for r, sh in enumerate(shards):
            xi, v, cell = state[r]
            n = counts[r]
            assert np.array_equal(xi[:n].cpu().numpy(), ow.xi[lo:lo + n])
            assert np.array_equal(v[:n].cpu().numpy().view(np.int64), ow.v[lo:lo + n].view(np.int64))
            assert np.array_equal(cell[:n].cpu().numpy() + sh.cell_lo, ow.cell_id[lo:lo + n])
            lo += n
    finally:
        for c in ctxs:
            c.close()


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


@pytest.mark.parametrize("case", ["log31", "from_zero", "negative", "narrow38", "wide3", "bins39", "bins200"])
def test_volume_spectrum_bin_search_variants(dev, case):
    """Both kernels of the product and both bin searches: up to 38 bins take lane-private columns (no atomics) and
    find the bin through a table over the high word of the volume when every edge is positive (bins far narrower
    and far wider than a table cell, values exactly on edges), by binary search otherwise; more bins take the
    atomic kernel.  Ragged odd length."""
    sdm = _sdm()
    rng = np.random.default_rng(7)
    n = 100_003
    v = np.exp(rng.normal(np.log(1e-15), 2.0, n))
    xi = rng.integers(0, 10**9, n).astype(np.int64)
    if case == "log31":
        edges = np.exp(np.linspace(np.log(1e-18), np.log(1e-12), 32))
    elif case == "from_zero":
        edges = np.linspace(0.0, 5e-15, 11)
    elif case == "negative":
        edges = np.linspace(-1e-15, 4e-15, 8)
        v[::7] *= -1.0
    elif case == "narrow38":
        edges = 1e-15 * (1.0 + np.arange(39) * 1e-9)     # 38 bins inside a few low-word steps of one high word
        v[: n // 2] = 1e-15 * (1.0 + rng.random(n // 2) * 39e-9)
    elif case == "wide3":
        edges = np.array([1e-300, 1e-16, 1e-14, 1e300])
    elif case == "bins39":
        edges = np.exp(np.linspace(np.log(1e-18), np.log(1e-12), 40))
    else:
        edges = np.exp(np.linspace(np.log(1e-18), np.log(1e-12), 201))
    v[:edges.size] = edges                                 # values exactly on the edges (the last one is outside)
    with sdm.SDMContext(n, 1, device=dev) as ctx:
        got = [t.cpu().numpy() for t in ctx.volume_spectrum(torch.from_numpy(xi).to(dev), torch.from_numpy(v).to(dev), edges)]
    want = oracle.volume_spectrum(xi, v, edges)
    assert want[0].sum() > 0
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


# ------------------------------------------------------------------------------------------- NEXT-3: efficiency table
def _eff_table():
    rng = np.random.default_rng(12)
    radius = np.exp(np.linspace(np.log(2e-9), np.log(2e-3), 11))
    table = rng.random((11, 6))
    table[:, 0] *= 0.1
    return radius, table


@pytest.mark.parametrize("which", ["random", "constant"])
def test_efficiency_table_kernel_bit_exact(dev, which):
    """SDM_KERNEL_GEOMETRIC_TABLE (R39): K on the device == the oracle's, bit for bit, on volumes that cover the whole
    radius grid, its outside, equal radii (p = 1) and a zero volume; a constant table == the geometric kernel."""
    sdm = _sdm()
    radius, table = _eff_table()
    if which == "constant":
        table = np.full_like(table, 0.625)
    rng = np.random.default_rng(3)
    n = 20_000
    vj = np.exp(rng.uniform(np.log(1e-27), np.log(1e-6), n))
    vk = np.exp(rng.uniform(np.log(1e-27), np.log(1e-6), n))
    vk[:100] = vj[:100]
    vj[100], vk[100] = 0.0, 1e-15
    vj[101:111] = 4.0 / 3.0 * np.pi * radius[:10] ** 3           # on the grid nodes
    okp = oracle.geometric_table(radius, table)
    want = np.array([oracle.kernel(okp, float(a), float(b)) for a, b in zip(vj, vk)])
    with sdm.SDMContext(1024, 1, device=dev) as ctx:
        with pytest.raises(sdm.SDMError):                           # no table installed yet
            ctx.kernel_eval(sdm.geometric_table(), torch.from_numpy(vj).to(dev), torch.from_numpy(vk).to(dev))
        ctx.set_collision_efficiency(radius, table)
        got = ctx.kernel_eval(sdm.geometric_table(), torch.from_numpy(vj).to(dev), torch.from_numpy(vk).to(dev)).cpu().numpy()
        assert np.array_equal(got.view(np.int64), want.view(np.int64))
        if which == "constant":
            geo = ctx.kernel_eval(sdm.geometric(0.625), torch.from_numpy(vj).to(dev), torch.from_numpy(vk).to(dev)).cpu().numpy()
            assert np.array_equal(got.view(np.int64), geo.view(np.int64))
        for bad_r, bad_t in (([1.0, 1.0], [[0, 1], [0, 1]]), ([1.0, 2.0], [[0, -1], [0, 1]]), ([1.0], [[0.0, 1.0]])):
            with pytest.raises(sdm.SDMError):
                ctx.set_collision_efficiency(bad_r, bad_t)
        ctx.set_collision_efficiency(None, None)
        with pytest.raises(sdm.SDMError):
            ctx.coalescence_step(torch.ones(4, dtype=torch.int64, device=dev), torch.ones(4, dtype=torch.float64, device=dev),
                                 torch.zeros(4, dtype=torch.int32, device=dev), 1, 1.0, 1.0, sdm.geometric_table(), 42, 0)


@pytest.mark.parametrize("path", ["general", "cell_sorted", "hybrid"])
@pytest.mark.parametrize("dV", [400.0, 0.04])
def test_efficiency_table_whole_steps(dev, path, dV):
    """whole steps with a tabulated efficiency (entries from 0 to 1: the early-out bounds use the table's maximum),
    p from << 1 to >> 1, debug outputs off, state bit for bit against the oracle"""
    sdm = _sdm()
    radius, table = _eff_table()
    w = W.small("cfg3", interleave=(path == "hybrid"))
    ow = w.copy()
    okp = oracle.geometric_table(radius, table)
    p = {"general": sdm.PATH_GENERAL, "cell_sorted": sdm.PATH_CELL_SORTED, "hybrid": sdm.PATH_HYBRID}[path]
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        ctx.set_path(p)
        ctx.set_collision_efficiency(radius, table)
        xi, v, cell = _to_dev(w, dev)
        for s in range(4):
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, dV, okp, 42, s)
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, dV, sdm.geometric_table(), 42, s)
            assert ctx.poll_error() == 0
            assert np.array_equal(xi.cpu().numpy(), ow.xi), f"step {s}"
            assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v.view(np.int64)), f"step {s}"
    assert not np.array_equal(ow.xi, w.xi)


# ------------------------------------------------------------------------------------------- NEXT-4: displacement
@pytest.mark.parametrize("n_off", [0, 1])
def test_displacement_against_oracle(dev, n_off):
    """sdm_displace / sdm_cell_id_from_positions vs the oracle (O8): positions and cell_id bit for bit over ten steps
    of the paper's single-eddy flow, including positions on cell edges, at the periodic seam, and (n_off = 1) arrays
    that are neither 16-byte aligned nor even in length."""
    sdm = _sdm()
    w = W.small("cfg3")
    nx, nz = 19, 17
    u, wv = W.single_eddy(nx, nz, courant_max=0.9)
    x, z = W.positions_in_cells(w.cell_id, nx, nz)
    x[:40] = np.arange(40) % nx                       # exactly on the edges
    z[40:80] = np.arange(40) % nz
    x[80:90] = np.nextafter(float(nx), 0.0)           # the last representable position before the seam
    x[90:100] = 0.0
    n = w.n_sd - 3 * n_off
    ox, oz = x[:n].copy(), z[:n].copy()
    ocell = oracle.cell_id_from_positions(ox, oz, nx, nz)
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        gx_all, gz_all = torch.from_numpy(x).to(dev), torch.from_numpy(z).to(dev)
        gc_all = torch.zeros(w.n_sd + 1, dtype=torch.int32, device=dev)
        gx, gz, gc = gx_all[n_off:n_off + n], gz_all[n_off:n_off + n], gc_all[n_off:n_off + n]
        ox, oz = x[n_off:n_off + n].copy(), z[n_off:n_off + n].copy()
        ocell = oracle.cell_id_from_positions(ox, oz, nx, nz)
        gu, gw = torch.from_numpy(u).to(dev), torch.from_numpy(wv).to(dev)
        ctx.cell_id_from_positions(gx, gz, nx, nz, cell_id=gc)
        assert np.array_equal(gc.cpu().numpy(), ocell)
        for step in range(10):
            dt = 1.0 if step % 2 == 0 else 0.37
            oracle.displace(ox, oz, ocell, nx, nz, u, wv, dt)
            ctx.displace(gx, gz, gc, nx, nz, gu, gw, dt)
            assert np.array_equal(gx.cpu().numpy().view(np.int64), ox.view(np.int64)), f"x step {step}"
            assert np.array_equal(gz.cpu().numpy().view(np.int64), oz.view(np.int64)), f"z step {step}"
            assert np.array_equal(gc.cpu().numpy(), ocell), f"cell_id step {step}"
        assert ctx.poll_error() == 0
        # the seam: a tiny negative coordinate folds to 0, a step of a whole period lands where it started
        sx = torch.tensor([1e-300, 0.25, nx - 0.25, 0.0], dtype=torch.float64, device=dev)
        sz = torch.tensor([0.5, 0.5, 0.5, 0.5], dtype=torch.float64, device=dev)
        sc = torch.zeros(4, dtype=torch.int32, device=dev)
        su = torch.full((nx * nz,), -2e-300, dtype=torch.float64, device=dev)
        ctx.displace(sx, sz, sc, nx, nz, su, torch.zeros_like(su), 1.0)
        hx, hz, hc = np.array([1e-300, 0.25, nx - 0.25, 0.0]), np.full(4, 0.5), np.zeros(4, np.int32)
        oracle.displace(hx, hz, hc, nx, nz, np.full(nx * nz, -2e-300), np.zeros(nx * nz), 1.0)
        assert sx.cpu().numpy().tolist() == hx.tolist() and hx[0] == 0.0 and hx[3] == 0.0
        assert sc.cpu().numpy().tolist() == hc.tolist()
        with pytest.raises(sdm.SDMError):
            ctx.displace(sx, sz, sc, 0, nz, su, su, 1.0)
        with pytest.raises(sdm.SDMError):
            ctx.displace(sx, sz, sc, nx, nz, su, su, 0.0)


def test_displacement_then_coalescence_time_loop(dev):
    """The 2-D loop the displacement exists for: displace, then one coalescence step on the
    cell_id it produced -- no longer sorted, so AUTO leaves the cell-sorted path -- for six steps against the oracle
    doing the same; state, positions and cell_id bit for bit."""
    sdm = _sdm()
    w = W.small("cfg3")
    ow = w.copy()
    nx, nz = 19, 17
    u, wv = W.single_eddy(nx, nz, courant_max=0.6)
    x, z = W.positions_in_cells(w.cell_id, nx, nz)
    ox, oz = x.copy(), z.copy()
    okp, kp = _okp(w), _gkp(w)
    paths = []
    with sdm.SDMContext(w.n_sd, w.n_cell, device=dev) as ctx:
        xi, v, cell = _to_dev(w, dev)
        gx, gz = torch.from_numpy(x).to(dev), torch.from_numpy(z).to(dev)
        gu, gw = torch.from_numpy(u).to(dev), torch.from_numpy(wv).to(dev)
        for s in range(6):
            oracle.coalescence_step(ow.xi, ow.v, ow.cell_id, w.n_cell, w.dt, w.dV, okp, 42, s)
            ctx.coalescence_step(xi, v, cell, w.n_cell, w.dt, w.dV, kp, 42, s)
            paths.append(ctx.last_path())
            oracle.displace(ox, oz, ow.cell_id, nx, nz, u, wv, w.dt)
            ctx.displace(gx, gz, cell, nx, nz, gu, gw, w.dt)
            assert ctx.poll_error() == 0
            assert np.array_equal(cell.cpu().numpy(), ow.cell_id), f"cell_id step {s}"
            assert np.array_equal(xi.cpu().numpy(), ow.xi), f"step {s}"
            assert np.array_equal(v.cpu().numpy().view(np.int64), ow.v.view(np.int64)), f"step {s}"
    assert paths[0] == sdm.PATH_CELL_SORTED and sdm.PATH_CELL_SORTED not in paths[1:]
    assert sdm.PATH_HYBRID in paths


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
