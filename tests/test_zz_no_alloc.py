"""sdm_remove_zero_multiplicity_static -- the entry point that allocates nothing (csrc/sdm_noalloc.cu: scratch in a
fixed device array inside the library) -- against the existing path (sdm_remove_zero_multiplicity through a context
and the caller's workspace) and against the oracle, bit for bit, on two calls in a row.

This file is collected LAST on purpose (pytest -x: a failure here hides nothing behind it) and
passes alone in a fresh process as well as after the other tests."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

import oracle  # noqa: E402

pytestmark = pytest.mark.gpu


def _state(n, zero_frac, seed):
    rng = np.random.default_rng(seed)
    xi = rng.integers(1, 10**9, n).astype(np.int64)
    xi[rng.random(n) < zero_frac] = 0
    v = rng.random(n) * 1e-12
    cell = np.sort(rng.integers(0, max(n // 50, 1), n)).astype(np.int32)
    return xi, v, cell


def _bits(a):
    return a.view(np.int64) if a.dtype == np.float64 else a


def _both(sdm, ctx, dev, xi, v, cell, n_out_dev):
    """The same input through the new entry point and the existing path; returns the two prefixes and the oracle's."""
    a = [torch.from_numpy(t.copy()).to(dev) for t in (xi, v, cell)]
    b = [torch.from_numpy(t.copy()).to(dev) for t in (xi, v, cell)]
    n = xi.shape[0]
    sdm.remove_zero_multiplicity_static(a[0], a[1], a[2], n_out_dev)       # asynchronous: the result stays on the device
    n_new = int(n_out_dev.item())
    n_old = ctx.remove_zero_multiplicity(b[0], b[1], b[2])
    o = [t.copy() for t in (xi, v, cell)]
    n_ora = oracle.remove_zero_multiplicity(o[0], o[1], o[2])
    assert n_new == n_old == n_ora == int((xi != 0).sum())
    for got, ref, want in zip(a, b, o):
        g = _bits(got[:n_new].cpu().numpy())
        assert np.array_equal(g, _bits(ref[:n_new].cpu().numpy()))      # the existing path
        assert np.array_equal(g, _bits(want[:n_new]))                   # the oracle
    return n_new


def test_static_entry_point_matches_existing_path_twice():
    import paper_2103_17238_b200 as sdm

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need one (there is no CPU fallback)")
    dev = torch.device("cuda", 0)
    assert sdm.static_max_n_sd() == 2 ** 26
    n_out_dev = torch.full((1,), -1, dtype=torch.int64, device=dev)
    n1, n2 = 1_000_003, 300_001   # several hundred tiles in several waves, ragged tails; the second call is SMALLER:
    with sdm.SDMContext(n1, n1, device=dev) as ctx:   # it must not see the first call's ticket or tile states
        k1 = _both(sdm, ctx, dev, *_state(n1, 0.30, 1), n_out_dev)
        k2 = _both(sdm, ctx, dev, *_state(n2, 0.02, 2), n_out_dev)
        assert 0 < k1 < n1 and 0 < k2 < n2
        # nothing to remove, everything to remove, a single entry, an empty array
        for n, frac, seed in ((70_001, 0.0, 3), (70_001, 1.0, 4), (1, 0.0, 5), (1, 1.0, 6)):
            _both(sdm, ctx, dev, *_state(n, frac, seed), n_out_dev)
        e = torch.empty(0, dtype=torch.int64, device=dev)
        sdm.remove_zero_multiplicity_static(e, e.double(), e.int(), n_out_dev)
        assert int(n_out_dev.item()) == 0


def test_static_entry_point_rejects_sizes_beyond_its_scratch():
    import paper_2103_17238_b200 as sdm

    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the gpu tests need one (there is no CPU fallback)")
    dev = torch.device("cuda", 0)
    xi = torch.ones(8, dtype=torch.int64, device=dev)
    v = torch.ones(8, dtype=torch.float64, device=dev)
    c = torch.zeros(8, dtype=torch.int32, device=dev)
    out = torch.full((1,), -7, dtype=torch.int64, device=dev)
    with pytest.raises(sdm.SDMError) as err:    # the size is checked before anything is touched
        sdm.remove_zero_multiplicity_static(xi, v, c, out, n_sd=sdm.static_max_n_sd() + 1)
    assert err.value.status == -5 and "2^26" in str(err.value)
    with pytest.raises(sdm.SDMError) as err:
        sdm.remove_zero_multiplicity_static(xi, v, c, out, n_sd=-1)
    assert err.value.status == -1
    torch.cuda.synchronize()
    assert int(out.item()) == -7 and int(xi.sum().item()) == 8
