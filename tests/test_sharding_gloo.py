"""Multi-GPU plan on CPU: world_size-2 `gloo` processes, each stepping its
shard of contiguous cells with the ORACLE (index_base = first array entry of the shard, reading R34), must
reproduce the unsharded oracle step bit for bit, and bench.py's whole-job aggregation (max time over ranks, sum of
units) must come out right.  No data-path collective exists: the only exchanges are the test's own gather and the
timing reduction."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import sdm_workloads as W  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _kp(w):
    return oracle.golovin(w.b) if w.kernel_kind == W.GOLOVIN else oracle.geometric(w.E)


def _worker(rank, world, port, name, n_steps, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        w = W.small(name)
        sh = W.shard(w, rank, world)
        sw = sh.work
        kp = _kp(sw)
        for s in range(n_steps):
            oracle.coalescence_step(sw.xi, sw.v, sw.cell_id, sw.n_cell, sw.dt, sw.dV, kp, sw.seed, s,
                                    index_base=sh.index_base)
        np.savez(os.path.join(out_dir, f"shard{rank}.npz"), xi=sw.xi, v=sw.v, lo=sh.index_base, cells=[sh.cell_lo, sh.cell_hi])
        # the bench's aggregation: max of the per-rank times, sum of the per-rank units
        ms, units = bench.aggregate_over_ranks(10.0 * (rank + 1), float(sw.n_sd * n_steps), dist, torch.device("cpu"))
        if rank == 0:
            np.save(os.path.join(out_dir, "agg.npy"), np.array([ms, units]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("name", ["cfg3", "cfg4s"])
def test_two_rank_shards_reproduce_the_unsharded_step(tmp_path, name):
    world, n_steps = 2, 3
    mp.spawn(_worker, args=(world, _free_port(), name, n_steps, str(tmp_path)), nprocs=world, join=True)
    w = W.small(name)
    kp = _kp(w)
    for s in range(n_steps):
        oracle.coalescence_step(w.xi, w.v, w.cell_id, w.n_cell, w.dt, w.dV, kp, w.seed, s)
    covered = 0
    cells = []
    for r in range(world):
        z = np.load(os.path.join(tmp_path, f"shard{r}.npz"))
        lo, n = int(z["lo"]), len(z["xi"])
        assert lo == covered                              # contiguous, no gaps, no overlap
        assert np.array_equal(z["xi"], w.xi[lo:lo + n])
        assert np.array_equal(z["v"].view(np.int64), w.v[lo:lo + n].view(np.int64))
        covered += n
        cells.append(tuple(int(c) for c in z["cells"]))
    assert covered == w.n_sd
    assert cells[0][0] == 0 and cells[-1][1] == w.n_cell and cells[0][1] == cells[1][0]
    ms, units = np.load(os.path.join(tmp_path, "agg.npy"))
    assert ms == 20.0                                     # max over ranks
    assert units == float(w.n_sd * n_steps)               # sum over ranks = the whole job


def test_shard_refuses_what_does_not_shard():
    with pytest.raises(ValueError):
        W.shard(W.small("cfg0"), 0, 2)                    # single-cell box: replicas only
    with pytest.raises(ValueError):
        W.shard(W.small("cfg3", interleave=True), 0, 2)   # not cell-major
