"""The N > 1 plumbing on CPU (gloo, world_size 2): track slices tile the time frame, the timing reduction is
a max over ranks, counts add up, and the sharded outputs of a strong-scaling run put back together are the
single-rank result (checked with the parity comparator).  The tracking step itself has no collective (DESIGN.md
"Multi-GPU")."""
import os
import socket

import numpy as np

import pytest
import torch
import torch.multiprocessing as mp

from paper_2003_03174_b200 import dist as D, parity as P


def test_track_slices_tile_the_frame():
    for n in (0, 1, 7, 500_000, 2_000_001):
        for world in (1, 2, 3, 8):
            parts = [D.track_slice(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    r, w = D.init("gloo")
    assert (r, w) == (rank, world)
    lo, hi = D.track_slice(1001, r, w)
    D.barrier()
    ms = D.max_over_ranks(10.0 + 5.0 * rank)           # the slower rank defines the step time
    total = D.sum_over_ranks(hi - lo)
    # strong scaling: every rank holds the results of its own slice of ONE frame; together they are the frame's
    full = _fake_result(1001)
    mine = {k: v[..., lo:hi] for k, v in full.items()}
    back = D.gather_sharded(mine, 1001)
    rep = P.compare(back, dict(full, margin=np.full(1001, np.inf)))
    ok = rep["ok"] and rep["n_assign_mismatch"] == 0 and all(np.array_equal(back[k], full[k]) for k in full)
    q.put((rank, ms, total, bool(ok)))
    D.shutdown()


def _fake_result(n):
    """A result-shaped dict from a fixed seed (the comparator holds none of the method's arithmetic)."""
    rng = np.random.default_rng(7)
    return dict(idx=rng.integers(-1, 1000, (6, n)).astype(np.int32), par=rng.normal(size=(5, n)), cov=np.abs(rng.normal(size=(15, n))),
                x=np.full(n, 364.0), sector=rng.integers(0, 18, n).astype(np.int32), chi2=np.abs(rng.normal(size=n)),
                n_matched=rng.integers(0, 7, n).astype(np.int32))


def test_two_ranks_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, 15.0, 1001.0, True), (1, 15.0, 1001.0, True)]
