"""World-size-2 gloo test of the multi-GPU plumbing: round-robin particle shards,
no data-path collective, max-over-ranks timing, summed attempt counters, gather to rank 0.  The traced
"kernel" here is the CPU oracle standing in for a rank's GPU, so the test also shows that sharding does not
change any particle's result."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_indices_partition():
    from paper_2605_16734_b200 import ensemble as E
    for n in (0, 1, 7, 100):
        for world in (1, 2, 3, 8):
            parts = [E.shard_indices(n, r, world) for r in range(world)]
            assert sorted(np.concatenate(parts).tolist()) == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
            vals = [np.stack([p * 2.0, p * 3.0]) for p in parts]
            full = E.unshard(vals, n)
            assert np.array_equal(full[0], np.arange(n) * 2.0) and np.array_equal(full[1], np.arange(n) * 3.0)
    with pytest.raises(ValueError):
        E.shard_indices(4, 2, 2)


def test_loss_fraction_curve():
    from paper_2605_16734_b200 import ensemble as E
    t = np.array([1.0, 0.2, 0.5, 1.0])
    st = np.array([0, 1, 1, 0])
    f = E.loss_fraction_curve(t, st, np.array([0.1, 0.2, 0.6, 1.0]))
    assert np.allclose(f, [0.0, 0.25, 0.5, 0.5])


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ["OMP_NUM_THREADS"] = "2"
    import torch.distributed as dist
    import oracle
    from paper_2605_16734_b200 import ensemble as E, workloads as W
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    fld, spec = W.make_field(0), W.make_spec(0)
    P = W.make_particles(0, 20)
    OF = oracle.OracleField(fld)
    mu = W.mu_from(P, OF.eval_B_many(P.s, P.theta, P.zeta)[:, 0])
    idx = E.shard_indices(P.n, rank, world)
    r = OF.trace(spec, P.s[idx], P.theta[idx], P.zeta[idx], P.vpar[idx], mu[idx], t_max=2e-6)
    attempts = int(r.n_acc.sum() + r.n_rej.sum())
    ms, total = E.reduce_timing(10.0 * (rank + 1), attempts)
    y = E.gather_to_rank0(r.y, P.n)
    if rank == 0:
        full = OF.trace(spec, P.s, P.theta, P.zeta, P.vpar, mu, t_max=2e-6)
        q.put((ms, total, int(full.n_acc.sum() + full.n_rej.sum()), bool(np.array_equal(y, full.y))))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shard_reduce_gather():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    ms, total, expect, same = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 20.0                  # max over ranks
    assert total == expect             # summed attempts equal the unsharded run's
    assert same                        # gathered shards reproduce the unsharded result bit for bit
