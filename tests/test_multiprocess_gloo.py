"""N>1 host logic on CPU: world_size-2 gloo processes.

The per-rank compute is stood in for by the oracle (tests may call it); what is under test is the
partitioning and the two collectives the multi-GPU paths use: a scalar SUM for the row-sharded
eval pass and a scalar MAX for the replicas-only training time."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist            # noqa: E402
import torch.multiprocessing as mp          # noqa: E402

from paper_2606_30497_b200 import sharding  # noqa: E402


def test_row_shard_covers_everything_once():
    for n in (0, 1, 127, 128, 129, 1000, 65536, 70001):
        for world in (1, 2, 3, 8):
            edges = [sharding.row_shard(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            for (a, b), (c, d) in zip(edges, edges[1:]):
                assert b == c and a <= b and c <= d
            for lo, hi in edges[:-1]:
                assert hi % 128 == 0 or hi == n


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import mlp_oracle as O
        from paper_2606_30497_b200 import datagen
        X, Y = datagen.make_dataset(n, 0.1)
        W1, W2 = O.init_weights(2, 32, 64)
        lo, hi = sharding.row_shard(n, rank, world)
        local = O.eval_loss(X[lo:hi], Y[lo:hi], W1, W2) if hi > lo else 0.0
        loss = sharding.combine_eval(local, hi - lo)
        slowest = sharding.max_over_ranks(10.0 + rank)
        q.put((rank, loss, slowest, lo, hi))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n", [1000, 4097])
def test_sharded_eval_and_replica_timing_world2(n):
    from oracle import mlp_oracle as O
    from paper_2606_30497_b200 import datagen
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=600) for _ in range(2))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    X, Y = datagen.make_dataset(n, 0.1)
    W1, W2 = O.init_weights(2, 32, 64)
    full = O.eval_loss(X, Y, W1, W2)
    assert res[0][3] == 0 and res[0][4] == res[1][3] and res[1][4] == n
    for _, loss, slowest, _, _ in res:
        assert abs(loss - full) <= 1e-12 * full
        assert slowest == 11.0
