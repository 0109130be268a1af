"""Host logic of the N > 1 path (batch sharding + the one all-gather), world_size 2, gloo, CPU.
The per-rank evaluation is a stand-in (no likelihood arithmetic on the CPU exists in the product)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1505_07674_b200.shard import loglike_sharded, shard_range


def test_shard_range_partitions_the_batch():
    for B in (0, 1, 2, 5, 16, 1023, 16384):
        for world in (1, 2, 3, 8):
            spans = [shard_range(B, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == B
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def _worker(rank, world, port, B, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    params = torch.arange(B * 3, dtype=torch.float32).reshape(B, 3)
    calls = []

    def evaluate(p):
        calls.append(p.shape[0])
        return -0.5 * (p * p).sum(dim=1)

    out = loglike_sharded(evaluate, params)
    q.put((rank, out.numpy(), calls))
    dist.destroy_process_group()


@pytest.mark.parametrize("B", [7, 8, 1])
def test_two_ranks_gather_the_whole_batch_in_order(B):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, B, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(60)
    want = -0.5 * (np.arange(B * 3, dtype=np.float32).reshape(B, 3) ** 2).sum(axis=1)
    for rank, out, calls in got:
        assert np.array_equal(out, want)
        lo, hi = shard_range(B, rank, 2)
        assert calls == ([hi - lo] if hi > lo else [])
