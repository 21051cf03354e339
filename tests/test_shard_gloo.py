"""World-size-2 CPU test (gloo) of the N>1 path: sharding by stream index needs no exchange.

Each rank derives its shard with the arithmetic bench.py / the package use, produces its columns
(the CPU oracle stands in for the GPU kernels here -- this is a test), and the gathered columns must
equal the single-process family: stream s is a function of (seed, s, block_len) only.
Also covers the max-over-ranks timing reduction.
"""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

import oracle  # noqa: E402
from paper_1307_5869_b200 import sharding  # noqa: E402

CASES = [("lfsr113", 12345, 2**40, 10), ("mrg32k3a", 12345, 2**76, 7), ("gm29", 1, 2**26, 5)]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, total_streams, rows, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ok = True
        for gen, seed, L, per_rank in CASES:
            # strong split of one family
            first, ns = sharding.shard_streams(total_streams, rank, world)
            mine, _ = oracle.streams(gen, seed, first, ns, L, rows, "u32")
            parts = [None] * world
            dist.all_gather_object(parts, (first, mine))
            parts.sort(key=lambda p: p[0])
            full = np.concatenate([p[1] for p in parts], axis=1)
            want, _ = oracle.streams(gen, seed, 0, total_streams, L, rows, "u32")
            ok &= np.array_equal(full, want)
            # weak split (bench.py --gpus N): rank r holds streams [r*per_rank, (r+1)*per_rank)
            first, ns = sharding.weak_shard(per_rank, rank)
            mine, _ = oracle.streams(gen, seed, first, ns, L, rows, "u32")
            want, _ = oracle.streams(gen, seed, 0, world * per_rank, L, rows, "u32")
            ok &= np.array_equal(mine, want[:, first:first + ns])
        slow = sharding.max_over_ranks(10.0 + rank)          # rank 1 is the slow one
        ok &= slow == 10.0 + (world - 1)
        dist.barrier()
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_cover_the_family_without_exchange():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, 13, 9, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = dict(q.get(timeout=10) for _ in range(2))
    assert got == {0: True, 1: True}


def test_shard_arithmetic():
    for total in (0, 1, 2, 7, 1024, 2**20 + 3):
        for world in (1, 2, 3, 8):
            spans = [sharding.shard_streams(total, r, world) for r in range(world)]
            assert spans[0][0] == 0 and sum(n for _, n in spans) == total
            for (f0, n0), (f1, _) in zip(spans, spans[1:]):
                assert f0 + n0 == f1
            assert max(n for _, n in spans) - min(n for _, n in spans) <= 1
    assert sharding.weak_shard(65536, 3) == (196608, 65536)
    assert sharding.max_over_ranks(3.5) == 3.5
