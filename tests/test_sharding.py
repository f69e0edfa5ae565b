"""Multi-process (gloo, world_size 2, CPU) tests of the sharding plumbing: patch partition, max-over-ranks timing
reduction, toplist gather on rank 0 and the block-toplist merge.  No GPU, no oracle."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1904_04873_b200 import sharding  # noqa: E402
from paper_1904_04873_b200.binding import CAND_DTYPE  # noqa: E402


def test_partition_covers_every_patch_once():
    for n, w in [(256, 1), (256, 2), (256, 8), (10, 4), (3, 8), (0, 2)]:
        seen = []
        for r in range(w):
            part = sharding.patches_of_rank(n, r, w)
            assert all(p % w == r for p in part)
            seen += part
        assert sorted(seen) == list(range(n))
    sizes = [len(sharding.patches_of_rank(256, r, 8)) for r in range(8)]
    assert max(sizes) - min(sizes) == 0
    with pytest.raises(ValueError):
        sharding.patches_of_rank(4, 2, 2)


def test_single_process_paths_are_identities():
    assert sharding.max_over_ranks(3.5) == 3.5
    assert sharding.sum_over_ranks(2.0) == 2.0
    recs = np.zeros(3, dtype=CAND_DTYPE)
    assert sharding.gather_toplists({4: recs})[4] is recs


def _records(indices, counts):
    r = np.zeros(len(indices), dtype=CAND_DTYPE)
    r["index"] = indices
    r["count"] = counts
    return r


def test_merge_block_toplists_orders_by_value_then_index():
    a = _records([5, 9, 40], [30, 30, 12])
    b = _records([7, 2, 41], [30, 29, 12])
    top = sharding.merge_block_toplists([a, b], k=5)
    assert top["index"].tolist() == [5, 7, 9, 2, 40]
    assert top["count"].tolist() == [30, 30, 30, 29, 12]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = sharding.patches_of_rank(7, rank, world)
        local = {p: _records([100 * p + 1, 100 * p], [50 - p, 50 - p]) for p in mine}
        ms = sharding.max_over_ranks(10.0 + rank, dist)
        total = sharding.sum_over_ranks(float(len(mine)), dist)
        got = sharding.gather_toplists(local, dist, dst=0)
        q.put((rank, ms, total, None if got is None else {k: v["index"].tolist() for k, v in got.items()}))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_reduction_and_gather():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = {}
    for _ in procs:
        rank, ms, total, got = q.get(timeout=120)
        out[rank] = (ms, total, got)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out[0][0] == 11.0 and out[1][0] == 11.0          # max over ranks on every rank
    assert out[0][1] == 7.0 and out[1][1] == 7.0            # all 7 patches were owned by somebody
    assert out[1][2] is None                                # only rank 0 receives the toplists
    assert sorted(out[0][2].keys()) == list(range(7))
    assert out[0][2][3] == [301, 300]
