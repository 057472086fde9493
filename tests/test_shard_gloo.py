"""Host-side logic of the N > 1 path: rows of H sharded over ranks, no data-path
collective.  Runs on CPU with the gloo backend, world_size 2 (and 3 for the ragged split).  The
per-rank "evaluation" is a stand-in that returns each row's index-dependent value: what is under
test is the slicing, the optional gather and the max-over-ranks timing rule, not the arithmetic
(that is the GPU parity suite)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2603_06010_b200 import shard


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_row_slices_partition_the_batch():
    for B in (0, 1, 2, 5, 64, 4096, 8191):
        for world in (1, 2, 3, 8):
            sl = shard.all_slices(B, world)
            assert sl[0][0] == 0 and sl[-1][1] == B
            assert all(sl[i][1] == sl[i + 1][0] for i in range(world - 1))
            sizes = [h - l for l, h in sl]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.row_slice(4, 2, 2)
    with pytest.raises(ValueError):
        shard.row_slice(-1, 0, 1)


def _worker(rank: int, world: int, port: int, B: int, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        H = torch.arange(B * 4, dtype=torch.float64).reshape(B, 4)  # same on every rank (replicated inputs)
        lo, hi = shard.row_slice(B, rank, world)
        out_local = -0.5 * (H[lo:hi] ** 2).sum(dim=1)               # stand-in for the rank's td_loglike_batch
        full = shard.gather_out(out_local, B)
        t = shard.max_over_ranks(10.0 + rank)
        q.put((rank, lo, hi, full.numpy().copy(), t))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,B", [(2, 64), (2, 7), (3, 8), (2, 1)])
def test_sharded_batch_gathers_to_the_unsharded_result(world, B):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, B, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = [q.get(timeout=120) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    H = np.arange(B * 4, dtype=np.float64).reshape(B, 4)
    want = -0.5 * (H ** 2).sum(axis=1)
    covered = np.zeros(B, dtype=int)
    for rank, lo, hi, full, t in got:
        assert np.array_equal(full, want)          # every rank sees the whole vector, bit for bit
        assert t == 10.0 + world - 1               # max over ranks
        covered[lo:hi] += 1
    assert np.all(covered == 1)                    # each row evaluated by exactly one rank
