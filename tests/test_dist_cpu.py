"""World-size-2 gloo test (CPU) of the slice-parallel plumbing used by bench.py --gpus N:
disjoint balanced slice shards, barrier, max/sum over ranks.  No data-path collective exists
(replicas only), so this is all the multi-GPU host logic there is."""
import os
import socket

import torch
import torch.multiprocessing as mp

from paper_1009_1380_b200 import dist as rdist


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_slices, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, lr, w = rdist.init("gloo")
    assert (r, w) == (rank, world)
    mine = list(rdist.shard_slices(n_slices, r, w))
    rdist.barrier()
    t_max = rdist.max_over_ranks(10.0 + rank)           # device time: max over ranks
    total = rdist.sum_over_ranks(float(len(mine)))
    out[rank] = (mine, t_max, total)
    torch.distributed.destroy_process_group()


def test_two_rank_slice_sharding_and_reductions():
    world, n_slices = 2, 33
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, _free_port(), n_slices, out), nprocs=world, join=True)
        got = dict(out)
    a, b = got[0][0], got[1][0]
    assert sorted(a + b) == list(range(n_slices)) and not set(a) & set(b)
    assert abs(len(a) - len(b)) <= 1
    assert got[0][1] == got[1][1] == 11.0
    assert got[0][2] == got[1][2] == float(n_slices)


def test_shard_edge_cases():
    assert list(rdist.shard_slices(0, 0, 4)) == []
    assert [len(rdist.shard_slices(5, r, 8)) for r in range(8)] == [1, 1, 1, 1, 1, 0, 0, 0]
    assert list(rdist.shard_slices(32, 3, 4)) == list(range(24, 32))
