"""N > 1 plumbing on CPU: two gloo ranks (no GPU).  The path has no data-path collective (envs are
independent); what is covered is the env partition and the benchmark's reductions."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_08098_b200 import sharding


@pytest.mark.parametrize("world,E", [(1, 7), (2, 256), (3, 16), (4, 5), (8, 3), (8, 1024)])
def test_env_blocks_partition_the_batch(world, E):
    blocks = [sharding.env_block(r, world, E) for r in range(world)]
    assert blocks[0][0] == 0 and blocks[-1][1] == E
    for (a0, a1), (b0, b1) in zip(blocks, blocks[1:]):
        assert a1 == b0 and a0 <= a1
    sizes = [b - a for a, b in blocks]
    assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)


def test_env_block_rejects_bad_rank():
    with pytest.raises(ValueError):
        sharding.env_block(2, 2, 8)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        e0, e1 = sharding.env_block(rank, world, 5)
        ms = 10.0 + 3.0 * rank                       # rank 1 is the slow one
        mx, sm = sharding.reduce_max_sum([ms], [float(e1 - e0), 100.0 * (rank + 1)], torch.device("cpu"))
        # strong scaling: the rank renders ITS envs of the one shared batch; the slices tile the whole keyframe
        from paper_2607_08098_b200 import scenes
        import hashlib
        spec = scenes.small(scenes.config(4), num_envs=5, height=24, width=32, num_keyframes=2)
        sc = scenes.make_scene(spec)
        mine = scenes.render_keyframe(sc, 1, envs=list(range(e0, e1)))
        whole = scenes.render_keyframe(sc, 1)
        same = all(torch.equal(mine[k], whole[k][e0:e1]) for k in mine)
        counts = sharding.gather_counts(1000 * (rank + 1) + (e1 - e0), torch.device("cpu"))
        out[rank] = (mx, sm, sharding.rank_seed(42, rank), same, counts, (e0, e1))
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reduce_max_time_and_sum_counters():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.get_context("spawn").Manager()        # not fork(): the test process is multi-threaded
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0][:2] == out[1][:2]
    mx, sm = out[0][:2]
    assert mx == [13.0] and sm == [5.0, 300.0]       # max time; all 5 envs accounted for; counters summed
    assert out[0][2] != out[1][2]                     # different batches per rank (weak scaling)
    # strong scaling (ShardedEvis): the ranks' renders are the slices of the one batch; the count all-gather (the only
    # collective of the sharded path) returns every rank's count to every rank, in rank order
    assert out[0][3] and out[1][3]
    assert out[0][4] == out[1][4] == [1003, 2002]
    assert out[0][5] == (0, 3) and out[1][5] == (3, 5)


def test_single_process_reduction_is_identity():
    assert sharding.reduce_max_sum([1.5], [2.0, 3.0], torch.device("cpu")) == ([1.5], [2.0, 3.0])
