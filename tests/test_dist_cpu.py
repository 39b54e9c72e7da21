"""N > 1 host logic on CPU: world_size-2 gloo run of the sharding and the max-over-ranks timing rule
(units are independent, no data-path collective)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_00760_b200 import shard, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, ret):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = synth.WORKLOADS["tiny"]
        mine = shard.rank_workload(w, rank)
        # every rank draws its own requests; the same rank always draws the same bytes
        K, _, _ = synth.make_inputs_np(1, 1, 1, 64, 128, 64, seed=mine.seed)
        digest = int(K.astype(np.uint64).sum())
        t = 1.0 + rank  # the slower rank decides
        mx = shard.max_over_ranks(t, world)
        thr = shard.job_throughput(10.0 * (rank + 1), t, world)
        owned = list(shard.shard_requests(7, rank, world))
        gathered = [None] * world
        dist.all_gather_object(gathered, (digest, owned, mine.seed))
        ret[rank] = (mx, thr, gathered)
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_sharding_and_timing():
    world, port = 2, _free_port()
    ret = mp.Manager().dict()
    mp.spawn(_worker, args=(world, port, ret), nprocs=world, join=True)
    for rank in range(world):
        mx, thr, gathered = ret[rank]
        assert mx == 2.0                      # max over ranks, identical on every rank
        assert thr == (10.0 + 20.0) / 2.0     # all ranks' units / the max time
        (d0, o0, s0), (d1, o1, s1) = gathered
        assert s0 != s1 and d0 != d1          # distinct requests per rank (weak scaling)
        assert sorted(o0 + o1) == list(range(7)) and not set(o0) & set(o1)  # disjoint cover (strong scaling)


def test_shard_requests_is_a_partition():
    for n in (1, 7, 8, 64):
        for world in (1, 2, 3, 8):
            parts = [list(shard.shard_requests(n, r, world)) for r in range(world)]
            flat = [x for p in parts for x in p]
            assert flat == list(range(n))
            assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


def test_single_rank_needs_no_process_group():
    assert shard.max_over_ranks(3.5, 1) == 3.5
    assert shard.job_throughput(8.0, 2.0, 1) == 4.0
