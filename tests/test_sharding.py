"""N>1 host logic on CPU with gloo, world_size 2: event sharding by global index and the
good-helicity mask agreement are the only multi-rank pieces of the path."""
import os

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2507_21039_b200 import sharding


def test_shard_ranges_cover_every_event_once():
    for total in (0, 1, 31, 32, 33, 1000, 65536, 524288 + 17):
        for world in (1, 2, 3, 8):
            seen = np.zeros(total, dtype=np.int32)
            prev_end = 0
            for r in range(world):
                first, n = sharding.shard_range(total, r, world)
                assert first == prev_end
                assert first % 32 == 0 or n == 0
                seen[first:first + n] += 1
                prev_end = first + n
            assert prev_end == total and np.all(seen == 1)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # each rank saw different good helicities on its shard; the agreed mask is their union
    mask = torch.zeros(16, dtype=torch.uint8)
    mask[[5, 6] if rank == 0 else [9, 10, 6]] = 1
    merged = sharding.merge_good_masks(mask)
    tmax = sharding.max_over_ranks(1.0 + rank)
    # sharded oracle evaluation reproduces the single-shard result (global Philox addressing)
    from oracle import binding as O
    total = 96
    first, n = sharding.shard_range(total, rank, world)
    p, w = O.rambo(2, first, n, (173.0, 173.0), 1500.0)
    q.put((rank, merged.tolist(), tmax, first, p.tolist()))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    expect = [0] * 16
    for k in (5, 6, 9, 10):
        expect[k] = 1
    assert res[0][1] == expect and res[1][1] == expect
    assert res[0][2] == 2.0 and res[1][2] == 2.0
    from oracle import binding as O
    full, _ = O.rambo(2, 0, 96, (173.0, 173.0), 1500.0)
    got = np.concatenate([np.array(res[0][4]), np.array(res[1][4])])
    assert res[0][3] == 0 and res[1][3] == 64          # 3 pages of 32 events: rank 0 takes two, rank 1 one
    assert np.array_equal(got, full)
