"""Multi-rank host logic on CPU: world_size 2, gloo.  No transport runs here (that needs the GPU); the ranks
exchange oracle results of the two id-range shares' stand-ins and the reduced tallies must be exact mod 2^64."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2506_00263_b200 import shard


def test_id_ranges_partition_the_source():
    for n in (1, 2, 31, 33, 100000, 10 ** 8 + 7):
        for world in (1, 2, 3, 4, 8):
            nxt = 0
            for r in range(world):
                lo, cnt = shard.id_range(n, r, world)
                assert lo == nxt and cnt >= 0
                nxt = lo + cnt
            assert nxt == n
            sizes = [shard.id_range(n, r, world)[1] for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def _fake_result(rank):
    rng = np.random.default_rng(100 + rank)
    big = np.int64(2 ** 62)                                   # two of these wrap around int64: the sum must stay exact mod 2^64
    return dict(flux=rng.integers(0, 2 ** 40, 23409).astype(np.int64) + big, coll=rng.integers(0, 2 ** 40, 23409).astype(np.int64),
                leak=rng.integers(0, 1000, 6).astype(np.int64),
                totals={"n_seg": int(rng.integers(0, 2 ** 50)), "digest": int(rng.integers(0, 2 ** 63)) * 2 + 1, "n_born": 5 + rank})


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = _fake_result(rank) if rank < 2 else None           # a rank with no share contributes zeros
    out = shard.allreduce_tallies(mine, template=_fake_result(0))
    (mx, sm) = shard.reduce_timing([10.0 + rank], [100.0 * (rank + 1)])
    if rank == 0:
        q.put((out, mx, sm))
    dist.barrier()
    dist.destroy_process_group()


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _run(world):
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = q.get()
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    return out


def test_allreduce_of_tallies_is_exact_world2():
    out, mx, sm = _run(2)
    ref = shard.merge_local([_fake_result(0), _fake_result(1)])
    for k in shard.SUM_KEYS:
        assert np.array_equal(out[k].view(np.uint64), ref[k].view(np.uint64)), k
    assert out["totals"] == ref["totals"]
    assert mx == [11.0] and sm == [300.0]


def test_rank_without_a_share_world3():
    out, mx, sm = _run(3)
    ref = shard.merge_local([_fake_result(0), _fake_result(1)])
    assert out["totals"] == ref["totals"] and np.array_equal(out["flux"], ref["flux"])
    assert mx == [12.0] and sm == [600.0]
