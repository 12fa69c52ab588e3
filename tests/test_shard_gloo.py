"""Multi-rank host logic on CPU: world_size 2 and 3, gloo.  The transport itself is done by the ORACLE here (the CUDA
library needs a GPU), through the same four-call stepping interface the library offers, so what is tested is the
exchange protocol of paper_2506_00263_b200.shard: id ranges, the per-generation 32-byte all-reduce, local population
control with the global ratio, the final int64 all-reduce of the tallies — against the oracle's un-sharded run."""
import os
import socket

import numpy as np
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2506_00263_b200 import shard
from paper_2506_00263_b200 import workloads as W


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


def _k_problem():
    return W.cfg1(n=6001, n_inactive=2, n_active=3)


def _fixed_problem():
    return W.cfg3(n=1501, n_ebins=100, n_grid=4000)


def _worker(rank, world, port, q):
    from oracle import orc
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    orc.lib().orc_set_threads(2)
    # one k-eigenvalue problem over `world` ranks
    p = _k_problem()
    eng = orc.Oracle(p)
    res = shard.run_k_eigenvalue_sharded(eng, p.n_particles, p.n_inactive, p.n_active, p.seed, rank, world)
    red = shard.allreduce_tallies(res)
    banks = [None] * world
    dist.all_gather_object(banks, res["bank"])
    eng.close()
    # one fixed source over `world` ranks; the last rank of a 3-rank world gets no share when n < world (not here) -> also test None
    pf = _fixed_problem()
    lo, cnt = shard.id_range(pf.n_particles, rank, world)
    engf = orc.Oracle(pf)
    part = engf.run_fixed_source_range(lo, cnt, pf.seed) if cnt else None
    redf = shard.allreduce_tallies(part, template=part)
    engf.close()
    (mx, sm) = shard.reduce_timing([10.0 + rank], [100.0 * (rank + 1)])
    if rank == 0:
        q.put((dict(res, **red), np.concatenate(banks), redf, mx, sm))
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
        p.join(120)
        assert p.exitcode == 0
    return out


def _check(world):
    from oracle import orc
    k, bank, f, mx, sm = _run(world)
    ref = orc.run(_k_problem())
    for key in ("flux", "coll", "leak", "gen_n", "gen_m", "gen_p", "gen_pc"):
        assert np.array_equal(np.asarray(k[key]).astype(np.int64), np.asarray(ref[key]).astype(np.int64)), key
    assert k["totals"] == ref["totals"]
    assert np.array_equal(k["gen_k"], ref["gen_k"]) and k["k_mean"] == ref["k_mean"] and k["k_std"] == ref["k_std"]
    assert np.array_equal(np.sort(bank.view(np.dtype((np.void, 48)))), np.sort(ref["bank"].view(np.dtype((np.void, 48)))))
    reff = orc.run(_fixed_problem())
    for key in ("flux", "coll", "leak"):
        assert np.array_equal(f[key], reff[key]), key
    assert f["totals"] == reff["totals"]
    assert mx == [10.0 + world - 1] and sm == [100.0 * world * (world + 1) / 2]


def test_sharded_runs_equal_the_unsharded_oracle_world2():
    _check(2)


def test_sharded_runs_equal_the_unsharded_oracle_world3():
    _check(3)


def test_shares_in_turn_on_one_process_equal_the_unsharded_oracle():
    """The same driver with every share in one process (how a single GPU emulates several): no collective at all."""
    from oracle import orc
    p = _k_problem()
    engines = [orc.Oracle(p) for _ in range(3)]
    parts = shard.run_k_eigenvalue_shares(engines, [(r, 3) for r in range(3)], p.n_particles, p.n_inactive, p.n_active, p.seed)
    for e in engines:
        e.close()
    ref = orc.run(p)
    m = shard.merge_local(parts)
    for key in ("flux", "coll", "leak"):
        assert np.array_equal(m[key], ref[key]), key
    assert m["totals"] == ref["totals"]
    assert np.array_equal(parts[0]["gen_k"], ref["gen_k"]) and np.array_equal(parts[1]["gen_p"], ref["gen_p"])
    bank = np.concatenate([x["bank"] for x in parts])
    assert np.array_equal(np.sort(bank.view(np.dtype((np.void, 48)))), np.sort(ref["bank"].view(np.dtype((np.void, 48)))))
