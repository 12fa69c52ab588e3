"""Multi-GPU plumbing (one process per GPU, torch.distributed): histories are independent given the
(id, generation, segment)-keyed RNG, so a fixed source shards by contiguous id ranges with NO collective on the
data path; the only exchange is one int64 all-reduce of the tallies at the end (PAPER.md:13, 17 use MPI
replication for the same purpose).  Integer fixed-point tallies make the reduced result bit-identical for any
number of ranks.  No transport arithmetic lives here."""
from __future__ import annotations

import numpy as np

SUM_KEYS = ("flux", "coll", "leak")


def id_range(n: int, rank: int, world: int):
    """Contiguous share [lo, lo + count) of source ids 0..n-1 for this rank (sizes differ by at most one)."""
    base, rem = divmod(n, world)
    return rank * base + min(rank, rem), base + (1 if rank < rem else 0)


def run_fixed_source_sharded(problem, n, seed, rank, world, device, **options):
    """This rank's share of a fixed-source run: ids lo..lo+count-1 on `device`.  Returns read_tallies() (local)."""
    from . import tdr
    lo, count = id_range(n, rank, world)
    if count == 0:
        return None
    P = tdr.Problem(problem, device=device, id_offset=lo, **options)
    try:
        P.run_fixed_source(count, seed)
        return P.read_tallies(history=False, bank=False)
    finally:
        P.close()


def merge_local(results):
    """Sum of per-shard results on one process (what the all-reduce computes across processes)."""
    results = [r for r in results if r is not None]
    out = {k: np.sum([r[k] for r in results], axis=0, dtype=np.int64) for k in SUM_KEYS}
    out["totals"] = {k: sum(r["totals"][k] for r in results) & 0xFFFFFFFFFFFFFFFF for k in results[0]["totals"]}
    return out


def allreduce_tallies(res, template=None, group=None):
    """Sum int64 tallies, leak and totals over all ranks (two's complement wrap-around = exact mod 2^64).
    `res` may be None on a rank that had no share; `template` then gives the array sizes."""
    import torch
    import torch.distributed as dist
    src = res if res is not None else template
    names = sorted(src["totals"])
    parts = [np.asarray(src[k], dtype=np.int64).ravel() for k in SUM_KEYS]
    parts.append(np.array([src["totals"][k] for k in names], dtype=np.uint64).view(np.int64))
    flat = np.concatenate(parts)
    if res is None:
        flat = np.zeros_like(flat)
    t = torch.from_numpy(flat.copy())
    if dist.get_backend(group) == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    flat = t.cpu().numpy()
    out, o = {}, 0
    for k in SUM_KEYS:
        m = np.asarray(src[k]).size
        out[k] = flat[o:o + m].reshape(np.asarray(src[k]).shape).copy(); o += m
    tot = flat[o:o + len(names)].view(np.uint64)
    out["totals"] = {k: int(v) for k, v in zip(names, tot)}
    return out


def reduce_timing(values_max, values_sum, device=None, group=None):
    """bench.py: max over ranks of the timings, sum over ranks of the work counts."""
    import torch
    import torch.distributed as dist
    mx = torch.tensor(values_max, dtype=torch.float64, device=device)
    sm = torch.tensor(values_sum, dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(mx, op=dist.ReduceOp.MAX, group=group)
        dist.all_reduce(sm, op=dist.ReduceOp.SUM, group=group)
    return mx.tolist(), sm.tolist()
