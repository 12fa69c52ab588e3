"""Multi-GPU plumbing (one process per GPU, torch.distributed).  Histories are independent given the (id, generation,
segment)-keyed RNG, so the path shards by contiguous id ranges (the paper's counterpart is MPI replication over
four V100s):

  * fixed source: each rank runs ids [lo, lo + count); NO collective on the data path; one int64 all-reduce of the tallies
    at the end;
  * k-eigenvalue: each rank holds a contiguous share of the source.  Per generation ONE exchange step — an all-reduce of
    four int64 (P, Pc, N_g, M_g: 32 bytes) — after which every rank forms the same k_g = P 2^-S / N_g and the same
    population-control ratio p = N / M_g and controls its OWN bank with it (sites never move); one int64 all-reduce of
    the tallies at the end.

Integer fixed-point sums make every result bit-identical for any number of ranks.  No transport arithmetic lives here:
the `engine` (a tdr.Problem; in the CPU tests the oracle's stand-in with the same four calls) does all of it."""
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


def run_k_eigenvalue_shares(engines, shares, n, n_inactive, n_active, seed, allreduce4=None, read=True):
    """ONE k-eigenvalue problem of n particles per generation (D2 in steps, include/tdr.h).  `engines` are the shares this
    process drives — one per process under torch.distributed, or several in turn on one GPU — and `shares` their
    (rank, world) pairs.  An engine offers k_begin / k_generation / k_population_control / k_end / scale / read_tallies
    (a tdr.Problem; in the CPU tests the oracle's stand-in).  `allreduce4(list of 4 ints) -> list` adds over the OTHER
    processes (None: this process holds every share).  Returns one read_tallies() per engine: per-generation arrays and k
    are global, tallies and bank are the share's."""
    n_gen = n_inactive + n_active
    for e, (rank, world) in zip(engines, shares):
        lo, count = id_range(n, rank, world)
        e.k_begin(lo, count, n_gen, seed)
    scale = engines[0].scale()
    gen_n, gen_m, gen_p, gen_pc, gen_k = [], [], [], [], []
    k_prev = 1.0
    for g in range(n_gen):
        last = g + 1 == n_gen
        sums = [0, 0, 0, 0]
        for e in engines:
            sums = [a + b for a, b in zip(sums, e.k_generation(g, g >= n_inactive, k_prev, last))]
        if allreduce4 is not None:
            sums = allreduce4(sums)                                   # the generation's ONE exchange step: 32 bytes
        P, Pc, N, M = sums
        if N == 0:
            raise RuntimeError("population died out")
        k = (float(P) * (1.0 / scale)) / float(N)                     # D2: identical on every rank
        gen_n.append(N); gen_m.append(M); gen_p.append(P); gen_pc.append(Pc); gen_k.append(k)
        if M == 0:
            raise RuntimeError(f"fission bank empty in generation {g}")
        if last:
            break
        for e in engines:
            e.k_population_control(g + 1, float(n) / float(M))         # the local bank, the global ratio
        k_prev = k
    out = []
    for e in engines:
        e.k_end(n_inactive, gen_n, gen_m, gen_p, gen_pc, gen_k)
        out.append(e.read_tallies(history=False, bank=True) if read else None)
    return out


def run_k_eigenvalue_sharded(engine, n, n_inactive, n_active, seed, rank, world, read=True):
    """This rank's share of one k-eigenvalue problem under torch.distributed (one process per GPU)."""
    return run_k_eigenvalue_shares([engine], [(rank, world)], n, n_inactive, n_active, seed,
                                   allreduce4=allreduce_int64 if world > 1 else None, read=read)[0]


def allreduce_int64(vals, group=None):
    """Sum a short list of Python ints over all ranks as int64 (exact)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([int(v) for v in vals], dtype=torch.int64)
    if dist.get_backend(group) == "nccl":
        t = t.cuda()
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return [int(v) for v in t.cpu().tolist()]


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
