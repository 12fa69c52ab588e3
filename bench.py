#!/usr/bin/env python
"""bench.py — particle-events/s (transport segments/s) and histories/s of the TDR transport hot path on B200.

Headline (N = 1): BASELINE.json configs[4] in full — the continuous-energy pin cell in k-eigenvalue mode at 1e8 particles per
generation, 1 inactive + 2 active generations (reading Q19) — the largest single-GPU workload.  A "step" is one
tdr_run_k_eigenvalue call: source, XS lookup, move, tally, collide / surface, remap, fission bank, population control and the
k update of every generation.  `value` is timed with the problem resident on the device; `e2e` goes through the C ABI from
HOST buffers (tdr_init_problem uploads the tables, tdr_read_tallies downloads the results) inside the timed region.
`workloads` carries all five configs x both remapping schemes (x the task decompositions on cfg4), each with segments/s,
histories/s, roofline and e2e, measured with fewer repetitions (stated per entry).
Multi-GPU (`--gpus N` under torchrun): ONE problem shared by the ranks (contiguous shares of the source, one 32-byte
all-reduce per generation, paper_2506_00263_b200.shard) -> "strong" scaling.
`--impl reference` times the CPU oracle on a bounded sample of the same workload.
`--workload cfgN --scheme S --decomposition D --stash T` times a single variant (the command the ncu profiles use)."""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "particle_events_per_sec"
UNIT = "segments/s"
# algorithmic bytes: state read + written + index traffic per transport segment under
# whole-population residency, plus the bank record written at fission and read at birth per history
BYTES_PER_SEGMENT = {"mg": 150.0, "ce": 160.0, "split": 380.0}
BYTES_PER_HISTORY = 96.0
ISSUE_PEAK = 148 * 4 * 32 * 1.965e9            # thread-instructions/s: 148 SM x 4 schedulers x 32 lanes x 1.965 GHz

# full sizes of BASELINE.json configs[0..4]
FULL = {
    "cfg0": dict(desc="cfg0: 1-group fixed source, infinite medium, 1e5 histories", kw={}, ce=False),
    "cfg1": dict(desc="cfg1: 7-group k-eigenvalue pin cell, 1e6 particles/gen, 20 inactive + 50 active generations", kw={}, ce=False),
    "cfg2": dict(desc="cfg2: 7-group k-eigenvalue 3-D 2x2 assemblies (C5G7 shape), 1e7 particles/gen, 6 + 18 generations, 51x51x9 mesh tally", kw={}, ce=False),
    "cfg3": dict(desc="cfg3: continuous-energy pin cell, fixed 14 MeV source, 1e7 histories, 100 energy bins", kw=dict(n=10000000, n_ebins=100), ce=True),
    "cfg4": dict(desc="cfg4: continuous-energy pin cell, k-eigenvalue, 1e8 particles/gen, 1 inactive + 2 active generations, 100 energy bins", kw={}, ce=True),
}
HEADLINE = "cfg4"
# (scheme, decomposition, stash) timed per workload; the first one of HEADLINE's list is the headline (the fastest on cfg4, profiles/throughput_r02.md)
VARIANTS = {
    "cfg0": [("stack", "fused", None), ("async", "fused", "index"), ("async", "hybrid", "shared")],
    "cfg1": [("stack", "fused", None), ("stack", "split", None), ("async", "fused", "index"), ("async", "hybrid", "shared"), ("async", "fused", "particle")],
    "cfg2": [("stack", "fused", None), ("async", "fused", "index"), ("async", "hybrid", "shared")],
    "cfg3": [("stack", "fused", None), ("async", "fused", "index"), ("async", "fused", "particle"), ("async", "hybrid", "shared")],
    "cfg4": [("stack", "fused", None), ("async", "fused", "index"), ("async", "hybrid", "shared"), ("async", "split", "index"), ("stack", "split", None)],
}


def vkey(v):
    return "/".join(x for x in v if x)


def peaks():
    try:
        d = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def profile_metrics():
    """Per-kernel numbers taken from the committed ncu captures (profiles/ncu_r02_kernel_metrics.csv): DRAM bytes and
    thread-instructions per transport segment for each (workload, variant).  Missing rows give null fields."""
    out = {}
    path = os.path.join(ROOT, "profiles", "ncu_r02_kernel_metrics.csv")
    if os.path.exists(path):
        for r in csv.DictReader(l for l in open(path) if not l.startswith("#")):
            out[(r["workload"], r["variant"])] = r
    return out


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(index)],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        mhz, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                mhz.append(float(r[0])); mx = float(r[1])
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        mhz.sort()
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": mx, "reasons": sorted(reasons), "samples": len(mhz)}


def input_bytes(problem):
    import numpy as np
    n = 0
    for d in (problem.geometry, problem.materials, problem.xs or {}):
        for v in d.values():
            n += v.nbytes if isinstance(v, np.ndarray) else 8
    return n


def output_bytes(res):
    import numpy as np
    return sum(v.nbytes for v in res.values() if isinstance(v, np.ndarray)) + 12 * 8 + 16


def make_problem(name, scale=1.0):
    from paper_2506_00263_b200 import workloads as W
    p = W.BY_NAME[name](**FULL[name]["kw"])
    if scale != 1.0:
        p.n_particles = max(1, int(p.n_particles * scale))
    return p


def histories_of(problem, res):
    return int(res["gen_n"].sum()) if problem.mode == "k" else int(res["totals"]["n_born"])


# ---------------------------------------------------------------------------------------------------- the oracle legs
def oracle_sample(name):
    """A bounded sample of the workload for the CPU oracle (about 10-20 s on the box's cores)."""
    from paper_2506_00263_b200 import workloads as W
    if name == "cfg4":
        return W.cfg4(n=1000000, n_inactive=1, n_active=2), "cfg4's problem at 1e6 particles/gen (1/100 of the workload's 1e8), 1 + 2 generations"
    if name == "cfg1":
        return W.cfg1(n=1000000, n_inactive=5, n_active=10), "cfg1 at 1e6 particles/gen, 5 + 10 of the 70 generations"
    if name == "cfg2":
        return W.cfg2(n=1000000, n_inactive=1, n_active=2), "cfg2 at 1e6 particles/gen, 1 + 2 generations"
    if name == "cfg3":
        return W.cfg3(n=1000000, n_ebins=100), "cfg3 at 1e6 of the 1e7 histories"
    return W.cfg0(), "cfg0 in full"


def time_oracle(problem, threads):
    from oracle import orc
    cores = orc.lib().orc_set_threads(threads)
    t0 = time.perf_counter()
    r = orc.run(problem)
    dt = time.perf_counter() - t0
    orc.lib().orc_set_threads(0)
    return r["totals"]["n_seg"] / dt, histories_of(problem, r) / dt, cores, dt, r


def cpu_baseline(name):
    """The oracle as it stands on the box's host cores: all cores on a bounded sample, and one core on a tenth of it."""
    from paper_2506_00263_b200 import workloads as W
    p, what = oracle_sample(name)
    v, h, cores, dt, r = time_oracle(p, 0)
    small = W.BY_NAME[name](**dict(FULL[name]["kw"], n=max(1000, p.n_particles // 16), **({"n_inactive": p.n_inactive, "n_active": p.n_active} if p.mode == "k" else {})))
    v1, h1, _, dt1, _ = time_oracle(small, 1)
    return {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": f"{what} ({r['totals']['n_seg']} segments, {dt:.1f} s)",
            "histories_per_sec": h,
            "one_core": {"value": v1, "unit": UNIT, "cores": 1, "histories_per_sec": h1,
                         "sample": f"the same problem at {small.n_particles} particles ({dt1:.1f} s)"}}, p, r


def run_reference(args, rank, world):
    """The oracle, as it stands, on the host cores; each step a bounded sample of the headline workload."""
    if rank != 0:
        return
    from oracle import orc
    name = args.workload or HEADLINE
    p, what = oracle_sample(name)
    if name == "cfg4":                       # keep K + W steps inside a few minutes: a fifth of the cpu_baseline sample per step
        p.n_particles = 200000
        what = "cfg4's problem at 2e5 particles/gen (1/500 of the workload's 1e8), 1 + 2 generations per step"
    cores = orc.lib().orc_set_threads(0)
    segs = hist = 0
    for _ in range(args.warmup):
        orc.run(p)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = orc.run(p)
        segs += r["totals"]["n_seg"]; hist += histories_of(p, r)
    dt = time.perf_counter() - t0
    v = segs / dt
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1), "higher_is_better": True, "scaling": "strong",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": FULL[name]["desc"], "sample": what},
                      "histories_per_sec": hist / dt,
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}))


# ---------------------------------------------------------------------------------------------------- the CUDA path
class Runner:
    def __init__(self, rank, world, local_rank, extra_opts=None):
        import torch
        self.extra_opts = dict(extra_opts or {})
        self.torch, self.rank, self.world, self.dev = torch, rank, world, f"cuda:{local_rank}"
        self.flush = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev)
        self.prof = profile_metrics()
        self.peak, self.peak_src = peaks()

    def barrier(self):
        if self.world > 1:
            import torch.distributed as dist
            dist.barrier()
        self.torch.cuda.synchronize()

    def run_once(self, P, prob):
        """One step.  world == 1: the library's own loop; world > 1: this rank's share of the one problem."""
        if self.world == 1:
            if prob.mode == "fixed":
                P.run_fixed_source(prob.n_particles, prob.seed)
            else:
                P.run_k_eigenvalue(prob.n_particles, prob.n_inactive, prob.n_active, prob.seed)
        else:
            from paper_2506_00263_b200 import shard
            if prob.mode == "fixed":
                lo, cnt = shard.id_range(prob.n_particles, self.rank, self.world)
                P.set_option("id_offset", lo)
                if cnt:
                    P.run_fixed_source(cnt, prob.seed)
            else:
                shard.run_k_eigenvalue_sharded(P, prob.n_particles, prob.n_inactive, prob.n_active, prob.seed, self.rank, self.world, read=False)

    def time_variant(self, name, prob, variant, steps, warmup, sample_clocks=False, e2e_steps=1):
        import torch.distributed as dist
        from paper_2506_00263_b200 import tdr
        torch = self.torch
        scheme, decomp, stash = variant
        if self.rank == 0:
            print(f"[bench] {name} {vkey(variant)}: {warmup} warm-up + {steps} timed step(s)", file=sys.stderr, flush=True)
        opts = dict(scheme=scheme, decomposition=decomp, keep_history=0, **({"stash": stash} if stash else {}), **self.extra_opts)
        P = tdr.Problem(prob, device=self.dev, time_kernels=1, **opts)
        for _ in range(warmup):
            self.run_once(P, prob)
        self.barrier()
        sampler = ClockSampler(int(self.dev.split(":")[1])) if (sample_clocks and self.rank == 0) else None
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        launches = 0; step_ms = 0.0; step_launches = 0
        e0.record()
        for _ in range(steps):
            self.flush.zero_()                                       # L2 flush between timed iterations
            self.run_once(P, prob)
            d = P.diagnostics()
            launches += d["kernel_launches"]; step_ms += d["step_ms"]; step_launches += d["step_launches"]
        e1.record()
        self.barrier()
        ms = e0.elapsed_time(e1)
        clocks = sampler.stop() if sampler else None
        res = P.read_tallies(history=False, bank=False)
        seg_local, hist_local = res["totals"]["n_seg"], histories_of(prob, res) if self.world == 1 else int(res["totals"]["n_born"])
        P.close()
        # e2e: host buffers in, host buffers out, through the C ABI (init uploads the tables, read_tallies downloads)
        self.barrier()
        t0 = time.perf_counter()
        bi = bo = 0
        for _ in range(e2e_steps):
            Q = tdr.Problem(prob, device=self.dev, **opts)
            self.run_once(Q, prob)
            r = Q.read_tallies(history=False, bank=False)
            bi, bo = input_bytes(prob), output_bytes(r)
            Q.close()
        self.barrier()
        e2e_s = time.perf_counter() - t0
        t = torch.tensor([ms, e2e_s, float(seg_local), float(hist_local), float(launches), step_ms], dtype=torch.float64, device=self.dev)
        if self.world > 1:
            mx = t.clone(); dist.all_reduce(mx, op=dist.ReduceOp.MAX)
            sm = t.clone(); dist.all_reduce(sm, op=dist.ReduceOp.SUM)
            ms, e2e_s, step_ms = mx[0].item(), mx[1].item(), mx[5].item()
            seg_step, hist_step, launches = sm[2].item(), sm[3].item(), sm[4].item()
        else:
            seg_step, hist_step = float(seg_local), float(hist_local)
        kind = "split" if decomp == "split" else ("ce" if FULL[name]["ce"] else "mg")
        alg_bytes = BYTES_PER_SEGMENT[kind] * seg_local + BYTES_PER_HISTORY * hist_local          # one step, this rank
        ach = (alg_bytes * steps / 1e9) / (step_ms / 1e3) if step_ms > 0 else 0.0
        kname = {"stack": {"fused": "k_step (+ k_drain)", "hybrid": "k_step + k_collide", "split": "k_event x 5"}[decomp],
                 "async": {"index": "k_async", "particle": "k_pstash", "shared": "k_cstash", None: "k_async"}[stash if decomp != "split" else "index"]}[scheme]
        pm = self.prof.get((name, vkey(variant)), {})
        traffic = float(pm["dram_bytes_per_segment"]) * seg_local / max(step_launches / max(steps, 1), 1) if pm.get("dram_bytes_per_segment") else None
        tips = float(pm["thread_inst_per_segment"]) if pm.get("thread_inst_per_segment") else None
        seg_rate_kernel = seg_local * steps / (step_ms / 1e3) if step_ms > 0 else 0.0
        entry = {
            "scheme": scheme, "decomposition": decomp, "stash": stash, "steps": steps, "warmup": warmup,
            "value": seg_step * steps / (ms / 1e3), "unit": UNIT, "histories_per_sec": hist_step * steps / (ms / 1e3), "ms_per_step": ms / max(steps, 1),
            "segments_per_step": seg_step, "histories_per_step": hist_step,
            "e2e": {"value": seg_step * e2e_steps / e2e_s, "unit": UNIT, "h2d_bytes_per_step": bi, "d2h_bytes_per_step": bo, "steps": e2e_steps},
            "gpu_launches": int(launches), "digest": f"{res['totals']['digest']:016x}", "k_mean": res["k_mean"] if prob.mode == "k" else None,
            "roofline": {"bound": "hbm", "kind": "modelled algorithmic bytes / measured kernel time (traffic = measured DRAM bytes)", "achieved": ach, "peak": self.peak, "unit": "GB/s", "frac": ach / self.peak, "traffic": traffic,
                         "peak_source": self.peak_src, "kernel": kname, "kernel_share_of_step": step_ms / ms if ms > 0 else None,
                         "avg_launch_us": 1e3 * step_ms / max(step_launches, 1),
                         "algorithmic_bytes_per_launch": alg_bytes * steps / max(step_launches, 1),
                         "model": f"{BYTES_PER_SEGMENT[kind]:.0f} B/segment + {BYTES_PER_HISTORY:.0f} B/history (DESIGN.md section 6); the in-flight "
                                  "window is L2- or shared-memory-resident, so measured DRAM traffic is far below it: see roofline_issue"},
            "roofline_issue": ({"bound": "alu", "unit": "thread-instructions/s", "achieved": seg_rate_kernel * tips, "peak": ISSUE_PEAK,
                                "frac": seg_rate_kernel * tips / ISSUE_PEAK, "thread_inst_per_segment": tips,
                                "source": f"profiles/ncu_r02_kernel_metrics.csv ({pm.get('commit', '?')})"} if tips else None),
        }
        return entry, clocks, res


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2506_00263_b200 import tdr
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    R = Runner(rank, world, local_rank, dict(kv.split("=", 1) for kv in args.opt))
    single = args.workload is not None
    head_name = args.workload or HEADLINE
    head_prob = make_problem(head_name, args.scale)
    if single:
        head_variants = [(args.scheme, args.decomposition, args.stash if args.scheme == "async" else None)]
    else:
        head_variants = VARIANTS[head_name]
    aux_steps, aux_warm = min(args.steps, 2), 1
    workloads, clocks, head_entry = {}, None, None
    # the headline workload: its first variant with K steps and W warm-ups, the other variants with fewer repetitions
    entries = {}
    for i, v in enumerate(head_variants):
        full = i == 0
        e, c, res = R.time_variant(head_name, head_prob, v, args.steps if full else aux_steps, args.warmup if full else aux_warm,
                                   sample_clocks=full, e2e_steps=min(args.steps, 2) if full else 1)
        entries[vkey(v)] = e
        if full:
            head_entry, clocks = e, c
    digests = {e["digest"] for e in entries.values()}
    workloads[head_name] = {"workload": FULL[head_name]["desc"], "variants": entries, "all_variants_bit_identical": len(digests) == 1}
    if not single and not args.headline_only:
        for name in ("cfg0", "cfg1", "cfg2", "cfg3"):
            prob = make_problem(name, args.scale)
            es = {}
            for v in VARIANTS[name]:
                try:
                    e, _, _ = R.time_variant(name, prob, v, aux_steps, aux_warm)
                except Exception as ex:                                # a side variant must not cost the headline its line
                    e = {"error": f"{type(ex).__name__}: {ex}", "value": 0.0}
                es[vkey(v)] = e
            workloads[name] = {"workload": FULL[name]["desc"], "variants": es,
                               "all_variants_bit_identical": len({e.get("digest", e.get("error")) for e in es.values()}) == 1}
    if rank == 0:
        e = head_entry
        best = {n: max(w["variants"], key=lambda k: w["variants"][k]["value"]) for n, w in workloads.items()}
        line = {"metric": METRIC, "value": e["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": e["ms_per_step"], "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": {"workload": FULL[head_name]["desc"] + ("" if args.scale == 1.0 else f" x {args.scale} particles"), "scheme": e["scheme"],
                           "decomposition": e["decomposition"], "stash": e["stash"], "particles": head_prob.n_particles,
                           "generations": head_prob.n_inactive + head_prob.n_active, "l2": "flushed between timed steps (256 MiB write)",
                           "sharding": "one problem, contiguous shares of the source per rank, one 32-byte all-reduce per generation" if world > 1 else "single GPU",
                           "other_variants": f"{aux_steps} timed step(s) after {aux_warm} warm-up each (see workloads)"},
                "histories_per_sec": e["histories_per_sec"], "e2e": e["e2e"], "gpu_launches": e["gpu_launches"], "clocks": clocks,
                "roofline": e["roofline"], "roofline_issue": e["roofline_issue"], "fastest_variant": best, "workloads": workloads}
        if world == 1 and not args.no_peaks:
            try:
                fp64, l2 = tdr.measure_peak("fp64"), tdr.measure_peak("l2")
                line["measured_peaks"] = {"fp64_dfma_tflops": fp64, "l2_copy_gbs": l2, "hbm_copy_gbs": R.peak, "how": "tdr_measure_peak micro-benchmarks (8 DFMA chains per thread; 16 MB -> 16 MB copy x 64); HBM from MEASURED_PEAKS.json",
                                          "issue_peak_thread_inst_per_s": ISSUE_PEAK}
            except Exception as ex:                                    # never lose the line over a micro-benchmark
                line["measured_peaks"] = {"error": str(ex)}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"], o_prob, o_res = cpu_baseline(head_name)
            # the oracle's sample against the CUDA path on the SAME sample: bit-exact parity inside the bench run
            P = tdr.Problem(o_prob, device=R.dev, scheme=e["scheme"], decomposition=e["decomposition"], keep_history=0, **({"stash": e["stash"]} if e["stash"] else {}))
            g = P.run(); P.close()
            import numpy as np
            ok = o_res["totals"] == g["totals"] and all(np.array_equal(o_res[k], g[k]) for k in ("flux", "coll", "leak", "gen_n", "gen_m", "gen_p", "gen_pc"))
            ok = ok and (len(o_res["gen_k"]) == 0 or bool(np.allclose(o_res["gen_k"], g["gen_k"], rtol=1e-12, atol=0)))
            line["parity_on_oracle_sample"] = {"ok": bool(ok), "checked": "totals + history digest, flux, coll, leak, per-generation N/M/P/Pc (bit-exact), k (1e-12) on the cpu_baseline sample"}
            if not ok:
                print(json.dumps(line)); raise SystemExit("parity on the oracle sample FAILED")
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=None, choices=sorted(FULL), help="time ONE workload/variant (profiling); default: the full bench")
    ap.add_argument("--scheme", default="async", choices=["stack", "async"])
    ap.add_argument("--decomposition", default="fused", choices=["fused", "split", "hybrid"])
    ap.add_argument("--stash", default="index", choices=["index", "particle", "shared"])
    ap.add_argument("--scale", type=float, default=1.0, help="scale the particle count of every workload (smoke runs)")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE", help="extra tdr_set_option for every variant timed (sweeps, profiling)")
    ap.add_argument("--headline-only", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-peaks", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1")); local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
