"""Throughput of the CUDA path on any of the five synthetic workloads (BASELINE.json configs[0..4]):
    python -m paper_2506_00263_b200.throughput cfg2 --n 10000000 --inactive 2 --active 4 --scheme async --decomposition fused
Prints one JSON line per (scheme, decomposition): segments/s, histories/s, device time of the run_* body (CUDA events
inside the library).  GPU only; no oracle is involved (parity is the tests' and bench.py's job)."""
from __future__ import annotations

import argparse
import json

from . import tdr, workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", choices=sorted(W.BY_NAME))
    ap.add_argument("--n", type=int, default=0)
    ap.add_argument("--inactive", type=int, default=-1)
    ap.add_argument("--active", type=int, default=-1)
    ap.add_argument("--ebins", type=int, default=0)
    ap.add_argument("--scheme", default="async,stack")
    ap.add_argument("--decomposition", default="fused,hybrid,split")
    ap.add_argument("--repeat", type=int, default=2)
    ap.add_argument("--option", action="append", default=[], help="key=value passed to tdr_set_option")
    a = ap.parse_args()
    kw = {}
    if a.n:
        kw["n"] = a.n
    if a.inactive >= 0:
        kw["n_inactive"] = a.inactive
    if a.active >= 0:
        kw["n_active"] = a.active
    if a.ebins:
        kw["n_ebins"] = a.ebins
    prob = W.BY_NAME[a.workload](**kw)
    extra = dict(o.split("=", 1) for o in a.option)
    for scheme in a.scheme.split(","):
        for decomp in a.decomposition.split(","):
            P = tdr.Problem(prob, scheme=scheme, decomposition=decomp, keep_history=0, **extra)
            best = None
            for _ in range(a.repeat):
                P.run_fixed_source(prob.n_particles, prob.seed) if prob.mode == "fixed" else \
                    P.run_k_eigenvalue(prob.n_particles, prob.n_inactive, prob.n_active, prob.seed)
                d = P.diagnostics()
                best = d["gpu_ms"] if best is None else min(best, d["gpu_ms"])
            r = P.read_tallies(history=False, bank=False)
            hist = int(r["gen_n"].sum()) if prob.mode == "k" else r["totals"]["n_born"]
            print(json.dumps({"workload": a.workload, "n": prob.n_particles, "generations": prob.n_inactive + prob.n_active,
                              "scheme": scheme, "decomposition": decomp, "segments": r["totals"]["n_seg"], "histories": hist,
                              "gpu_ms": best, "segments_per_sec": r["totals"]["n_seg"] / best * 1e3, "histories_per_sec": hist / best * 1e3,
                              "k_mean": r["k_mean"], "kernel_launches": d["kernel_launches"], "digest": r["totals"]["digest"]}), flush=True)
            P.close()


if __name__ == "__main__":
    main()
