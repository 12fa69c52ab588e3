"""Helpers shared by the GPU parity tests: run both sides on the same seeded workload and compare."""
import numpy as np


def assert_same(o, g, what=""):
    """o = oracle result, g = CUDA result.  Integers bit-exact; bank/history as sorted multisets; k to 1e-12."""
    assert o["totals"] == g["totals"], (what, o["totals"], g["totals"])
    for k in ("flux", "coll", "leak", "gen_n", "gen_m", "gen_p", "gen_pc"):
        assert np.array_equal(o[k], g[k]), (what, k)
    assert len(o["gen_k"]) == len(g["gen_k"])
    if len(o["gen_k"]):
        assert np.allclose(o["gen_k"], g["gen_k"], rtol=1e-12, atol=0), (what, "gen_k")
        assert abs(o["k_mean"] - g["k_mean"]) <= 1e-12 * abs(o["k_mean"]) and abs(o["k_std"] - g["k_std"]) <= 1e-12 * max(abs(o["k_std"]), 1e-300) + 1e-18
    if "hist_id" in g and len(o["hist_id"]):
        a = np.sort(np.rec.fromarrays([o["hist_id"], o["hist_nseg"], o["hist_ncoll"]]), order=["f0", "f1", "f2"])
        b = np.sort(np.rec.fromarrays([g["hist_id"], g["hist_nseg"], g["hist_ncoll"]]), order=["f0", "f1", "f2"])
        assert len(a) == len(b) and np.array_equal(a, b), (what, "per-history event counts")
    if "bank" in g:
        assert np.array_equal(np.sort(o["bank"].view(np.dtype((np.void, 48)))), np.sort(g["bank"].view(np.dtype((np.void, 48))))), (what, "bank multiset")


_ORACLE_CACHE = {}


def _problem_key(p):
    import hashlib
    h = hashlib.sha1()
    for d in (p.geometry, p.materials, p.xs or {}):
        for k in sorted(d):
            v = d[k]
            h.update(k.encode()); h.update(np.ascontiguousarray(v).tobytes() if isinstance(v, np.ndarray) else repr(v).encode())
    return (p.mode, p.n_particles, p.n_inactive, p.n_active, p.seed, h.hexdigest())


def oracle_result(problem):
    """The oracle's result for this problem, computed once per test session (many variants are compared with the same run)."""
    from oracle import orc
    k = _problem_key(problem)
    if k not in _ORACLE_CACHE:
        if len(_ORACLE_CACHE) > 24:
            _ORACLE_CACHE.pop(next(iter(_ORACLE_CACHE)))
        _ORACLE_CACHE[k] = orc.run(problem)
    return _ORACLE_CACHE[k]


def run_both(problem, **options):
    from paper_2506_00263_b200 import tdr
    o = oracle_result(problem)
    P = tdr.Problem(problem, **options)
    try:
        g = P.run()
        d = P.diagnostics()
    finally:
        P.close()
    return o, g, d
