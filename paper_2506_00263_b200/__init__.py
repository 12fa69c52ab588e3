"""paper_2506_00263_b200 — event-based Monte Carlo neutron transport with thread-data remapping
(arxiv 2506.00263) as hand-written CUDA for B200 (sm_100a), behind the C ABI in include/tdr.h.

  workloads  seeded synthetic inputs (shared with the test oracle; no method arithmetic)
  tdr        ctypes binding of libtdr.so (loads the CUDA library; no CPU fallback)
  build      in-tree nvcc build
  shard      multi-GPU plumbing: id-range sharding of a fixed source, int64 all-reduce of tallies
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "tdr", "build", "shard"]


def __getattr__(name):
    if name in ("tdr", "build", "shard"):
        import importlib
        return importlib.import_module("." + name, __name__)
    raise AttributeError(name)
