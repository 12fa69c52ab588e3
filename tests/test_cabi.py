"""CPU-side checks of the boundary: the library builds, loads and exports every symbol include/tdr.h declares."""
import os
import re

from paper_2506_00263_b200 import tdr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "tdr.h")).read()
    declared = sorted(set(re.findall(r"\b(tdr_[a-z_]+)\s*\(", header)))
    assert set(declared) == set(tdr.EXPORTS), declared
    L = tdr.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_struct_layouts_match_header_sizes():
    import ctypes as C
    assert tdr.SITE_DTYPE.itemsize == 48
    assert C.sizeof(tdr.tdr_sizes) == 32
    assert C.sizeof(tdr.tdr_diag) == 8 * 2 + 64 + 24 + 16 + 8


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2506_00263_b200")
    bad = re.compile(r"^\s*(from|import)\s+oracle|orc\.h|liborc|orc_[a-z]+\s*\(", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not bad.search(open(os.path.join(dirpath, f)).read()), f
    assert not bad.search(open(os.path.join(ROOT, "include", "tdr.h")).read())
    # and the oracle never touches the CUDA side
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "libtdr" not in src and "tdr_" not in src and "import tdr" not in src, f


def test_no_gpu_means_loud_failure():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2506_00263_b200 import workloads as W
    with pytest.raises(RuntimeError):
        tdr.Problem(W.cfg0())
