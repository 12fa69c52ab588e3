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


def _init_rc(problem):
    """tdr_init_problem's return code for a (possibly broken) problem; input validation runs before any CUDA call."""
    import ctypes as C
    keep = []
    g = tdr._fill(tdr.tdr_geometry(), problem.geometry, keep)
    m = tdr._fill(tdr.tdr_materials(), problem.materials, keep)
    x = tdr._fill(tdr.tdr_xs_tables(), problem.xs, keep) if problem.xs is not None else None
    h = C.c_void_p()
    rc = tdr.lib().tdr_init_problem(C.byref(g), C.byref(m), C.byref(x) if x is not None else None, C.byref(h))
    if rc == 0:
        tdr.lib().tdr_free_problem(h)
    return rc


def test_init_rejects_out_of_range_tables_with_einval():
    """Every index table is dereferenced on the device, so init range-checks it on the host (TDR_EINVAL = -1)."""
    import numpy as np
    from paper_2506_00263_b200 import workloads as W
    EINVAL = -1

    def broken(make, edit):
        p = make()
        edit(p)
        return _init_rc(p)

    mk2 = lambda: W.cfg2(n=10)
    assert broken(mk2, lambda p: p.geometry["cell_univ"].__setitem__((0, 0, 0), 7)) == EINVAL        # universe out of range
    assert broken(mk2, lambda p: p.geometry["univ_mat"].__setitem__((0, 0), 9)) == EINVAL            # material out of range
    assert broken(mk2, lambda p: p.geometry["univ_radius"].__setitem__((0, 0), 0.7)) == EINVAL       # radius >= pitch/2
    assert broken(mk2, lambda p: p.geometry["xplanes"].__setitem__(3, 0.5)) == EINVAL                # planes not ascending
    assert broken(mk2, lambda p: p.geometry["mesh_z"].__setitem__(4, 1.0)) == EINVAL                 # mesh not ascending
    assert broken(mk2, lambda p: p.geometry.__setitem__("src_index", 7)) == EINVAL                   # group >= G
    assert broken(mk2, lambda p: p.geometry["bc"].__setitem__(0, 3)) == EINVAL
    mk3 = lambda: W.cfg3(n=10, n_grid=500)
    assert broken(mk3, lambda p: p.materials["mat_nuc"].__setitem__((0, 0), 3)) == EINVAL            # nuclide out of range
    assert broken(mk3, lambda p: p.materials["mat_nnuc"].__setitem__(1, 5)) == EINVAL
    assert broken(mk3, lambda p: p.xs["energy"].__setitem__(10, p.xs["energy"][9])) == EINVAL        # grid not increasing
    assert broken(mk3, lambda p: p.geometry["e_edges"].__setitem__(2, 0.0)) == EINVAL
    mk4 = lambda: W.cfg4(n=10, n_grid=500)
    assert broken(mk4, lambda p: p.geometry.__setitem__("src_index", 3)) == EINVAL                   # Watt nuclide out of range
    mk5 = lambda: W.general_cells("k", n=10)                                                          # general cells (readings C1-C6)
    assert broken(mk5, lambda p: p.geometry["cell_surf"].__setitem__((0, 0), 9)) == EINVAL           # surface out of range
    assert broken(mk5, lambda p: p.geometry["cell_surf"].__setitem__((1, 1), 0)) == EINVAL           # a cell naming no surface
    assert broken(mk5, lambda p: p.geometry["cell_mat"].__setitem__(2, 5)) == EINVAL
    assert broken(mk5, lambda p: p.geometry["surf_kind"].__setitem__(0, 3)) == EINVAL
    assert broken(mk5, lambda p: p.geometry["surf_coef"].__setitem__((0, 3), -0.5)) == EINVAL        # negative radius
    assert broken(mk5, lambda p: p.geometry["univ_ncell"].__setitem__(2, 9)) == EINVAL               # cells beyond the table
    # untouched problems pass validation (the return code is then 0 on a GPU box, TDR_ECUDA = -3 without a device)
    for mk in (mk2, mk3, mk4, mk5, W.cfg0, lambda: W.cfg1(n=10), lambda: W.slab(1.0, 2.0, n=10), lambda: W.ce_slowing_down(n=10)):
        assert _init_rc(mk()) in (0, -3)
