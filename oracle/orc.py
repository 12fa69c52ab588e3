"""ctypes binding of the CPU oracle (TEST INFRASTRUCTURE ONLY — see oracle/orc.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this module.  It never imports the CUDA package's binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.environ.get("ORC_LIB") or os.path.join(HERE, "liborc.so")     # ORC_LIB: tests/mutation_check.py loads a mutant
MAX_RINGS, MAX_NUC, T_COUNT = 4, 4, 16
TOTAL_NAMES = ["n_seg", "n_coll", "n_cross", "n_abs", "n_fis", "n_leak", "n_born", "n_dropped",
               "n_dirfail", "digest", "n_sites", "n_census", "n_roulette"]
SITE_DTYPE = np.dtype([("x", "<f8"), ("y", "<f8"), ("z", "<f8"), ("id", "<u8"), ("ix", "<i2"), ("iy", "<i2"),
                       ("iz", "<i2"), ("mx", "<i2"), ("my", "<i2"), ("mz", "<i2"), ("ring", "u1"),
                       ("src", "u1"), ("depth", "u1"), ("it", "u1")])
assert SITE_DTYPE.itemsize == 48

PD, PI = C.POINTER(C.c_double), C.POINTER(C.c_int32)


def build(force=False):
    src = os.path.join(HERE, "orc.c")
    if os.environ.get("ORC_LIB"):
        return LIB
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(src), os.path.getmtime(os.path.join(HERE, "orc.h"))):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC",
                               src, "-o", LIB, "-lm"])
    return LIB


class Geometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("xplanes", PD), ("yplanes", PD), ("zplanes", PD), ("cx", PD), ("cy", PD), ("cell_univ", PI),
                ("bc", C.c_int32 * 6), ("n_univ", C.c_int32), ("univ_nrings", PI), ("univ_radius", PD), ("univ_mat", PI),
                ("mesh_n", C.c_int32 * 3), ("mesh_x", PD), ("mesh_y", PD), ("mesh_z", PD),
                ("by_group", C.c_int32), ("n_ebins", C.c_int32), ("e_edges", PD),
                ("src_kind", C.c_int32), ("src_lo", C.c_double * 3), ("src_hi", C.c_double * 3),
                ("src_dir_kind", C.c_int32), ("src_dir", C.c_double * 3),
                ("src_energy_kind", C.c_int32), ("src_index", C.c_int32), ("src_energy", C.c_double),
                ("tally_scale_log2", C.c_int32), ("n_tbins", C.c_int32), ("t_edges", PD),
                ("implicit_capture", C.c_int32), ("w_roulette", C.c_double), ("w_survive", C.c_double),
                ("n_surf", C.c_int32), ("surf_kind", PI), ("surf_coef", PD), ("n_cell", C.c_int32), ("univ_cell0", PI), ("univ_ncell", PI),
                ("cell_nsurf", PI), ("cell_surf", PI), ("cell_mat", PI)]


class Materials(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("G", C.c_int32), ("sig_t", PD), ("sig_s", PD), ("sig_f", PD), ("nu", PD),
                ("chi", PD), ("mat_nnuc", PI), ("mat_nuc", PI), ("mat_dens", PD), ("speed", PD)]


class XsTables(C.Structure):
    _fields_ = [("n_grid", C.c_int32), ("n_nuc", C.c_int32), ("energy", PD), ("A", PD), ("sig_s", PD), ("sig_c", PD),
                ("sig_f", PD), ("nu", PD), ("watt_a", PD), ("watt_b", PD)]


class Sizes(C.Structure):
    _fields_ = [("n_bins", C.c_uint64), ("n_gen", C.c_uint64), ("n_hist", C.c_uint64), ("n_bank", C.c_uint64)]


class Tallies(C.Structure):
    _fields_ = [("flux", C.c_void_p), ("coll", C.c_void_p), ("leak", C.c_int64 * 6), ("totals", C.c_uint64 * T_COUNT),
                ("k_mean", C.c_double), ("k_std", C.c_double), ("gen_n", C.c_void_p), ("gen_m", C.c_void_p),
                ("gen_p", C.c_void_p), ("gen_pc", C.c_void_p), ("gen_k", C.c_void_p), ("hist_id", C.c_void_p),
                ("hist_nseg", C.c_void_p), ("hist_ncoll", C.c_void_p), ("bank", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(LIB)
        L.orc_init_problem.argtypes = [C.POINTER(Geometry), C.POINTER(Materials), C.POINTER(XsTables), C.POINTER(C.c_void_p)]
        L.orc_run_fixed_source.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64]
        L.orc_run_k_eigenvalue.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint64]
        L.orc_run_fixed_source_range.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64]
        L.orc_k_begin.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint64]
        L.orc_k_generation.argtypes = [C.c_void_p, C.c_uint32, C.c_int, C.c_double, C.c_int, C.POINTER(C.c_int64)]
        L.orc_k_popctrl.argtypes = [C.c_void_p, C.c_uint32, C.c_double, C.POINTER(C.c_uint64)]
        L.orc_k_end.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.orc_tally_sizes.argtypes = [C.c_void_p, C.POINTER(Sizes)]
        L.orc_read_tallies.argtypes = [C.c_void_p, C.POINTER(Tallies)]
        L.orc_free_problem.argtypes = [C.c_void_p]
        L.orc_free_problem.restype = None
        L.orc_set_threads.argtypes = [C.c_int]
        L.orc_philox.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.orc_philox.restype = None
        L.orc_draw.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_draw.restype = C.c_double
        L.orc_derive_id.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_derive_id.restype = C.c_uint64
        L.orc_det_log.argtypes = [C.c_double]
        L.orc_det_log.restype = C.c_double
        L.orc_iso_dir.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, PD]
        L.orc_watt.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_double, C.c_double]
        L.orc_watt.restype = C.c_double
        L.orc_scatter_ce.argtypes = [C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint32, C.c_double, C.c_double, PD, PD, PD]
        L.orc_scatter_ce.restype = None
        L.orc_dist_cyl.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int]
        L.orc_dist_cyl.restype = C.c_double
        L.orc_surf_eval.argtypes = [C.c_int, PD, C.c_double, C.c_double, C.c_double]
        L.orc_surf_eval.restype = C.c_double
        L.orc_surf_dist.argtypes = [C.c_int, PD] + [C.c_double] * 6 + [C.c_int]
        L.orc_surf_dist.restype = C.c_double
        L.orc_grid_index.argtypes = [PD, C.c_int32, C.c_double]
        L.orc_grid_index.restype = C.c_int32
        _lib = L
    return _lib


def _pd(a):
    return a.ctypes.data_as(PD)


def _pi(a):
    return a.ctypes.data_as(PI)


def _fill(struct, d, keep):
    for name, ctype in struct._fields_:
        if name not in d:
            continue
        v = d[name]
        if ctype is PD:
            a = np.ascontiguousarray(v, dtype=np.float64); keep.append(a); setattr(struct, name, _pd(a))
        elif ctype is PI:
            a = np.ascontiguousarray(v, dtype=np.int32); keep.append(a); setattr(struct, name, _pi(a))
        elif isinstance(v, np.ndarray) or isinstance(v, (list, tuple)):
            setattr(struct, name, ctype(*[x.item() if hasattr(x, "item") else x for x in np.asarray(v).ravel()]))
        else:
            setattr(struct, name, v)
    return struct


class Oracle:
    """One problem instance of the oracle; results as numpy arrays."""

    def __init__(self, problem):
        self.problem = problem
        keep = []
        g = _fill(Geometry(), problem.geometry, keep)
        m = _fill(Materials(), problem.materials, keep)
        x = _fill(XsTables(), problem.xs, keep) if problem.xs is not None else None
        self.h = C.c_void_p()
        rc = lib().orc_init_problem(C.byref(g), C.byref(m), C.byref(x) if x is not None else None, C.byref(self.h))
        if rc:
            raise RuntimeError(f"orc_init_problem failed: {rc}")

    def run(self, n=None, n_inactive=None, n_active=None, seed=None):
        p = self.problem
        n = p.n_particles if n is None else n
        seed = p.seed if seed is None else seed
        if p.mode == "fixed":
            rc = lib().orc_run_fixed_source(self.h, n, seed)
        else:
            rc = lib().orc_run_k_eigenvalue(self.h, n, p.n_inactive if n_inactive is None else n_inactive,
                                            p.n_active if n_active is None else n_active, seed)
        if rc:
            raise RuntimeError(f"oracle run failed: {rc}")
        return self.read()

    def run_fixed_source_range(self, first_id, n, seed):
        rc = lib().orc_run_fixed_source_range(self.h, first_id, n, seed)
        if rc:
            raise RuntimeError(f"oracle run failed: {rc}")
        return self.read()

    # D2 in steps: the same four calls the CUDA library offers, so that the multi-process driver can be tested on CPU
    def k_begin(self, first_id, n_local, n_gen, seed):
        rc = lib().orc_k_begin(self.h, first_id, n_local, n_gen, seed)
        if rc:
            raise RuntimeError(f"orc_k_begin failed: {rc}")

    def k_generation(self, gen, active, k_prev, last):
        sums = (C.c_int64 * 4)()
        rc = lib().orc_k_generation(self.h, gen, int(active), k_prev, int(last), sums)
        if rc:
            raise RuntimeError(f"orc_k_generation failed: {rc}")
        return list(sums)

    def k_population_control(self, gen_next, pr):
        n = C.c_uint64()
        rc = lib().orc_k_popctrl(self.h, gen_next, pr, C.byref(n))
        if rc:
            raise RuntimeError(f"orc_k_popctrl failed: {rc}")
        return n.value

    def k_end(self, n_inactive, gen_n, gen_m, gen_p, gen_pc, gen_k):
        a = [np.ascontiguousarray(gen_n, np.uint64), np.ascontiguousarray(gen_m, np.uint64), np.ascontiguousarray(gen_p, np.int64),
             np.ascontiguousarray(gen_pc, np.int64), np.ascontiguousarray(gen_k, np.float64)]
        rc = lib().orc_k_end(self.h, len(a[0]), n_inactive, *[x.ctypes.data for x in a])
        if rc:
            raise RuntimeError(f"orc_k_end failed: {rc}")

    def scale(self):
        return float(2 ** int(self.problem.geometry["tally_scale_log2"]))

    def read_tallies(self, history=True, bank=True):
        return self.read()

    def read(self):
        s = Sizes()
        lib().orc_tally_sizes(self.h, C.byref(s))
        out = dict(flux=np.zeros(s.n_bins, np.int64), coll=np.zeros(s.n_bins, np.int64),
                   gen_n=np.zeros(s.n_gen, np.uint64), gen_m=np.zeros(s.n_gen, np.uint64),
                   gen_p=np.zeros(s.n_gen, np.int64), gen_pc=np.zeros(s.n_gen, np.int64), gen_k=np.zeros(s.n_gen, np.float64),
                   hist_id=np.zeros(s.n_hist, np.uint64), hist_nseg=np.zeros(s.n_hist, np.uint32),
                   hist_ncoll=np.zeros(s.n_hist, np.uint32), bank=np.zeros(s.n_bank, SITE_DTYPE))
        t = Tallies()
        for k, a in out.items():
            setattr(t, k, a.ctypes.data)
        rc = lib().orc_read_tallies(self.h, C.byref(t))
        if rc:
            raise RuntimeError(f"orc_read_tallies failed: {rc}")
        out["leak"] = np.array(list(t.leak), np.int64)
        out["totals"] = {n: int(t.totals[i]) for i, n in enumerate(TOTAL_NAMES)}
        out["k_mean"], out["k_std"] = t.k_mean, t.k_std
        return out

    def close(self):
        if self.h:
            lib().orc_free_problem(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def run(problem, **kw):
    o = Oracle(problem)
    try:
        return o.run(**kw)
    finally:
        o.close()
