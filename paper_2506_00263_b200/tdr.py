"""Thin ctypes binding of libtdr.so (include/tdr.h).  Argument marshalling only: every step of the
transport path runs in the CUDA kernels.  torch supplies device memory (the workspace) and the stream.
There is no CPU fallback: a missing library or device raises."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from . import build as _build

MAX_RINGS, MAX_NUC, T_COUNT = 4, 4, 16
TOTAL_NAMES = ["n_seg", "n_coll", "n_cross", "n_abs", "n_fis", "n_leak", "n_born", "n_dropped",
               "n_dirfail", "digest", "n_sites", "n_census", "n_roulette"]
SITE_DTYPE = np.dtype([("x", "<f8"), ("y", "<f8"), ("z", "<f8"), ("id", "<u8"), ("ix", "<i2"), ("iy", "<i2"),
                       ("iz", "<i2"), ("mx", "<i2"), ("my", "<i2"), ("mz", "<i2"), ("ring", "u1"),
                       ("src", "u1"), ("depth", "u1"), ("it", "u1")])
PD, PI = C.POINTER(C.c_double), C.POINTER(C.c_int32)


class tdr_geometry(C.Structure):
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


class tdr_materials(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("G", C.c_int32), ("sig_t", PD), ("sig_s", PD), ("sig_f", PD), ("nu", PD),
                ("chi", PD), ("mat_nnuc", PI), ("mat_nuc", PI), ("mat_dens", PD), ("speed", PD)]


class tdr_xs_tables(C.Structure):
    _fields_ = [("n_grid", C.c_int32), ("n_nuc", C.c_int32), ("energy", PD), ("A", PD), ("sig_s", PD), ("sig_c", PD),
                ("sig_f", PD), ("nu", PD), ("watt_a", PD), ("watt_b", PD)]


class tdr_sizes(C.Structure):
    _fields_ = [("n_bins", C.c_uint64), ("n_gen", C.c_uint64), ("n_hist", C.c_uint64), ("n_bank", C.c_uint64)]


class tdr_tallies(C.Structure):
    _fields_ = [("flux", C.c_void_p), ("coll", C.c_void_p), ("leak", C.c_int64 * 6), ("totals", C.c_uint64 * T_COUNT),
                ("k_mean", C.c_double), ("k_std", C.c_double), ("gen_n", C.c_void_p), ("gen_m", C.c_void_p),
                ("gen_p", C.c_void_p), ("gen_pc", C.c_void_p), ("gen_k", C.c_void_p), ("hist_id", C.c_void_p),
                ("hist_nseg", C.c_void_p), ("hist_ncoll", C.c_void_p), ("bank", C.c_void_p)]


class tdr_diag(C.Structure):
    _fields_ = [("kernel_launches", C.c_uint64), ("iterations", C.c_uint64), ("events", C.c_uint64 * 8),
                ("spills", C.c_uint64), ("fetches", C.c_uint64), ("make_work_calls", C.c_uint64),
                ("gpu_ms", C.c_double), ("step_ms", C.c_double), ("step_launches", C.c_uint64)]


EXPORTS = ["tdr_init_problem", "tdr_set_option", "tdr_workspace_bytes", "tdr_bind_workspace", "tdr_run_fixed_source",
           "tdr_run_k_eigenvalue", "tdr_tally_sizes", "tdr_read_tallies", "tdr_read_diagnostics", "tdr_free_problem",
           "tdr_last_error", "tdr_dev_det_log", "tdr_dev_draw", "tdr_k_begin", "tdr_k_generation", "tdr_k_population_control", "tdr_k_end", "tdr_measure_peak", "tdr_dev_popctrl", "tdr_dev_popctrl_noalloc"]

_lib = None


def lib():
    """Load libtdr.so (building it in-tree if the sources are newer).  Raises if it cannot be loaded."""
    global _lib
    if _lib is None:
        path = os.environ.get("TDR_LIB") or (_build.build() if os.path.exists(_build.CSRC) else _build.LIB)   # TDR_LIB: a developer's trial build
        L = C.CDLL(path)
        L.tdr_init_problem.argtypes = [C.POINTER(tdr_geometry), C.POINTER(tdr_materials), C.POINTER(tdr_xs_tables), C.POINTER(C.c_void_p)]
        L.tdr_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_char_p]
        L.tdr_workspace_bytes.argtypes = [C.c_void_p, C.c_uint64, C.POINTER(C.c_uint64)]
        L.tdr_bind_workspace.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
        L.tdr_run_fixed_source.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64]
        L.tdr_run_k_eigenvalue.argtypes = [C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint64]
        L.tdr_k_begin.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint32, C.c_uint64]
        L.tdr_k_generation.argtypes = [C.c_void_p, C.c_uint32, C.c_int, C.c_double, C.c_int, C.POINTER(C.c_int64)]
        L.tdr_k_population_control.argtypes = [C.c_void_p, C.c_uint32, C.c_double, C.POINTER(C.c_uint64)]
        L.tdr_k_end.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tdr_measure_peak.argtypes = [C.c_int, C.POINTER(C.c_double), C.c_void_p]
        L.tdr_tally_sizes.argtypes = [C.c_void_p, C.POINTER(tdr_sizes)]
        L.tdr_read_tallies.argtypes = [C.c_void_p, C.POINTER(tdr_tallies)]
        L.tdr_read_diagnostics.argtypes = [C.c_void_p, C.POINTER(tdr_diag)]
        L.tdr_free_problem.argtypes = [C.c_void_p]
        L.tdr_free_problem.restype = None
        L.tdr_last_error.restype = C.c_char_p
        L.tdr_dev_det_log.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
        L.tdr_dev_draw.argtypes = [C.c_uint64, C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_uint64, C.c_void_p]
        for f in (L.tdr_dev_popctrl, L.tdr_dev_popctrl_noalloc):
            f.argtypes = [C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_void_p, C.c_uint64, C.c_uint32, C.c_double, C.c_void_p]
        _lib = L
    return _lib


class TdrError(RuntimeError):
    def __init__(self, code, what):
        super().__init__(f"{what}: code {code}: {lib().tdr_last_error().decode()}")
        self.code = code


def _check(rc, what):
    if rc != 0:
        raise TdrError(rc, what)


def _fill(struct, d, keep):
    for name, ctype in struct._fields_:
        if name not in d:
            continue
        v = d[name]
        if ctype is PD:
            a = np.ascontiguousarray(v, dtype=np.float64); keep.append(a); setattr(struct, name, a.ctypes.data_as(PD))
        elif ctype is PI:
            a = np.ascontiguousarray(v, dtype=np.int32); keep.append(a); setattr(struct, name, a.ctypes.data_as(PI))
        elif isinstance(v, (np.ndarray, list, tuple)):
            setattr(struct, name, ctype(*[x.item() if hasattr(x, "item") else x for x in np.asarray(v).ravel()]))
        else:
            setattr(struct, name, v)
    return struct


class Problem:
    """init_problem / run_fixed_source / run_k_eigenvalue / read_tallies on one CUDA device."""

    def __init__(self, problem, device="cuda:0", **options):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2506_00263_b200 needs a CUDA device: there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.problem = problem
        keep = []
        g = _fill(tdr_geometry(), problem.geometry, keep)
        m = _fill(tdr_materials(), problem.materials, keep)
        x = _fill(tdr_xs_tables(), problem.xs, keep) if problem.xs is not None else None
        self.h = C.c_void_p()
        _check(lib().tdr_init_problem(C.byref(g), C.byref(m), C.byref(x) if x is not None else None, C.byref(self.h)), "tdr_init_problem")
        self.ws = None
        for k, v in options.items():
            self.set_option(k, v)

    def set_option(self, key, value):
        _check(lib().tdr_set_option(self.h, str(key).encode(), str(value).encode()), f"tdr_set_option({key})")

    def _bind(self, n):
        need = C.c_uint64()
        _check(lib().tdr_workspace_bytes(self.h, n, C.byref(need)), "tdr_workspace_bytes")
        if self.ws is None or self.ws.numel() < need.value:
            self.ws = None
            self.ws = self.torch.empty(need.value + 256, dtype=self.torch.uint8, device=self.device)
        ptr = (self.ws.data_ptr() + 255) & ~255
        stream = self.torch.cuda.current_stream(self.device).cuda_stream
        _check(lib().tdr_bind_workspace(self.h, ptr, need.value, stream), "tdr_bind_workspace")

    def run_fixed_source(self, n_particles, seed):
        self._bind(n_particles)
        _check(lib().tdr_run_fixed_source(self.h, n_particles, seed), "tdr_run_fixed_source")

    def run_k_eigenvalue(self, n_particles, n_inactive, n_active, seed):
        self._bind(n_particles)
        _check(lib().tdr_run_k_eigenvalue(self.h, n_particles, n_inactive, n_active, seed), "tdr_run_k_eigenvalue")

    # D2 in steps (one problem on several GPUs; paper_2506_00263_b200.shard drives these)
    def k_begin(self, first_id, n_local, n_gen, seed):
        self._bind(max(n_local, 1))
        _check(lib().tdr_k_begin(self.h, first_id, n_local, n_gen, seed), "tdr_k_begin")

    def k_generation(self, gen, active, k_prev, last):
        sums = (C.c_int64 * 4)()
        _check(lib().tdr_k_generation(self.h, gen, int(active), k_prev, int(last), sums), "tdr_k_generation")
        return list(sums)

    def k_population_control(self, gen_next, pr):
        n = C.c_uint64()
        _check(lib().tdr_k_population_control(self.h, gen_next, pr, C.byref(n)), "tdr_k_population_control")
        return n.value

    def k_end(self, n_inactive, gen_n, gen_m, gen_p, gen_pc, gen_k):
        a = [np.ascontiguousarray(gen_n, np.uint64), np.ascontiguousarray(gen_m, np.uint64), np.ascontiguousarray(gen_p, np.int64),
             np.ascontiguousarray(gen_pc, np.int64), np.ascontiguousarray(gen_k, np.float64)]
        _check(lib().tdr_k_end(self.h, len(a[0]), n_inactive, *[x.ctypes.data for x in a]), "tdr_k_end")

    def scale(self):
        return float(2 ** int(self.problem.geometry["tally_scale_log2"]))

    def run(self, n=None, n_inactive=None, n_active=None, seed=None):
        p = self.problem
        n = p.n_particles if n is None else n
        seed = p.seed if seed is None else seed
        if p.mode == "fixed":
            self.run_fixed_source(n, seed)
        else:
            self.run_k_eigenvalue(n, p.n_inactive if n_inactive is None else n_inactive,
                                  p.n_active if n_active is None else n_active, seed)
        return self.read_tallies()

    def read_tallies(self, history=True, bank=True):
        s = tdr_sizes()
        _check(lib().tdr_tally_sizes(self.h, C.byref(s)), "tdr_tally_sizes")
        out = dict(flux=np.zeros(s.n_bins, np.int64), coll=np.zeros(s.n_bins, np.int64),
                   gen_n=np.zeros(s.n_gen, np.uint64), gen_m=np.zeros(s.n_gen, np.uint64),
                   gen_p=np.zeros(s.n_gen, np.int64), gen_pc=np.zeros(s.n_gen, np.int64), gen_k=np.zeros(s.n_gen, np.float64))
        if history:
            out.update(hist_id=np.zeros(s.n_hist, np.uint64), hist_nseg=np.zeros(s.n_hist, np.uint32), hist_ncoll=np.zeros(s.n_hist, np.uint32))
        if bank:
            out.update(bank=np.zeros(s.n_bank, SITE_DTYPE))
        t = tdr_tallies()
        for k, a in out.items():
            setattr(t, k, a.ctypes.data)
        _check(lib().tdr_read_tallies(self.h, C.byref(t)), "tdr_read_tallies")
        out["leak"] = np.array(list(t.leak), np.int64)
        out["totals"] = {n: int(t.totals[i]) for i, n in enumerate(TOTAL_NAMES)}
        out["k_mean"], out["k_std"] = t.k_mean, t.k_std
        return out

    def diagnostics(self):
        d = tdr_diag()
        _check(lib().tdr_read_diagnostics(self.h, C.byref(d)), "tdr_read_diagnostics")
        return dict(kernel_launches=d.kernel_launches, iterations=d.iterations, events=list(d.events), spills=d.spills,
                    fetches=d.fetches, make_work_calls=d.make_work_calls, gpu_ms=d.gpu_ms, step_ms=d.step_ms,
                    step_launches=d.step_launches)

    def close(self):
        if getattr(self, "h", None):
            lib().tdr_free_problem(self.h)
            self.h = C.c_void_p()
        self.ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def dev_det_log(x):
    """x: torch cuda float64 tensor -> det_log(x) computed by the device primitive."""
    import torch
    out = torch.empty_like(x)
    _check(lib().tdr_dev_det_log(x.data_ptr(), out.data_ptr(), x.numel(), torch.cuda.current_stream().cuda_stream), "tdr_dev_det_log")
    return out


def dev_draw(seed, ids, gen, seg, purpose, j):
    import torch
    out = torch.empty(ids.numel(), dtype=torch.float64, device=ids.device)
    _check(lib().tdr_dev_draw(seed, ids.data_ptr(), gen, seg, purpose, j, out.data_ptr(), ids.numel(), torch.cuda.current_stream().cuda_stream), "tdr_dev_draw")
    return out


def measure_peak(what):
    """what: "fp64" -> DFMA TFLOP/s, "l2" -> L2-resident copy GB/s, measured on the current device by the library's micro-benchmarks."""
    import torch
    v = C.c_double()
    _check(lib().tdr_measure_peak({"fp64": 0, "l2": 1}[what], C.byref(v), torch.cuda.current_stream().cuda_stream), "tdr_measure_peak")
    return v.value


def dev_popctrl(bank, next_cap, seed, gen_next, pr, noalloc=False):
    """Population control on a device array of 48-byte sites (torch uint8 tensor of shape [n, 48]).  Returns (next sites
    [min(total, next_cap), 48] uint8, total).  noalloc=True: the entry point that allocates nothing (static device scratch,
    at most TDR_NOALLOC_MAX_SITES sites); the output tensors are still the caller's."""
    import torch
    n = bank.shape[0]
    nxt = torch.empty((next_cap, 48), dtype=torch.uint8, device=bank.device)
    cnt = torch.zeros(1, dtype=torch.int64, device=bank.device)
    f = lib().tdr_dev_popctrl_noalloc if noalloc else lib().tdr_dev_popctrl
    _check(f(bank.data_ptr(), n, nxt.data_ptr(), next_cap, cnt.data_ptr(), seed, gen_next, float(pr), torch.cuda.current_stream().cuda_stream),
           "tdr_dev_popctrl_noalloc" if noalloc else "tdr_dev_popctrl")
    total = int(cnt.item())
    return nxt[:min(total, next_cap)], total
