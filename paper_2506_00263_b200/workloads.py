"""Seeded synthetic workloads (inputs only — none of the method's arithmetic lives here).

Both the CPU oracle (oracle/) and the CUDA library are fed from this module; it imports
neither.  The five workloads stand in for the paper's inputs, which are not available
(C5G7-TD cross sections and pin map; MC/DC's continuous-energy library and
examples/fixed_source/inf_pin_ce/input.py).  They take the *shape* of those
workloads as BASELINE.json configs[0..4] describe them; the recipe is stated in DESIGN.md
section 4.  Problem seed 0x25060263 (numpy PCG64), run seed 1.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

MAX_RINGS = 4
MAX_NUC = 4
MAX_CSURF = 6
PROBLEM_SEED = 0x25060263
INF = float("inf")


@dataclass
class Problem:
    name: str
    geometry: dict
    materials: dict
    xs: Optional[dict]
    mode: str                       # "fixed" | "k"
    n_particles: int
    n_inactive: int = 0
    n_active: int = 0
    seed: int = 1
    notes: dict = field(default_factory=dict)


def _f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _i32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.int32))


def geometry(xplanes, yplanes, zplanes, cell_univ, universes, bc, mesh=None, by_group=0,
             e_edges=None, src_kind=0, src_lo=(0, 0, 0), src_hi=(0, 0, 0), src_dir=None,
             src_energy=("group", 0), scale_log2=24, cx=None, cy=None, t_edges=None, implicit=None, surfaces=None):
    """universes: list of (radii ascending, materials innermost..background), or ("cells", [(signed surfaces, material), ...]) for a
    universe of general cells (readings C1-C6): each cell is the intersection of half-spaces of `surfaces`
    = [(kind, a, b, c, d)], kind "plane" | "sphere" | "zcyl", named +(s+1) for the side f >= 0 and -(s+1) for f < 0."""
    xp, yp, zp = _f64(xplanes), _f64(yplanes), _f64(zplanes)
    nx, ny, nz = len(xp) - 1, len(yp) - 1, len(zp) - 1
    if cx is None:
        cx = [0.5 * (xp[i] + xp[i + 1]) if np.isfinite(xp[i]) and np.isfinite(xp[i + 1]) else 0.0 for i in range(nx)]
    if cy is None:
        cy = [0.5 * (yp[i] + yp[i + 1]) if np.isfinite(yp[i]) and np.isfinite(yp[i + 1]) else 0.0 for i in range(ny)]
    nr = _i32([-1 if u[0] == "cells" else len(u[0]) for u in universes])
    rad = np.zeros((len(universes), MAX_RINGS))
    mat = np.zeros((len(universes), MAX_RINGS + 1), dtype=np.int32)
    cell0, ncell, cell_ns, cell_sf, cell_mat = np.zeros(len(universes), np.int32), np.zeros(len(universes), np.int32), [], [], []
    for k, (radii, mats) in enumerate(universes):
        if radii == "cells":
            cell0[k], ncell[k] = len(cell_ns), len(mats)
            for sf, m in mats:
                assert 1 <= len(sf) <= MAX_CSURF and all(r != 0 and abs(r) <= len(surfaces) for r in sf)
                cell_ns.append(len(sf)); cell_sf.append(list(sf) + [0] * (MAX_CSURF - len(sf))); cell_mat.append(m)
            continue
        assert len(mats) == len(radii) + 1 and len(radii) <= MAX_RINGS
        rad[k, :len(radii)] = radii
        mat[k, :len(mats)] = mats
    if mesh is None:
        mesh = ([xp[0], xp[-1]], [yp[0], yp[-1]], [zp[0], zp[-1]])
    ekind = {"group": 0, "mono": 1, "watt": 2}[src_energy[0]]
    g = dict(nx=nx, ny=ny, nz=nz, xplanes=xp, yplanes=yp, zplanes=zp, cx=_f64(cx), cy=_f64(cy),
             cell_univ=_i32(cell_univ).reshape(nz, ny, nx), bc=_i32(bc), n_univ=len(universes),
             univ_nrings=nr, univ_radius=_f64(rad), univ_mat=_i32(mat),
             mesh_n=_i32([len(mesh[0]) - 1, len(mesh[1]) - 1, len(mesh[2]) - 1]),
             mesh_x=_f64(mesh[0]), mesh_y=_f64(mesh[1]), mesh_z=_f64(mesh[2]),
             by_group=int(by_group), n_ebins=(len(e_edges) - 1 if e_edges is not None else 0),
             e_edges=_f64(e_edges if e_edges is not None else [0.0]),
             src_kind=int(src_kind), src_lo=_f64(src_lo), src_hi=_f64(src_hi),
             src_dir_kind=0 if src_dir is None else 1, src_dir=_f64(src_dir if src_dir is not None else (0, 0, 1)),
             src_energy_kind=ekind,
             src_index=int(src_energy[1]) if ekind != 1 else 0,
             src_energy=float(src_energy[1]) if ekind == 1 else 0.0,
             tally_scale_log2=int(scale_log2),
             n_tbins=(len(t_edges) - 1 if t_edges is not None else 0), t_edges=_f64(t_edges if t_edges is not None else [0.0]),
             implicit_capture=0 if implicit is None else 1, w_roulette=0.0 if implicit is None else float(implicit[0]),
             w_survive=0.0 if implicit is None else float(implicit[1]))
    if surfaces:
        kinds = {"plane": 0, "sphere": 1, "zcyl": 2}
        g.update(n_surf=len(surfaces), surf_kind=_i32([kinds[t[0]] for t in surfaces]), surf_coef=_f64([list(t[1:5]) for t in surfaces]),
                 n_cell=len(cell_ns), univ_cell0=_i32(cell0), univ_ncell=_i32(ncell), cell_nsurf=_i32(cell_ns), cell_surf=_i32(cell_sf),
                 cell_mat=_i32(cell_mat))
    return g


def mg_materials(sig_t, sig_s, sig_f, nu, chi, speed=None):
    sig_t = _f64(sig_t)
    n_mat, G = sig_t.shape
    d = dict(n_mat=n_mat, G=G, sig_t=sig_t, sig_s=_f64(sig_s).reshape(n_mat, G, G), sig_f=_f64(sig_f).reshape(n_mat, G),
             nu=_f64(nu).reshape(n_mat, G), chi=_f64(chi).reshape(n_mat, G))
    if speed is not None:
        d["speed"] = _f64(speed).reshape(G)                  # time-dependent runs: speed of each group
    return d


def ce_materials(mats):
    """mats: list of list of (nuclide index, atom density)."""
    n_mat = len(mats)
    nn = _i32([len(m) for m in mats])
    nuc = np.zeros((n_mat, MAX_NUC), dtype=np.int32)
    dens = np.zeros((n_mat, MAX_NUC))
    for k, m in enumerate(mats):
        for j, (n, d) in enumerate(m):
            nuc[k, j] = n
            dens[k, j] = d
    return dict(n_mat=n_mat, G=0, mat_nnuc=nn, mat_nuc=_i32(nuc), mat_dens=_f64(dens))


# --------------------------------------------------------------------------- pins / small problems
def infinite_medium(sig_t, sig_s, sig_f=None, nu=None, chi=None, mode="fixed", n=100000,
                    n_inactive=0, n_active=0, seed=1, by_group=0):
    """Infinite homogeneous medium, point isotropic source at the origin, group 0."""
    sig_t = np.atleast_1d(_f64(sig_t))
    G = len(sig_t)
    sig_s = _f64(sig_s).reshape(1, G, G)
    sig_f = np.zeros((1, G)) if sig_f is None else _f64(sig_f).reshape(1, G)
    nu = np.zeros((1, G)) if nu is None else _f64(nu).reshape(1, G)
    chi = np.eye(1, G) if chi is None else _f64(chi).reshape(1, G)
    geo = geometry([-INF, INF], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6, by_group=by_group)
    return Problem("infinite_medium", geo, mg_materials(sig_t.reshape(1, G), sig_s, sig_f, nu, chi), None,
                   mode, n, n_inactive, n_active, seed)


def cfg0(n=100000, seed=1):
    """configs[0]: 1-group fixed source, St=1.0, Ss=0.7, analog capture."""
    p = infinite_medium([1.0], [[0.7]], n=n, seed=seed)
    p.name = "cfg0"
    return p


def slab(sig_t, L, n=100000, seed=1):
    """Purely absorbing slab 0<x<L, mono-directional +x source at x=0, vacuum at x=L."""
    geo = geometry([0.0, L], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6,
                   src_dir=(1.0, 0.0, 0.0))
    mats = mg_materials([[sig_t]], [[[0.0]]], [[0.0]], [[0.0]], [[1.0]])
    return Problem("slab", geo, mats, None, "fixed", n, seed=seed)


def slab_mesh(sig_t, sig_s, L, axis=0, direction=(1.0, 0.0, 0.0), start=0.0, lattice=None, mesh=None, n=100000, seed=1):
    """1-group slab 0 < r[axis] < L (vacuum faces, infinite in the other two axes), mono-directional point source at
    r[axis] = start; `lattice` = interior lattice planes along the axis, `mesh` = tally planes along the axis (they need
    not coincide with the lattice planes)."""
    planes = [[-INF, INF], [-INF, INF], [-INF, INF]]
    planes[axis] = [0.0] + list(lattice or []) + [L]
    ncell = len(planes[axis]) - 1
    mp = [[-INF, INF], [-INF, INF], [-INF, INF]]
    mp[axis] = list(mesh) if mesh is not None else [0.0, L]
    src = [0.0, 0.0, 0.0]
    src[axis] = start
    geo = geometry(planes[0], planes[1], planes[2], [0] * ncell, [((), (0,))], [0] * 6, mesh=tuple(mp),
                   src_lo=tuple(src), src_dir=direction)
    mats = mg_materials([[sig_t]], [[[sig_s]]], [[0.0]], [[0.0]], [[1.0]])
    return Problem("slab_mesh", geo, mats, None, "fixed", n, seed=seed)


def two_region(kind="pin", n=200000, seed=1):
    """Volume-ratio pin: one group, the same S_t = 1.0 and S_s = 0.7 everywhere, uniform isotropic box
    source, all faces reflective, so the flux is flat; absorption in the fuel rings is booked as fission with nu = 0
    (no children), in the moderator as capture, so n_fis / (n_fis + n_abs) = fuel volume fraction.
    kind: "pin" (cfg1's cell), "lattice" (3 x 3 cells: lattice-plane crossings reset the ring), "zones" (two axial zones
    with different universes: a z crossing re-locates the ring), "rings" (two nested rings, fuel in the annulus)."""
    h, R = 0.63, 0.54
    mats = mg_materials([[1.0], [1.0]], [[[0.7]], [[0.7]]], [[0.3], [0.0]], [[0.0], [0.0]], [[1.0], [1.0]])
    pi = float(np.pi)
    if kind == "pin":
        geo = geometry([-h, h], [-h, h], [-INF, INF], [0], [((R,), (0, 1))], [1, 1, 1, 1, 0, 0],
                       src_kind=1, src_lo=(-h, -h, 0.0), src_hi=(h, h, 0.0))
        frac = pi * R * R / (4 * h * h)
    elif kind == "lattice":
        xp = [-3 * h, -h, h, 3 * h]
        geo = geometry(xp, xp, [-INF, INF], [0] * 9, [((R,), (0, 1))], [1, 1, 1, 1, 0, 0],
                       src_kind=1, src_lo=(-3 * h, -3 * h, 0.0), src_hi=(3 * h, 3 * h, 0.0))
        frac = pi * R * R / (4 * h * h)
    elif kind == "zones":
        # three zones: pin R, bare moderator (a universe without rings), thin pin R2
        R2 = 0.30
        geo = geometry([-h, h], [-h, h], [0.0, 1.0, 2.5, 3.0], [0, 1, 2], [((R,), (0, 1)), ((), (1,)), ((R2,), (0, 1))], [1] * 6,
                       src_kind=1, src_lo=(-h, -h, 0.0), src_hi=(h, h, 3.0))
        frac = (pi * R * R * 1.0 + pi * R2 * R2 * 0.5) / (4 * h * h * 3.0)
    elif kind == "rings":
        R1 = 0.25
        geo = geometry([-h, h], [-h, h], [-INF, INF], [0], [((R1, R), (1, 0, 1))], [1, 1, 1, 1, 0, 0],
                       src_kind=1, src_lo=(-h, -h, 0.0), src_hi=(h, h, 0.0))
        frac = pi * (R * R - R1 * R1) / (4 * h * h)
    elif kind == "strips":
        # two lattice cells of the SAME universe of general cells, split by the plane X = 0.2 of the cell frame: a particle that
        # goes through the lattice plane leaves the moderator strip of one cell and enters the fuel strip of the next
        geo = geometry([-1.0, 0.0, 1.0], [-1.0, 1.0], [-1.0, 1.0], [0, 0], [("cells", [((-1,), 0), ((+1,), 1)])], [1] * 6,
                       src_kind=1, src_lo=(-1.0, -1.0, -1.0), src_hi=(1.0, 1.0, 1.0), surfaces=[("plane", 1.0, 0.0, 0.0, 0.2)])
        frac = 0.7
    elif kind == "two_universes":
        # two universes of general cells side by side whose cell lists name the materials in opposite order: fuel inside the
        # sphere of the first, fuel OUTSIDE the (smaller) sphere of the second
        surf = [("sphere", 0.0, 0.0, 0.0, 0.45), ("sphere", 0.1, 0.0, 0.0, 0.3)]
        geo = geometry([-1.0, 0.0, 1.0], [-0.5, 0.5], [-0.5, 0.5], [0, 1], [("cells", [((-1,), 0), ((+1,), 1)]), ("cells", [((-2,), 1), ((+2,), 0)])],
                       [1] * 6, src_kind=1, src_lo=(-1.0, -0.5, -0.5), src_hi=(1.0, 0.5, 0.5), surfaces=surf)
        frac = (4.0 / 3.0 * pi * 0.45 ** 3 + (1.0 - 4.0 / 3.0 * pi * 0.3 ** 3)) / 2.0
    elif kind in ("sphere", "halfspace", "offcyl", "shell", "lens", "lattice_cells"):
        # general cells (readings C1-C6): "fuel" (material 0) is a cell, or several, of a universe of general cells
        c = 1.0                                                # half width of the cube; z is finite here (spheres)
        box = dict(bc=[1] * 6, src_kind=1, src_lo=(-c, -c, -c), src_hi=(c, c, c))
        if kind == "sphere":                                   # a sphere off the cell centre
            surf = [("sphere", 0.1, -0.2, 0.15, 0.7)]
            cells = [((-1,), 0), ((+1,), 1)]
            frac = 4.0 / 3.0 * pi * 0.7 ** 3 / 8.0
        elif kind == "halfspace":                              # an oblique plane X + 2Y + 2Z = 0.9 (unit normal times 3)
            surf = [("plane", 1.0, 2.0, 2.0, 0.9)]
            cells = [((-1,), 0), ((+1,), 1)]
            frac = None                                        # by quadrature in the test
        elif kind == "offcyl":                                 # a z-cylinder whose axis is not the cell's
            surf = [("zcyl", 0.25, -0.3, 0.0, 0.6)]
            cells = [((+1,), 1), ((-1,), 0)]                   # (cell order must not matter)
            frac = pi * 0.36 * 2.0 / 8.0
        elif kind == "shell":                                  # fuel = the shell between two concentric spheres, cut by a plane
            surf = [("sphere", 0.0, 0.0, 0.0, 0.4), ("sphere", 0.0, 0.0, 0.0, 0.9), ("plane", 0.0, 0.0, 1.0, 0.0)]
            cells = [((-1,), 1), ((+1, -2, +3), 0), ((+1, -2, -3), 1), ((+2,), 1)]
            frac = 0.5 * 4.0 / 3.0 * pi * (0.9 ** 3 - 0.4 ** 3) / 8.0
        elif kind == "lens":                                   # fuel = the intersection of two spheres (two surfaces met at once on its rim)
            surf = [("sphere", -0.3, 0.0, 0.0, 0.7), ("sphere", 0.3, 0.0, 0.0, 0.7)]
            cells = [((-1, -2), 0), ((-1, +2), 1), ((+1, -2), 1), ((+1, +2), 1)]
            hcap = 0.7 - 0.3
            frac = 2.0 * (pi * hcap * hcap * (3 * 0.7 - hcap) / 3.0) / 8.0
        else:                                                  # 2 x 2 lattice: general cells next to a ring universe
            surf = [("sphere", 0.0, 0.0, 0.0, 0.45)]
            cells = [((-1,), 0), ((+1,), 1)]
            geo = geometry([-1.0, 0.0, 1.0], [-1.0, 0.0, 1.0], [-0.5, 0.5], [0, 1, 1, 0], [("cells", cells), ((0.3,), (0, 1))], [1] * 6,
                           src_kind=1, src_lo=(-1.0, -1.0, -0.5), src_hi=(1.0, 1.0, 0.5), surfaces=surf)
            frac = (2 * 4.0 / 3.0 * pi * 0.45 ** 3 + 2 * pi * 0.09 * 1.0) / 4.0
        if kind != "lattice_cells":
            geo = geometry([-c, c], [-c, c], [-c, c], [0], [("cells", cells)], surfaces=surf, **box)
    else:
        raise ValueError(kind)
    p = Problem("two_region_" + kind, geo, mats, None, "fixed", n, seed=seed)
    p.notes["fuel_volume_fraction"] = frac
    return p


def ce_two_nuclide_medium(order=(0, 1), mode="k", n=20000, n_inactive=3, n_active=17, seed=1, scatter=True, n_ebins=None):
    """Infinite medium of two nuclides with energy-independent cross sections (CE collision pin): nuclide 0 = scatterer /
    absorber (A = 12), nuclide 1 = fissile (A = 200, nu = 2, Watt a = 0.9e6, b = 2.0e-6).  `order` = the order in which
    the material lists them (results must not depend on it statistically)."""
    n_grid = 64
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    E[0], E[-1] = 1e-5, 2e7
    s = np.array([[2.0], [1.0]]) * (1.0 if scatter else 0.0) * np.ones((2, n_grid))
    c = np.array([[1.0], [0.5]]) * np.ones((2, n_grid))
    f = np.array([[0.0], [1.5]]) * np.ones((2, n_grid))
    xs = dict(n_grid=n_grid, n_nuc=2, energy=_f64(E), A=_f64([12.0, 200.0]), sig_s=_f64(s), sig_c=_f64(c), sig_f=_f64(f),
              nu=_f64([0.0, 2.0]), watt_a=_f64([1.0, 0.9e6]), watt_b=_f64([1.0, 2.0e-6]))
    dens = {0: 0.5, 1: 0.3}
    edges = [1e-5, 2e7] if n_ebins is None else n_ebins
    geo = geometry([-INF, INF], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6, e_edges=edges,
                   src_energy=("watt", 1) if mode == "k" else ("mono", 1e6))
    mats = ce_materials([[(order[0], dens[order[0]]), (order[1], dens[order[1]])]])
    p = Problem("ce_two_nuclide", geo, mats, xs, mode, n, n_inactive, n_active, seed)
    p.notes.update(N=dens, sig_s=(2.0 if scatter else 0.0, 1.0 if scatter else 0.0), sig_c=(1.0, 0.5), sig_f=(0.0, 1.5), nu=2.0,
                   watt=(0.9e6, 2.0e-6))
    return p


def ce_lerp_absorber(E0, n=100000, seed=1):
    """Pure absorber whose capture cross section is tabulated on a COARSE grid, mono-energetic source between grid points
    (or outside the grid): pins the X2 interpolation and clamping.  sigma_c = 8, 2, 4, 1 b at 1, 10, 100, 1000 eV; N = 0.4."""
    xs = dict(n_grid=4, n_nuc=1, energy=_f64([1.0, 10.0, 100.0, 1000.0]), A=_f64([10.0]), sig_s=_f64(np.zeros((1, 4))),
              sig_c=_f64([[8.0, 2.0, 4.0, 1.0]]), sig_f=_f64(np.zeros((1, 4))), nu=_f64([0.0]), watt_a=_f64([1.0]), watt_b=_f64([1.0]))
    geo = geometry([-INF, INF], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6, e_edges=[1e-3, 1e5],
                   src_energy=("mono", E0))
    return Problem("ce_lerp_absorber", geo, ce_materials([[(0, 0.4)]]), xs, "fixed", n, seed=seed)


def td_medium(sig_t, sig_s, speed, t_edges, sig_f=0.0, nu=0.0, n=100000, seed=1):
    """Time-dependent pin: one-group infinite medium, point source at t_edges[0], time-mesh tally, census at
    t_edges[-1].  With removal rate S_a v the population is N(t) = exp(-S_a v t) (k_inf = 0), so the track length in a time
    bin and the census fraction have closed forms."""
    geo = geometry([-INF, INF], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6, t_edges=t_edges)
    mats = mg_materials([[sig_t]], [[[sig_s]]], [[sig_f]], [[nu]], [[1.0]], speed=[speed])
    return Problem("td_medium", geo, mats, None, "fixed", n, seed=seed)


def td_ce_absorber(E0, t_edges, n=100000, seed=1):
    """Continuous-energy pure absorber (sigma_c = 2 b flat, N = 0.5), mono-energetic source: pins the speed law v(E)."""
    xs = dict(n_grid=4, n_nuc=1, energy=_f64([1e-5, 1.0, 1e3, 2e7]), A=_f64([10.0]), sig_s=_f64(np.zeros((1, 4))),
              sig_c=_f64(np.full((1, 4), 2.0)), sig_f=_f64(np.zeros((1, 4))), nu=_f64([0.0]), watt_a=_f64([1.0]), watt_b=_f64([1.0]))
    geo = geometry([-INF, INF], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6, e_edges=[1e-5, 2e7],
                   src_energy=("mono", E0), t_edges=t_edges)
    return Problem("td_ce_absorber", geo, ce_materials([[(0, 0.5)]]), xs, "fixed", n, seed=seed)


def cfg3_td(n=1000000, n_tbins=128, t_max=3.0e-6, seed=1, n_grid=50000, sigf0=None):
    """The paper's own continuous-energy experiment: the infinite pin cell with a uniform 14 MeV source
    at t = 0, a time-mesh tally of 1 ... 128 bins and a census at t_max.  One energy bin."""
    geo, mats, xs = _ce_pin(1, n_grid, ("mono", 14e6), CE_SIGF0 if sigf0 is None else sigf0)
    geo["n_tbins"] = int(n_tbins)
    geo["t_edges"] = _f64(np.linspace(0.0, t_max, n_tbins + 1))
    return Problem("cfg3_td", geo, mats, xs, "fixed", n, seed=seed)


def with_implicit_capture(problem, w_roulette=0.25, w_survive=0.5):
    """The same fixed-source problem with implicit capture and weight roulette (readings W1-W4)."""
    assert problem.mode == "fixed"
    problem.geometry.update(implicit_capture=1, w_roulette=float(w_roulette), w_survive=float(w_survive))
    problem.name += "_ic"
    return problem


def _mg_material(rng, G, kind):
    """One synthetic G-group material (recipe: DESIGN.md section 4, cfg1)."""
    sig_t = rng.uniform(0.2, 2.0, G)
    c = rng.uniform(0.50, 0.90, G) if kind == "fuel" else rng.uniform(0.90, 0.995, G)
    P = np.zeros((G, G))
    for g in range(G):
        if g >= 4:
            P[g, g - 1] = 0.05 * rng.uniform()
        P[g, g] = 1.0
        for j in range(1, G - g):
            P[g, g + j] = 0.5 ** j * rng.uniform(0.5, 1.0)
        P[g] /= P[g].sum()
    sig_s = (c * sig_t)[:, None] * P
    sig_a = sig_t - sig_s.sum(axis=1)
    if kind == "fuel":
        sig_f = rng.uniform(0.3, 0.7, G) * sig_a
        nu = rng.uniform(2.3, 2.7, G)
    elif kind == "chamber":
        sig_f = 0.01 * sig_a
        nu = np.full(G, 2.4)
    else:
        sig_f = np.zeros(G)
        nu = np.zeros(G)
    chi = np.zeros(G)
    chi[:3] = (0.60, 0.30, 0.10)
    return sig_t, sig_s, sig_f, nu, chi


def _mg_set(kinds, G=7, seed=PROBLEM_SEED):
    rng = np.random.default_rng(seed)
    parts = [_mg_material(rng, G, k) for k in kinds]
    return mg_materials(*[np.stack([p[i] for p in parts]) for i in range(5)])


def cfg1(n=1000000, n_inactive=20, n_active=50, seed=1, identical_materials=False):
    """configs[1]: 7-group k-eigenvalue 2-D pin cell, reflective."""
    h = 0.63
    geo = geometry([-h, h], [-h, h], [-INF, INF], [0], [((0.54,), (0, 1))], [1, 1, 1, 1, 0, 0],
                   by_group=1, src_kind=1, src_lo=(-h, -h, 0.0), src_hi=(h, h, 0.0))
    mats = _mg_set(["fuel", "fuel"] if identical_materials else ["fuel", "mod"])
    if identical_materials:
        for k in ("sig_t", "sig_s", "sig_f", "nu", "chi"):
            mats[k][1] = mats[k][0]
    return Problem("cfg1", geo, mats, None, "k", n, n_inactive, n_active, seed)


def general_cells(mode="k", n=40003, n_inactive=1, n_active=2, seed=1, n_ebins=None):
    """Universes of general cells (readings C1-C6) in a k-eigenvalue or fixed-source run: a 2 x 2 x 2 lattice with
    vacuum on +x, +z and reflection elsewhere; universe 0 = a fuel sphere cut by an oblique plane (two fuel cells) inside
    moderator, universe 1 = cfg1's ring pin, universe 2 = a fuel lens (two spheres) beside an off-axis guide cylinder.
    7-group materials of cfg1; with n_ebins the continuous-energy pin cell of cfg3 / cfg4 in the same geometry."""
    surf = [("sphere", 0.05, -0.04, 0.0, 0.5), ("plane", 1.0, 1.0, 2.0, 0.1),                   # universe 0
            ("sphere", -0.15, 0.0, 0.1, 0.42), ("sphere", 0.15, 0.0, 0.1, 0.42), ("zcyl", 0.0, 0.52, 0.0, 0.08)]   # universe 2
    u0 = ("cells", [((-1, -2), 0), ((-1, +2), 0), ((+1,), 1)])
    u2 = ("cells", [((-3, -4), 0), ((-5,), 1), ((+3, +4, +5), 1), ((-3, +4), 1), ((+3, -4), 1)])
    xp = [-0.63, 0.63, 1.89]; zp = [-0.6, 0.6, 1.8]
    cu = [0, 1, 2, 0, 1, 2, 0, 1]
    kw = dict(src_kind=1, src_lo=(xp[0], xp[0], zp[0]), src_hi=(xp[-1], xp[-1], zp[-1]), surfaces=surf, mesh=(xp, xp, [zp[0], zp[-1]]))
    bc = [1, 0, 1, 1, 1, 0]
    universes = [u0, ((0.54,), (0, 1)), u2]
    if n_ebins is None:
        geo = geometry(xp, xp, zp, cu, universes, bc, by_group=1, **kw)
        return Problem("general_cells_" + mode, geo, _mg_set(["fuel", "mod"]), None, mode, n, n_inactive if mode == "k" else 0, n_active if mode == "k" else 0, seed)
    base = cfg4(n=n, n_inactive=n_inactive, n_active=n_active, seed=seed, n_ebins=n_ebins) if mode == "k" else cfg3(n=n, n_ebins=n_ebins, seed=seed)
    g0 = base.geometry
    geo = geometry(xp, xp, zp, cu, universes, bc, e_edges=g0["e_edges"], src_energy=("watt", 2) if mode == "k" else ("mono", 14.0e6), **kw)
    return Problem("general_cells_ce_" + mode, geo, base.materials, base.xs, mode, n, base.n_inactive, base.n_active, seed)


def cfg2(n=10000000, n_inactive=6, n_active=18, seed=1):
    """configs[2]: 7-group k-eigenvalue, 3-D 2x2 assemblies in C5G7 *shape* (own pin rule)."""
    pitch, npin = 1.26, 51
    xp = np.arange(npin + 1) * pitch
    zp = [0.0, 64.26, 85.68]
    # materials: 0..3 fuels A-D, 4 guide tube, 5 fission chamber, 6 moderator
    mats = _mg_set(["fuel", "fuel", "fuel", "fuel", "mod", "chamber", "mod"])
    universes = [((0.54,), (m, 6)) for m in range(6)] + [((), (6,))]
    MOD = 6
    cu = np.full((2, npin, npin), MOD, dtype=np.int32)
    for ay in range(2):
        for ax in range(2):
            for j in range(17):
                for i in range(17):
                    if (i, j) == (8, 8):
                        u = 5
                    elif i in (2, 5, 8, 11, 14) and j in (2, 5, 8, 11, 14):
                        u = 4
                    elif ax == ay:
                        u = 0
                    else:
                        t = min(i, j, 16 - i, 16 - j)
                        u = 1 if t == 0 else (2 if t <= 3 else 3)
                    cu[0, ay * 17 + j, ax * 17 + i] = u
    mz = np.linspace(0.0, 85.68, 10)
    mz[-1] = 85.68
    geo = geometry(xp, xp, zp, cu, universes, [1, 0, 1, 0, 1, 0], mesh=(xp, xp, mz), by_group=0,
                   src_kind=1, src_lo=(0.0, 0.0, 0.0), src_hi=(42.84, 42.84, 64.26))
    return Problem("cfg2", geo, mats, None, "k", n, n_inactive, n_active, seed)


# --------------------------------------------------------------------------- continuous energy
def ce_tables(n_grid=50000, n_res=200, sigf0=2.5, res_fis=0.05, seed=PROBLEM_SEED):
    """3 synthetic nuclides (A=1,16,238) on a log grid 1e-5 eV .. 2e7 eV."""
    rng = np.random.default_rng(seed + 1)
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    E[0], E[-1] = 1e-5, 2e7
    inv_v = np.sqrt(0.0253 / E)
    z = np.zeros(n_grid)
    s = [np.full(n_grid, 20.0), np.full(n_grid, 3.8), np.full(n_grid, 9.0)]
    c = [0.332 * inv_v, 1e-4 * inv_v, 2.7 * inv_v]
    f = [z.copy(), z.copy(), sigf0 * inv_v + 0.3 * (E > 1e6)]
    lo, hi = np.searchsorted(E, 1.0), np.searchsorted(E, 1e3)
    idx = rng.integers(lo, hi, n_res)
    gg = 0.023
    for Er, xi in zip(E[idx], rng.uniform(size=n_res)):
        gn = 2e-3 * (0.1 + 2 * xi * xi) * np.sqrt(Er)
        gt = gn + gg
        s0 = 2.608e6 / Er * (gn / gt)
        x = 2.0 * (E - Er) / gt
        lor = 1.0 / (1.0 + x * x)
        s[2] = s[2] + s0 * (gn / gt) * lor
        cap = s0 * (gg / gt) * np.sqrt(Er / E) * lor
        c[2] = c[2] + cap
        f[2] = f[2] + res_fis * cap
    return dict(n_grid=n_grid, n_nuc=3, energy=_f64(E), A=_f64([1.0, 16.0, 238.0]),
                sig_s=_f64(np.stack(s)), sig_c=_f64(np.stack(c)), sig_f=_f64(np.stack(f)),
                nu=_f64([0.0, 0.0, 2.43]), watt_a=_f64([1.0, 1.0, 0.988e6]), watt_b=_f64([1.0, 1.0, 2.249e-6]))


def _ce_pin(n_ebins, n_grid, src_energy, sigf0, res_fis=None):
    h = 0.63
    xs = ce_tables(n_grid=n_grid, sigf0=sigf0, res_fis=CE_RES_FIS if res_fis is None else res_fis)
    E = xs["energy"]
    edges = E[np.round(np.arange(n_ebins + 1) * (n_grid - 1) / n_ebins).astype(int)]
    geo = geometry([-h, h], [-h, h], [-INF, INF], [0], [((0.54,), (0, 1))], [1, 1, 1, 1, 0, 0],
                   e_edges=edges, src_kind=1, src_lo=(-h, -h, 0.0), src_hi=(h, h, 0.0), src_energy=src_energy)
    mats = ce_materials([[(2, 0.022), (1, 0.044)], [(0, 0.0668), (1, 0.0334)]])
    return geo, mats, xs


CE_RES_FIS = 0.4
CE_SIGF0 = 8.0   # thermal fission scale of the A=238 nuclide, tuned so k_inf < 1 (reading Q17)


def cfg3(n=1000000, n_ebins=100, seed=1, n_grid=50000, sigf0=CE_SIGF0):
    """configs[3]: continuous-energy infinite pin cell, fixed 14 MeV source, energy-mesh tally."""
    geo, mats, xs = _ce_pin(n_ebins, n_grid, ("mono", 14e6), sigf0)
    return Problem("cfg3", geo, mats, xs, "fixed", n, seed=seed)


def cfg4(n=100000000, n_inactive=1, n_active=2, n_ebins=100, seed=1, n_grid=50000, sigf0=CE_SIGF0):
    """configs[4]: the same pin cell in k-eigenvalue mode (generation-0 source: Watt of nuclide 2)."""
    geo, mats, xs = _ce_pin(n_ebins, n_grid, ("watt", 2), sigf0)
    return Problem("cfg4", geo, mats, xs, "k", n, n_inactive, n_active, seed)


def ce_slowing_down(A=1.0, n=100000, n_grid=2000, seed=1, n_ebins=7):
    """Pure scatterer of mass A (tiny 1/v capture), infinite medium, 1 MeV source: kinematics pin."""
    E = np.exp(np.linspace(np.log(1e-5), np.log(2e7), n_grid))
    xs = dict(n_grid=n_grid, n_nuc=1, energy=_f64(E), A=_f64([A]), sig_s=_f64(np.full((1, n_grid), 20.0)),
              sig_c=_f64(np.zeros((1, n_grid))), sig_f=_f64(np.zeros((1, n_grid))),
              nu=_f64([0.0]), watt_a=_f64([1.0]), watt_b=_f64([1.0]))
    xs["sig_c"][0, :200] = 1e6        # absorb once thermal so histories end
    edges = 10.0 ** np.arange(-1, n_ebins)            # decade bins 0.1 eV .. 1e6 eV
    geo = geometry([-INF, INF], [-INF, INF], [-INF, INF], [0], [((), (0,))], [0] * 6, e_edges=edges,
                   src_energy=("mono", 1e6))
    return Problem("ce_slowing_down", geo, ce_materials([[(0, 0.05)]]), xs, "fixed", n, seed=seed)


BY_NAME = {"cfg0": cfg0, "cfg1": cfg1, "cfg2": cfg2, "cfg3": cfg3, "cfg4": cfg4}
