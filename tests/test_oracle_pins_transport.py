"""Pins of the oracle's TRANSPORT loop against things other than itself (second table).

What each one fixes (oracle/orc.c line ranges in DESIGN.md section 5):
  * volume-ratio pins           -> ring / material bookkeeping after cylinder, lattice-plane and zone crossings (G7)
  * azimuth pins                -> the rotation of the CE scatter about the incoming direction, both branches (T6)
  * two-nuclide medium          -> nuclide and reaction selection, CE nu*Sigma_f, fission multiplicity, Watt birth from a site
  * absorbing slab with a mesh  -> mesh-plane distances, mesh index updates, per-bin track-length flux (closed form)
  * scattering slab vs Peierls  -> isotropic scatter + both leak faces + per-bin flux and collisions, against a deterministic
                                   collision-probability solution of the slab integral equation (scipy E_n functions)
  * Kolmogorov-Smirnov          -> the per-history path length is exactly Exp(Sigma_a)
  * Python replay with geometry -> every segment of 100 pin-cell histories recomputed from the raw draws (P12 i)
  * fission chains              -> fixed-source secondaries (LIFO stack, derive_id tags, depth cap)
CPU only.
"""
import ctypes as C
import math

import numpy as np
import pytest
from scipy import special, stats

from oracle import orc
from paper_2506_00263_b200 import workloads as W

L = orc.lib()
S24 = float(2 ** 24)


# ------------------------------------------------------------------ G7: ring / material bookkeeping
@pytest.mark.parametrize("kind", ["pin", "lattice", "zones", "rings"])
def test_flat_flux_absorption_splits_by_volume(kind):
    """Same S_t and S_s everywhere + uniform source + reflective faces => flat flux, so the share of absorptions that
    happen inside the fuel rings (booked as nu = 0 fissions) is the fuel volume fraction pi r^2 / p^2.  A ring that is
    not updated at a cylinder crossing, not reset at a lattice-plane crossing or not re-located at a zone crossing
    moves this share by many sigma."""
    n = 200000
    p = W.two_region(kind, n=n)
    r = orc.run(p)
    T = r["totals"]
    assert T["n_born"] == n and T["n_sites"] == 0 and T["n_leak"] == 0 and T["n_fis"] + T["n_abs"] == n
    f = p.notes["fuel_volume_fraction"]
    assert abs(T["n_fis"] / n - f) < 4 * math.sqrt(f * (1 - f) / n), (kind, T["n_fis"] / n, f)
    # and the flat flux itself: track length per source = 1 / S_a
    assert abs(r["flux"][0] / S24 / n - 1 / 0.3) < 4 * (1 / 0.3) / math.sqrt(n)
    assert T["n_cross"] > n


# ------------------------------------------------------------------ T6: CE scatter rotation
def _frame(d):
    """Any right-handed orthonormal pair perpendicular to d (Gram-Schmidt against the axis least aligned with d)."""
    d = np.asarray(d, float)
    a = np.eye(3)[int(np.argmin(np.abs(d)))]
    e1 = a - (a @ d) * d
    e1 /= np.linalg.norm(e1)
    return e1, np.cross(d, e1)


@pytest.mark.parametrize("din", [(0.6, 0.0, 0.8), (0.36, -0.48, 0.8), (-0.7, 0.1, -0.7071067811865476), (1.0, 0.0, 0.0),
                                 (0.0, 0.0, 1.0), (0.0, 0.0, -1.0), (3e-6, -4e-6, 1.0), (6e-6, 8e-6, -1.0)])
@pytest.mark.parametrize("A", [1.0, 16.0])
def test_ce_scatter_azimuth_is_uniform_about_the_incoming_direction(din, A):
    """For a FIXED incoming direction the outgoing one must have (i) polar cosine exactly mu_lab of the two-body
    kinematics about it and (ii) a uniform azimuth about it — including the |w| ~ 1 branch of the rotation.  A swapped
    component or a wrong sign in either branch breaks (i) or skews (ii)."""
    d = np.array(din, float)
    d /= np.linalg.norm(d)
    e1, e2 = _frame(d)
    n = 20000
    di = (C.c_double * 3)(*d)
    Eo, do = C.c_double(), (C.c_double * 3)()
    phi = np.empty(n)
    # T6 treats a direction with 1 - w^2 <= 1e-10 as exactly +-z (polar cosine then off by up to ~1e-5), and just above
    # that switch 1 - w*w loses ~6 digits to cancellation
    tol_mu = 1e-12 if (1.0 - d[2] * d[2] > 1e-6 or d[0] == d[1] == 0.0) else 2e-5
    for i in range(n):
        L.orc_scatter_ce(21, i, 0, 3, A, 1.0e6, di, C.byref(Eo), do)
        o = np.array(do[:])
        mu_cm = 2.0 * L.orc_draw(21, i, 0, 3, 2, 0) - 1.0                    # purpose 2 = ENERGY, j = 0
        mu_lab = (1.0 + A * mu_cm) / math.sqrt(A * A + 2.0 * A * mu_cm + 1.0)
        assert abs(o @ o - 1.0) < 1e-14
        assert abs(o @ d - mu_lab) < tol_mu, (i, o @ d, mu_lab)
        assert abs(Eo.value / 1.0e6 - (A * A + 2.0 * A * mu_cm + 1.0) / (A + 1.0) ** 2) < 1e-14
        phi[i] = math.atan2(o @ e2, o @ e1)
    tol = 4 * math.sqrt(0.5 / n)
    for k in (1, 2, 3):
        assert abs(np.cos(k * phi).mean()) < tol and abs(np.sin(k * phi).mean()) < tol, (din, k)
    assert stats.kstest((phi + math.pi) / (2 * math.pi), "uniform").pvalue > 1e-3


# ------------------------------------------------------------------ T6: CE nuclide / reaction selection, nu, Watt at birth
def _two_nuclide_expect(p):
    N, ss, sc, sf = p.notes["N"], p.notes["sig_s"], p.notes["sig_c"], p.notes["sig_f"]
    St = sum(N[i] * (ss[i] + sc[i] + sf[i]) for i in (0, 1))
    return dict(St=St, cap=sum(N[i] * sc[i] for i in (0, 1)) / St, fis=sum(N[i] * sf[i] for i in (0, 1)) / St,
                sca=sum(N[i] * ss[i] for i in (0, 1)) / St, kinf=N[1] * p.notes["nu"] * sf[1] / sum(N[i] * (sc[i] + sf[i]) for i in (0, 1)))


@pytest.mark.parametrize("order", [(0, 1), (1, 0)])
def test_ce_two_nuclide_medium_reaction_rates_and_kinf(order):
    """Energy-independent cross sections: capture / fission / scatter shares of all collisions are N sigma_x / S_t summed
    over the nuclides, collisions per history S_t / S_a, k_inf = N nu sigma_f / S_a.  A wrong nuclide (order, running sum),
    swapped sigma_c / sigma_f, or nu of the wrong nuclide each move one of them by many sigma."""
    p = W.ce_two_nuclide_medium(order=order, n=40000, n_inactive=2, n_active=18)
    r = orc.run(p)
    e = _two_nuclide_expect(p)
    T = r["totals"]
    nc, nh = T["n_coll"], T["n_born"]
    for got, ref in ((T["n_abs"] / nc, e["cap"]), (T["n_fis"] / nc, e["fis"]), (1 - (T["n_abs"] + T["n_fis"]) / nc, e["sca"])):
        assert abs(got - ref) < 4 * math.sqrt(ref * (1 - ref) / nc), (got, ref)
    pa = e["cap"] + e["fis"]                                       # collisions per history: geometric
    assert abs(nc / nh - 1 / pa) < 4 * math.sqrt((1 - pa) / pa ** 2 / nh)
    assert abs(r["k_mean"] - e["kinf"]) < 4 * r["k_std"] and r["k_std"] < 0.005
    # fission multiplicity floor(nu / k_prev + xi): sites per fission averaged over a generation = nu / k_prev
    g = len(r["gen_k"]) - 1
    assert abs(r["gen_pc"].sum() / r["gen_p"].sum() - 1) < 0.01    # collision estimator of k agrees (P7)
    assert abs(T["n_sites"] / T["n_fis"] - np.mean(p.notes["nu"] / np.concatenate([[1.0], r["gen_k"][:g]]))) < 0.02
    assert T["n_born"] == T["n_abs"] + T["n_fis"] == int(r["gen_n"].sum())


@pytest.mark.parametrize("E0,sigma", [(32.5, 2.5), (4.6, 5.6), (550.0, 2.5), (5000.0, 1.0), (0.5, 8.0)])
def test_ce_cross_section_interpolation_and_clamping(E0, sigma):
    """X2: linear interpolation between the two bracketing grid points, constant extrapolation outside the grid.  In a
    pure absorber the mean path is 1 / (N sigma(E0)) with sigma(E0) worked out by hand from the 4-point table."""
    n = 100000
    r = orc.run(W.ce_lerp_absorber(E0, n=n))
    mean = 1.0 / (0.4 * sigma)
    assert abs(r["flux"][0] / S24 / n - mean) < 4 * mean / math.sqrt(n)
    assert r["totals"]["n_abs"] == r["totals"]["n_coll"] == n


def test_tally_overflow_is_an_error_not_a_wrap():
    """N5: a fixed-point sum that leaves int64 is ORC_EOVERFLOW (-6)."""
    p = W.infinite_medium([1e-4], [[0.0]], n=100000)
    p.geometry["tally_scale_log2"] = 40                       # 1e5 histories x 1e4 cm x 2^40 = 1.1e21 > 2^63
    with pytest.raises(RuntimeError, match="-6"):
        orc.run(p)


def _watt_cdf(a, b, edges):
    E = np.linspace(0.0, 40e6, 2000001)
    pdf = np.exp(-E / a) * np.sinh(np.sqrt(b * E))
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (pdf[1:] + pdf[:-1]) * np.diff(E))])
    return np.interp(edges, E, cdf / cdf[-1])


@pytest.mark.parametrize("order", [(0, 1), (1, 0)])
def test_births_from_fission_sites_have_the_fissioned_nuclides_watt_spectrum(order):
    """No scattering: every history flies once at its birth energy, so the track-length flux per energy bin is the birth
    spectrum.  In generations >= 1 all births come from bank sites, whose `src` names the fissioned nuclide (index 1, listed
    SECOND in the problem's nuclide table): bin shares must follow Watt(a_1, b_1) (numerical integral of the density)."""
    edges = [1e-5, 0.3e6, 1.0e6, 2.0e6, 4.0e6, 2e7]
    p = W.ce_two_nuclide_medium(order=order, n=60000, n_inactive=1, n_active=4, scatter=False, n_ebins=edges)
    r = orc.run(p)
    f = r["flux"].astype(float)
    share = f / f.sum()
    a, b = p.notes["watt"]
    ref = np.diff(_watt_cdf(a, b, np.array(edges)))
    nh = int(r["gen_n"][1:].sum())
    assert np.all(np.abs(share - ref) < 4 * np.sqrt(ref * (1 - ref) / nh) * 1.5 + 1e-4), (share, ref)
    assert r["totals"]["n_seg"] == r["totals"]["n_coll"] == r["totals"]["n_born"]


# ------------------------------------------------------------------ mesh tally: closed form in an absorbing slab
@pytest.mark.parametrize("axis,direction,start", [(0, (1.0, 0.0, 0.0), 0.0), (0, (-1.0, 0.0, 0.0), 2.0), (1, (0.0, 1.0, 0.0), 0.0),
                                                  (2, (0.0, 0.0, -1.0), 2.0), (0, (0.6, 0.8, 0.0), 0.0), (2, (0.28, -0.0, 0.96), 0.0)])
def test_absorbing_slab_flux_per_mesh_bin(axis, direction, start):
    """Uncollided beam in a pure absorber: track length per source in mesh bin [a, b] (along the beam's axis component c)
    is (exp(-S a/|c|) - exp(-S b/|c|)) / S, measured from the entry face.  The mesh planes do not coincide with the lattice
    planes (three lattice cells, seven uneven mesh bins), so mesh and lattice crossings interleave."""
    S, Lx, n = 1.3, 2.0, 100000
    mesh = [0.0, 0.11, 0.4, 0.75, 1.0, 1.31, 1.9, 2.0]
    p = W.slab_mesh(S, 0.0, Lx, axis=axis, direction=direction, start=start, lattice=[0.5, 1.25], mesh=mesh, n=n)
    r = orc.run(p)
    c = abs(direction[axis])
    edges = np.array(mesh) if direction[axis] > 0 else Lx - np.array(mesh)
    ref = np.abs(np.diff(np.exp(-S * edges / c))) / S
    got = r["flux"] / S24 / n
    width = np.diff(mesh) / c
    assert np.all(np.abs(got - ref) < 4 * np.sqrt(width * ref / n) + 1e-7), (got, ref)
    t = math.exp(-S * Lx / c)
    face = 2 * axis + (1 if direction[axis] > 0 else 0)
    assert abs(r["leak"][face] / n - t) < 4 * math.sqrt(t * (1 - t) / n) and r["leak"].sum() == r["leak"][face]
    assert int(r["coll"].sum()) == r["totals"]["n_coll"] << 24 == r["totals"]["n_abs"] << 24


# ------------------------------------------------------------------ scattering slab vs the slab integral equation
def _slab_collision_probability(St, c, Lx, ncell=2000):
    """Deterministic reference: normally incident beam on a slab with isotropic scattering (ratio c).  Collisions per
    source in fine cells solve C = C0 + c P C with first-flight collision probabilities from exponential integrals E3
    (flat source per cell, error O(h^2))."""
    x = np.linspace(0.0, Lx, ncell + 1)
    tau = St * np.diff(x)                                    # optical widths
    t0, t1 = St * x[:-1], St * x[1:]                         # optical positions of the cell edges
    E3 = lambda z: special.expn(3, np.maximum(z, 0.0))
    C0 = np.exp(-t0) - np.exp(-t1)
    # P[i, j] = probability that a neutron emitted isotropically and uniformly in cell j collides next in cell i
    P = np.empty((ncell, ncell))
    for j in range(ncell):
        d = np.where(np.arange(ncell) > j, t0 - t1[j], t0[j] - t1)       # optical gap between cell i and cell j
        d = np.maximum(d, 0.0)
        P[:, j] = (E3(d) - E3(d + tau) - E3(d + tau[j]) + E3(d + tau + tau[j])) / (2.0 * tau[j])
        P[j, j] = 1.0 - (1.0 - 2.0 * E3(tau[j])) / (2.0 * tau[j])
    Ct = np.linalg.solve(np.eye(ncell) - c * P, C0)
    escR = (E3(St * Lx - t1) - E3(St * Lx - t0)) / (2.0 * tau)
    escL = (E3(t0) - E3(t1)) / (2.0 * tau)
    T = math.exp(-St * Lx) + c * float(escR @ Ct)
    R = c * float(escL @ Ct)
    return x, Ct, T, R


def test_scattering_slab_matches_the_integral_transport_solution():
    """Isotropic scattering in a finite slab has no closed form, but the slab integral equation can be solved to 1e-6
    deterministically.  Pins, together: the isotropic direction law (the E_n kernels are its angular integrals), plane
    distances in both directions, both leak faces, the scatter / capture split, and the per-bin flux and collision tallies
    on a mesh that does not coincide with the lattice planes."""
    St, c, Lx, n = 1.0, 0.8, 2.0, 400000
    mesh = [0.0, 0.11, 0.4, 0.75, 1.0, 1.31, 1.9, 2.0]
    p = W.slab_mesh(St, c * St, Lx, lattice=[0.5, 1.25], mesh=mesh, n=n)
    r = orc.run(p)
    x, Ct, T, R = _slab_collision_probability(St, c, Lx)
    A = 1.0 - T - R
    assert abs((1 - c) * Ct.sum() - A) < 1e-5                                 # the reference balances
    for got, ref in ((r["leak"][1] / n, T), (r["leak"][0] / n, R), (r["totals"]["n_abs"] / n, A)):
        assert abs(got - ref) < 4 * math.sqrt(ref * (1 - ref) / n), (got, ref)
    cum = np.concatenate([[0.0], np.cumsum(Ct)])
    ref_bin = np.diff(np.interp(mesh, x, cum))                                # collisions per source per mesh bin
    coll = r["coll"] / S24 / n
    flux = r["flux"] / S24 / n
    # per-history collision counts in a bin are small integers with variance < ~3x the mean here
    assert np.all(np.abs(coll - ref_bin) < 4 * np.sqrt(3 * ref_bin / n)), (coll, ref_bin)
    assert np.all(np.abs(flux - ref_bin / St) < 4 * np.sqrt(3 * ref_bin / n) / St), (flux, ref_bin / St)
    assert abs(r["totals"]["n_coll"] / n - Ct.sum()) < 4 * math.sqrt(3 * Ct.sum() / n)


# ------------------------------------------------------------------ P2: the path length of a history is Exp(S_a)
def test_path_length_per_history_is_exponential_ks():
    """In an infinite medium the total path of a history is a geometric sum of Exp(S_t) flights = exactly Exp(S_a).
    2000 single-history runs (seeds 1..2000, id 0): Kolmogorov-Smirnov against the exponential law."""
    o = orc.Oracle(W.cfg0(n=1))
    paths = np.array([o.run(seed=s)["flux"][0] / S24 for s in range(1, 2001)])
    o.close()
    assert stats.kstest(paths, "expon", args=(0, 1 / 0.3)).pvalue > 1e-3
    assert abs((paths > 1 / 0.3).mean() - math.exp(-1)) < 4 * math.sqrt(math.exp(-1) * (1 - math.exp(-1)) / 2000)


# ------------------------------------------------------------------ P12(i): replay of pin-cell histories from raw draws
def _replay_pin_cell(p, seed, ids, gen=0):
    """Independent replay (plain Python floats = IEEE doubles, no fused operations) of two-group pin-cell histories from
    the raw draws: returns per-history (n_seg, n_coll) and the integer flux / collision tallies by group."""
    g, m = p.geometry, p.materials
    h = float(g["xplanes"][1])
    R = float(g["univ_radius"][0, 0])
    G = m["G"]
    flux, coll, out = [0] * G, [0] * G, []
    draw = lambda i, seg, pur, j: L.orc_draw(seed, i, gen, seg, pur, j)

    def iso(i, seg):
        a = 0
        while True:
            v1, v2 = 2.0 * draw(i, seg, 3, 2 * a) - 1.0, 2.0 * draw(i, seg, 3, 2 * a + 1) - 1.0
            s = v1 * v1 + v2 * v2
            if s < 1.0:
                t = 2.0 * math.sqrt(1.0 - s)
                return v1 * t, v2 * t, 1.0 - 2.0 * s
            a += 1

    for i in ids:
        x = -h + draw(i, 0, 5, 0) * (h - -h)
        y = -h + draw(i, 0, 5, 1) * (h - -h)
        ring = 0 if x * x + y * y < R * R else 1
        u, v, w = iso(i, 0)
        grp, seg, nc = 0, 0, 0
        while True:
            seg += 1
            mat = int(g["univ_mat"][0, ring])
            St = float(m["sig_t"][mat, grp])
            dc = -L.orc_det_log(draw(i, seg, 0, 0)) / St
            cand = {}
            if u > 0.0: cand["x"] = (h - x) / u
            elif u < 0.0: cand["x"] = (-h - x) / u
            if v > 0.0: cand["y"] = (h - y) / v
            elif v < 0.0: cand["y"] = (-h - y) / v
            a_, b_, c_ = u * u + v * v, x * u + y * v, (x * x + y * y) - R * R
            if a_ != 0.0:
                disc = b_ * b_ - a_ * c_
                if ring == 0:
                    cand["out"] = max((-b_ + math.sqrt(max(disc, 0.0))) / a_, 0.0)
                elif b_ < 0.0 and disc > 0.0:
                    cand["in"] = max((-b_ - math.sqrt(disc)) / a_, 0.0)
            ds = min(cand.values())
            hit = dc < ds
            d = dc if hit else ds
            x, y = x + d * u, y + d * v
            flux[grp] += round(d * S24)                       # round-half-even, as llrint
            if hit:
                nc += 1
                coll[grp] += 1 << 24
                sst = 0.0
                for b in range(G):
                    sst = sst + float(m["sig_s"][mat, grp, b])
                r_ = draw(i, seg, 1, 1) * St
                if r_ < sst:
                    t_ = draw(i, seg, 2, 0) * sst
                    acc, ng = 0.0, G - 1
                    for b in range(G):
                        acc = acc + float(m["sig_s"][mat, grp, b])
                        if t_ < acc:
                            ng = b
                            break
                    grp = ng
                    u, v, w = iso(i, seg)
                else:
                    break                                     # capture or nu = 0 fission: the history ends
            else:
                if cand.get("x") == d:
                    x = h if u > 0.0 else -h
                    u = -u
                if cand.get("y") == d:
                    y = h if v > 0.0 else -h
                    v = -v
                if cand.get("out") == d: ring = 1
                if cand.get("in") == d: ring = 0
        out.append((i, seg, nc))
    return out, flux, coll


def test_replay_of_pin_cell_histories_from_raw_draws():
    """P12(i) with geometry: 100 histories of a two-group pin cell (cylinder, reflective box, group transfer) are
    recomputed segment by segment in Python from the raw draws; per-history segment and collision counts and the integer
    tallies by group must be identical (the replay calls the oracle's pinned det_log and draw entry points only)."""
    rng = np.random.default_rng(12)
    sig_t = np.array([[0.9, 1.6], [1.2, 2.1]])
    ss = np.array([[[0.35, 0.30], [0.05, 0.90]], [[0.55, 0.60], [0.10, 1.80]]])
    mats = W.mg_materials(sig_t, ss, [[0.1, 0.3], [0.0, 0.0]], np.zeros((2, 2)), [[1.0, 0.0], [1.0, 0.0]])
    h = 0.63
    geo = W.geometry([-h, h], [-h, h], [-W.INF, W.INF], [0], [((0.54,), (0, 1))], [1, 1, 1, 1, 0, 0], by_group=1,
                     src_kind=1, src_lo=(-h, -h, 0.0), src_hi=(h, h, 0.0))
    p = W.Problem("replay_pin", geo, mats, None, "fixed", 100, seed=int(rng.integers(1, 2 ** 40)))
    r = orc.run(p)
    hist, flux, coll = _replay_pin_cell(p, p.seed, range(100))
    got = sorted(zip(r["hist_id"].tolist(), r["hist_nseg"].tolist(), r["hist_ncoll"].tolist()))
    assert got == sorted(hist)
    assert r["flux"].tolist() == flux and r["coll"].tolist() == coll
    assert sum(s for _, s, _ in hist) == r["totals"]["n_seg"] > 1000 and r["totals"]["n_cross"] > 500


# ------------------------------------------------------------------ D1: fixed-source secondaries
def test_fission_chain_progeny_in_a_subcritical_medium():
    """Fixed source with fission: every source neutron starts a branching process with k_inf = nu S_f / S_a = 0.6, so the
    histories per source neutron are 1 / (1 - k_inf) = 2.5 (variance sigma_offspring^2 / (1 - m)^3 = 10).  Pins the
    secondary stack, the derived ids (all distinct) and the multiplicity floor(nu + xi)."""
    n = 100000
    p = W.infinite_medium([1.0], [[0.5]], [0.2], [1.5], mode="fixed", n=n)
    r = orc.run(p)
    T = r["totals"]
    assert abs(T["n_born"] / n - 2.5) < 4 * math.sqrt(10.0 / n)
    assert T["n_born"] == n + T["n_sites"] and T["n_dropped"] == 0 and T["n_born"] == T["n_abs"] + T["n_fis"]
    assert abs(T["n_sites"] / T["n_fis"] - 1.5) < 4 * 0.5 / math.sqrt(T["n_fis"])
    assert len(np.unique(r["hist_id"])) == len(r["hist_id"]) == T["n_born"]
    assert abs(r["flux"][0] / S24 / n - 2.5 / 0.5) < 4 * math.sqrt(10.0 / n) / 0.5 * 1.5


def test_depth_cap_ends_supercritical_chains():
    """k_inf = 1.02: chains that survive 200 generations are cut (children dropped and counted); the run terminates and
    balances exactly."""
    n = 300
    p = W.infinite_medium([1.0], [[0.5]], [0.34], [1.5], mode="fixed", n=n)
    r = orc.run(p)
    T = r["totals"]
    assert T["n_dropped"] > 0
    assert T["n_born"] == n + T["n_sites"] == T["n_abs"] + T["n_fis"]
    assert len(np.unique(r["hist_id"])) == T["n_born"]


def test_population_control_ids_are_distinct_and_population_is_unbiased():
    """D2: copies of a bank site get ids derive_id(site id, g+1, 0, 2048 + r): all starters of the last generation must
    be distinct, and E[N_{g+1}] = N (m = floor(N/M + xi) per site)."""
    p = W.infinite_medium([1.0], [[0.5]], [0.2], [2.6], mode="k", n=30000, n_inactive=2, n_active=6)
    r = orc.run(p)
    assert len(np.unique(r["hist_id"])) == len(r["hist_id"]) == int(r["gen_n"][-1])
    assert np.all(np.abs(r["gen_n"].astype(float) - 30000) < 4 * math.sqrt(30000 * 0.25) + 1)
    assert len(np.unique(r["bank"]["id"])) == len(r["bank"])


# ------------------------------------------------------------------ TD: time-dependent fixed source
@pytest.mark.parametrize("c", [0.0, 0.7])
def test_time_dependent_population_decays_exponentially(c):
    """One-group infinite medium, speed v: collisions do not change the speed, so the population is N(t) = exp(-S_a v t)
    whatever the scattering ratio.  Track length per source in the time bin [a, b] = (exp(-S_a v a) - exp(-S_a v b)) / S_a,
    the census fraction is exp(-S_a v t_max).  Pins the time advance, the time-edge candidate, the time-bin index and census."""
    St, v, n = 1.0, 2.5, 200000
    Sa = St * (1 - c)
    edges = np.array([0.0, 0.05, 0.2, 0.21, 0.5, 0.9, 1.2])
    r = orc.run(W.td_medium(St, c * St, v, edges, n=n))
    T = r["totals"]
    ref = -np.diff(np.exp(-Sa * v * edges)) / Sa
    got = r["flux"] / S24 / n
    assert np.all(np.abs(got - ref) < 4 * np.sqrt(np.diff(edges) * v * ref / n) + 1e-7), (got, ref)
    surv = math.exp(-Sa * v * edges[-1])
    assert abs(T["n_census"] / n - surv) < 4 * math.sqrt(surv * (1 - surv) / n)
    assert T["n_born"] == T["n_abs"] + T["n_census"] == n and T["n_leak"] == 0
    assert abs(r["coll"].sum() / S24 / n - St * ref.sum()) < 4 * math.sqrt(3 * St * ref.sum() / n)


def test_time_dependent_fission_chain_growth():
    """Supercritical medium: the expected population grows as exp((nu S_f - S_a) v t); the census count pins secondaries that
    inherit their parent's time (a child restarted at t = 0 would never reach the census in time)."""
    St, Ss, Sf, nu, v, n = 1.0, 0.5, 0.3, 2.5, 1.0, 100000
    Sa = St - Ss
    alpha = (nu * Sf - Sa) * v
    edges = np.linspace(0.0, 3.0, 7)
    r = orc.run(W.td_medium(St, Ss, v, edges, sig_f=Sf, nu=nu, n=n))
    T = r["totals"]
    grow = math.exp(alpha * edges[-1])
    assert abs(T["n_census"] / n - grow) < 0.03 * grow                     # branching-process variance: a few sigma at 1e5
    ref = np.diff(np.exp(alpha * edges)) / alpha * v                        # integral of N(t) v dt per bin
    got = r["flux"] / S24 / n
    assert np.all(np.abs(got / ref - 1) < 0.03), (got, ref)
    assert T["n_born"] == n + T["n_sites"] == T["n_abs"] + T["n_fis"] + T["n_census"]


@pytest.mark.parametrize("E0", [0.0253, 1.0e6])
def test_time_dependent_speed_law_of_continuous_energy(E0):
    """v = 1.3831592e6 cm/s x sqrt(E / eV) (TD1): 2200 m/s at 0.0253 eV.  In a flat pure absorber the census fraction at
    t_max is exp(-S v t_max); t_max is set to one mean lifetime 1 / (S v) with v from the textbook value."""
    v = 2.19991e5 if E0 == 0.0253 else 1.3831592e9
    S = 0.5 * 2.0
    tmax = 1.0 / (S * v)
    edges = np.linspace(0.0, tmax, 5)
    n = 100000
    r = orc.run(W.td_ce_absorber(E0, edges, n=n))
    surv = math.exp(-1.0)
    assert abs(r["totals"]["n_census"] / n - surv) < 4 * math.sqrt(surv * (1 - surv) / n) + 2e-4
    ref = -np.diff(np.exp(-S * v * edges)) / S
    assert np.all(np.abs(r["flux"] / S24 / n - ref) < 4 * np.sqrt(ref * ref / n) + 1e-3 * ref)


def test_time_mesh_resolution_does_not_change_the_physics():
    """The paper's sweep: time-mesh widths 1, 2, ... 128.  A finer mesh adds time-edge crossings (each one a
    segment, so the random streams differ) but must not change any expectation: the summed flux, the collisions and the
    census of the CE pin cell agree within statistics for every width."""
    n, out = 20000, []
    for nt in (1, 8, 128):
        r = orc.run(W.cfg3_td(n=n, n_tbins=nt, n_grid=4000))
        T = r["totals"]
        assert T["n_born"] == T["n_abs"] + T["n_fis"] + T["n_census"] + T["n_leak"] and T["n_census"] > 0
        assert len(r["flux"]) == nt and int(r["coll"].sum()) == T["n_coll"] << 24
        out.append((r["flux"].sum() / S24 / n, T["n_coll"] / n, T["n_census"] / n, T["n_born"] / n))
    for a in out[1:]:
        assert np.allclose(a, out[0], rtol=0.1), out                   # branching-process noise at 2e4 sources


# ------------------------------------------------------------------ W: implicit capture + weight roulette
def test_implicit_capture_keeps_every_expectation_and_cuts_the_variance():
    """Capture by weight reduction and roulette below w_roulette change no expectation: flux per source 1 / S_a and
    collisions per source S_t / S_a in the infinite medium, with nobody captured in the analog way and every history
    ended by the roulette; the spread over batches is smaller than the analog one."""
    n = 100000
    r = orc.run(W.with_implicit_capture(W.cfg0(n=n)))
    T = r["totals"]
    assert T["n_abs"] == 0 and T["n_roulette"] == n == T["n_born"]
    assert abs(r["flux"][0] / S24 / n - 1 / 0.3) < 4 * (1 / 0.3) / math.sqrt(n)
    assert abs(r["coll"][0] / S24 / n - 1 / 0.3) < 4 * math.sqrt(0.7 / 0.09 / n)
    o = orc.Oracle(W.cfg0(n=500)); a = np.array([o.run(seed=s)["coll"][0] for s in range(1, 41)]) / S24 / 500; o.close()
    o = orc.Oracle(W.with_implicit_capture(W.cfg0(n=500))); b = np.array([o.run(seed=s)["coll"][0] for s in range(1, 41)]) / S24 / 500; o.close()
    assert b.std() < 0.8 * a.std(), (a.std(), b.std())


def test_implicit_capture_in_the_scattering_slab_matches_the_integral_equation():
    """Weighted scores per mesh bin against the deterministic slab solution: the weight after each collision, the scores
    that carry it and the roulette are all in play; the analog run of the same slab is the second witness."""
    St, c, Lx, n = 1.0, 0.8, 2.0, 400000
    mesh = [0.0, 0.11, 0.4, 0.75, 1.0, 1.31, 1.9, 2.0]
    r = orc.run(W.with_implicit_capture(W.slab_mesh(St, c * St, Lx, lattice=[0.5, 1.25], mesh=mesh, n=n), 0.1, 0.3))
    x, Ct, T, R = _slab_collision_probability(St, c, Lx)
    cum = np.concatenate([[0.0], np.cumsum(Ct)])
    ref_bin = np.diff(np.interp(mesh, x, cum))
    coll, flux = r["coll"] / S24 / n, r["flux"] / S24 / n
    assert np.all(np.abs(coll - ref_bin) < 4 * np.sqrt(3 * ref_bin / n)), (coll, ref_bin)
    assert np.all(np.abs(flux - ref_bin / St) < 4 * np.sqrt(3 * ref_bin / n) / St), (flux, ref_bin / St)
    assert r["totals"]["n_abs"] == 0 and r["totals"]["n_roulette"] > 0
    assert r["totals"]["n_born"] == r["totals"]["n_roulette"] + r["totals"]["n_leak"]


@pytest.mark.parametrize("ce", [False, True])
def test_implicit_capture_with_fission_chains(ce):
    """Fission stays analog under implicit capture (W3) and children inherit the weight (W1): flux per source neutron is
    1 / (S_a - nu S_f) in a sub-critical infinite medium, multigroup and continuous energy."""
    n = 100000
    if ce:
        p = W.ce_two_nuclide_medium(mode="fixed", n=n)
        ref = 1.0 / (0.5 * 1.0 + 0.3 * 2.0 - 0.3 * 2.0 * 1.5)
    else:
        p = W.infinite_medium([1.0], [[0.5]], [0.2], [1.5], mode="fixed", n=n)
        ref = 1.0 / (0.5 - 1.5 * 0.2)
    a = orc.run(p)
    r = orc.run(W.with_implicit_capture(p))
    assert abs(r["flux"].sum() / S24 / n - ref) < 0.03 * ref and abs(a["flux"].sum() / S24 / n - ref) < 0.03 * ref
    T = r["totals"]
    assert T["n_abs"] == 0 and T["n_born"] == n + T["n_sites"] == T["n_fis"] + T["n_roulette"]


# ------------------------------------------------------------------ C: general cells (readings C1-C6)
def _halfspace_fraction():
    """Volume fraction of the cube [-1, 1]^3 with X + 2 Y + 2 Z < 0.9, by quadrature (independent of the oracle)."""
    g = np.linspace(-1, 1, 2001); g = 0.5 * (g[1:] + g[:-1])
    Y, Z = np.meshgrid(g, g, indexing="ij")
    xmax = np.clip(0.9 - 2 * Y - 2 * Z, -1, 1)                 # X runs from -1 to xmax
    return float(np.mean(xmax + 1) / 2)


@pytest.mark.parametrize("kind", ["sphere", "halfspace", "offcyl", "shell", "lens", "lattice_cells", "strips", "two_universes"])
def test_general_cells_split_a_flat_flux_by_volume(kind):
    """The flat-flux volume pin on universes of general cells: a wrong root or side in the distance to a sphere, plane or
    cylinder, a cell search that ignores the crossed surface, a missed tie on the rim of the lens or a missed re-location at a
    lattice plane moves the share of absorptions in the fuel cells by many sigma (or loses particles)."""
    n = 200000
    p = W.two_region(kind, n=n)
    r = orc.run(p)
    T = r["totals"]
    assert T["n_born"] == n and T["n_leak"] == 0 and T["n_fis"] + T["n_abs"] == n
    f = p.notes["fuel_volume_fraction"] if kind != "halfspace" else _halfspace_fraction()
    assert abs(T["n_fis"] / n - f) < 4 * math.sqrt(f * (1 - f) / n), (kind, T["n_fis"] / n, f)
    assert abs(r["flux"][0] / S24 / n - 1 / 0.3) < 4 * (1 / 0.3) / math.sqrt(n)
    assert T["n_cross"] > n / 2


def test_surface_distance_lands_on_the_surface_and_is_the_first_hit():
    """orc_surf_dist against a brute-force march of the surface function (sign changes of orc_surf_eval along the ray), for
    all three kinds from both sides."""
    rng = np.random.default_rng(11)
    PDc = C.POINTER(C.c_double)
    for kind, co in ((0, [0.3, -0.5, 0.8, 0.2]), (1, [0.1, -0.2, 0.3, 0.9]), (2, [-0.2, 0.1, 0.0, 0.7])):
        ca = (C.c_double * 4)(*co)
        hits = 0
        for _ in range(300):
            r0 = rng.uniform(-1.5, 1.5, 3); d = rng.normal(size=3); d /= np.linalg.norm(d)
            f0 = L.orc_surf_eval(kind, ca, *r0)
            neg = f0 < 0
            dist = L.orc_surf_dist(kind, ca, *r0, *d, int(neg))
            ts = np.linspace(0, 6, 6001)[1:]
            fs = np.array([L.orc_surf_eval(kind, ca, *(r0 + t * d)) for t in ts])
            change = np.nonzero((fs < 0) != neg)[0]
            if len(change) == 0:
                assert dist == math.inf or dist > 6 - 2e-3, (kind, r0, d, dist)
                continue
            hits += 1
            assert abs(dist - ts[change[0]]) < 2e-3, (kind, r0, d, dist, ts[change[0]])
            assert abs(L.orc_surf_eval(kind, ca, *(r0 + dist * d))) < 1e-9
        assert hits > 50


def test_sphere_of_absorber_in_a_void_transmits_exp_minus_sigma_r():
    """A point source at the centre of a purely absorbing sphere (S = 1.3, R = 0.8) inside a void with vacuum faces: the
    share that leaks is exp(-S R) whatever the direction (pins the outward root and the cell change sphere -> void)."""
    n, S, R = 100000, 1.3, 0.8
    geo = W.geometry([-2, 2], [-2, 2], [-2, 2], [0], [("cells", [((-1,), 0), ((+1,), 1)])], [0] * 6, surfaces=[("sphere", 0.0, 0.0, 0.0, R)])
    mats = W.mg_materials([[S], [0.0]], [[[0.0]], [[0.0]]], [[0.0], [0.0]], [[0.0], [0.0]], [[1.0], [1.0]])
    r = orc.run(W.Problem("sphere_void", geo, mats, None, "fixed", n))
    t = math.exp(-S * R)
    assert abs(r["totals"]["n_leak"] / n - t) < 4 * math.sqrt(t * (1 - t) / n)
    assert r["totals"]["n_cross"] >= r["totals"]["n_leak"] * 2                # sphere surface, then the box face
