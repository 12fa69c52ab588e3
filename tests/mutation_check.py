#!/usr/bin/env python
"""Mutation check of the oracle's pins (not a pytest file; run by hand:  python tests/mutation_check.py [name ...]).

For every one-line mutation of oracle/orc.c listed below: build the mutant into a temporary shared object, point the
oracle binding at it (ORC_LIB) and run the CPU pins (tests/test_oracle_pins.py, tests/test_oracle_pins_transport.py)
until the first failure.  A mutant is KILLED when a pin fails (or the mutant errors out / runs away and is stopped);
it SURVIVES when every pin still passes — a survivor is either an equivalent program (stated in the table) or a hole.
Writes tests/golden/mutation_report.txt.  Only oracle/ and tests/ are touched; the CUDA path is not involved.
"""
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "orc.c")
PINS = ["tests/test_oracle_pins.py", "tests/test_oracle_pins_transport.py"]

# (name, text in orc.c, replacement, what it breaks)
MUTANTS = [
    ("csg_plane_side", "if (negative_side ? !(den > 0.0) : !(den < 0.0)) return INFINITY;", "if (negative_side ? !(den < 0.0) : !(den > 0.0)) return INFINITY;", "C3 plane reachable from the wrong side"),
    ("csg_inside_root", "d = (-qb + sqrt(disc)) / qa;", "d = (-qb - sqrt(disc)) / qa;", "C3 leaving root of a sphere / cylinder"),
    ("csg_outside_root", "d = (-qb - sqrt(disc)) / qa;", "d = (-qb + sqrt(disc)) / qa;", "C3 entering root of a sphere / cylinder"),
    ("csg_sphere_z", "oz = kind == 1 ? Z - co[2] : 0.0", "oz = kind == 1 ? Z + co[2] : 0.0", "C3 sphere centre z"),
    ("csg_eval_plane", "if (kind == 0) return ((co[0] * X + co[1] * Y) + co[2] * Z) - co[3];", "if (kind == 0) return ((co[0] * X + co[1] * Y) + co[2] * Z) + co[3];", "C2 plane function"),
    ("csg_eval_cyl", "return (ox * ox + oy * oy) - co[3] * co[3];", "return (ox * ox + oy * oy) - co[3];", "C2 cylinder function"),
    ("csg_crossed_side", "if ((crossed >> i & 1u) && abs(rf) - 1 == sf) neg = !(rf < 0);", "if ((crossed >> i & 1u) && abs(rf) - 1 == sf) neg = (rf < 0);", "C4 a crossed surface keeps its old side"),
    ("csg_tie_first_only", "for (int j = 0; j < ncs; j++) if (dcs[j] == d) crossed |= 1u << j;", "for (int j = 0; j < ncs; j++) if (dcs[j] == d) { crossed |= 1u << j; break; }", "C6 only the first of several surfaces met at once is crossed (EQUIVALENT in practice: ties have measure zero)"),
    ("csg_candidate", "for (int j = 0; j < ncs; j++) if (dcs[j] < ds) ds = dcs[j];", "for (int j = 1; j < ncs; j++) if (dcs[j] < ds) ds = dcs[j];", "C5 the cell's first surface is not a candidate"),
    ("csg_relocate_xy", "{ if (moved_xy || nu2 != univ) q->ring = locate_in_universe(", "{ if (nu2 != univ) q->ring = locate_in_universe(", "C6 no re-location at a lattice plane between cells of the same general universe"),
    ("csg_material", "return p->cell_mat[p->univ_cell0[univ] + ring];", "return p->cell_mat[ring];", "C1 material of a cell: universe offset dropped"),
    ("rot_swap_uv", "un = mul * u + k * ((u * w) * cphi - v * sphi);", "un = mul * u + k * ((v * w) * cphi - u * sphi);", "T6 rotation: u/v swapped in the first component"),
    ("rot_sign_vn", "vn = mul * v + k * ((v * w) * cphi + u * sphi);", "vn = mul * v + k * ((v * w) * cphi - u * sphi);", "T6 rotation: sign of the sin(phi) term of v'"),
    ("rot_sign_wn", "wn = mul * w - (k * ow) * cphi;", "wn = mul * w + (k * ow) * cphi;", "T6 rotation: sign of the w' correction"),
    ("rot_pole_sign", "wn = (w > 0.0) ? mul : -mul;", "wn = mul;", "T6 |w| ~ 1 branch: sign for w < 0"),
    ("rot_mirror_sphi", "sphi = (2.0 * v1 * v2) / s; break; }", "sphi = -(2.0 * v1 * v2) / s; break; }", "T6 azimuth mirrored (EQUIVALENT: -phi is as uniform as phi)"),
    ("mul_formula", "double mul = (1.0 + A * mu) / sqrt(q);", "double mul = (A + mu) / sqrt(q);", "T6 lab cosine"),
    ("eout_formula", "*E_out = E * (q / ((A + 1.0) * (A + 1.0)));", "*E_out = E * (q / ((A + 1.0) * (A - 1.0)));", "T6 outgoing energy"),
    ("nuclide_pick", "if (r < acc) { n = k; break; }", "if (r > acc) { n = k; break; }", "T6 nuclide selection comparison"),
    ("nuclide_sum", "acc = acc + p->mat_dens[mat * ORC_MAX_NUC + k] * st[k];", "acc = acc + p->mat_dens[mat * ORC_MAX_NUC + k] * ss[k];", "T6 nuclide running sum over N sigma_t"),
    ("reaction_swap", "else if (r2 < ss[n] + sc[n]) kind = 1; else kind = 2;", "else if (r2 < ss[n] + sc[n]) kind = 2; else kind = 1;", "T6 capture / fission swapped"),
    ("nu_wrong_nuclide", "nu = p->nuc_nu[fnuc]; src = fnuc;", "nu = p->nuc_nu[p->mat_nuc[mat * ORC_MAX_NUC]]; src = fnuc;", "nu of the material's first nuclide"),
    ("src_is_position", "nu = p->nuc_nu[fnuc]; src = fnuc;", "nu = p->nuc_nu[fnuc]; src = n;", "bank src = position in the material list, not the nuclide index"),
    ("ce_nsf", "nsf = nsf + N * (p->nuc_nu[nuc] * sf[n]);", "nsf = nsf + N * (p->nuc_nu[nuc] * sc[n]);", "T5 CE nu Sigma_f built from sigma_c"),
    ("lerp_fraction", "double f = (El - p->grid[i]) / (p->grid[i + 1] - p->grid[i]);", "double f = (p->grid[i + 1] - El) / (p->grid[i + 1] - p->grid[i]);", "X2 interpolation fraction"),
    ("lerp_clamp", "if (El > p->grid[p->n_grid - 1]) El = p->grid[p->n_grid - 1];", "", "X2 clamp above the grid"),
    ("sigma_t_sum", "st[n] = (ss[n] + sc[n]) + sf[n];", "st[n] = (ss[n] + sc[n]);", "X2 sigma_t without fission"),
    ("ring_out", "if (dout == d) q->ring += 1;", "if (dout == d) q->ring += 0;", "G7 ring after leaving a cylinder"),
    ("ring_in", "if (din == d) q->ring -= 1;", "if (din == d) q->ring -= 0;", "G7 ring after entering a cylinder"),
    ("ring_reset_xy", "if (moved_xy) q->ring = p->univ_nr[nu2];", "if (moved_xy) q->ring = 0;", "G7 ring after a lattice-plane crossing"),
    ("ring_relocate_z", "else if (nu2 != univ) q->ring = locate_ring(p, nu2, q->x - p->cx[q->ix], q->y - p->cy[q->iy]);", "", "G7 ring after a zone crossing into another universe"),
    ("locate_ring_cmp", "if (r2 < R * R) return r; }", "if (r2 < R) return r; }", "G2 ring search at birth"),
    ("mesh_inc", "if (q->mx + 1 < p->mesh_n[0]) q->mx += 1; }", "if (q->mx + 1 < p->mesh_n[0]) q->mx += 0; }", "T7 mesh index +x"),
    ("mesh_dec", "if (q->mx > 0) q->mx -= 1; } }", "if (q->mx > 0) q->mx -= 0; } }", "T7 mesh index -x"),
    ("mesh_dist_z", "if (dmz < ds) ds = dmz;", "", "T3 mesh-plane candidate (z) dropped"),
    ("mesh_dist_y", "if (dmy < ds) ds = dmy;", "", "T3 mesh-plane candidate (y) dropped"),
    ("mesh_bin_index", "+ q->mx) * p->n_e + e;   /* TD4", "+ q->mx) * p->n_e;   /* TD4", "T5 energy offset of the bin"),
    ("plane_dist_neg", "if (c < 0.0) return (lo - x) / c;", "if (c < 0.0) return (x - lo) / c;", "G3 plane distance for c < 0"),
    ("cyl_inside_root", "d = (-b + sqrt(disc)) / a;", "d = (-b - sqrt(disc)) / a;", "G4 leaving root"),
    ("cyl_c_term", "double c = (X * X + Y * Y) - R * R;", "double c = (X * X + Y * Y) - R;", "G4 constant term"),
    ("reflect_x", "if (p->bc[1]) q->u = -u0;", "if (p->bc[1]) q->u = u0;", "G7 reflection at +x"),
    ("leak_face", "else { alive = 0; c->leak[1] += 1; } } else { q->ix += 1;", "else { alive = 0; c->leak[0] += 1; } } else { q->ix += 1;", "G7 leak booked on the wrong face"),
    ("tie_rule", "int collide = dcoll < ds;", "int collide = dcoll <= ds;", "G5 tie rule (EQUIVALENT in practice: ties have measure zero)"),
    ("advance", "q->x = q->x + d * u0;", "q->x = q->x + d * v0;", "G6 advance"),
    ("flux_score", "const double wd = p->implicit ? q->wgt * d : d;", "const double wd = p->implicit ? q->wgt * d : dcoll;", "T5 scores the collision distance, not the flight"),
    ("pc_score", "c->Pc += fixp(p, nsf / St);", "c->Pc += fixp(p, nsf);", "T6 collision estimator of k"),
    ("p_score", "c->P += fixp(p, d * nsf);", "c->P += fixp(p, d * St);", "T5 track-length estimator of k"),
    ("mg_select", "if (r < sst) kind = 0; else if (r < sst + p->sig_c[mat * p->G + q->g]) kind = 1; else kind = 2;", "if (r < sst) kind = 0; else if (r < p->sig_c[mat * p->G + q->g]) kind = 1; else kind = 2;", "T6 MG capture threshold"),
    ("mg_cdf_transposed", "acc = acc + m->sig_s[(k * G + a) * G + b]; p->scdf[(k * G + a) * G + b] = acc;", "acc = acc + m->sig_s[(k * G + b) * G + a]; p->scdf[(k * G + a) * G + b] = acc;", "X1 scatter matrix transposed"),
    ("sample_cdf_cmp", "for (int k = 0; k < n; k++) if (t < cdf[k]) return k;", "for (int k = 0; k < n; k++) if (t > cdf[k]) return k;", "X1 cdf search"),
    ("multiplicity", "int n = (int)floor(nu_eff + orc_draw(seed, q->id, gen, seg, PUR_MULT, 0));", "int n = (int)floor(nu_eff);", "T6 multiplicity without the random rounding"),
    ("k_prev_unused", "double nu_eff = c->kmode ? nu / c->k_prev : nu;", "double nu_eff = nu;", "T6 multiplicity not normalised by k"),
    ("child_tag", "s.id = orc_derive_id(seed, q->id, gen, seg, (uint32_t)k);", "s.id = orc_derive_id(seed, q->id, gen, seg, 0u);", "R4 children share one id"),
    ("child_depth", "s.depth = (uint8_t)(c->kmode ? 0 : q->depth + 1);", "s.depth = (uint8_t)(c->kmode ? 0 : q->depth);", "D1 depth never grows (cap never reached)"),
    ("secondaries_lost", "while (!c.err && c.stack.n > 0) {", "while (0) {", "D1 secondaries never run"),
    ("popctrl_round", "int m = (int)floor(pr + orc_draw(p->kseed, b->id, gen_next, 0, PUR_POPCTRL, 0));", "int m = (int)floor(pr + 0.5);", "D2 deterministic rounding in population control"),
    ("popctrl_tag", "cp.id = orc_derive_id(p->kseed, b->id, gen_next, 0, 2048u + (uint32_t)r);", "cp.id = orc_derive_id(p->kseed, b->id, gen_next, 0, 2048u);", "R4 copies of a site share one id"),
    ("k_formula", "double k = ((double)sums[0] * (1.0 / p->scale)) / (double)sums[2];", "double k = ((double)sums[1] * (1.0 / p->scale)) / (double)sums[2];", "D2 k from the collision estimator (EQUIVALENT within statistics: both estimators are unbiased)"),
    ("watt_cos2", "cos2 = (v1 * v1) / s; break; }", "cos2 = (v1 * v1); break; }", "B3 Watt cos^2"),
    ("watt_shift", "return (W + aab / 4.0) + (2.0 * x2 - 1.0) * sqrt(aab * W);", "return (W + aab / 2.0) + (2.0 * x2 - 1.0) * sqrt(aab * W);", "B3 Watt shift term"),
    ("iso_w", "out[0] = v1 * t; out[1] = v2 * t; out[2] = 1.0 - 2.0 * s;", "out[0] = v1 * t; out[1] = v2 * t; out[2] = 1.0 - s;", "B2 Marsaglia w"),
    ("unit_shift", "uint64_t u52 = (((uint64_t)hi << 32) | lo) >> 12;", "uint64_t u52 = (((uint64_t)hi << 32) | lo) >> 13;", "N3 bit count"),
    ("philox_key", "k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;", "k0 += 0x9E3779B9u; k1 += 0xBB67AE86u;", "R1 Weyl constant"),
    ("det_log_coeff", "for (int k = 9; k >= 1; k--) p = fma(p, z, 1.0 / (double)(2 * k + 1));", "for (int k = 9; k >= 2; k--) p = fma(p, z, 1.0 / (double)(2 * k + 1));", "N4 series short by a term"),
    ("grid_index_cmp", "if (grid[mid] <= E) lo = mid; else hi = mid;", "if (grid[mid] < E) lo = mid; else hi = mid;", "X2 index at a grid point"),
    ("ebin_search", "if (p->e_edges[mid] <= q->E) lo = mid; else hi = mid; }", "if (p->e_edges[mid] <= q->E) hi = mid; else lo = mid; }", "T5 energy-bin search"),
    ("birth_box", "pos[a] = p->src_lo[a] + orc_draw(c->seed, i, c->gen, 0, PUR_POS, (uint32_t)a) * (p->src_hi[a] - p->src_lo[a]);", "pos[a] = p->src_lo[a] + orc_draw(c->seed, i, c->gen, 0, PUR_POS, 0u) * (p->src_hi[a] - p->src_lo[a]);", "B1 one draw for all three coordinates"),
]


def run_one(name, old, new, workdir):
    src = open(SRC).read()
    if src.count(old) != 1:
        return "SKIPPED (pattern found %d times)" % src.count(old), 0.0
    c = os.path.join(workdir, name + ".c")
    so = os.path.join(workdir, name + ".so")
    open(c, "w").write(src.replace(old, new))
    subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-I", os.path.join(ROOT, "oracle"), c, "-o", so, "-lm"])
    env = dict(os.environ, ORC_LIB=so)
    t0 = time.time()
    try:
        r = subprocess.run([sys.executable, "-m", "pytest", *PINS, "-x", "-q", "-m", "not gpu", "-p", "no:cacheprovider"], cwd=ROOT, env=env,
                           capture_output=True, text=True, timeout=600)
    except subprocess.TimeoutExpired:
        return "KILLED (runaway: stopped after 600 s)", time.time() - t0
    dt = time.time() - t0
    if r.returncode == 0:
        return "SURVIVED", dt
    first = [ln for ln in r.stdout.splitlines() if ln.startswith("FAILED") or ln.startswith("ERROR")]
    return "KILLED by " + (first[0].split(" ", 1)[1].split(" - ")[0] if first else "a crash"), dt


def main():
    only = set(sys.argv[1:])
    lines = []
    with tempfile.TemporaryDirectory() as wd:
        for name, old, new, what in MUTANTS:
            if only and name not in only:
                continue
            res, dt = run_one(name, old, new, wd)
            line = f"{name:18s} | {what:95s} | {res}"
            print(line, f"({dt:.0f} s)", flush=True)
            lines.append(line)
    if not only:
        with open(os.path.join(ROOT, "tests", "golden", "mutation_report.txt"), "w") as f:
            f.write("# written by tests/mutation_check.py (calls only oracle/ and the CPU pins)\n")
            f.write("\n".join(lines) + "\n")
    bad = [ln for ln in lines if "SURVIVED" in ln and "EQUIVALENT" not in ln]
    print(f"{len(lines)} mutants, {len(bad)} unexplained survivors")
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
