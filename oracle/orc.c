/* orc.c — TEST INFRASTRUCTURE ONLY: plain history-based CPU oracle (see orc.h).
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC orc.c -o liborc.so -lm
 * Section letters (N,R,G,X,B,T,D) refer to DESIGN.md section 3.
 */
#include "orc.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <omp.h>

/* ------------------------------------------------------------------ R1: Philox4x32-10 */
void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; r++) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

enum { PUR_DIST = 0, PUR_SELECT = 1, PUR_ENERGY = 2, PUR_DIR = 3, PUR_MULT = 4, PUR_POS = 5,
       PUR_POPCTRL = 6, PUR_CLOSEOUT = 7, PUR_IDDERIVE = 15 };
#define MAX_ATTEMPT 1024

static void block(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, uint32_t purpose,
                  uint32_t pair, uint32_t out[4]) {
  uint32_t ctr[4], key[2];
  uint32_t blk = (purpose << 12) | (pair & 0xFFFu);
  ctr[0] = (uint32_t)id; ctr[1] = (uint32_t)(id >> 32);
  ctr[2] = (gen & 0xFFFFu) | (blk << 16); ctr[3] = seg;
  key[0] = (uint32_t)seed; key[1] = (uint32_t)(seed >> 32);
  orc_philox(ctr, key, out);
}

/* N3: 52 random bits -> xi in (0,1), symmetric about 1/2 */
static double to_unit(uint32_t lo, uint32_t hi) {
  uint64_t u52 = (((uint64_t)hi << 32) | lo) >> 12;
  return (double)(2 * u52 + 1) * 0x1p-53;
}

double orc_draw(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, uint32_t purpose, uint32_t j) {
  uint32_t w[4];
  block(seed, id, gen, seg, purpose, j >> 1, w);
  return (j & 1u) ? to_unit(w[2], w[3]) : to_unit(w[0], w[1]);
}

/* R4 */
uint64_t orc_derive_id(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, uint32_t tag) {
  uint32_t w[4];
  block(seed, id, gen, seg, PUR_IDDERIVE, tag, w);
  return ((uint64_t)w[1] << 32) | w[0];
}

/* ------------------------------------------------------------------ N4: det_log */
double orc_det_log(double x) {
  uint64_t bits; memcpy(&bits, &x, 8);
  int e = (int)((bits >> 52) & 0x7FF) - 1022;
  uint64_t mb = (bits & 0x000FFFFFFFFFFFFFull) | 0x3FE0000000000000ull;
  double m; memcpy(&m, &mb, 8);                 /* m in [1/2, 1) */
  if (m < 0x1.6a09e667f3bcdp-1) { m = 2.0 * m; e = e - 1; }
  double f = m - 1.0;
  double s = f / (2.0 + f);
  double z = s * s;
  double p = 1.0 / 21.0;
  for (int k = 9; k >= 1; k--) p = fma(p, z, 1.0 / (double)(2 * k + 1));
  double t = (s * z) * p;
  double r = 2.0 * (s + t);
  double de = (double)e;
  return (de * 0x1.62e42fee00000p-1) + ((de * 0x1.a39ef35793c76p-33) + r);
}

/* ------------------------------------------------------------------ B2: isotropic direction */
int orc_iso_dir(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, double out[3]) {
  for (uint32_t a = 0; a < MAX_ATTEMPT; a++) {
    double v1 = 2.0 * orc_draw(seed, id, gen, seg, PUR_DIR, 2 * a) - 1.0;
    double v2 = 2.0 * orc_draw(seed, id, gen, seg, PUR_DIR, 2 * a + 1) - 1.0;
    double s = v1 * v1 + v2 * v2;
    if (s < 1.0) {
      double t = 2.0 * sqrt(1.0 - s);
      out[0] = v1 * t; out[1] = v2 * t; out[2] = 1.0 - 2.0 * s;
      return 0;
    }
  }
  out[0] = 0.0; out[1] = 0.0; out[2] = 1.0;
  return 1;
}

/* B3: Watt spectrum, birth draws (seg = 0) */
double orc_watt(uint64_t seed, uint64_t id, uint32_t gen, double a, double b) {
  double cos2 = 1.0;
  for (uint32_t t = 0; t < MAX_ATTEMPT; t++) {
    double v1 = 2.0 * orc_draw(seed, id, gen, 0, PUR_ENERGY, 8 + 2 * t) - 1.0;
    double v2 = 2.0 * orc_draw(seed, id, gen, 0, PUR_ENERGY, 9 + 2 * t) - 1.0;
    double s = v1 * v1 + v2 * v2;
    if (s < 1.0 && s > 0.0) { cos2 = (v1 * v1) / s; break; }
  }
  double l0 = orc_det_log(orc_draw(seed, id, gen, 0, PUR_ENERGY, 0));
  double l1 = orc_det_log(orc_draw(seed, id, gen, 0, PUR_ENERGY, 1));
  double x2 = orc_draw(seed, id, gen, 0, PUR_ENERGY, 2);
  double W = -a * (l0 + l1 * cos2);
  double aab = (a * a) * b;
  return (W + aab / 4.0) + (2.0 * x2 - 1.0) * sqrt(aab * W);
}

/* T6 scatter CE: target at rest, isotropic in CM */
void orc_scatter_ce(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, double A, double E,
                    const double d[3], double *E_out, double o[3]) {
  double u = d[0], v = d[1], w = d[2];
  double mu = 2.0 * orc_draw(seed, id, gen, seg, PUR_ENERGY, 0) - 1.0;
  double q = (A * A + (2.0 * A) * mu) + 1.0;
  *E_out = E * (q / ((A + 1.0) * (A + 1.0)));
  double mul = (1.0 + A * mu) / sqrt(q);
  double cphi = 1.0, sphi = 0.0;
  for (uint32_t t = 0; t < MAX_ATTEMPT; t++) {
    double v1 = 2.0 * orc_draw(seed, id, gen, seg, PUR_DIR, 2 * t) - 1.0;
    double v2 = 2.0 * orc_draw(seed, id, gen, seg, PUR_DIR, 2 * t + 1) - 1.0;
    double s = v1 * v1 + v2 * v2;
    if (s < 1.0 && s > 0.0) { cphi = (v1 * v1 - v2 * v2) / s; sphi = (2.0 * v1 * v2) / s; break; }
  }
  double om = 1.0 - mul * mul; if (om < 0.0) om = 0.0;
  double ow = 1.0 - w * w;
  double un, vn, wn;
  if (ow > 1e-10) {
    double k = sqrt(om / ow);
    un = mul * u + k * ((u * w) * cphi - v * sphi);
    vn = mul * v + k * ((v * w) * cphi + u * sphi);
    wn = mul * w - (k * ow) * cphi;
  } else {
    double k = sqrt(om);
    un = k * cphi; vn = k * sphi; wn = (w > 0.0) ? mul : -mul;
  }
  double n = sqrt((un * un + vn * vn) + wn * wn);
  o[0] = un / n; o[1] = vn / n; o[2] = wn / n;
}

/* G4: distance to a z-cylinder of radius R about the origin of (X,Y) */
double orc_dist_cyl(double X, double Y, double u, double v, double R, int inside) {
  double a = u * u + v * v;
  if (a == 0.0) return INFINITY;
  double b = X * u + Y * v;
  double c = (X * X + Y * Y) - R * R;
  double disc = b * b - a * c;
  double d;
  if (inside) {
    if (disc < 0.0) disc = 0.0;
    d = (-b + sqrt(disc)) / a;
  } else {
    if (b >= 0.0) return INFINITY;
    if (disc <= 0.0) return INFINITY;
    d = (-b - sqrt(disc)) / a;
  }
  if (d < 0.0) d = 0.0;
  return d;
}

/* C2: the surface function; a point with f < 0 is on the negative side (inside a sphere or cylinder) */
double orc_surf_eval(int kind, const double *co, double X, double Y, double Z) {
  if (kind == 0) return ((co[0] * X + co[1] * Y) + co[2] * Z) - co[3];
  const double ox = X - co[0], oy = Y - co[1];
  if (kind == 1) { const double oz = Z - co[2]; return ((ox * ox + oy * oy) + oz * oz) - co[3] * co[3]; }
  return (ox * ox + oy * oy) - co[3] * co[3];
}

/* C3: distance along (u,v,w) to the surface for a particle KNOWN to be on the given side (the side comes from the cell's
 * definition, not from the sign of f: a particle that has just crossed sits on the surface up to rounding).  Plane: reachable
 * only when moving towards it.  Sphere / cylinder: G4's two roots with the full quadratic. */
double orc_surf_dist(int kind, const double *co, double X, double Y, double Z, double u, double v, double w, int negative_side) {
  double d;
  if (kind == 0) {
    const double den = (co[0] * u + co[1] * v) + co[2] * w;
    if (negative_side ? !(den > 0.0) : !(den < 0.0)) return INFINITY;
    d = (co[3] - ((co[0] * X + co[1] * Y) + co[2] * Z)) / den;
  } else {
    const double ox = X - co[0], oy = Y - co[1], oz = kind == 1 ? Z - co[2] : 0.0, wz = kind == 1 ? w : 0.0;
    const double qa = (u * u + v * v) + wz * wz;
    if (qa == 0.0) return INFINITY;
    const double qb = (ox * u + oy * v) + oz * wz;
    const double qc = ((ox * ox + oy * oy) + oz * oz) - co[3] * co[3];
    double disc = qb * qb - qa * qc;
    if (negative_side) {
      if (disc < 0.0) disc = 0.0;
      d = (-qb + sqrt(disc)) / qa;
    } else {
      if (qb >= 0.0) return INFINITY;
      if (disc <= 0.0) return INFINITY;
      d = (-qb - sqrt(disc)) / qa;
    }
  }
  if (d < 0.0) d = 0.0;
  return d;
}

/* X2: largest i with grid[i] <= E (E clamped to the grid), capped at n-2 */
int32_t orc_grid_index(const double *grid, int32_t n, double E) {
  if (E < grid[0]) E = grid[0];
  if (E > grid[n - 1]) E = grid[n - 1];
  int32_t lo = 0, hi = n - 1;                   /* invariant grid[lo] <= E, (hi==n-1 or grid[hi] > E) */
  while (hi - lo > 1) {
    int32_t mid = lo + (hi - lo) / 2;
    if (grid[mid] <= E) lo = mid; else hi = mid;
  }
  if (lo > n - 2) lo = n - 2;
  return lo;
}

/* ------------------------------------------------------------------ problem */
typedef struct { uint64_t *id; uint32_t *nseg, *ncoll; size_t n, cap; } histvec;   /* per-history records */

struct orc_problem {
  int nx, ny, nz, bc[6], n_univ, mesh_n[3], by_group, n_e, S, n_t;           /* n_t: time bins (0 = time-independent) */
  int implicit; double w_roulette, w_survive;                                /* W: implicit capture + roulette */
  double *xp, *yp, *zp, *cx, *cy, *univ_rad, *mesh[3], *e_edges, *t_edges, *speed;
  int32_t *cell_univ, *univ_nr, *univ_mat;
  int n_surf, n_cell; int32_t *surf_kind, *univ_cell0, *univ_ncell, *cell_nsurf, *cell_surf, *cell_mat; double *surf_coef;   /* C: general cells */
  int src_kind, src_dir_kind, src_energy_kind, src_index;
  double src_lo[3], src_hi[3], src_dir[3], src_energy, scale;
  int n_mat, G;
  double *sig_t, *sig_f, *nu, *sst, *sig_c, *scdf, *chicdf, *nusigf;
  int32_t *mat_nnuc, *mat_nuc; double *mat_dens;
  int n_grid, n_nuc;
  double *grid, *A, *xs_s, *xs_c, *xs_f, *nuc_nu, *wa, *wb;
  /* results */
  uint64_t n_bins;
  int64_t *flux, *coll, leak[6];
  uint64_t totals[ORC_T_COUNT];
  uint64_t n_gen, *gen_n, *gen_m; int64_t *gen_p, *gen_pc; double *gen_k, k_mean, k_std;
  uint64_t n_hist, *hist_id; uint32_t *hist_nseg, *hist_ncoll;
  uint64_t n_bank; orc_site *bank;
  int ran;
  /* D2 in steps: this process's source share, its bank, its history records */
  uint64_t k_first, n_ksrc, n_kbank, kseed; orc_site *ksrc, *kbank; histvec khist;
};

static void *dup_mem(const void *src, size_t bytes) {
  void *p = malloc(bytes ? bytes : 1);
  if (p && src && bytes) memcpy(p, src, bytes);
  return p;
}
#define DUPD(src, n) ((double *)dup_mem((src), sizeof(double) * (size_t)(n)))
#define DUPI(src, n) ((int32_t *)dup_mem((src), sizeof(int32_t) * (size_t)(n)))

static void free_results(orc_problem *p) {
  free(p->flux); free(p->coll); free(p->gen_n); free(p->gen_m); free(p->gen_p); free(p->gen_pc);
  free(p->gen_k); free(p->hist_id); free(p->hist_nseg); free(p->hist_ncoll); free(p->bank);
  p->flux = p->coll = NULL; p->gen_n = p->gen_m = NULL; p->gen_p = p->gen_pc = NULL; p->gen_k = NULL;
  p->hist_id = NULL; p->hist_nseg = p->hist_ncoll = NULL; p->bank = NULL;
  p->n_gen = p->n_hist = p->n_bank = 0; p->ran = 0;
}

void orc_free_problem(orc_problem *p) {
  if (!p) return;
  free_results(p);
  free(p->xp); free(p->yp); free(p->zp); free(p->cx); free(p->cy); free(p->univ_rad);
  for (int a = 0; a < 3; a++) free(p->mesh[a]);
  free(p->e_edges); free(p->t_edges); free(p->speed); free(p->cell_univ); free(p->univ_nr); free(p->univ_mat);
  free(p->surf_kind); free(p->univ_cell0); free(p->univ_ncell); free(p->cell_nsurf); free(p->cell_surf); free(p->cell_mat); free(p->surf_coef);
  free(p->sig_t); free(p->sig_f); free(p->nu); free(p->sst); free(p->sig_c); free(p->scdf);
  free(p->chicdf); free(p->nusigf); free(p->mat_nnuc); free(p->mat_nuc); free(p->mat_dens);
  free(p->grid); free(p->A); free(p->xs_s); free(p->xs_c); free(p->xs_f); free(p->nuc_nu);
  free(p->wa); free(p->wb);
  free(p->ksrc); free(p->kbank); free(p->khist.id); free(p->khist.nseg); free(p->khist.ncoll);
  free(p);
}

int orc_init_problem(const orc_geometry *g, const orc_materials *m, const orc_xs_tables *x, orc_problem **out) {
  if (!g || !m || !out) return ORC_EINVAL;
  if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->n_univ < 1 || m->n_mat < 1) return ORC_EINVAL;
  if (g->nx > 32767 || g->ny > 32767 || g->nz > 32767) return ORC_EINVAL;
  if (m->G == 0 && !x) return ORC_EINVAL;
  if (g->tally_scale_log2 < 0 || g->tally_scale_log2 > 40) return ORC_EINVAL;
  orc_problem *p = (orc_problem *)calloc(1, sizeof(*p));
  if (!p) return ORC_ENOMEM;
  p->nx = g->nx; p->ny = g->ny; p->nz = g->nz; memcpy(p->bc, g->bc, sizeof p->bc);
  p->xp = DUPD(g->xplanes, g->nx + 1); p->yp = DUPD(g->yplanes, g->ny + 1); p->zp = DUPD(g->zplanes, g->nz + 1);
  p->cx = DUPD(g->cx, g->nx); p->cy = DUPD(g->cy, g->ny);
  p->cell_univ = DUPI(g->cell_univ, (size_t)g->nx * g->ny * g->nz);
  p->n_univ = g->n_univ; p->univ_nr = DUPI(g->univ_nrings, g->n_univ);
  p->univ_rad = DUPD(g->univ_radius, g->n_univ * ORC_MAX_RINGS);
  p->univ_mat = DUPI(g->univ_mat, g->n_univ * (ORC_MAX_RINGS + 1));
  const double *mp[3] = { g->mesh_x, g->mesh_y, g->mesh_z };
  const double *lp[3] = { p->xp, p->yp, p->zp };
  const int ln[3] = { g->nx, g->ny, g->nz };
  for (int a = 0; a < 3; a++) {
    if (g->mesh_n[a] < 1 || g->mesh_n[a] > 32767) { orc_free_problem(p); return ORC_EINVAL; }
    p->mesh_n[a] = g->mesh_n[a]; p->mesh[a] = DUPD(mp[a], g->mesh_n[a] + 1);
    if (!(p->mesh[a][0] <= lp[a][0]) || !(p->mesh[a][g->mesh_n[a]] >= lp[a][ln[a]])) { orc_free_problem(p); return ORC_EINVAL; }
  }
  p->n_surf = g->n_surf; p->n_cell = g->n_cell;
  if (p->n_surf > 0) {
    if (!g->surf_kind || !g->surf_coef || !g->univ_cell0 || !g->univ_ncell || !g->cell_nsurf || !g->cell_surf || !g->cell_mat || g->n_cell < 1) { orc_free_problem(p); return ORC_EINVAL; }
    p->surf_kind = DUPI(g->surf_kind, g->n_surf); p->surf_coef = DUPD(g->surf_coef, 4 * g->n_surf);
    p->univ_cell0 = DUPI(g->univ_cell0, g->n_univ); p->univ_ncell = DUPI(g->univ_ncell, g->n_univ);
    p->cell_nsurf = DUPI(g->cell_nsurf, g->n_cell); p->cell_surf = DUPI(g->cell_surf, g->n_cell * ORC_MAX_CSURF); p->cell_mat = DUPI(g->cell_mat, g->n_cell);
    for (int k = 0; k < g->n_surf; k++) if (p->surf_kind[k] < 0 || p->surf_kind[k] > 2 || (p->surf_kind[k] > 0 && !(p->surf_coef[4 * k + 3] > 0.0))) { orc_free_problem(p); return ORC_EINVAL; }
    for (int k = 0; k < g->n_cell; k++) {
      if (p->cell_nsurf[k] < 1 || p->cell_nsurf[k] > ORC_MAX_CSURF || p->cell_mat[k] < 0 || p->cell_mat[k] >= m->n_mat) { orc_free_problem(p); return ORC_EINVAL; }
      for (int j = 0; j < p->cell_nsurf[k]; j++) { int r = p->cell_surf[k * ORC_MAX_CSURF + j]; if (r == 0 || abs(r) > g->n_surf) { orc_free_problem(p); return ORC_EINVAL; } }
    }
  }
  for (int u = 0; u < g->n_univ; u++) {
    if (p->univ_nr[u] == -1 && p->n_surf > 0) {
      if (p->univ_cell0[u] < 0 || p->univ_ncell[u] < 1 || p->univ_ncell[u] > 255 || p->univ_cell0[u] + p->univ_ncell[u] > p->n_cell) { orc_free_problem(p); return ORC_EINVAL; }
    } else if (p->univ_nr[u] < 0 || p->univ_nr[u] > ORC_MAX_RINGS) { orc_free_problem(p); return ORC_EINVAL; }
  }
  p->G = m->G; p->n_mat = m->n_mat; p->by_group = g->by_group;
  if (p->G > 0) p->n_e = g->by_group ? p->G : 1;
  else { if (g->n_ebins < 1) { orc_free_problem(p); return ORC_EINVAL; } p->n_e = g->n_ebins; p->e_edges = DUPD(g->e_edges, g->n_ebins + 1); }
  p->src_kind = g->src_kind; p->src_dir_kind = g->src_dir_kind; p->src_energy_kind = g->src_energy_kind;
  p->src_index = g->src_index; p->src_energy = g->src_energy;
  memcpy(p->src_lo, g->src_lo, 24); memcpy(p->src_hi, g->src_hi, 24); memcpy(p->src_dir, g->src_dir, 24);
  p->S = g->tally_scale_log2; p->scale = ldexp(1.0, p->S);
  p->implicit = g->implicit_capture != 0; p->w_roulette = g->w_roulette; p->w_survive = g->w_survive;     /* W */
  if (p->implicit && !(p->w_roulette > 0.0 && p->w_survive >= p->w_roulette)) { orc_free_problem(p); return ORC_EINVAL; }
  p->n_t = g->n_tbins;                                                  /* TD: time mesh */
  if (p->n_t < 0 || p->n_t > 255) { orc_free_problem(p); return ORC_EINVAL; }
  if (p->n_t > 0) {
    if (!g->t_edges || (p->G > 0 && !m->speed)) { orc_free_problem(p); return ORC_EINVAL; }
    p->t_edges = DUPD(g->t_edges, p->n_t + 1);
    for (int k = 0; k < p->n_t; k++) if (!(p->t_edges[k] < p->t_edges[k + 1])) { orc_free_problem(p); return ORC_EINVAL; }
    if (p->G > 0) p->speed = DUPD(m->speed, p->G);
  }
  p->n_bins = (uint64_t)(p->n_t > 0 ? p->n_t : 1) * p->mesh_n[0] * p->mesh_n[1] * p->mesh_n[2] * p->n_e;
  if (p->G > 0) {                                                    /* X1 */
    int G = p->G, M = p->n_mat;
    p->sig_t = DUPD(m->sig_t, M * G); p->sig_f = DUPD(m->sig_f, M * G); p->nu = DUPD(m->nu, M * G);
    p->sst = DUPD(NULL, M * G); p->sig_c = DUPD(NULL, M * G); p->nusigf = DUPD(NULL, M * G);
    p->scdf = DUPD(NULL, M * G * G); p->chicdf = DUPD(NULL, M * G);
    for (int k = 0; k < M; k++) {
      double cc = 0.0;
      for (int a = 0; a < G; a++) {
        double acc = 0.0;
        for (int b = 0; b < G; b++) { acc = acc + m->sig_s[(k * G + a) * G + b]; p->scdf[(k * G + a) * G + b] = acc; }
        p->sst[k * G + a] = acc;
        double sa = p->sig_t[k * G + a] - acc;
        p->sig_c[k * G + a] = sa - p->sig_f[k * G + a];
        p->nusigf[k * G + a] = p->nu[k * G + a] * p->sig_f[k * G + a];
        cc = cc + m->chi[k * G + a]; p->chicdf[k * G + a] = cc;
      }
    }
  } else {
    p->mat_nnuc = DUPI(m->mat_nnuc, p->n_mat); p->mat_nuc = DUPI(m->mat_nuc, p->n_mat * ORC_MAX_NUC);
    p->mat_dens = DUPD(m->mat_dens, p->n_mat * ORC_MAX_NUC);
    p->n_grid = x->n_grid; p->n_nuc = x->n_nuc;
    if (p->n_grid < 2) { orc_free_problem(p); return ORC_EINVAL; }
    p->grid = DUPD(x->energy, x->n_grid); p->A = DUPD(x->A, x->n_nuc);
    size_t t = (size_t)x->n_nuc * x->n_grid;
    p->xs_s = DUPD(x->sig_s, t); p->xs_c = DUPD(x->sig_c, t); p->xs_f = DUPD(x->sig_f, t);
    p->nuc_nu = DUPD(x->nu, x->n_nuc); p->wa = DUPD(x->watt_a, x->n_nuc); p->wb = DUPD(x->watt_b, x->n_nuc);
  }
  *out = p;
  return ORC_OK;
}

/* ------------------------------------------------------------------ particle + per-thread context */
typedef struct {
  double x, y, z, u, v, w, E, t, wgt;
  int g, ix, iy, iz, ring, mx, my, mz, depth, it;
  uint64_t id; uint32_t seg, ncoll;
} part;

typedef struct { orc_site *v; size_t n, cap; } sitevec;

typedef struct {
  const orc_problem *p;
  uint64_t seed; uint32_t gen; int kmode, active; double k_prev;
  int64_t *flux, *coll, leak[6];
  __int128 P, Pc;
  uint64_t tot[ORC_T_COUNT];
  sitevec bank, stack; double *stack_t, *stack_w; size_t stack_t_cap;     /* time (TD5) and weight (W1) of secondary stack.v[i] */
  histvec hist; int keep_hist;
  int err;
} ctx;

static int push_site(sitevec *s, const orc_site *r) {
  if (s->n == s->cap) {
    size_t nc = s->cap ? 2 * s->cap : 1024;
    orc_site *nv = (orc_site *)realloc(s->v, nc * sizeof(orc_site));
    if (!nv) return 1;
    s->v = nv; s->cap = nc;
  }
  s->v[s->n++] = *r;
  return 0;
}

static int find_bin(const double *pl, int n, double x) {       /* G2 lower-inclusive */
  int k = 0;
  for (int i = 1; i < n; i++) if (pl[i] <= x) k = i;
  return k;
}

static int locate_ring(const orc_problem *p, int univ, double X, double Y) {
  int nr = p->univ_nr[univ];
  double r2 = X * X + Y * Y;
  for (int r = 0; r < nr; r++) { double R = p->univ_rad[univ * ORC_MAX_RINGS + r]; if (r2 < R * R) return r; }
  return nr;
}

/* C4: the cell of a general universe that holds the point: the first cell all of whose half-spaces hold.  A surface in
 * `crossed` (bit j = surface slot j of cell `from`) is not evaluated: the particle has just gone through it, so it is on
 * the side opposite to the one cell `from` names.  -1: no cell (undefined geometry). */
static int locate_cell(const orc_problem *p, int univ, double X, double Y, double Z, int from, unsigned crossed) {
  const int c0 = p->univ_cell0[univ], nc = p->univ_ncell[univ];
  for (int k = 0; k < nc; k++) {
    const int cell = c0 + k; int ok = 1;
    for (int j = 0; j < p->cell_nsurf[cell] && ok; j++) {
      const int r = p->cell_surf[cell * ORC_MAX_CSURF + j], sf = abs(r) - 1, want_neg = r < 0;
      int neg = -1;
      if (from >= 0)
        for (int i = 0; i < p->cell_nsurf[from]; i++) {
          const int rf = p->cell_surf[from * ORC_MAX_CSURF + i];
          if ((crossed >> i & 1u) && abs(rf) - 1 == sf) neg = !(rf < 0);
        }
      if (neg < 0) neg = orc_surf_eval(p->surf_kind[sf], p->surf_coef + 4 * sf, X, Y, Z) < 0.0;
      ok = neg == want_neg;
    }
    if (ok) return k;
  }
  return -1;
}

/* ring (or cell) of a point in a universe, by coordinates (G2, C4) */
static int locate_in_universe(const orc_problem *p, int univ, double X, double Y, double Z) {
  if (p->univ_nr[univ] < 0) return locate_cell(p, univ, X, Y, Z, -1, 0u);
  return locate_ring(p, univ, X, Y);
}

static int material_of(const orc_problem *p, int univ, int ring) {
  if (p->univ_nr[univ] < 0) return p->cell_mat[p->univ_cell0[univ] + ring];
  return p->univ_mat[univ * (ORC_MAX_RINGS + 1) + ring];
}

static int sample_cdf(const double *cdf, int n, double xi) {   /* X1 */
  double t = xi * cdf[n - 1];
  for (int k = 0; k < n; k++) if (t < cdf[k]) return k;
  return n - 1;
}

static int64_t fixp(const orc_problem *p, double v) { return (int64_t)llrint(v * p->scale); }   /* N5 */

static double plane_dist(double lo, double hi, double x, double c) {   /* G3 */
  if (c > 0.0) return (hi - x) / c;
  if (c < 0.0) return (lo - x) / c;
  return INFINITY;
}

/* B: birth of a primary source particle i, or from a site */
static void birth_common(ctx *c, part *q, int src, int from_site) {
  const orc_problem *p = c->p;
  q->seg = 0; q->ncoll = 0; q->E = 0.0; q->g = 0;
  if (!from_site && p->src_dir_kind == 1) { q->u = p->src_dir[0]; q->v = p->src_dir[1]; q->w = p->src_dir[2]; }
  else { double d[3]; c->tot[ORC_T_NDIRFAIL] += orc_iso_dir(c->seed, q->id, c->gen, 0, d); q->u = d[0]; q->v = d[1]; q->w = d[2]; }
  if (from_site) {
    if (p->G > 0) q->g = sample_cdf(p->chicdf + src * p->G, p->G, orc_draw(c->seed, q->id, c->gen, 0, PUR_ENERGY, 0));
    else q->E = orc_watt(c->seed, q->id, c->gen, p->wa[src], p->wb[src]);
  } else if (p->src_energy_kind == 0) q->g = p->src_index;
  else if (p->src_energy_kind == 1) q->E = p->src_energy;
  else q->E = orc_watt(c->seed, q->id, c->gen, p->wa[p->src_index], p->wb[p->src_index]);
  c->tot[ORC_T_NBORN] += 1;
}

static void birth_primary(ctx *c, part *q, uint64_t i) {                /* i = source id (D1: first_id + index) */
  const orc_problem *p = c->p;
  q->id = i; q->depth = 0;
  q->it = 0; q->t = p->n_t > 0 ? p->t_edges[0] : 0.0;                   /* TD5: emitted at the first time edge */
  q->wgt = 1.0;                                                         /* W1 */
  double pos[3];
  for (int a = 0; a < 3; a++) {
    if (p->src_kind == 0) pos[a] = p->src_lo[a];
    else pos[a] = p->src_lo[a] + orc_draw(c->seed, i, c->gen, 0, PUR_POS, (uint32_t)a) * (p->src_hi[a] - p->src_lo[a]);
  }
  q->x = pos[0]; q->y = pos[1]; q->z = pos[2];
  q->ix = find_bin(p->xp, p->nx, q->x); q->iy = find_bin(p->yp, p->ny, q->y); q->iz = find_bin(p->zp, p->nz, q->z);
  q->mx = find_bin(p->mesh[0], p->mesh_n[0], q->x); q->my = find_bin(p->mesh[1], p->mesh_n[1], q->y);
  q->mz = find_bin(p->mesh[2], p->mesh_n[2], q->z);
  int univ = p->cell_univ[((size_t)q->iz * p->ny + q->iy) * p->nx + q->ix];
  q->ring = locate_in_universe(p, univ, q->x - p->cx[q->ix], q->y - p->cy[q->iy], q->z);
  if (q->ring < 0) { c->err = ORC_ELOST; q->ring = 0; }
  birth_common(c, q, 0, 0);
}

static void birth_site(ctx *c, part *q, const orc_site *s, double t, double wgt) {
  q->id = s->id; q->depth = s->depth; q->t = t; q->it = s->it; q->wgt = wgt;
  q->x = s->x; q->y = s->y; q->z = s->z;
  q->ix = s->ix; q->iy = s->iy; q->iz = s->iz; q->mx = s->mx; q->my = s->my; q->mz = s->mz; q->ring = s->ring;
  birth_common(c, q, s->src, 1);
}

/* ------------------------------------------------------------------ T: one history, birth to death */
static void record_death(ctx *c, const part *q) {
  uint32_t ctr[4] = { (uint32_t)q->id, (uint32_t)(q->id >> 32), q->ncoll, q->seg - q->ncoll };
  uint32_t key[2] = { q->seg, 0x7D12u }, w[4];
  orc_philox(ctr, key, w);
  c->tot[ORC_T_DIGEST] += ((uint64_t)w[1] << 32) | w[0];
  if (c->keep_hist) {
    histvec *h = &c->hist;
    if (h->n == h->cap) {
      size_t nc = h->cap ? 2 * h->cap : 4096;
      h->id = (uint64_t *)realloc(h->id, nc * 8); h->nseg = (uint32_t *)realloc(h->nseg, nc * 4);
      h->ncoll = (uint32_t *)realloc(h->ncoll, nc * 4); h->cap = nc;
      if (!h->id || !h->nseg || !h->ncoll) { c->err = ORC_ENOMEM; return; }
    }
    h->id[h->n] = q->id; h->nseg[h->n] = q->seg; h->ncoll[h->n] = q->ncoll; h->n++;
  }
}

static void transport(ctx *c, part *q) {
  const orc_problem *p = c->p;
  const uint64_t seed = c->seed; const uint32_t gen = c->gen;
  int alive = 1;
  while (alive) {
    if (q->seg >= (1u << 24)) { c->err = ORC_ELOST; return; }
    q->seg += 1;                                                        /* R3 */
    const uint32_t seg = q->seg;
    int univ = p->cell_univ[((size_t)q->iz * p->ny + q->iy) * p->nx + q->ix];
    int mat = material_of(p, univ, q->ring);
    /* T1 */
    double St = 0.0, nsf = 0.0;
    double ss[ORC_MAX_NUC], sc[ORC_MAX_NUC], sf[ORC_MAX_NUC], st[ORC_MAX_NUC];
    int nn = 0;
    if (p->G > 0) { St = p->sig_t[mat * p->G + q->g]; nsf = p->nusigf[mat * p->G + q->g]; }
    else {
      double El = q->E; if (El < p->grid[0]) El = p->grid[0]; if (El > p->grid[p->n_grid - 1]) El = p->grid[p->n_grid - 1];
      int i = orc_grid_index(p->grid, p->n_grid, El);
      double f = (El - p->grid[i]) / (p->grid[i + 1] - p->grid[i]);
      nn = p->mat_nnuc[mat];
      for (int n = 0; n < nn; n++) {
        int nuc = p->mat_nuc[mat * ORC_MAX_NUC + n]; double N = p->mat_dens[mat * ORC_MAX_NUC + n];
        const double *ts = p->xs_s + (size_t)nuc * p->n_grid, *tc = p->xs_c + (size_t)nuc * p->n_grid, *tf = p->xs_f + (size_t)nuc * p->n_grid;
        ss[n] = ts[i] + f * (ts[i + 1] - ts[i]);
        sc[n] = tc[i] + f * (tc[i + 1] - tc[i]);
        sf[n] = tf[i] + f * (tf[i + 1] - tf[i]);
        st[n] = (ss[n] + sc[n]) + sf[n];
        St = St + N * st[n];
        nsf = nsf + N * (p->nuc_nu[nuc] * sf[n]);
      }
    }
    /* T2 */
    double dcoll = INFINITY;
    if (St > 0.0) dcoll = -orc_det_log(orc_draw(seed, q->id, gen, seg, PUR_DIST, 0)) / St;
    /* T3 */
    const double u0 = q->u, v0 = q->v, w0 = q->w;
    double dx = plane_dist(p->xp[q->ix], p->xp[q->ix + 1], q->x, u0);
    double dy = plane_dist(p->yp[q->iy], p->yp[q->iy + 1], q->y, v0);
    double dz = plane_dist(p->zp[q->iz], p->zp[q->iz + 1], q->z, w0);
    double dout = INFINITY, din = INFINITY;
    int nr = p->univ_nr[univ];
    if (nr > 0) {
      double X = q->x - p->cx[q->ix], Y = q->y - p->cy[q->iy];
      if (q->ring < nr) dout = orc_dist_cyl(X, Y, u0, v0, p->univ_rad[univ * ORC_MAX_RINGS + q->ring], 1);
      if (q->ring > 0) din = orc_dist_cyl(X, Y, u0, v0, p->univ_rad[univ * ORC_MAX_RINGS + q->ring - 1], 0);
    }
    double dcs[ORC_MAX_CSURF]; int ncs = 0, gcell = -1;                 /* C5: the surfaces of the current general cell */
    if (nr < 0) {
      gcell = p->univ_cell0[univ] + q->ring; ncs = p->cell_nsurf[gcell];
      const double X = q->x - p->cx[q->ix], Y = q->y - p->cy[q->iy];
      for (int j = 0; j < ncs; j++) {
        const int r = p->cell_surf[gcell * ORC_MAX_CSURF + j], sf = abs(r) - 1;
        dcs[j] = orc_surf_dist(p->surf_kind[sf], p->surf_coef + 4 * sf, X, Y, q->z, u0, v0, w0, r < 0);
      }
    }
    double dmx = plane_dist(p->mesh[0][q->mx], p->mesh[0][q->mx + 1], q->x, u0);
    double dmy = plane_dist(p->mesh[1][q->my], p->mesh[1][q->my + 1], q->y, v0);
    double dmz = plane_dist(p->mesh[2][q->mz], p->mesh[2][q->mz + 1], q->z, w0);
    double vel = 0.0, dtm = INFINITY;                                   /* TD1, TD2: speed and distance to the next time edge */
    if (p->n_t > 0) {
      vel = p->G > 0 ? p->speed[q->g] : 1.3831592e6 * sqrt(q->E);
      dtm = (p->t_edges[q->it + 1] - q->t) * vel;
    }
    double ds = dx;
    if (dy < ds) ds = dy;
    if (dz < ds) ds = dz;
    if (dout < ds) ds = dout;
    if (din < ds) ds = din;
    for (int j = 0; j < ncs; j++) if (dcs[j] < ds) ds = dcs[j];
    if (dmx < ds) ds = dmx;
    if (dmy < ds) ds = dmy;
    if (dmz < ds) ds = dmz;
    if (dtm < ds) ds = dtm;
    int collide = dcoll < ds;                                           /* G5: surface wins ties */
    double d = collide ? dcoll : ds;
    if (!(d < INFINITY)) { c->err = ORC_ELOST; return; }
    /* T4 */
    q->x = q->x + d * u0; q->y = q->y + d * v0; q->z = q->z + d * w0;
    if (p->n_t > 0) q->t = q->t + d / vel;                              /* TD3 */
    c->tot[ORC_T_NSEG] += 1;
    /* T5 */
    int e = -1;
    if (p->G > 0) e = p->by_group ? q->g : 0;
    else if (q->E >= p->e_edges[0] && q->E < p->e_edges[p->n_e]) {
      int lo = 0, hi = p->n_e;
      while (hi - lo > 1) { int mid = lo + (hi - lo) / 2; if (p->e_edges[mid] <= q->E) lo = mid; else hi = mid; }
      e = lo;
    }
    size_t bin = 0;
    if (e >= 0) bin = (((((size_t)q->it * p->mesh_n[2] + q->mz) * p->mesh_n[1] + q->my) * p->mesh_n[0]) + q->mx) * p->n_e + e;   /* TD4: it = 0 without a time mesh */
    const double wd = p->implicit ? q->wgt * d : d;                     /* W2: scores carry the weight (1 in analog runs) */
    if (c->active && e >= 0 && __builtin_add_overflow(c->flux[bin], fixp(p, wd), &c->flux[bin])) { c->err = ORC_EOVERFLOW; return; }   /* N5 */
    if (c->kmode) c->P += fixp(p, d * nsf);
    if (collide) {
      /* T6 */
      q->ncoll += 1; c->tot[ORC_T_NCOLL] += 1;
      if (c->active && e >= 0 && __builtin_add_overflow(c->coll[bin], fixp(p, p->implicit ? q->wgt : 1.0), &c->coll[bin])) { c->err = ORC_EOVERFLOW; return; }
      if (c->kmode) c->Pc += fixp(p, nsf / St);
      int kind;                                                         /* 0 scatter 1 capture 2 fission */
      int fnuc = 0; double nu = 0.0; int src = mat;
      if (p->G > 0) {
        double r = orc_draw(seed, q->id, gen, seg, PUR_SELECT, 1) * St;
        double sst = p->sst[mat * p->G + q->g];
        if (r < sst) kind = 0; else if (r < sst + p->sig_c[mat * p->G + q->g]) kind = 1; else kind = 2;
        if (p->implicit) {                                               /* W3: capture by weight, then scatter or fission */
          const double snc = St - p->sig_c[mat * p->G + q->g];
          if (snc > 0.0) {
            q->wgt = q->wgt * (snc / St);
            kind = (orc_draw(seed, q->id, gen, seg, PUR_SELECT, 1) * snc < sst) ? 0 : 2;
          } else kind = 1;
        }
        nu = p->nu[mat * p->G + q->g];
      } else {
        double r = orc_draw(seed, q->id, gen, seg, PUR_SELECT, 0) * St;
        double acc = 0.0; int n = nn - 1;
        for (int k = 0; k < nn; k++) { acc = acc + p->mat_dens[mat * ORC_MAX_NUC + k] * st[k]; if (r < acc) { n = k; break; } }
        fnuc = p->mat_nuc[mat * ORC_MAX_NUC + n];
        double r2 = orc_draw(seed, q->id, gen, seg, PUR_SELECT, 1) * st[n];
        if (r2 < ss[n]) kind = 0; else if (r2 < ss[n] + sc[n]) kind = 1; else kind = 2;
        if (p->implicit) {                                               /* W3 */
          const double snc = st[n] - sc[n];
          if (snc > 0.0) {
            q->wgt = q->wgt * (snc / st[n]);
            kind = (orc_draw(seed, q->id, gen, seg, PUR_SELECT, 1) * snc < ss[n]) ? 0 : 2;
          } else kind = 1;
        }
        nu = p->nuc_nu[fnuc]; src = fnuc;
      }
      if (kind == 0) {
        if (p->G > 0) {
          q->g = sample_cdf(p->scdf + (mat * p->G + q->g) * p->G, p->G, orc_draw(seed, q->id, gen, seg, PUR_ENERGY, 0));
          double dd[3]; c->tot[ORC_T_NDIRFAIL] += orc_iso_dir(seed, q->id, gen, seg, dd);
          q->u = dd[0]; q->v = dd[1]; q->w = dd[2];
        } else {
          double din3[3] = { q->u, q->v, q->w }, dd[3], En;
          orc_scatter_ce(seed, q->id, gen, seg, p->A[fnuc], q->E, din3, &En, dd);
          q->E = En; q->u = dd[0]; q->v = dd[1]; q->w = dd[2];
        }
      } else if (kind == 1) { alive = 0; c->tot[ORC_T_NABS] += 1; }
      else {
        alive = 0; c->tot[ORC_T_NFIS] += 1;
        double nu_eff = c->kmode ? nu / c->k_prev : nu;
        int n = (int)floor(nu_eff + orc_draw(seed, q->id, gen, seg, PUR_MULT, 0));
        if (n > 64) n = 64;
        if (!c->kmode && q->depth >= 200) { c->tot[ORC_T_NDROPPED] += (uint64_t)n; n = 0; }
        for (int k = 0; k < n; k++) {
          orc_site s; memset(&s, 0, sizeof s);
          s.x = q->x; s.y = q->y; s.z = q->z; s.id = orc_derive_id(seed, q->id, gen, seg, (uint32_t)k);
          s.ix = (int16_t)q->ix; s.iy = (int16_t)q->iy; s.iz = (int16_t)q->iz;
          s.mx = (int16_t)q->mx; s.my = (int16_t)q->my; s.mz = (int16_t)q->mz;
          s.ring = (uint8_t)q->ring; s.src = (uint8_t)src; s.depth = (uint8_t)(c->kmode ? 0 : q->depth + 1);
          s.it = (uint8_t)q->it;                                        /* TD5: secondaries inherit the time */
          if (!c->kmode) {
            if (c->stack.n >= c->stack_t_cap) {
              size_t nc = c->stack_t_cap ? 2 * c->stack_t_cap : 1024;
              double *nt = (double *)realloc(c->stack_t, nc * sizeof(double)), *nw = (double *)realloc(c->stack_w, nc * sizeof(double));
              if (!nt || !nw) { c->err = ORC_ENOMEM; return; }
              c->stack_t = nt; c->stack_w = nw; c->stack_t_cap = nc;
            }
            c->stack_t[c->stack.n] = q->t; c->stack_w[c->stack.n] = q->wgt;
          }
          if (push_site(c->kmode ? &c->bank : &c->stack, &s)) { c->err = ORC_ENOMEM; return; }
        }
        c->tot[ORC_T_NSITES] += (uint64_t)n;
      }
    } else {
      /* T7 / G7: every candidate at exactly distance d is crossed */
      c->tot[ORC_T_NCROSS] += 1;
      int moved_xy = 0, moved_z = 0;
      if (dx == d) {
        if (u0 > 0.0) { q->x = p->xp[q->ix + 1]; if (q->ix + 1 == p->nx) { if (p->bc[1]) q->u = -u0; else { alive = 0; c->leak[1] += 1; } } else { q->ix += 1; moved_xy = 1; } }
        else { q->x = p->xp[q->ix]; if (q->ix == 0) { if (p->bc[0]) q->u = -u0; else { alive = 0; c->leak[0] += 1; } } else { q->ix -= 1; moved_xy = 1; } }
      }
      if (dy == d) {
        if (v0 > 0.0) { q->y = p->yp[q->iy + 1]; if (q->iy + 1 == p->ny) { if (p->bc[3]) q->v = -v0; else { alive = 0; c->leak[3] += 1; } } else { q->iy += 1; moved_xy = 1; } }
        else { q->y = p->yp[q->iy]; if (q->iy == 0) { if (p->bc[2]) q->v = -v0; else { alive = 0; c->leak[2] += 1; } } else { q->iy -= 1; moved_xy = 1; } }
      }
      if (dz == d) {
        if (w0 > 0.0) { q->z = p->zp[q->iz + 1]; if (q->iz + 1 == p->nz) { if (p->bc[5]) q->w = -w0; else { alive = 0; c->leak[5] += 1; } } else { q->iz += 1; moved_z = 1; } }
        else { q->z = p->zp[q->iz]; if (q->iz == 0) { if (p->bc[4]) q->w = -w0; else { alive = 0; c->leak[4] += 1; } } else { q->iz -= 1; moved_z = 1; } }
      }
      if (dout == d) q->ring += 1;
      if (din == d) q->ring -= 1;
      if (moved_xy || moved_z) {
        int nu2 = p->cell_univ[((size_t)q->iz * p->ny + q->iy) * p->nx + q->ix];
        if (p->univ_nr[nu2] < 0) { if (moved_xy || nu2 != univ) q->ring = locate_in_universe(p, nu2, q->x - p->cx[q->ix], q->y - p->cy[q->iy], q->z); }
        else if (moved_xy) q->ring = p->univ_nr[nu2];
        else if (nu2 != univ) q->ring = locate_ring(p, nu2, q->x - p->cx[q->ix], q->y - p->cy[q->iy]);
        if (q->ring < 0) { c->err = ORC_ELOST; return; }
      } else if (ncs > 0) {                                             /* C6: through one or more surfaces of a general cell */
        unsigned crossed = 0u;
        for (int j = 0; j < ncs; j++) if (dcs[j] == d) crossed |= 1u << j;
        if (crossed) {
          q->ring = locate_cell(p, univ, q->x - p->cx[q->ix], q->y - p->cy[q->iy], q->z, gcell, crossed);
          if (q->ring < 0) { c->err = ORC_ELOST; return; }
        }
      }
      if (dmx == d) { if (u0 > 0.0) { q->x = p->mesh[0][q->mx + 1]; if (q->mx + 1 < p->mesh_n[0]) q->mx += 1; } else { q->x = p->mesh[0][q->mx]; if (q->mx > 0) q->mx -= 1; } }
      if (dmy == d) { if (v0 > 0.0) { q->y = p->mesh[1][q->my + 1]; if (q->my + 1 < p->mesh_n[1]) q->my += 1; } else { q->y = p->mesh[1][q->my]; if (q->my > 0) q->my -= 1; } }
      if (dmz == d) { if (w0 > 0.0) { q->z = p->mesh[2][q->mz + 1]; if (q->mz + 1 < p->mesh_n[2]) q->mz += 1; } else { q->z = p->mesh[2][q->mz]; if (q->mz > 0) q->mz -= 1; } }
      if (!alive) c->tot[ORC_T_NLEAK] += 1;
      if (dtm == d) {                                                   /* TD3: time edge; the last one is the census */
        q->t = p->t_edges[q->it + 1]; q->it += 1;
        if (q->it == p->n_t && alive) { alive = 0; c->tot[ORC_T_NCENSUS] += 1; }
      }
    }
    /* W4 closeout (the fifth event of the paper's decomposed scheme): weight roulette for the next segment */
    if (p->implicit && alive && q->wgt < p->w_roulette) {
      if (orc_draw(seed, q->id, gen, seg, PUR_CLOSEOUT, 0) * p->w_survive < q->wgt) q->wgt = p->w_survive;
      else { alive = 0; c->tot[ORC_T_NROULETTE] += 1; }
    }
  }
  record_death(c, q);
}

/* ------------------------------------------------------------------ D: drivers */
static int g_threads = 0;
int orc_set_threads(int n) { g_threads = n > 0 ? n : 0; return g_threads ? g_threads : omp_get_max_threads(); }

typedef struct { __int128 P, Pc; sitevec bank; int err; } batch_out;

/* one batch of histories: sources are primary indices [0,n_src) (sites == NULL) or sites[0..n_src) */
static void run_batch(orc_problem *p, uint64_t seed, uint32_t gen, int kmode, int active, double k_prev, uint64_t first_id,
                      uint64_t n_src, const orc_site *sites, int keep_hist, histvec *hist_all, batch_out *out) {
  int nt = g_threads ? g_threads : omp_get_max_threads();
  out->P = 0; out->Pc = 0; out->bank.v = NULL; out->bank.n = out->bank.cap = 0; out->err = 0;
#pragma omp parallel num_threads(nt)
  {
    ctx c; memset(&c, 0, sizeof c);
    c.p = p; c.seed = seed; c.gen = gen; c.kmode = kmode; c.active = active; c.k_prev = k_prev; c.keep_hist = keep_hist;
    c.flux = (int64_t *)calloc(p->n_bins, 8); c.coll = (int64_t *)calloc(p->n_bins, 8);
    if (!c.flux || !c.coll) c.err = ORC_ENOMEM;
#pragma omp for schedule(dynamic, 256)
    for (uint64_t i = 0; i < n_src; i++) {
      if (c.err) continue;
      part q;
      if (sites) birth_site(&c, &q, &sites[i], 0.0, 1.0); else birth_primary(&c, &q, first_id + i);
      transport(&c, &q);
      while (!c.err && c.stack.n > 0) {                 /* D1: secondaries, LIFO, to extinction */
        orc_site s = c.stack.v[--c.stack.n];
        birth_site(&c, &q, &s, c.stack_t[c.stack.n], c.stack_w[c.stack.n]);
        transport(&c, &q);
      }
    }
#pragma omp critical
    {
      if (c.err && !out->err) out->err = c.err;
      if (!c.err) {
        for (uint64_t b = 0; b < p->n_bins; b++)                 /* N5: every tally sum is checked against int64 */
          if (__builtin_add_overflow(p->flux[b], c.flux[b], &p->flux[b]) || __builtin_add_overflow(p->coll[b], c.coll[b], &p->coll[b])) out->err = ORC_EOVERFLOW;
        for (int f = 0; f < 6; f++) p->leak[f] += c.leak[f];
        for (int t = 0; t < ORC_T_COUNT; t++) p->totals[t] += c.tot[t];
        out->P += c.P; out->Pc += c.Pc;
        for (size_t k = 0; k < c.bank.n && !out->err; k++) if (push_site(&out->bank, &c.bank.v[k])) out->err = ORC_ENOMEM;
        if (keep_hist && c.hist.n) {
          size_t need = hist_all->n + c.hist.n;
          if (need > hist_all->cap) {
            size_t nc = need * 2;
            hist_all->id = (uint64_t *)realloc(hist_all->id, nc * 8); hist_all->nseg = (uint32_t *)realloc(hist_all->nseg, nc * 4);
            hist_all->ncoll = (uint32_t *)realloc(hist_all->ncoll, nc * 4); hist_all->cap = nc;
          }
          memcpy(hist_all->id + hist_all->n, c.hist.id, c.hist.n * 8);
          memcpy(hist_all->nseg + hist_all->n, c.hist.nseg, c.hist.n * 4);
          memcpy(hist_all->ncoll + hist_all->n, c.hist.ncoll, c.hist.n * 4);
          hist_all->n = need;
        }
      }
    }
    free(c.flux); free(c.coll); free(c.bank.v); free(c.stack.v); free(c.stack_t); free(c.stack_w); free(c.hist.id); free(c.hist.nseg); free(c.hist.ncoll);
  }
}

static int alloc_results(orc_problem *p, uint64_t n_gen) {
  free_results(p);
  p->flux = (int64_t *)calloc(p->n_bins, 8); p->coll = (int64_t *)calloc(p->n_bins, 8);
  memset(p->leak, 0, sizeof p->leak); memset(p->totals, 0, sizeof p->totals);
  p->k_mean = 0.0; p->k_std = 0.0;
  if (n_gen) {
    p->gen_n = (uint64_t *)calloc(n_gen, 8); p->gen_m = (uint64_t *)calloc(n_gen, 8);
    p->gen_p = (int64_t *)calloc(n_gen, 8); p->gen_pc = (int64_t *)calloc(n_gen, 8); p->gen_k = (double *)calloc(n_gen, 8);
  }
  return (p->flux && p->coll) ? ORC_OK : ORC_ENOMEM;
}

static int fits_i64(__int128 v) { return v < ((__int128)1 << 63) && v > -((__int128)1 << 63); }

/* D1 over the id range [first_id, first_id + n): one share of a source split over several processes */
int orc_run_fixed_source_range(orc_problem *p, uint64_t first_id, uint64_t n, uint64_t seed) {
  if (!p) return ORC_EINVAL;
  int rc = alloc_results(p, 0); if (rc) return rc;
  histvec h; memset(&h, 0, sizeof h);
  batch_out o;
  run_batch(p, seed, 0, 0, 1, 1.0, first_id, n, NULL, n <= 2000000, &h, &o);
  free(o.bank.v);
  p->hist_id = h.id; p->hist_nseg = h.nseg; p->hist_ncoll = h.ncoll; p->n_hist = h.n;
  if (o.err) return o.err;
  p->ran = 1;
  return ORC_OK;
}

int orc_run_fixed_source(orc_problem *p, uint64_t n, uint64_t seed) { return orc_run_fixed_source_range(p, 0, n, seed); }

/* D2 in steps, so that one problem can be shared by several processes: every process holds a contiguous
 * share of the source, runs its generation, the (P, Pc, N, M) sums are added over the processes, and every process
 * controls its own bank with the global p = N / M.  orc_run_k_eigenvalue is the same loop with one share. */
int orc_k_begin(orc_problem *p, uint64_t first_id, uint64_t n_local, uint32_t n_gen, uint64_t seed) {
  if (!p || n_gen == 0 || n_gen > 65535 || p->n_t > 0 || p->implicit) return ORC_EINVAL;      /* the time mesh belongs to fixed-source runs */
  int rc = alloc_results(p, n_gen); if (rc) return rc;
  free(p->ksrc); free(p->kbank); p->ksrc = NULL; p->kbank = NULL; p->n_kbank = 0;
  p->k_first = first_id; p->n_ksrc = n_local; p->kseed = seed;
  memset(&p->khist, 0, sizeof p->khist);
  return ORC_OK;
}

/* one generation over this process's share; sums = { P, Pc, N_local, M_local } */
int orc_k_generation(orc_problem *p, uint32_t gen, int active, double k_prev, int keep_hist, int64_t sums[4]) {
  if (!p || !sums) return ORC_EINVAL;
  batch_out o;
  free(p->kbank); p->kbank = NULL; p->n_kbank = 0;
  run_batch(p, p->kseed, gen, 1, active, k_prev, p->k_first, p->n_ksrc, p->ksrc, keep_hist && p->n_ksrc <= 2000000, &p->khist, &o);
  if (o.err) { free(o.bank.v); return o.err; }
  if (!fits_i64(o.P) || !fits_i64(o.Pc)) { free(o.bank.v); return ORC_EOVERFLOW; }
  p->kbank = o.bank.v; p->n_kbank = o.bank.n;
  sums[0] = (int64_t)o.P; sums[1] = (int64_t)o.Pc; sums[2] = (int64_t)p->n_ksrc; sums[3] = (int64_t)o.bank.n;
  return ORC_OK;
}

/* population control of this process's bank with the global ratio pr = N / M: m = floor(pr + xi) copies per site */
int orc_k_popctrl(orc_problem *p, uint32_t gen_next, double pr, uint64_t *n_next) {
  if (!p || !n_next) return ORC_EINVAL;
  sitevec nx; memset(&nx, 0, sizeof nx);
  for (size_t s = 0; s < p->n_kbank; s++) {
    const orc_site *b = &p->kbank[s];
    int m = (int)floor(pr + orc_draw(p->kseed, b->id, gen_next, 0, PUR_POPCTRL, 0));
    if (m > 2048) m = 2048;
    for (int r = 0; r < m; r++) {
      orc_site cp = *b; cp.id = orc_derive_id(p->kseed, b->id, gen_next, 0, 2048u + (uint32_t)r);
      if (push_site(&nx, &cp)) { free(nx.v); return ORC_ENOMEM; }
    }
  }
  free(p->ksrc); p->ksrc = nx.v; p->n_ksrc = nx.n;
  *n_next = nx.n;
  return ORC_OK;
}

/* store the per-generation results (global sums) and close the run; the last bank stays readable */
int orc_k_end(orc_problem *p, uint32_t n_gen, uint32_t n_inactive, const uint64_t *gen_n, const uint64_t *gen_m, const int64_t *gen_p,
              const int64_t *gen_pc, const double *gen_k) {
  if (!p) return ORC_EINVAL;
  for (uint32_t g = 0; g < n_gen; g++) { p->gen_n[g] = gen_n[g]; p->gen_m[g] = gen_m[g]; p->gen_p[g] = gen_p[g]; p->gen_pc[g] = gen_pc[g]; p->gen_k[g] = gen_k[g]; }
  p->n_gen = n_gen;
  free(p->bank); p->bank = p->kbank; p->n_bank = p->n_kbank; p->kbank = NULL; p->n_kbank = 0;
  free(p->ksrc); p->ksrc = NULL; p->n_ksrc = 0;
  p->hist_id = p->khist.id; p->hist_nseg = p->khist.nseg; p->hist_ncoll = p->khist.ncoll; p->n_hist = p->khist.n;
  memset(&p->khist, 0, sizeof p->khist);
  const uint32_t n_active = n_gen - n_inactive;
  double sum = 0.0;
  for (uint32_t g = n_inactive; g < n_gen; g++) sum = sum + p->gen_k[g];
  p->k_mean = n_active ? sum / (double)n_active : 0.0;
  double var = 0.0;
  for (uint32_t g = n_inactive; g < n_gen; g++) { double dk = p->gen_k[g] - p->k_mean; var = var + dk * dk; }
  p->k_std = n_active > 1 ? sqrt((var / (double)(n_active - 1)) / (double)n_active) : 0.0;
  p->ran = 1;
  return ORC_OK;
}

int orc_run_k_eigenvalue(orc_problem *p, uint64_t n, uint32_t n_inactive, uint32_t n_active, uint64_t seed) {
  if (!p || n == 0 || (uint64_t)n_inactive + n_active == 0 || (uint64_t)n_inactive + n_active > 65535) return ORC_EINVAL;
  uint32_t n_gen = n_inactive + n_active;
  int rc = orc_k_begin(p, 0, n, n_gen, seed); if (rc) return rc;
  uint64_t *gn = (uint64_t *)calloc(n_gen, 8), *gm = (uint64_t *)calloc(n_gen, 8);
  int64_t *gp = (int64_t *)calloc(n_gen, 8), *gpc = (int64_t *)calloc(n_gen, 8);
  double *gk = (double *)calloc(n_gen, 8);
  double k_prev = 1.0;
  uint32_t done = 0;
  for (uint32_t g = 0; g < n_gen && !rc; g++) {
    int64_t sums[4];
    int last = (g + 1 == n_gen);
    rc = orc_k_generation(p, g, g >= n_inactive, k_prev, last, sums);
    if (rc) break;
    double k = ((double)sums[0] * (1.0 / p->scale)) / (double)sums[2];       /* D2 */
    gn[g] = (uint64_t)sums[2]; gm[g] = (uint64_t)sums[3]; gp[g] = sums[0]; gpc[g] = sums[1]; gk[g] = k;
    done = g + 1;
    if (sums[3] == 0) { rc = ORC_ESTATE; break; }
    if (last) break;
    /* population control: m = floor(N/M + xi) copies per site, unit weights */
    double pr = (double)n / (double)sums[3];
    uint64_t n_next = 0;
    rc = orc_k_popctrl(p, g + 1, pr, &n_next);
    k_prev = k;
    if (!rc && n_next == 0) rc = ORC_ESTATE;
  }
  if (!rc) rc = orc_k_end(p, n_gen, n_inactive, gn, gm, gp, gpc, gk);
  else { for (uint32_t g = 0; g < done; g++) { p->gen_n[g] = gn[g]; p->gen_m[g] = gm[g]; p->gen_p[g] = gp[g]; p->gen_pc[g] = gpc[g]; p->gen_k[g] = gk[g]; } p->n_gen = done; }
  free(gn); free(gm); free(gp); free(gpc); free(gk);
  return rc;
}

int orc_tally_sizes(const orc_problem *p, orc_sizes *o) {
  if (!p || !o) return ORC_EINVAL;
  o->n_bins = p->n_bins; o->n_gen = p->n_gen; o->n_hist = p->n_hist; o->n_bank = p->n_bank;
  return ORC_OK;
}

int orc_read_tallies(const orc_problem *p, orc_tallies *t) {
  if (!p || !t) return ORC_EINVAL;
  if (!p->ran) return ORC_ESTATE;
  if (t->flux) memcpy(t->flux, p->flux, p->n_bins * 8);
  if (t->coll) memcpy(t->coll, p->coll, p->n_bins * 8);
  memcpy(t->leak, p->leak, sizeof p->leak); memcpy(t->totals, p->totals, sizeof p->totals);
  t->k_mean = p->k_mean; t->k_std = p->k_std;
  if (t->gen_n) memcpy(t->gen_n, p->gen_n, p->n_gen * 8);
  if (t->gen_m) memcpy(t->gen_m, p->gen_m, p->n_gen * 8);
  if (t->gen_p) memcpy(t->gen_p, p->gen_p, p->n_gen * 8);
  if (t->gen_pc) memcpy(t->gen_pc, p->gen_pc, p->n_gen * 8);
  if (t->gen_k) memcpy(t->gen_k, p->gen_k, p->n_gen * 8);
  if (t->hist_id) memcpy(t->hist_id, p->hist_id, p->n_hist * 8);
  if (t->hist_nseg) memcpy(t->hist_nseg, p->hist_nseg, p->n_hist * 4);
  if (t->hist_ncoll) memcpy(t->hist_ncoll, p->hist_ncoll, p->n_hist * 4);
  if (t->bank) memcpy(t->bank, p->bank, p->n_bank * sizeof(orc_site));
  return ORC_OK;
}
