/* orc.h — TEST INFRASTRUCTURE ONLY.
 *
 * History-based CPU oracle for the event-based Monte Carlo transport hot path of
 * arxiv 2506.00263 ("a single iteration of the typical history-based
 * execution loop ... a single segment of transport"; PAPER.md:121 move + tallies,
 * collision, surface crossing; PAPER.md:101 k-eigenvalue cycles with population
 * control; PAPER.md:67 order-independent hash RNG).  The paper fixes the structure of
 * the loop, not the physics formulas: every formula follows the numbered readings in
 * DESIGN.md section 3 (N = numerics, R = RNG keying, G = geometry, X = cross sections,
 * B = birth, T = transport segment, D = drivers).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  It shares no source, header or table with the CUDA path
 * (paper_2506_00263_b200/csrc, include/tdr.h); the struct layouts below are declared
 * here independently.
 *
 * Parity pins (tests/test_oracle_pins.py): Philox block vs cuRAND host generator;
 * det_log vs libm; closed forms (collisions/history = St/Sa, flux = 1/Sa, k_inf,
 * multigroup k_inf eigenvalue, slab transmission exp(-St L)); exact integer balance;
 * CE kinematics means; Watt mean; brute-force replay of histories from raw draws.
 * Parity unpinned: heterogeneous k and flux shapes of the pin-cell / C5G7-shape / CE
 * workloads (no printed values exist in the paper).
 */
#ifndef ORC_H
#define ORC_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define ORC_MAX_RINGS 4
#define ORC_MAX_NUC 4
#define ORC_MAX_CSURF 6

enum { ORC_OK = 0, ORC_EINVAL = -1, ORC_ENOMEM = -2, ORC_ECAPACITY = -4, ORC_ELOST = -5,
       ORC_EOVERFLOW = -6, ORC_ESTATE = -7 };

typedef struct orc_geometry {
  int32_t nx, ny, nz;
  const double *xplanes, *yplanes, *zplanes; /* nx+1, ny+1, nz+1 ascending; ends may be +-inf */
  const double *cx, *cy;                     /* nx, ny: cylinder axes of each lattice column */
  const int32_t *cell_univ;                  /* [nz][ny][nx] universe index */
  int32_t bc[6];                             /* -x,+x,-y,+y,-z,+z : 0 vacuum, 1 reflective */
  int32_t n_univ;
  const int32_t *univ_nrings;                /* n_univ */
  const double *univ_radius;                 /* n_univ*ORC_MAX_RINGS ascending */
  const int32_t *univ_mat;                   /* n_univ*(ORC_MAX_RINGS+1): ring 0..nrings */
  int32_t mesh_n[3];
  const double *mesh_x, *mesh_y, *mesh_z;    /* mesh_n[a]+1 planes covering the domain */
  int32_t by_group;                          /* MG: energy axis of the tally = group */
  int32_t n_ebins;                           /* CE: energy bins (>=1) */
  const double *e_edges;                     /* CE: n_ebins+1 ascending */
  int32_t src_kind;                          /* 0 point (src_lo), 1 box */
  double src_lo[3], src_hi[3];
  int32_t src_dir_kind;                      /* 0 isotropic, 1 fixed src_dir */
  double src_dir[3];
  int32_t src_energy_kind;                   /* 0 group, 1 mono, 2 watt(of nuclide src_index) */
  int32_t src_index;                         /* group or nuclide */
  double src_energy;
  int32_t tally_scale_log2;
  int32_t n_tbins;                           /* time-dependent fixed source: time bins (0 = time-independent) */
  const double *t_edges;                     /* n_tbins+1 ascending; t_edges[0] = emission time, t_edges[n_tbins] = census */
  int32_t implicit_capture;                  /* fixed source: capture by weight reduction + weight roulette (the closeout event) */
  double w_roulette, w_survive;              /* roulette below w_roulette; survivors get w_survive */
  /* general cells (readings C1-C6): a universe with univ_nrings[u] == -1 is a list of cells, each the
   * intersection of up to ORC_MAX_CSURF half-spaces of surfaces given in the frame of the lattice cell
   * (X = x - cx[ix], Y = y - cy[iy], Z = z); the particle's `ring` then holds its cell within the universe */
  int32_t n_surf;
  const int32_t *surf_kind;                  /* n_surf: 0 plane aX + bY + cZ = d; 1 sphere centre (a,b,c) radius d; 2 z-cylinder axis (a,b) radius d */
  const double *surf_coef;                   /* n_surf*4: a, b, c, d */
  int32_t n_cell;
  const int32_t *univ_cell0, *univ_ncell;    /* n_univ: first cell / number of cells (<= 255) of a general universe */
  const int32_t *cell_nsurf;                 /* n_cell: 1..ORC_MAX_CSURF */
  const int32_t *cell_surf;                  /* n_cell*ORC_MAX_CSURF: +(s+1) = the side f_s >= 0, -(s+1) = the side f_s < 0 */
  const int32_t *cell_mat;                   /* n_cell */
} orc_geometry;

typedef struct orc_materials {
  int32_t n_mat;
  int32_t G;                                 /* 0 => continuous energy */
  const double *sig_t, *sig_s, *sig_f, *nu, *chi; /* MG: [m][g], [m][g][g'], [m][g] ... */
  const int32_t *mat_nnuc;                   /* CE: n_mat */
  const int32_t *mat_nuc;                    /* CE: n_mat*ORC_MAX_NUC */
  const double *mat_dens;                    /* CE: n_mat*ORC_MAX_NUC */
  const double *speed;                       /* MG, time-dependent runs: speed of group g (cm per time unit), [G] */
} orc_materials;

typedef struct orc_xs_tables {
  int32_t n_grid, n_nuc;
  const double *energy;                      /* n_grid strictly increasing */
  const double *A;                           /* n_nuc */
  const double *sig_s, *sig_c, *sig_f;       /* [nuc][n_grid] */
  const double *nu, *watt_a, *watt_b;        /* n_nuc */
} orc_xs_tables;

typedef struct orc_site {                    /* 48 bytes */
  double x, y, z;
  uint64_t id;
  int16_t ix, iy, iz, mx, my, mz;
  uint8_t ring, src, depth, it;             /* it: time bin (time-dependent fixed source), else 0 */
} orc_site;

typedef struct orc_sizes {
  uint64_t n_bins;      /* flux / coll length = mesh bins * energy bins */
  uint64_t n_gen;       /* generations run (0 for fixed source) */
  uint64_t n_hist;      /* per-history records available */
  uint64_t n_bank;      /* sites in the last fission bank */
} orc_sizes;

enum { ORC_T_NSEG = 0, ORC_T_NCOLL, ORC_T_NCROSS, ORC_T_NABS, ORC_T_NFIS, ORC_T_NLEAK,
       ORC_T_NBORN, ORC_T_NDROPPED, ORC_T_NDIRFAIL, ORC_T_DIGEST, ORC_T_NSITES, ORC_T_NCENSUS, ORC_T_NROULETTE, ORC_T_COUNT = 16 };

typedef struct orc_tallies {                 /* all buffers caller-allocated; NULL = skip */
  int64_t *flux, *coll;                      /* n_bins */
  int64_t leak[6];
  uint64_t totals[ORC_T_COUNT];
  double k_mean, k_std;
  uint64_t *gen_n, *gen_m;                   /* n_gen */
  int64_t *gen_p, *gen_pc;                   /* n_gen */
  double *gen_k;                             /* n_gen */
  uint64_t *hist_id; uint32_t *hist_nseg, *hist_ncoll; /* n_hist */
  orc_site *bank;                            /* n_bank */
} orc_tallies;

typedef struct orc_problem orc_problem;

int orc_init_problem(const orc_geometry *, const orc_materials *, const orc_xs_tables *, orc_problem **out);
int orc_run_fixed_source(orc_problem *, uint64_t n_particles, uint64_t seed);
int orc_run_k_eigenvalue(orc_problem *, uint64_t n_particles, uint32_t n_inactive, uint32_t n_active, uint64_t seed);
/* one share of a run split over several processes by contiguous id ranges */
int orc_run_fixed_source_range(orc_problem *, uint64_t first_id, uint64_t n_particles, uint64_t seed);
int orc_k_begin(orc_problem *, uint64_t first_id, uint64_t n_local, uint32_t n_gen, uint64_t seed);
int orc_k_generation(orc_problem *, uint32_t gen, int active, double k_prev, int keep_hist, int64_t sums[4]); /* P, Pc, N_local, M_local */
int orc_k_popctrl(orc_problem *, uint32_t gen_next, double pr, uint64_t *n_next);
int orc_k_end(orc_problem *, uint32_t n_gen, uint32_t n_inactive, const uint64_t *gen_n, const uint64_t *gen_m, const int64_t *gen_p,
              const int64_t *gen_pc, const double *gen_k);
int orc_tally_sizes(const orc_problem *, orc_sizes *out);
int orc_read_tallies(const orc_problem *, orc_tallies *out);
void orc_free_problem(orc_problem *);
int orc_set_threads(int n);                  /* returns threads that will be used */

/* unit-level entry points used only by the pins */
void orc_philox(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
double orc_draw(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, uint32_t purpose, uint32_t j);
uint64_t orc_derive_id(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, uint32_t tag);
double orc_det_log(double x);
int orc_iso_dir(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, double out[3]);
double orc_watt(uint64_t seed, uint64_t id, uint32_t gen, double a, double b);
void orc_scatter_ce(uint64_t seed, uint64_t id, uint32_t gen, uint32_t seg, double A, double E,
                    const double dir_in[3], double *E_out, double dir_out[3]);
double orc_dist_cyl(double X, double Y, double u, double v, double R, int inside);
/* readings C2, C3: value of the surface function (negative inside) and distance to the surface from the given side */
double orc_surf_eval(int kind, const double *coef, double X, double Y, double Z);
double orc_surf_dist(int kind, const double *coef, double X, double Y, double Z, double u, double v, double w, int negative_side);
int32_t orc_grid_index(const double *grid, int32_t n, double E);

#ifdef __cplusplus
}
#endif
#endif
