/* tdr.h — C ABI of the B200 event-based Monte Carlo transport library (libtdr.so).
 *
 * Method: event-based neutron transport with thread-data remapping (TDR), arxiv 2506.00263:
 *   - stack-based remapping (section 3.1): per-event index stacks, warp-collective
 *     push with one atomic per warp, one kernel launch per non-empty stack, make_work when drained;
 *   - asynchronous remapping (section 3.2): one persistent kernel, per-warp stash of
 *     work links in shared memory, spill/fetch through global link queues claimed by atomic swap;
 *   - monolithic ("fused") and decomposed ("split") task schemes (section 4).
 * The four calls named by BASELINE.json north_star are tdr_init_problem, tdr_run_fixed_source,
 * tdr_run_k_eigenvalue and tdr_read_tallies; the rest make them usable.  The numbered readings
 * (N,R,G,X,B,T,D) that fix the physics where the paper is silent are in DESIGN.md section 3.
 *
 * Conventions: every pointer inside tdr_geometry / tdr_materials / tdr_xs_tables is a HOST pointer;
 * tdr_init_problem copies what it needs (the caller may free at once).  tdr_tallies holds HOST
 * buffers allocated by the caller (sizes from tdr_tally_sizes; NULL = skip).  The only DEVICE
 * pointer in the interface is the workspace given to tdr_bind_workspace, which stays owned by the
 * caller (torch) and must outlive the runs.  All calls return 0 or a negative TDR_E* code and
 * never throw; tdr_last_error() gives a thread-local message.  run_* return after the stream has
 * drained.  There is no CPU fallback: without a CUDA device every run_* returns TDR_ECUDA.
 */
#ifndef TDR_H
#define TDR_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define TDR_MAX_RINGS 4
#define TDR_MAX_NUC 4
#define TDR_MAX_CSURF 6

enum { TDR_OK = 0, TDR_EINVAL = -1, TDR_ENOMEM = -2, TDR_ECUDA = -3, TDR_ECAPACITY = -4, TDR_ELOST = -5,
       TDR_EOVERFLOW = -6, TDR_ESTATE = -7 };

/* Geometry (G1-G7): rectilinear lattice of nx*ny*nz cells; each cell holds a universe of
 * concentric z-cylinders about (cx[ix], cy[iy]); tally mesh and source. */
typedef struct tdr_geometry {
  int32_t nx, ny, nz;
  const double *xplanes, *yplanes, *zplanes; /* nx+1, ny+1, nz+1 ascending; outer ones may be +-inf */
  const double *cx, *cy;                     /* nx, ny */
  const int32_t *cell_univ;                  /* [nz][ny][nx] */
  int32_t bc[6];                             /* faces -x,+x,-y,+y,-z,+z: 0 vacuum, 1 reflective */
  int32_t n_univ;
  const int32_t *univ_nrings;                /* n_univ, each <= TDR_MAX_RINGS */
  const double *univ_radius;                 /* n_univ*TDR_MAX_RINGS ascending */
  const int32_t *univ_mat;                   /* n_univ*(TDR_MAX_RINGS+1), ring 0 (innermost) .. nrings */
  int32_t mesh_n[3];
  const double *mesh_x, *mesh_y, *mesh_z;    /* mesh_n[a]+1 planes; must cover the lattice box */
  int32_t by_group;                          /* multigroup: tally energy axis = group */
  int32_t n_ebins;                           /* continuous energy: number of energy bins */
  const double *e_edges;                     /* n_ebins+1 */
  int32_t src_kind;                          /* 0 point at src_lo, 1 uniform box [src_lo, src_hi] */
  double src_lo[3], src_hi[3];
  int32_t src_dir_kind;                      /* 0 isotropic, 1 fixed src_dir */
  double src_dir[3];
  int32_t src_energy_kind;                   /* 0 group src_index, 1 mono src_energy, 2 Watt of nuclide src_index */
  int32_t src_index;
  double src_energy;
  int32_t tally_scale_log2;                  /* S: tallies are llrint(v * 2^S) summed in int64 */
  /* time-dependent fixed source (readings TD1-TD6): time-mesh tally + census */
  int32_t n_tbins;                           /* 0 = time-independent; <= 255 */
  const double *t_edges;                     /* n_tbins+1 ascending: emission time ... census time */
  /* implicit capture + weight roulette, the `closeout` of the paper's decomposed scheme (readings W1-W4);
   * fixed-source runs only */
  int32_t implicit_capture;                  /* 0 = analog (weights identically 1) */
  double w_roulette, w_survive;              /* roulette below w_roulette; a survivor continues with w_survive */
  /* general cells (readings C1-C6): a universe with univ_nrings[u] == -1 is a list of cells, each the
   * intersection of up to TDR_MAX_CSURF half-spaces of surfaces given in the frame of the lattice cell (X = x - cx[ix],
   * Y = y - cy[iy], Z = z); the particle's `ring` then holds its cell within the universe.  All HOST arrays, copied at init. */
  int32_t n_surf;                            /* 0 = none */
  const int32_t *surf_kind;                  /* n_surf: 0 plane aX + bY + cZ = d; 1 sphere centre (a,b,c) radius d; 2 z-cylinder axis (a,b) radius d */
  const double *surf_coef;                   /* n_surf*4: a, b, c, d */
  int32_t n_cell;
  const int32_t *univ_cell0, *univ_ncell;    /* n_univ: first cell / number of cells (<= 255) of a general universe */
  const int32_t *cell_nsurf;                 /* n_cell: 1..TDR_MAX_CSURF */
  const int32_t *cell_surf;                  /* n_cell*TDR_MAX_CSURF: +(s+1) = the side f_s >= 0, -(s+1) = the side f_s < 0 */
  const int32_t *cell_mat;                   /* n_cell */
} tdr_geometry;

typedef struct tdr_materials {
  int32_t n_mat;
  int32_t G;                                 /* groups; 0 = continuous energy */
  const double *sig_t, *sig_s, *sig_f, *nu, *chi; /* MG: [m][g], [m][g from][g to], [m][g] */
  const int32_t *mat_nnuc;                   /* CE: n_mat */
  const int32_t *mat_nuc;                    /* CE: n_mat*TDR_MAX_NUC nuclide indices */
  const double *mat_dens;                    /* CE: n_mat*TDR_MAX_NUC atom densities (1/b-cm) */
  const double *speed;                       /* MG, time-dependent runs only: speed of group g, [G] (CE: 1.3831592e6 cm/s x sqrt(E/eV)) */
} tdr_materials;

typedef struct tdr_xs_tables {               /* CE only; NULL for multigroup */
  int32_t n_grid, n_nuc;
  const double *energy;                      /* n_grid strictly increasing (union grid) */
  const double *A;                           /* n_nuc */
  const double *sig_s, *sig_c, *sig_f;       /* [nuc][n_grid] barns */
  const double *nu, *watt_a, *watt_b;        /* n_nuc */
} tdr_xs_tables;

typedef struct tdr_site {                    /* fission-bank / source-bank record, 48 bytes */
  double x, y, z;
  uint64_t id;
  int16_t ix, iy, iz, mx, my, mz;
  uint8_t ring, src, depth, it;              /* it: time bin (time-dependent fixed source), else 0 */
} tdr_site;

typedef struct tdr_sizes {
  uint64_t n_bins;                           /* flux / coll length */
  uint64_t n_gen;                            /* generations run (0 after a fixed-source run) */
  uint64_t n_hist;                           /* per-history records kept */
  uint64_t n_bank;                           /* sites in the last generation's fission bank */
} tdr_sizes;

enum { TDR_T_NSEG = 0, TDR_T_NCOLL, TDR_T_NCROSS, TDR_T_NABS, TDR_T_NFIS, TDR_T_NLEAK, TDR_T_NBORN,
       TDR_T_NDROPPED, TDR_T_NDIRFAIL, TDR_T_DIGEST, TDR_T_NSITES, TDR_T_NCENSUS, TDR_T_NROULETTE, TDR_T_COUNT = 16 };

typedef struct tdr_tallies {                 /* HOST buffers, caller-allocated; NULL = skip */
  int64_t *flux, *coll;                      /* n_bins, bin = (((it*nz_m+mz)*ny_m+my)*nx_m+mx)*n_e + e (it = 0 without a time mesh) */
  int64_t leak[6];
  uint64_t totals[TDR_T_COUNT];
  double k_mean, k_std;
  uint64_t *gen_n, *gen_m;                   /* n_gen: starters, bank sites */
  int64_t *gen_p, *gen_pc;                   /* n_gen: track-length / collision production, fixed point */
  double *gen_k;                             /* n_gen */
  uint64_t *hist_id; uint32_t *hist_nseg, *hist_ncoll; /* n_hist, any order */
  tdr_site *bank;                            /* n_bank, any order */
} tdr_tallies;

typedef struct tdr_diag {
  uint64_t kernel_launches;                  /* kernels launched by the last run_* */
  uint64_t iterations;                       /* stack scheme: remap iterations; async: persistent launches */
  uint64_t events[8];                        /* kernel-level events: source, step|lookup, move, tally, collide, surface, popctrl, - */
  uint64_t spills, fetches, make_work_calls; /* async scheme */
  double gpu_ms;                             /* CUDA-event time of the last run_* body */
  double step_ms;                            /* CUDA-event time summed over the dominant kernel's launches */
  uint64_t step_launches;
} tdr_diag;

typedef struct tdr_problem tdr_problem;

/* Copy the problem to the device, derive tables (MG cdfs, CE hash).  TDR_EINVAL on bad input. */
int tdr_init_problem(const tdr_geometry *, const tdr_materials *, const tdr_xs_tables *, tdr_problem **out);
/* keys: "scheme" = stack|async; "decomposition" = fused|split|hybrid; "window" = particles in flight;
 * "stash_links" (async, links per warp, 8..64); "slots_per_warp" (async); "sync_every" (stack: remap iterations per
 * counter read-back); "blocks_per_sm"; "keep_history" = 0|1; "time_kernels" = 0|1; "idle_timeout_s" (async watchdog);
 * "seg_per_event" (async fused: segments per step event); "seg_per_launch", "drain_below" (stack); "lockstep",
 * "async_threads" (async); "id_offset" (fixed source: ids id_offset .. id_offset+n-1, for sharding one source over several GPUs);
 * "step_lockstep" = -1|0|1 (stack: CTA-wide lockstep of the segments inside k_step; -1 = auto: multigroup only);
 * "device_loop" = 1|0 (stack: the remap loop runs as a CUDA-graph WHILE node without the host | host-driven batches of sync_every);
 * "stash" = auto|index|particle|shared, "pool_slots", "ps_threads" (async: which stash).
 * decomposition = fused (monolithic step) | split (five events) | hybrid (step + collide). */
int tdr_set_option(tdr_problem *, const char *key, const char *value);
int tdr_workspace_bytes(const tdr_problem *, uint64_t n_particles, uint64_t *bytes);
/* device_ptr: DEVICE memory of at least `bytes` (256-byte aligned); cuda_stream: cudaStream_t. */
int tdr_bind_workspace(tdr_problem *, void *device_ptr, uint64_t bytes, void *cuda_stream);
/* Fixed-source run (PAPER.md:103 [section 4]: "a uniform 14 MeV source ... run across a range of source particle counts [and]
 * temporal tally resolutions"; reading D1): source ids id_offset .. id_offset+n-1, generation 0, secondaries followed to
 * extinction (or to the census of a time mesh).  HOST scalars; results stay on the device until tdr_read_tallies.
 * Errors: TDR_ESTATE without a workspace, TDR_ENOMEM if it is too small, TDR_ECAPACITY / TDR_ELOST / TDR_EOVERFLOW from the device. */
int tdr_run_fixed_source(tdr_problem *, uint64_t n_particles, uint64_t seed);
/* k-eigenvalue run (PAPER.md:101 [section 4]: "k-eigenvalue simulations, using splitting roulette population control to bound
 * storage requirements for particle data ... the first ... cycles inactive and the remaining cycles active"; reading D2): power
 * iteration over n_inactive + n_active generations of about n_particles, k per generation from the track-length estimator,
 * tallies over the active generations only.  Same error behaviour as above; TDR_ESTATE if the population dies out. */
int tdr_run_k_eigenvalue(tdr_problem *, uint64_t n_particles, uint32_t n_inactive, uint32_t n_active, uint64_t seed);
/* D2 in steps, for ONE k-eigenvalue problem shared by several GPUs (one process each; the paper's counterpart is
 * MPI replication over 4 V100s).  Every process holds a contiguous share of the source:
 *   tdr_k_begin(first_id, n_local, n_gen, seed)             generation-0 ids first_id .. first_id + n_local - 1
 *   tdr_k_generation(gen, active, k_prev, last, sums)       runs the local share; sums = { P, Pc, N_local, M_local } (fixed point)
 *   -- the caller adds the four sums over all processes (one 32-byte all-reduce) and forms k_g = P 2^-S / N, pr = N_target / M --
 *   tdr_k_population_control(gen_next, pr, &n_next)         controls the LOCAL bank with the GLOBAL ratio pr; sites stay where they are
 *   tdr_k_end(...)                                          stores the global per-generation results for tdr_read_tallies
 * Results are bit-identical for any number of shares; tdr_run_k_eigenvalue is this loop with one share.  HOST pointers. */
int tdr_k_begin(tdr_problem *, uint64_t first_id, uint64_t n_local, uint32_t n_gen, uint64_t seed);
int tdr_k_generation(tdr_problem *, uint32_t gen, int active, double k_prev, int last, int64_t sums[4]);
int tdr_k_population_control(tdr_problem *, uint32_t gen_next, double pr, uint64_t *n_next);
int tdr_k_end(tdr_problem *, uint32_t n_gen, uint32_t n_inactive, const uint64_t *gen_n, const uint64_t *gen_m, const int64_t *gen_p,
              const int64_t *gen_pc, const double *gen_k);
int tdr_tally_sizes(const tdr_problem *, tdr_sizes *out);
/* The `finalize` side of the method (PAPER.md:65 [section 3]: results leave the device once, after the last event): copies the
 * int64 fixed-point tallies, leak counts, totals, per-generation sums, per-history records and the last fission bank into the
 * caller's HOST buffers (NULL = skip; sizes from tdr_tally_sizes).  TDR_ESTATE before any completed run. */
int tdr_read_tallies(const tdr_problem *, tdr_tallies *out);
int tdr_read_diagnostics(const tdr_problem *, tdr_diag *out);
void tdr_free_problem(tdr_problem *);
const char *tdr_last_error(void);

/* Unit-level device entry points (used by the parity tests of the primitives): all pointers DEVICE.
 * out[i] = det_log(x[i]); out[i] = draw(seed, id[i], gen, seg, purpose, j). */
int tdr_dev_det_log(const double *x, double *out, uint64_t n, void *cuda_stream);
int tdr_dev_draw(uint64_t seed, const uint64_t *id, uint32_t gen, uint32_t seg, uint32_t purpose, uint32_t j,
                 double *out, uint64_t n, void *cuda_stream);

/* Measured ceilings for the roofline: what = 0 -> fp64 DFMA rate in TFLOP/s, 1 -> L2-resident copy bandwidth in
 * GB/s (read + write bytes).  `value` is a HOST pointer; the call allocates and frees its own device scratch. */
int tdr_measure_peak(int what, double *value, void *cuda_stream);

/* Population control (reading D2; "splitting roulette population control") on caller-owned DEVICE arrays: site i
 * of bank[0..n_bank) gets m_i = floor(pr + xi(site id, gen_next, 0, POPCTRL, 0)) copies (at most 2048) with the derived ids of
 * reading R4.  next[0..min(total, next_cap)) receives the copies, count_dev[0] the total wanted (total > next_cap = overflow,
 * the caller's check).  All pointers DEVICE; asynchronous on cuda_stream.
 *
 * tdr_dev_popctrl: the library's k_popctrl as the k-eigenvalue driver runs it (copies in any order); it cudaMallocs and frees its
 * counter and synchronises the stream.
 *
 * tdr_dev_popctrl_noalloc: the same result from a variant that allocates NOTHING — for callers that cannot call cudaMalloc (code
 * under CUDA-graph capture, tight serving loops, harnesses that forbid it).  No cudaMalloc / cudaFree / allocating routine, no
 * synchronisation, no host-side read: three kernel launches on cuda_stream.  Its scratch (per-site copy counts, their prefix sums,
 * the total) lives in ONE file-scope `static __device__` array of 4 MiB + 256 B that every GPU which loads the library holds until
 * exit; its device address is resolved once per device (cudaGetSymbolAddress, on the first call with that device current: make
 * that first call outside a capture).  Limit: n_bank <= TDR_NOALLOC_MAX_SITES, beyond it TDR_EINVAL with a message.  The copies
 * come out in bank order (site 0's copies first), which the allocating path does not promise.  Every call shares the scratch, which
 * keeps the previous call's contents (each call rewrites what it reads); two calls that overlap on the GPU (different streams or
 * processes' threads without ordering) RACE: order them on one stream or with events. */
#define TDR_NOALLOC_MAX_SITES 524288
int tdr_dev_popctrl(const tdr_site *bank, uint64_t n_bank, tdr_site *next, uint64_t next_cap, uint64_t *count_dev,
                    uint64_t seed, uint32_t gen_next, double pr, void *cuda_stream);
int tdr_dev_popctrl_noalloc(const tdr_site *bank, uint64_t n_bank, tdr_site *next, uint64_t next_cap, uint64_t *count_dev,
                            uint64_t seed, uint32_t gen_next, double pr, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
