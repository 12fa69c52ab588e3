// tdr_api.cu — C ABI (include/tdr.h) and host drivers (D1 fixed source, D2 k-eigenvalue) of libtdr.so.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -fmad=false -lineinfo -shared -Xcompiler -fPIC
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>
#include <nvtx3/nvToolsExt.h>      // header-only NVTX 3: ranges around runs, generations and population control (no-ops without a tool)
#include "tdr_stack.cuh"
#include "tdr_split.cuh"
#include "tdr_async.cuh"
#include "tdr_pstash.cuh"
#include "tdr_cstash.cuh"
#include "tdr_peaks.cuh"

static thread_local char g_err[512] = "";
struct NvtxRange { explicit NvtxRange(const char *name) { nvtxRangePushA(name); } ~NvtxRange() { nvtxRangePop(); } };

static int fail(int code, const char *fmt, ...) {
  va_list ap; va_start(ap, fmt); vsnprintf(g_err, sizeof g_err, fmt, ap); va_end(ap);
  return code;
}
#define CK(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(TDR_ECUDA, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); } while (0)

struct tdr_problem {
  DevProb dp;
  std::vector<void *> dev_allocs;          // problem tables (cudaMalloc'd at init)
  bool ce = false;
  int S = 24;
  // options
  int scheme = 0;                          // 0 stack, 1 async
  int split = 0;                           // 0 fused, 1 split, 2 hybrid (step + collide events)
  u64 window = 1ull << 20;
  int stash_links = 8;
  int blocks_per_sm = 0;                   // 0 = occupancy query
  int keep_history = -1;                   // -1 auto (n <= 2e6)
  int time_kernels = 0;
  int lockstep = 1, async_threads = 512;   // async scheme: CTA-wide lockstep phase; threads per CTA (256 or 512)
  int seg_per_launch = 0;                  // stack fused/hybrid: segments per particle per k_step launch; 0 = auto (6 multigroup, 12 continuous energy)
  int force_spill = 0;                     // async stress option (tests): warps always believe another one is starved
  int seg_per_event = 0;                   // async fused: segments per step event before remapping; 0 = auto (2 multigroup, 5 continuous energy)
  int slots_per_warp = 128;                // async scheme: window slots a warp may claim for itself
  int idle_timeout_s = 30;                 // async scheme watchdog (seconds without progress while idle)
  u64 id_offset = 0;                       // fixed source: ids id_offset .. id_offset + n - 1
  int drain_below = 65536;                 // stack scheme, k-mode: population below which the tail is drained in one launch
  int sync_every = 6;                      // stack scheme: remap iterations launched per counter read-back
  int stash = -1;                          // async scheme: -1 = auto (multigroup: 2, continuous energy: 0); 0 = index stash per warp (slot numbers; state SoA in global memory), 1 = whole-particle stash per warp, 2 = whole-particle stash shared by the CTA
  int pool_slots = 64;                     // particle stash: particle slots per warp
  int ps_threads = PS_THREADS;             // particle stash: threads per CTA
  u64 bank_cap_opt = 0;                    // tests: fission-bank capacity in sites (0 = 2.5 n + 4096)
  u64 arena_links_opt = 0;                 // tests: global link arena of the asynchronous scheme (0 = 2 W/32 + 4096)
  // workspace
  char *ws = nullptr; u64 ws_bytes = 0; cudaStream_t stream = nullptr;
  // carved pointers (valid during/after a run)
  Soa soa; u32 *stacks[EV_COUNT]; u64 *ctr; DevOut out; tdr_site *bank, *srcbank, *sec; double *sec_time = nullptr, *sec_w = nullptr;
  u64 bank_cap = 0, src_cap = 0, sec_cap = 0, hist_cap = 0, W = 0;
  u64 *hist_id; u32 *hist_nseg, *hist_ncoll;
  AsyncMem am; PsMem pm;
  // results on host
  bool ran = false;
  std::vector<u64> gen_n, gen_m; std::vector<i64> gen_p, gen_pc; std::vector<double> gen_k;
  double k_mean = 0, k_std = 0; u64 n_hist = 0, n_bank = 0;
  tdr_diag diag;
  int num_sms = 148;
  u64 *h_ctr = nullptr;                    // pinned readback
  // D2 in steps
  u64 k_first = 0, k_nsrc = 0, k_seed = 0, k_last_bank = 0; u32 k_ngen = 0; bool k_keep = false; double k_clock_ms = 0;
  std::vector<cudaEvent_t> ev_pool; size_t ev_used = 0;
  // stack scheme, device-driven remap loop: a CUDA graph with one WHILE node (built per run), its capture stream, and the
  // DevRun the graph's kernels read
  int device_loop = 1;
  int step_lockstep = -1;                  // stack fused/hybrid: the CTA's warps run the segments of a k_step tile in lockstep; -1 = auto (multigroup only)
  cudaGraph_t sg_graph = nullptr; cudaGraphExec_t sg_exec = nullptr; cudaStream_t sg_capture = nullptr; int sg_per_pass = 0;
  DevRun *run_dev = nullptr;
};

static void drop_stack_graph(tdr_problem *p) {
  if (p->sg_exec) { cudaGraphExecDestroy(p->sg_exec); p->sg_exec = nullptr; }
  if (p->sg_graph) { cudaGraphDestroy(p->sg_graph); p->sg_graph = nullptr; }
}

const char *tdr_last_error(void) { return g_err; }

template <class T>
static int upload(tdr_problem *p, const T *src, size_t n, const T **dst) {
  void *d = nullptr;
  size_t bytes = (n ? n : 1) * sizeof(T);
  CK(cudaMalloc(&d, bytes));
  p->dev_allocs.push_back(d);
  if (n) CK(cudaMemcpy(d, src, n * sizeof(T), cudaMemcpyHostToDevice));
  *dst = (const T *)d;
  return 0;
}

void tdr_free_problem(tdr_problem *p) {
  if (!p) return;
  for (void *d : p->dev_allocs) cudaFree(d);
  for (cudaEvent_t e : p->ev_pool) cudaEventDestroy(e);
  drop_stack_graph(p);
  if (p->sg_capture) cudaStreamDestroy(p->sg_capture);
  if (p->h_ctr) cudaFreeHost(p->h_ctr);
  delete p;
}

int tdr_init_problem(const tdr_geometry *g, const tdr_materials *m, const tdr_xs_tables *x, tdr_problem **out) {
  if (!g || !m || !out) return fail(TDR_EINVAL, "null argument");
  if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->n_univ < 1 || m->n_mat < 1) return fail(TDR_EINVAL, "empty geometry or materials");
  if (g->nx > 32767 || g->ny > 32767 || g->nz > 32767) return fail(TDR_EINVAL, "lattice too large for 16-bit indices");
  if (m->n_mat > 255 || m->G > 255 || m->G < 0) return fail(TDR_EINVAL, "too many materials or groups");
  if (m->G == 0 && !x) return fail(TDR_EINVAL, "continuous energy needs xs_tables");
  if (g->tally_scale_log2 < 0 || g->tally_scale_log2 > 40) return fail(TDR_EINVAL, "tally_scale_log2 out of range");
  if (g->n_tbins < 0 || g->n_tbins > 255) return fail(TDR_EINVAL, "n_tbins in [0,255]");
  if (g->implicit_capture && !(g->w_roulette > 0.0 && g->w_survive >= g->w_roulette)) return fail(TDR_EINVAL, "implicit capture needs 0 < w_roulette <= w_survive");
  if (g->n_tbins > 0) {
    if (!g->t_edges) return fail(TDR_EINVAL, "time mesh without t_edges");
    for (int k = 0; k < g->n_tbins; k++) if (!(g->t_edges[k] < g->t_edges[k + 1])) return fail(TDR_EINVAL, "time edges are not strictly ascending");
    if (m->G > 0 && !m->speed) return fail(TDR_EINVAL, "a multigroup time-dependent run needs group speeds");
    if (m->G > 0) for (int a = 0; a < m->G; a++) if (!(m->speed[a] > 0.0)) return fail(TDR_EINVAL, "group speeds must be positive");
  }
  const double *mp[3] = { g->mesh_x, g->mesh_y, g->mesh_z };
  const double *lp[3] = { g->xplanes, g->yplanes, g->zplanes };
  const int ln[3] = { g->nx, g->ny, g->nz };
  if (!g->xplanes || !g->yplanes || !g->zplanes || !g->cx || !g->cy || !g->cell_univ || !g->univ_nrings || !g->univ_radius ||
      !g->univ_mat || !mp[0] || !mp[1] || !mp[2]) return fail(TDR_EINVAL, "null geometry array");
  for (int a = 0; a < 3; a++) {
    if (g->mesh_n[a] < 1 || g->mesh_n[a] > 32767) return fail(TDR_EINVAL, "bad mesh size");
    if (!(mp[a][0] <= lp[a][0]) || !(mp[a][g->mesh_n[a]] >= lp[a][ln[a]])) return fail(TDR_EINVAL, "tally mesh must cover the lattice box");
  }
  // every index table is dereferenced on the device: range-check it here (a bad index would be an illegal address there)
  for (int a = 0; a < 3; a++) {
    for (int k = 0; k < ln[a]; k++) if (!(lp[a][k] < lp[a][k + 1])) return fail(TDR_EINVAL, "lattice planes of axis %d are not strictly ascending", a);
    for (int k = 0; k < g->mesh_n[a]; k++) if (!(mp[a][k] < mp[a][k + 1])) return fail(TDR_EINVAL, "mesh planes of axis %d are not strictly ascending", a);
  }
  if (g->n_surf < 0 || g->n_surf > 32767) return fail(TDR_EINVAL, "bad surface count");
  if (g->n_surf > 0) {                          // general cells: every index the device follows is checked here
    if (!g->surf_kind || !g->surf_coef || !g->univ_cell0 || !g->univ_ncell || !g->cell_nsurf || !g->cell_surf || !g->cell_mat || g->n_cell < 1)
      return fail(TDR_EINVAL, "general cells: null table");
    for (int k = 0; k < g->n_surf; k++)
      if (g->surf_kind[k] < 0 || g->surf_kind[k] > 2 || (g->surf_kind[k] > 0 && !(g->surf_coef[4 * k + 3] > 0.0))) return fail(TDR_EINVAL, "surface %d: bad kind or radius", k);
    for (int k = 0; k < g->n_cell; k++) {
      if (g->cell_nsurf[k] < 1 || g->cell_nsurf[k] > TDR_MAX_CSURF) return fail(TDR_EINVAL, "cell %d: 1..%d surfaces", k, TDR_MAX_CSURF);
      if (g->cell_mat[k] < 0 || g->cell_mat[k] >= m->n_mat) return fail(TDR_EINVAL, "cell %d names material %d of %d", k, g->cell_mat[k], m->n_mat);
      for (int j = 0; j < g->cell_nsurf[k]; j++) { const int r = g->cell_surf[k * TDR_MAX_CSURF + j]; if (r == 0 || abs(r) > g->n_surf) return fail(TDR_EINVAL, "cell %d names surface %d of %d", k, r, g->n_surf); }
    }
  }
  for (int u = 0; u < g->n_univ; u++) {
    const int nr = g->univ_nrings[u];
    if (nr == -1 && g->n_surf > 0) {
      if (g->univ_cell0[u] < 0 || g->univ_ncell[u] < 1 || g->univ_ncell[u] > 255 || g->univ_cell0[u] + g->univ_ncell[u] > g->n_cell) return fail(TDR_EINVAL, "universe %d: bad cell range", u);
      continue;
    }
    if (nr < 0 || nr > TDR_MAX_RINGS) return fail(TDR_EINVAL, "bad ring count");
    for (int r = 0; r < nr; r++) {
      const double R = g->univ_radius[u * TDR_MAX_RINGS + r];
      if (!(R > 0.0) || (r > 0 && !(R > g->univ_radius[u * TDR_MAX_RINGS + r - 1]))) return fail(TDR_EINVAL, "radii of universe %d are not positive and ascending", u);
    }
    for (int r = 0; r <= nr; r++) {
      const int mt = g->univ_mat[u * (TDR_MAX_RINGS + 1) + r];
      if (mt < 0 || mt >= m->n_mat) return fail(TDR_EINVAL, "universe %d names material %d of %d", u, mt, m->n_mat);
    }
  }
  for (int iz = 0; iz < g->nz; iz++) for (int iy = 0; iy < g->ny; iy++) for (int ix = 0; ix < g->nx; ix++) {
    const int u = g->cell_univ[((size_t)iz * g->ny + iy) * g->nx + ix];
    if (u < 0 || u >= g->n_univ) return fail(TDR_EINVAL, "cell (%d,%d,%d) names universe %d of %d", ix, iy, iz, u, g->n_univ);
    const int nr = g->univ_nrings[u];
    if (nr > 0) {                             // G7: a particle on a cell face is outside every ring
      const double R = g->univ_radius[u * TDR_MAX_RINGS + nr - 1];
      const double hx0 = g->cx[ix] - g->xplanes[ix], hx1 = g->xplanes[ix + 1] - g->cx[ix], hy0 = g->cy[iy] - g->yplanes[iy], hy1 = g->yplanes[iy + 1] - g->cy[iy];
      if (!(R < hx0) || !(R < hx1) || !(R < hy0) || !(R < hy1)) return fail(TDR_EINVAL, "outer radius of universe %d reaches the face of cell (%d,%d)", u, ix, iy);
    }
  }
  for (int f = 0; f < 6; f++) if (g->bc[f] != 0 && g->bc[f] != 1) return fail(TDR_EINVAL, "bc must be 0 (vacuum) or 1 (reflective)");
  if (g->src_kind < 0 || g->src_kind > 1 || g->src_dir_kind < 0 || g->src_dir_kind > 1 || g->src_energy_kind < 0 || g->src_energy_kind > 2)
    return fail(TDR_EINVAL, "bad source kind");
  if (m->G > 0) {
    if (!m->sig_t || !m->sig_s || !m->sig_f || !m->nu || !m->chi) return fail(TDR_EINVAL, "null multigroup table");
    if (g->src_energy_kind != 0 || g->src_index < 0 || g->src_index >= m->G) return fail(TDR_EINVAL, "multigroup source must name a group below G");
    // the table is staged to shared memory by every kernel: it has to fit beside the private tallies and the stash
    if ((size_t)m->n_mat * m->G * (MGROW(m->G) + 1) * sizeof(double) > 96 * 1024) return fail(TDR_EINVAL, "multigroup table too large for shared memory (n_mat*G*(G+6)*8 > 96 KB)");
  } else {
    if (!m->mat_nnuc || !m->mat_nuc || !m->mat_dens || !x->energy || !x->A || !x->sig_s || !x->sig_c || !x->sig_f || !x->nu || !x->watt_a || !x->watt_b)
      return fail(TDR_EINVAL, "null continuous-energy table");
    if (x->n_grid < 2 || x->n_nuc < 1 || x->n_nuc > 255) return fail(TDR_EINVAL, "bad CE tables");
    for (int k = 0; k < m->n_mat; k++) {
      if (m->mat_nnuc[k] < 1 || m->mat_nnuc[k] > TDR_MAX_NUC) return fail(TDR_EINVAL, "material %d has %d nuclides (1..%d)", k, m->mat_nnuc[k], TDR_MAX_NUC);
      for (int n = 0; n < m->mat_nnuc[k]; n++)
        if (m->mat_nuc[k * TDR_MAX_NUC + n] < 0 || m->mat_nuc[k * TDR_MAX_NUC + n] >= x->n_nuc) return fail(TDR_EINVAL, "material %d names nuclide %d of %d", k, m->mat_nuc[k * TDR_MAX_NUC + n], x->n_nuc);
    }
    for (int i = 0; i + 1 < x->n_grid; i++) if (!(x->energy[i] < x->energy[i + 1])) return fail(TDR_EINVAL, "energy grid is not strictly increasing at %d", i);
    if (g->n_ebins < 1 || !g->e_edges) return fail(TDR_EINVAL, "continuous energy needs n_ebins >= 1 and e_edges");
    for (int i = 0; i < g->n_ebins; i++) if (!(g->e_edges[i] < g->e_edges[i + 1])) return fail(TDR_EINVAL, "energy-bin edges are not strictly ascending");
    if (g->src_energy_kind == 0) return fail(TDR_EINVAL, "continuous-energy source must be mono or Watt");
    if (g->src_energy_kind == 2 && (g->src_index < 0 || g->src_index >= x->n_nuc)) return fail(TDR_EINVAL, "Watt source names nuclide %d of %d", g->src_index, x->n_nuc);
  }
  int dev_count = 0;
  if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) return fail(TDR_ECUDA, "no CUDA device: this library has no CPU fallback");
  tdr_problem *p = new tdr_problem();
  memset(&p->dp, 0, sizeof p->dp); memset(&p->diag, 0, sizeof p->diag); memset(&p->soa, 0, sizeof p->soa);
  DevProb &D = p->dp;
  int rc = 0;
#define UP(src, n, dst) if (!rc) rc = upload(p, src, (size_t)(n), &dst)
  D.nx = g->nx; D.ny = g->ny; D.nz = g->nz; D.n_univ = g->n_univ; D.G = m->G; D.n_mat = m->n_mat; D.by_group = g->by_group;
  memcpy(D.bc, g->bc, sizeof D.bc); memcpy(D.mesh_n, g->mesh_n, sizeof D.mesh_n);
  UP(g->xplanes, g->nx + 1, D.xp); UP(g->yplanes, g->ny + 1, D.yp); UP(g->zplanes, g->nz + 1, D.zp);
  UP(g->cx, g->nx, D.cx); UP(g->cy, g->ny, D.cy);
  UP(g->cell_univ, (size_t)g->nx * g->ny * g->nz, D.cell_univ);
  UP(g->univ_nrings, g->n_univ, D.univ_nr); UP(g->univ_radius, g->n_univ * TDR_MAX_RINGS, D.univ_rad);
  UP(g->univ_mat, g->n_univ * (TDR_MAX_RINGS + 1), D.univ_mat);
  for (int a = 0; a < 3; a++) UP(mp[a], g->mesh_n[a] + 1, D.mesh[a]);
  D.n_surf = g->n_surf; D.n_cell = g->n_surf > 0 ? g->n_cell : 0;
  if (g->n_surf > 0) {
    UP(g->surf_kind, g->n_surf, D.surf_kind); UP(g->surf_coef, 4 * g->n_surf, D.surf_coef);
    UP(g->univ_cell0, g->n_univ, D.univ_cell0); UP(g->univ_ncell, g->n_univ, D.univ_ncell);
    UP(g->cell_nsurf, g->n_cell, D.cell_nsurf); UP(g->cell_surf, g->n_cell * TDR_MAX_CSURF, D.cell_surf); UP(g->cell_mat, g->n_cell, D.cell_mat);
  }
  D.n_t = g->n_tbins; D.implicit = g->implicit_capture != 0; D.w_roulette = g->w_roulette; D.w_survive = g->w_survive;
  if (D.n_t > 0) { UP(g->t_edges, D.n_t + 1, D.t_edges); if (m->G > 0) UP(m->speed, m->G, D.speed); }
  D.src_kind = g->src_kind; D.src_dir_kind = g->src_dir_kind; D.src_energy_kind = g->src_energy_kind; D.src_index = g->src_index;
  memcpy(D.src_lo, g->src_lo, 24); memcpy(D.src_hi, g->src_hi, 24); memcpy(D.src_dir, g->src_dir, 24);
  D.src_energy = g->src_energy; D.scale = ldexp(1.0, g->tally_scale_log2); p->S = g->tally_scale_log2;
  p->ce = (m->G == 0);
  if (!p->ce) {
    D.n_e = g->by_group ? m->G : 1;
    // X1: derived rows [sig_t, sig_s_tot, sig_c, nu*sig_f, nu, cdf...] + chi cdf
    int G = m->G, M = m->n_mat, row = MGROW(G);
    std::vector<double> t((size_t)M * G * row + (size_t)M * G);
    for (int k = 0; k < M; k++) {
      double cc = 0.0;
      for (int a = 0; a < G; a++) {
        double *r = &t[(size_t)(k * G + a) * row];
        double acc = 0.0;
        for (int b = 0; b < G; b++) { acc = acc + m->sig_s[(k * G + a) * G + b]; r[5 + b] = acc; }
        double st = m->sig_t[k * G + a], sf = m->sig_f[k * G + a], nu = m->nu[k * G + a];
        double sa = st - acc;
        r[0] = st; r[1] = acc; r[2] = sa - sf; r[3] = nu * sf; r[4] = nu;
        cc = cc + m->chi[k * G + a]; t[(size_t)M * G * row + k * G + a] = cc;
      }
    }
    D.mg_doubles = (int)t.size();
    UP(t.data(), t.size(), D.mg);
  } else {
    if (g->n_ebins < 1 || x->n_grid < 2 || x->n_nuc < 1 || x->n_nuc > 255) { tdr_free_problem(p); return fail(TDR_EINVAL, "bad CE tables"); }
    D.n_e = g->n_ebins; UP(g->e_edges, g->n_ebins + 1, D.e_edges);
    D.n_grid = x->n_grid; D.n_nuc = x->n_nuc;
    UP(m->mat_nnuc, m->n_mat, D.mat_nnuc); UP(m->mat_nuc, m->n_mat * TDR_MAX_NUC, D.mat_nuc); UP(m->mat_dens, m->n_mat * TDR_MAX_NUC, D.mat_dens);
    UP(x->energy, x->n_grid, D.grid); UP(x->A, x->n_nuc, D.A); UP(x->nu, x->n_nuc, D.nuc_nu); UP(x->watt_a, x->n_nuc, D.wa); UP(x->watt_b, x->n_nuc, D.wb);
    std::vector<double4> rec((size_t)x->n_nuc * x->n_grid);
    for (size_t i = 0; i < rec.size(); i++) rec[i] = make_double4(x->sig_s[i], x->sig_c[i], x->sig_f[i], 0.0);
    UP(rec.data(), rec.size(), D.xs);
    D.grid_lo = x->energy[0]; D.grid_hi = x->energy[x->n_grid - 1];
    if (!(D.grid_lo > 0.0)) { tdr_free_problem(p); return fail(TDR_EINVAL, "energy grid must be positive"); }
    // X3: bucket = top bits (exponent + 7 mantissa bits) of E; hash[b] = largest i with grid[i] <= lower edge of b
    u64 blo, bhi; memcpy(&blo, &D.grid_lo, 8); memcpy(&bhi, &D.grid_hi, 8);
    D.hash_bmin = (u32)(blo >> 45); D.hash_n = (u32)(bhi >> 45) - D.hash_bmin + 1;
    std::vector<u32> h(D.hash_n + 1 + ((D.hash_n + 1) & 1u));            // (an even number of words: staged to shared memory as doubles)
    int i = 0;
    for (u32 b = 0; b <= D.hash_n; b++) {
      u64 eb = ((u64)(D.hash_bmin + b)) << 45; double edge; memcpy(&edge, &eb, 8);
      while (i + 1 < x->n_grid && x->energy[i + 1] <= edge) i++;
      h[b] = (u32)i;
    }
    if (!h.empty()) h.back() = h[D.hash_n];
    UP(h.data(), h.size(), D.hash);
    if (h.size() * 4 > 64 * 1024) { tdr_free_problem(p); return fail(TDR_EINVAL, "energy grid spans too many binades for the staged hash (%zu bytes)", h.size() * 4); }
    D.mg = reinterpret_cast<const double *>(D.hash); D.mg_doubles = (int)(h.size() / 2);   // the block k_step, k_drain and k_async stage to shared memory (stage_mg)
  }
#undef UP
  if (rc) { tdr_free_problem(p); return rc; }
  D.n_bins = (u64)(D.n_t > 0 ? D.n_t : 1) * D.mesh_n[0] * D.mesh_n[1] * D.mesh_n[2] * D.n_e;
  cudaDeviceProp prop; int dev = 0; cudaGetDevice(&dev);
  if (cudaGetDeviceProperties(&prop, dev) == cudaSuccess) p->num_sms = prop.multiProcessorCount;
  if (cudaMallocHost((void **)&p->h_ctr, 64 * sizeof(u64)) != cudaSuccess) { tdr_free_problem(p); return fail(TDR_ECUDA, "cudaMallocHost failed"); }
  *out = p;
  return TDR_OK;
}

int tdr_set_option(tdr_problem *p, const char *key, const char *value) {
  if (!p || !key || !value) return fail(TDR_EINVAL, "null argument");
  std::string k(key), v(value);
  if (k == "scheme") { if (v == "stack") p->scheme = 0; else if (v == "async") p->scheme = 1; else return fail(TDR_EINVAL, "scheme must be stack|async"); }
  else if (k == "decomposition") { if (v == "fused") p->split = 0; else if (v == "split") p->split = 1; else if (v == "hybrid") p->split = 2; else return fail(TDR_EINVAL, "decomposition must be fused|split|hybrid"); }
  else if (k == "window") { long long w = atoll(value); if (w < 32) return fail(TDR_EINVAL, "window too small"); if (w > 0xFFFFFFC0ll) return fail(TDR_EINVAL, "window above 2^32 - 64: slot indices are 32-bit"); p->window = (u64)w; }
  else if (k == "stash_links") { int n = atoi(value); if (n < 8 || n > 64) return fail(TDR_EINVAL, "stash_links in [8,64]"); p->stash_links = n; }
  else if (k == "blocks_per_sm") p->blocks_per_sm = atoi(value);
  else if (k == "keep_history") p->keep_history = atoi(value);
  else if (k == "time_kernels") p->time_kernels = atoi(value);
  else if (k == "lockstep") p->lockstep = atoi(value) != 0;
  else if (k == "async_threads") { int n = atoi(value); if (n < 64 || n > TDR_ASYNC_MAXT || n % 32) return fail(TDR_EINVAL, "async_threads: a multiple of 32 in [64,%d]", TDR_ASYNC_MAXT); p->async_threads = n; }
  else if (k == "seg_per_launch") { int n = atoi(value); if (n < 0 || n > 1024) return fail(TDR_EINVAL, "seg_per_launch in [0,1024]"); p->seg_per_launch = n; }
  else if (k == "force_spill") p->force_spill = atoi(value) != 0;
  else if (k == "seg_per_event") { int n = atoi(value); if (n < 0 || n > 1024) return fail(TDR_EINVAL, "seg_per_event in [0,1024]"); p->seg_per_event = n; }
  else if (k == "slots_per_warp") { int n = atoi(value); if (n < 32 || n > 4096) return fail(TDR_EINVAL, "slots_per_warp in [32,4096]"); p->slots_per_warp = n; }
  else if (k == "idle_timeout_s") { int n = atoi(value); if (n < 1 || n > 3600) return fail(TDR_EINVAL, "idle_timeout_s in [1,3600]"); p->idle_timeout_s = n; }
  else if (k == "id_offset") p->id_offset = strtoull(value, nullptr, 10);
  else if (k == "drain_below") { int n = atoi(value); if (n < 0) return fail(TDR_EINVAL, "drain_below >= 0"); p->drain_below = n; }
  else if (k == "stash") { if (v == "auto") p->stash = -1; else if (v == "index") p->stash = 0; else if (v == "particle") p->stash = 1; else if (v == "shared") p->stash = 2; else return fail(TDR_EINVAL, "stash must be auto|index|particle|shared"); }
  else if (k == "pool_slots") { int n = atoi(value); if (n < 32 || n > PS_RING || n % 8) return fail(TDR_EINVAL, "pool_slots: a multiple of 8 in [32,%d]", PS_RING); p->pool_slots = n; }
  else if (k == "ps_threads") { int n = atoi(value); if (n < 32 || n > PS_THREADS || n % 32) return fail(TDR_EINVAL, "ps_threads: a multiple of 32 in [32,%d]", PS_THREADS); p->ps_threads = n; }
  else if (k == "bank_cap") p->bank_cap_opt = strtoull(value, nullptr, 10);
  else if (k == "arena_links") p->arena_links_opt = strtoull(value, nullptr, 10);
  else if (k == "device_loop") p->device_loop = atoi(value) != 0;
  else if (k == "step_lockstep") { int n = atoi(value); if (n < -1 || n > 1) return fail(TDR_EINVAL, "step_lockstep: -1 (auto), 0 or 1"); p->step_lockstep = n; }
  else if (k == "sync_every") { int n = atoi(value); if (n < 1 || n > 1024) return fail(TDR_EINVAL, "sync_every in [1,1024]"); p->sync_every = n; }
  else return fail(TDR_EINVAL, "unknown option %s", key);
  return TDR_OK;
}

// ---------------------------------------------------------------------------------- workspace layout
struct Carver {
  char *base; u64 off = 0;
  template <class T> T *take(u64 n) { off = (off + 255) & ~255ull; T *r = base ? (T *)(base + off) : nullptr; off += n * sizeof(T); return r; }
};

static u64 window_for(const tdr_problem *p, u64 n) {
  u64 cap = n + n / 4 + 4096;                 // k-mode population floats around n
  u64 w = p->window < cap ? p->window : cap;
  return (w + 31) & ~31ull;
}

static u64 layout(tdr_problem *p, u64 n, char *base, bool assign) {
  Carver c; c.base = base;
  u64 W = window_for(p, n);
  Soa s; memset(&s, 0, sizeof s);
  s.x = c.take<double>(W); s.y = c.take<double>(W); s.z = c.take<double>(W);
  s.u = c.take<double>(W); s.v = c.take<double>(W); s.w = c.take<double>(W);
  s.E = c.take<double>(p->ce ? W : 1);
  s.t = p->dp.n_t > 0 ? c.take<double>(W) : nullptr;
  s.wgt = p->dp.implicit ? c.take<double>(W) : nullptr;
  s.id = c.take<u64>(W); s.loc0 = c.take<u64>(W); s.loc1 = c.take<u64>(W);
  s.seg = c.take<u32>(W); s.ncoll = c.take<u32>(W);
  s.s_sigt = c.take<double>(W); s.s_nsf = c.take<double>(W); s.s_d = c.take<double>(W); s.s_f = c.take<double>(W);
  s.s_flags = c.take<u32>(W); s.s_gi = c.take<u32>(W);
  u32 *st[EV_COUNT];
  for (int e = 0; e < EV_COUNT; e++) st[e] = c.take<u32>(W);
  u64 *ctr = c.take<u64>(C_COUNT);
  DevRun *run_dev = c.take<DevRun>(1);
  DevOut o;
  o.flux = c.take<u64>(p->dp.n_bins); o.coll = c.take<u64>(p->dp.n_bins); o.leak = c.take<u64>(6);
  o.totals = c.take<u64>(TDR_T_COUNT); o.PPc = c.take<u64>(2); o.err = c.take<int>(1);
  u64 bank_cap = p->bank_cap_opt ? p->bank_cap_opt : 2 * n + n / 2 + 4096, src_cap = n + n / 4 + 4096, sec_cap = W + (1ull << 20);
  tdr_site *bank = c.take<tdr_site>(bank_cap), *src = c.take<tdr_site>(src_cap), *sec = c.take<tdr_site>(sec_cap);
  double *sec_time = p->dp.n_t > 0 ? c.take<double>(sec_cap) : nullptr, *sec_w = p->dp.implicit ? c.take<double>(sec_cap) : nullptr;
  u64 hist_cap = 16 * (n < 2000000 ? n : 2000000) + 4096;
  u64 *hid = c.take<u64>(hist_cap); u32 *hs = c.take<u32>(hist_cap), *hc = c.take<u32>(hist_cap);
  AsyncMem am; async_layout(c, W, sec_cap, p->arena_links_opt, am);
  PsMem pm; pstash_layout(c, W, p->arena_links_opt, p->dp.n_t > 0, p->dp.implicit != 0, pm);
  if (assign) {
    p->W = W; p->soa = s; memcpy(p->stacks, st, sizeof st); p->ctr = ctr; p->run_dev = run_dev; p->out = o;
    p->bank = bank; p->srcbank = src; p->sec = sec; p->sec_time = sec_time; p->sec_w = sec_w; p->bank_cap = bank_cap; p->src_cap = src_cap; p->sec_cap = sec_cap;
    p->hist_cap = hist_cap; p->hist_id = hid; p->hist_nseg = hs; p->hist_ncoll = hc; p->am = am; p->pm = pm;
  }
  return (c.off + 255) & ~255ull;
}

int tdr_workspace_bytes(const tdr_problem *p, uint64_t n, uint64_t *bytes) {
  if (!p || !bytes || n == 0) return fail(TDR_EINVAL, "bad argument");
  *bytes = layout(const_cast<tdr_problem *>(p), n, nullptr, false);
  return TDR_OK;
}

int tdr_bind_workspace(tdr_problem *p, void *ptr, uint64_t bytes, void *stream) {
  if (!p || !ptr || ((uintptr_t)ptr & 255)) return fail(TDR_EINVAL, "workspace must be a 256-byte aligned device pointer");
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess || at.type != cudaMemoryTypeDevice) { cudaGetLastError(); return fail(TDR_EINVAL, "workspace is not device memory"); }
  p->ws = (char *)ptr; p->ws_bytes = bytes; p->stream = (cudaStream_t)stream;
  return TDR_OK;
}

// ---------------------------------------------------------------------------------- launch helpers
// grid = SMs x resident CTAs; 0 when the kernel cannot be launched with this much dynamic shared memory (the callers turn that
// into TDR_EINVAL).  Above the default 48 KB the kernel is opted in to large shared memory first.
template <class K>
static int grid_for(tdr_problem *p, K kernel, size_t smem, int threads = 256) {
  if (smem > 48 * 1024 && cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) { cudaGetLastError(); return 0; }
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem) != cudaSuccess || occ < 1) { cudaGetLastError(); return 0; }
  const int bps = p->blocks_per_sm > 0 ? p->blocks_per_sm : occ;
  return p->num_sms * bps;
}
#define GRID_OR_FAIL(g, what) do { if ((g) < 1) return fail(TDR_EINVAL, "%s: the kernel does not fit an SM with %zu bytes of dynamic shared memory (smaller multigroup table, fewer tally bins below 257, fewer stash_links or threads)", what, smem); } while (0)

struct KTimer {                                   // optional CUDA-event bracket around the dominant kernel's launches
  tdr_problem *p; bool on;
  int n;                                          // launches inside the bracket (they run back to back on the stream)
  KTimer(tdr_problem *p_, bool dominant, int n_ = 1) : p(p_), on(p_->time_kernels && dominant), n(n_) {
    if (!on) return;
    while (p->ev_pool.size() < p->ev_used + 2) { cudaEvent_t e; cudaEventCreate(&e); p->ev_pool.push_back(e); }
    cudaEventRecord(p->ev_pool[p->ev_used], p->stream);
  }
  ~KTimer() { if (on) { cudaEventRecord(p->ev_pool[p->ev_used + 1], p->stream); p->ev_used += 2; p->diag.step_launches += n; } }
};

static void collect_kernel_times(tdr_problem *p) {
  double ms = 0;
  for (size_t i = 0; i + 1 < p->ev_used; i += 2) { float t = 0; cudaEventElapsedTime(&t, p->ev_pool[i], p->ev_pool[i + 1]); ms += t; }
  p->diag.step_ms = ms; p->ev_used = 0;
}

static int check_dev_err(tdr_problem *p, int code) {
  if (code == 0) return 0;
  const char *w = code == TDR_ECAPACITY ? "bank/stack/arena capacity exceeded" : code == TDR_ELOST ? "lost particle (no finite distance or segment overflow)" :
                  code == TDR_EOVERFLOW ? "a fixed-point tally left int64 (lower tally_scale_log2)" : "device error";
  return fail(code, "%s", w);
}

#define LAUNCH_CHECK() CK(cudaGetLastError())

// ---------------------------------------------------------------------------------- stack scheme: one remap iteration
// The kernels of remap iteration `it` on stream st: the monolithic step (fused), step + collide (hybrid) or the five event
// kernels in flow order (split; one kernel per event stack, a kernel whose stack is empty returns at once).  DEV selects
// where the kernels find their DevRun (TDR_BIND_RUN); `cap_blocks` bounds the grids by the population where it is known.
struct StackGrids { int step, coll, ev[EV_COUNT]; };

template <bool CE, bool DEV, bool EXT>
static void stack_grids(tdr_problem *p, size_t smem, StackGrids &g) {
  memset(&g, 0, sizeof g);
  if (p->split == 1) {
    g.ev[EV_LOOKUP] = grid_for(p, k_event<CE, EV_LOOKUP, DEV, EXT>, smem); g.ev[EV_MOVE] = grid_for(p, k_event<CE, EV_MOVE, DEV, EXT>, smem);
    g.ev[EV_TALLY] = grid_for(p, k_event<CE, EV_TALLY, DEV, EXT>, smem); g.ev[EV_COLLIDE] = grid_for(p, k_event<CE, EV_COLLIDE, DEV, EXT>, smem);
    g.ev[EV_SURFACE] = grid_for(p, k_event<CE, EV_SURFACE, DEV, EXT>, smem);
  } else if (p->split == 2) { g.step = grid_for(p, k_step<CE, true, DEV, EXT>, smem); g.coll = grid_for(p, k_collide<CE, DEV, EXT>, smem); }
  else g.step = grid_for(p, k_step<CE, false, DEV, EXT>, smem);
}

template <bool CE, bool DEV, bool EXT>
static int remap_iteration(tdr_problem *p, const DevRun &R, cudaStream_t st, size_t smem, const StackGrids &G, u64 it, int cap_blocks) {
  u64 *ctr = p->ctr;
  const DevRun *Rp = DEV ? p->run_dev : nullptr;
  auto cap = [&](int g) { return g < cap_blocks ? g : cap_blocks; };
  const u32 spl = (u32)(p->seg_per_launch ? p->seg_per_launch : (CE ? 12 : 6));
  const int sls = p->step_lockstep < 0 ? !CE : p->step_lockstep;       // segment lockstep inside k_step: multigroup only by default
  if (p->split == 1) {
    StackSet K; for (int e = 0; e < EV_COUNT; e++) K.s[e] = p->stacks[e];
    K.cnt = ctr + C_STACK0;
    k_event<CE, EV_LOOKUP, DEV, EXT><<<cap(G.ev[EV_LOOKUP]), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, K, EV_SURFACE);
    k_event<CE, EV_MOVE, DEV, EXT><<<cap(G.ev[EV_MOVE]), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, K, EV_LOOKUP);
    k_event<CE, EV_TALLY, DEV, EXT><<<cap(G.ev[EV_TALLY]), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, K, EV_MOVE);
    k_event<CE, EV_COLLIDE, DEV, EXT><<<cap(G.ev[EV_COLLIDE]), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, K, EV_TALLY);
    k_event<CE, EV_SURFACE, DEV, EXT><<<cap(G.ev[EV_SURFACE]), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, K, EV_COLLIDE);
    return 5;
  }
  // fused / hybrid: two index stacks, three rotating counters (in, out, the one to clear)
  if (DEV) {                                       // the kernels derive the iteration's pointers themselves: bases only
    if (p->split == 2) {
      k_step<CE, true, true, EXT><<<G.step, 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, p->stacks[0], ctr, p->stacks[1], nullptr, nullptr, p->stacks[2], nullptr, nullptr, spl, sls);
      k_collide<CE, true, EXT><<<G.coll, 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, p->stacks[2], ctr, p->stacks[0], reinterpret_cast<u64 *>(p->stacks[1]));
      return 2;
    }
    k_step<CE, false, true, EXT><<<G.step, 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, p->stacks[0], ctr, p->stacks[1], nullptr, nullptr, nullptr, nullptr, nullptr, spl, sls);
    return 1;
  }
  const int in = (int)(it % 3), out = (int)((it + 1) % 3), zr = (int)((it + 2) % 3);
  if (p->split == 2) {
    u64 *cc = ctr + C_STACK0 + 3 + (it & 1), *cz = ctr + C_STACK0 + 3 + ((it + 1) & 1);      // collide-stack counters
    k_step<CE, true, DEV, EXT><<<cap(G.step), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, p->stacks[it & 1], ctr + C_STACK0 + in,
                                                          p->stacks[(it + 1) & 1], ctr + C_STACK0 + out, ctr + C_STACK0 + zr, p->stacks[2], cc, cz, spl, sls);
    k_collide<CE, DEV, EXT><<<cap(G.coll), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, p->stacks[2], cc, p->stacks[(it + 1) & 1], ctr + C_STACK0 + out);
    return 2;
  }
  k_step<CE, false, DEV, EXT><<<cap(G.step), 256, smem, st>>>(p->dp, p->out, R, Rp, p->soa, p->stacks[it & 1], ctr + C_STACK0 + in,
                                                         p->stacks[(it + 1) & 1], ctr + C_STACK0 + out, ctr + C_STACK0 + zr, nullptr, nullptr, nullptr, spl, sls);
  return 1;
}

// the device-driven loop: graph = one WHILE node; body = ONE remap iteration + k_loop_ctl, so the condition (extinct, short
// enough to drain, error) is tested after every iteration.  Captured once per run on the library's own capture stream.
template <bool CE, bool EXT>
static int build_stack_graph(tdr_problem *p, size_t smem) {
  drop_stack_graph(p);
  if (!p->sg_capture) CK(cudaStreamCreateWithFlags(&p->sg_capture, cudaStreamNonBlocking));
  CK(cudaGraphCreate(&p->sg_graph, 0));
  cudaGraphConditionalHandle h;
  CK(cudaGraphConditionalHandleCreate(&h, p->sg_graph, 1, cudaGraphCondAssignDefault));
  cudaGraphNodeParams np = { cudaGraphNodeTypeConditional }; np.conditional.handle = h; np.conditional.type = cudaGraphCondTypeWhile; np.conditional.size = 1;
  cudaGraphNode_t node;
  CK(cudaGraphAddNode(&node, p->sg_graph, nullptr, 0, &np));
  cudaGraph_t body = np.conditional.phGraph_out[0];
  StackGrids G; stack_grids<CE, true, EXT>(p, smem, G);
  GRID_OR_FAIL(p->split == 1 ? G.ev[EV_MOVE] : G.step, "stack scheme");
  DevRun none; memset(&none, 0, sizeof none);
  CK(cudaStreamBeginCaptureToGraph(p->sg_capture, body, nullptr, nullptr, 0, cudaStreamCaptureModeRelaxed));
  const int per_pass = remap_iteration<CE, true, EXT>(p, none, p->sg_capture, smem, G, 0, 1 << 30);
  LoopCtl c; c.ctr = p->ctr; c.R = p->run_dev; c.split = p->split == 1; c.drain_below = (u64)p->drain_below;
  k_loop_ctl<<<1, 32, 0, p->sg_capture>>>(c, h);
  cudaGraph_t captured = nullptr;
  cudaError_t e = cudaStreamEndCapture(p->sg_capture, &captured);
  if (e != cudaSuccess) { drop_stack_graph(p); return fail(TDR_ECUDA, "capture of the remap loop failed: %s", cudaGetErrorString(e)); }
  e = cudaGraphInstantiate(&p->sg_exec, p->sg_graph, 0);
  if (e != cudaSuccess) { drop_stack_graph(p); return fail(TDR_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e)); }
  p->sg_per_pass = per_pass;
  return 0;
}

// ---------------------------------------------------------------------------------- stack scheme, one generation
// dynamic shared memory = [staged table (multigroup rows | continuous energy: hash buckets + energy edges) | private tally words];
// staged = false: a continuous-energy kernel that reads the block from global memory instead (stage_mg)
static size_t smem_bytes(const tdr_problem *p, bool staged = true) {
  size_t priv = p->dp.n_bins <= PRIV_MAX_BINS ? (size_t)p->dp.n_bins * 16 : 0;
  return ((p->ce && !staged) ? 0 : (size_t)p->dp.mg_doubles * sizeof(double)) + priv;
}

template <bool CE, bool EXT>
static int run_stack(tdr_problem *p, DevRun R) {
  cudaStream_t st = p->stream;
  const size_t smem = smem_bytes(p);
  u64 *ctr = p->ctr; u64 *h = p->h_ctr;
  const int g_src = grid_for(p, k_source<CE>, smem);
  GRID_OR_FAIL(g_src, "stack scheme");
  const u64 W = p->W;
  u64 h_src_next = 0, h_sec_tail = 0, h_sec_head = 0;
  auto source = [&](u32 *stack, u64 *count, u64 n_sec, u64 n) -> int {
    k_source<CE><<<g_src, 256, smem, st>>>(p->dp, p->out, R, p->soa, stack, count, h_sec_head, n_sec, h_src_next, n);
    LAUNCH_CHECK(); p->diag.kernel_launches++; p->diag.events[0] += n;
    h_sec_head += n_sec; h_src_next += n - n_sec;
    return 0;
  };
  int rc;
  const bool split = p->split == 1, dev = p->device_loop != 0;
  // the live stack between iterations: stacks[it & 1] with counter it % 3 (fused, hybrid), the LOOKUP stack (split)
  auto live_stack = [&](u64 it) { return split ? p->stacks[EV_LOOKUP] : p->stacks[it & 1]; };
  auto live_count = [&](u64 it) { return ctr + C_STACK0 + (split ? (u64)EV_LOOKUP : it % 3); };
  u64 n0 = R.src_total < W ? R.src_total : W;
  u64 it = 0, passes_seen = 0;
  if ((rc = source(live_stack(0), live_count(0), 0, n0))) return rc;
  u64 n_in = n0;
  StackGrids G;
  if (dev) { if (!p->sg_exec && (rc = build_stack_graph<CE, EXT>(p, smem))) return rc; }
  else {
    stack_grids<CE, false, EXT>(p, smem, G);
    GRID_OR_FAIL(split ? G.ev[EV_MOVE] : G.step, "stack scheme");
  }
  for (;;) {
    R.sec_limit = h_sec_tail; R.sec_head0 = h_sec_head;
    if (dev) {
      // one graph launch runs remap iterations until the population is extinct (or short enough to drain, or an error is
      // flagged); the host comes back for the tail drain, for a refill of an empty window, or to finish
      CK(cudaMemcpyAsync(p->run_dev, &R, sizeof R, cudaMemcpyHostToDevice, st));      // (pageable source: staged before the call returns)
      { KTimer tb(p, true, 0); CK(cudaGraphLaunch(p->sg_exec, st)); }
    } else {
      // the out count never exceeds the in count (dead lanes are reborn in place), so n_in bounds every launch of
      // this batch: launch `batch` remap iterations back to back and read the counters once
      const int batch = n_in * 4 > W ? 1 : p->sync_every;
      u64 blocks64 = (n_in + 255) / 256; int cap_blocks = blocks64 > (1u << 30) ? (1 << 30) : (int)blocks64;
      if (cap_blocks < 1) cap_blocks = 1;
      KTimer tb(p, true, 0);                              // one event pair per batch: the launches run back to back
      for (int b = 0; b < batch; b++) {
        const int nk = remap_iteration<CE, false, EXT>(p, R, st, smem, G, it, cap_blocks);
        LAUNCH_CHECK(); p->diag.kernel_launches += nk; p->diag.step_launches += p->time_kernels ? nk : 0;
        it++; p->diag.iterations++;
      }
    }
    CK(cudaMemcpyAsync(h, ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));
    if (dev) {
      const u64 np = h[C_PENDING] - passes_seen; passes_seen = h[C_PENDING];
      it = h[C_PENDING]; p->diag.iterations += np;
      p->diag.kernel_launches += np * (p->sg_per_pass + 1); p->diag.step_launches += p->time_kernels ? np * (p->sg_per_pass + 1) : 0;
    }
    if ((rc = check_dev_err(p, (int)h[C_COUNT - 1]))) return rc;
    const u64 alive = h[C_STACK0 + (split ? (u64)EV_LOOKUP : it % 3)];
    n_in = alive;
    h_sec_tail = h[C_SEC_TAIL];
    h_src_next = h[C_SRC_NEXT] < R.src_total ? h[C_SRC_NEXT] : R.src_total;
    h_sec_head = h[C_SEC_HEAD] < R.sec_limit ? h[C_SEC_HEAD] : R.sec_limit;          // claims past the limit got nothing
    if (dev) h_sec_head = h[C_SEC_HEAD];                                              // (k_loop_ctl has already given them back)
    const u64 pend = h_sec_tail - h_sec_head, rem = R.src_total - h_src_next;
    if (R.kmode && rem == 0 && alive > 0 && alive <= (u64)p->drain_below) {
      // tail drain: the few particles left are followed to their death in ONE launch (k_drain).  Also under the five-event
      // decomposition: after a whole iteration every survivor waits on the LOOKUP stack, i.e. at the start of a segment.
      const int blocks = (int)((alive + 63) / 64);
      if (smem > 48 * 1024) CK(cudaFuncSetAttribute(k_drain<CE, EXT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      { KTimer td(p, true); k_drain<CE, EXT><<<blocks, 64, smem, st>>>(p->dp, p->out, R, p->soa, live_stack(it), live_count(it)); }
      LAUNCH_CHECK(); p->diag.kernel_launches++; p->diag.iterations++;
      CK(cudaMemcpyAsync(h, ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
      CK(cudaStreamSynchronize(st));
      if ((rc = check_dev_err(p, (int)h[C_COUNT - 1]))) return rc;
      break;
    }
    if (alive == 0) {
      if (pend + rem == 0) break;
      u64 n = pend + rem < W ? pend + rem : W, n_sec = pend < n ? pend : n;
      R.sec_limit = h_sec_tail; R.sec_head0 = h_sec_head;
      if ((rc = source(live_stack(it), live_count(it), n_sec, n))) return rc;
      n_in = n;
    } else if (!dev && h[C_SEC_HEAD] != h_sec_head) {
      h[33] = h_sec_head;                                   // clamp the overshoot of the claim cursor (the limit grows later)
      CK(cudaMemcpyAsync(ctr + C_SEC_HEAD, h + 33, 8, cudaMemcpyHostToDevice, st));
      CK(cudaStreamSynchronize(st));
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------- asynchronous scheme, one generation
template <bool CE, int MODE, bool EXT>
static int launch_async(tdr_problem *p, const DevRun &R, size_t smem, int threads) {
  int grid = grid_for(p, k_async<CE, MODE, EXT>, smem, threads);
  GRID_OR_FAIL(grid, "asynchronous scheme");
  KTimer t(p, true);
  k_async<CE, MODE, EXT><<<grid, threads, smem, p->stream>>>(p->dp, p->out, R, p->soa, p->am, p->pm, p->stash_links, (u64)p->idle_timeout_s * 1000000000ull,
                                                        (u32)p->slots_per_warp, p->lockstep, (u32)(p->seg_per_event ? p->seg_per_event : (CE ? 5 : 2)));
  return 0;
}

template <bool CE>
static int run_async(tdr_problem *p, DevRun R) {
  cudaStream_t st = p->stream;
  const int threads = p->async_threads;
  const size_t smem = smem_bytes(p) + (threads / 32) * (size_t)STASH_WORDS(p->stash_links) * 4;
  R.defer_death = 1; R.outstanding = p->ctr + C_PENDING; R.slot_next = p->ctr + C_STACK0; R.starved = p->ctr + C_STARVED; R.W = p->W;
  if (!R.kmode) { k_ps_init<<<64, 256, 0, st>>>(p->pm, R.outstanding, R.src_total, R.starved, p->force_spill ? (1ull << 40) : 0ull); LAUNCH_CHECK(); }   // the links of secondaries
  k_async_init<<<64, 256, 0, st>>>(p->am, R.outstanding, R.src_total, R.slot_next, R.starved, p->force_spill ? (1ull << 40) : 0ull);
  LAUNCH_CHECK();
  const bool ext = p->dp.n_t > 0 || p->dp.implicit || p->dp.n_surf > 0;           // the build with the time mesh / weights compiled in (ProbX)
  int lrc;
  if (ext) lrc = p->split == 1 ? launch_async<CE, 1, true>(p, R, smem, threads) : p->split == 2 ? launch_async<CE, 2, true>(p, R, smem, threads) : launch_async<CE, 0, true>(p, R, smem, threads);
  else lrc = p->split == 1 ? launch_async<CE, 1, false>(p, R, smem, threads) : p->split == 2 ? launch_async<CE, 2, false>(p, R, smem, threads) : launch_async<CE, 0, false>(p, R, smem, threads);
  if (lrc) return lrc;
  LAUNCH_CHECK(); p->diag.kernel_launches += 2; p->diag.iterations++;
  u64 *h = p->h_ctr;
  CK(cudaMemcpyAsync(h, p->ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(h + 40, p->am.actr, AC_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  p->diag.spills += h[40 + AC_SPILLS]; p->diag.fetches += h[40 + AC_FETCHES]; p->diag.make_work_calls += h[40 + AC_MAKEWORK];
  p->diag.events[1] += h[40 + AC_EVENTS]; p->diag.events[0] += R.src_total;
  int rc;
  if ((int)h[C_COUNT - 1] == TDR_ELOST && h[40 + AC_DBG + 5])
    return fail(TDR_ELOST, "async watchdog: warp %llu busy too long: link count %llu ev %llu nrun %llu nfree %llu iter %llu events %llu delta %lld outstanding %llu",
                h[40 + AC_DBG], h[41 + AC_DBG], h[42 + AC_DBG], h[43 + AC_DBG], h[44 + AC_DBG], h[45 + AC_DBG], h[46 + AC_DBG], (long long)h[47 + AC_DBG], h[C_PENDING]);
  if ((rc = check_dev_err(p, (int)h[C_COUNT - 1]))) return rc;
  if (h[C_PENDING] != 0) return fail(TDR_ESTATE, "asynchronous scheme left %llu particles outstanding", h[C_PENDING]);
  return 0;
}

// ---------------------------------------------------------------------------------- asynchronous scheme, whole-particle stash
template <bool CE, int MODE>
static int launch_pstash(tdr_problem *p, const DevRun &R, size_t smem, int threads) {
  auto kernel = k_pstash<CE, MODE>;
  CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int bps = p->blocks_per_sm;
  if (bps <= 0) { if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, threads, smem) != cudaSuccess || bps < 1) return fail(TDR_EINVAL, "particle stash: %zu bytes of shared memory per CTA do not fit an SM (fewer pool_slots or ps_threads)", smem); }
  KTimer t(p, true);
  kernel<<<p->num_sms * bps, threads, smem, p->stream>>>(p->dp, p->out, R, p->pm, p->pool_slots, (u64)p->idle_timeout_s * 1000000000ull);
  return 0;
}

template <bool CE>
static int run_pstash(tdr_problem *p, DevRun R) {
  cudaStream_t st = p->stream;
  const int threads = p->ps_threads;
  const size_t smem = smem_bytes(p, false) + (threads / 32) * PsPool<CE>::bytes(p->pool_slots);
  if (smem > 227 * 1024) return fail(TDR_EINVAL, "particle stash needs %zu bytes of shared memory per CTA (limit 227 KB)", smem);
  R.defer_death = 1; R.outstanding = p->ctr + C_PENDING; R.starved = p->ctr + C_STARVED; R.W = p->W;
  k_ps_init<<<64, 256, 0, st>>>(p->pm, R.outstanding, R.src_total, R.starved, p->force_spill ? (1ull << 40) : 0ull);
  LAUNCH_CHECK();
  int rc = p->split == 2 ? launch_pstash<CE, 2>(p, R, smem, threads) : launch_pstash<CE, 0>(p, R, smem, threads);
  if (rc) return rc;
  LAUNCH_CHECK(); p->diag.kernel_launches += 2; p->diag.iterations++;
  u64 *h = p->h_ctr;
  CK(cudaMemcpyAsync(h, p->ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(h + 40, p->pm.ctr, PC_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  p->diag.spills += h[40 + PC_SPILLS]; p->diag.fetches += h[40 + PC_FETCHES]; p->diag.make_work_calls += h[40 + PC_EV_BIRTH];
  p->diag.events[0] += h[40 + PC_LN_BIRTH]; p->diag.events[2] += h[40 + PC_LN_MOVE]; p->diag.events[4] += h[40 + PC_LN_COLLIDE];
  p->diag.events[1] += h[40 + PC_EV_MOVE] + h[40 + PC_EV_COLLIDE] + h[40 + PC_EV_BIRTH];     // warp-level events (32 lanes each at best)
  if ((rc = check_dev_err(p, (int)h[C_COUNT - 1]))) return rc;
  if (!R.kmode && (h[C_PENDING] != 0 || h[40 + PC_GWORK] != 0))
    return fail(TDR_ESTATE, "particle stash left %llu particles outstanding, %llu links queued", h[C_PENDING], h[40 + PC_GWORK]);
  return 0;
}

// ---------------------------------------------------------------------------------- asynchronous scheme, stash shared by the CTA
template <bool CE, int MODE>
static int launch_cstash(tdr_problem *p, const DevRun &R, size_t smem, int threads, int ns) {
  auto kernel = k_cstash<CE, MODE>;
  CK(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int bps = p->blocks_per_sm;
  if (bps <= 0) { if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bps, kernel, threads, smem) != cudaSuccess || bps < 1) return fail(TDR_EINVAL, "shared stash: %zu bytes of shared memory per CTA do not fit an SM (fewer pool_slots or ps_threads)", smem); }
  KTimer t(p, true);
  kernel<<<p->num_sms * bps, threads, smem, p->stream>>>(p->dp, p->out, R, p->pm, ns, (u64)p->idle_timeout_s * 1000000000ull);
  return 0;
}

template <bool CE>
static int run_cstash(tdr_problem *p, DevRun R) {
  cudaStream_t st = p->stream;
  const int threads = p->ps_threads <= CS_THREADS ? p->ps_threads : CS_THREADS;
  const int ns = p->pool_slots * (threads / 32);
  if (ns > 32768) return fail(TDR_EINVAL, "shared stash: more than 32768 slots per CTA");
  const size_t smem = smem_bytes(p, false) + CsPool<CE>::bytes(ns);
  if (smem > 227 * 1024) return fail(TDR_EINVAL, "shared stash needs %zu bytes of shared memory per CTA (limit 227 KB)", smem);
  R.defer_death = 1; R.outstanding = p->ctr + C_PENDING; R.starved = p->ctr + C_STARVED; R.W = p->W;
  k_ps_init<<<64, 256, 0, st>>>(p->pm, R.outstanding, R.src_total, R.starved, p->force_spill ? (1ull << 40) : 0ull);
  LAUNCH_CHECK();
  int rc = p->split == 2 ? launch_cstash<CE, 2>(p, R, smem, threads, ns) : launch_cstash<CE, 0>(p, R, smem, threads, ns);
  if (rc) return rc;
  LAUNCH_CHECK(); p->diag.kernel_launches += 2; p->diag.iterations++;
  u64 *h = p->h_ctr;
  CK(cudaMemcpyAsync(h, p->ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(h + 40, p->pm.ctr, PC_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  p->diag.spills += h[40 + PC_SPILLS]; p->diag.fetches += h[40 + PC_FETCHES]; p->diag.make_work_calls += h[40 + PC_EV_BIRTH];
  p->diag.events[0] += h[40 + PC_LN_BIRTH]; p->diag.events[2] += h[40 + PC_LN_MOVE]; p->diag.events[4] += h[40 + PC_LN_COLLIDE];
  p->diag.events[1] += h[40 + PC_EV_MOVE] + h[40 + PC_EV_COLLIDE] + h[40 + PC_EV_BIRTH];
  if ((rc = check_dev_err(p, (int)h[C_COUNT - 1]))) return rc;
  if (!R.kmode && (h[C_PENDING] != 0 || h[40 + PC_GWORK] != 0))
    return fail(TDR_ESTATE, "shared stash left %llu particles outstanding, %llu links queued", h[C_PENDING], h[40 + PC_GWORK]);
  return 0;
}

static int overflow_check(tdr_problem *p);
static int run_async_any(tdr_problem *p, DevRun &R);

// one generation (or the whole fixed-source run) under the selected scheme
static int run_generation(tdr_problem *p, DevRun &R) {
  NvtxRange nvtx(R.kmode ? "tdr generation" : "tdr fixed-source transport");
  cudaStream_t st = p->stream;
  CK(cudaMemsetAsync(p->ctr, 0, C_COUNT * 8, st));
  CK(cudaMemsetAsync(p->out.PPc, 0, 16, st));
  R.src_next = p->ctr + C_SRC_NEXT; R.sec_tail = p->ctr + C_SEC_TAIL; R.sec_head = p->ctr + C_SEC_HEAD;
  R.bank_count = p->ctr + C_BANK; R.hist_count = p->ctr + C_HIST;
  R.sec = p->sec; R.sec_time = p->sec_time; R.sec_w = p->sec_w; R.sec_cap = p->sec_cap; R.sec_limit = 0; R.sec_head0 = 0;
  R.bank = p->bank; R.bank_cap = p->bank_cap; R.err = p->out.err;
  R.hist_id = p->hist_id; R.hist_nseg = p->hist_nseg; R.hist_ncoll = p->hist_ncoll;
  if (p->scheme == 0) {
    const bool ext = p->dp.n_t > 0 || p->dp.implicit || p->dp.n_surf > 0;
    int rc = p->ce ? (ext ? run_stack<true, true>(p, R) : run_stack<true, false>(p, R)) : (ext ? run_stack<false, true>(p, R) : run_stack<false, false>(p, R));
    return rc ? rc : overflow_check(p);
  }
  { int rc = run_async_any(p, R); return rc ? rc : overflow_check(p); }
}

static int overflow_check(tdr_problem *p) {
  if (p->dp.n_bins <= PRIV_MAX_BINS) return 0;               // block-private tallies are checked at every flush; the scheme's own read-back saw the flag
  k_overflow_check<<<64, 256, 0, p->stream>>>(p->out.flux, p->out.coll, p->dp.n_bins, p->out.err);
  LAUNCH_CHECK();
  CK(cudaMemcpyAsync(p->h_ctr + 32, p->out.err, sizeof(int), cudaMemcpyDeviceToHost, p->stream)); CK(cudaStreamSynchronize(p->stream));
  return check_dev_err(p, *(int *)(p->h_ctr + 32));
}

static int run_async_any(tdr_problem *p, DevRun &R) {
  // auto: the shared particle stash where the path is instruction bound (multigroup); the index stash where it is bound by
  // cross-section gathers and wants the L1 that a particle stash would take (continuous energy) — DESIGN.md section 6
  const bool ext = p->dp.n_t > 0 || p->dp.implicit || p->dp.n_surf > 0;
  if (ext && p->stash > 0) return fail(TDR_EINVAL, "time-dependent, implicit-capture and general-cell runs use the index stash (stash = auto|index)");
  const int stash = p->stash >= 0 ? p->stash : ((p->ce || ext) ? 0 : 2);
  if (stash == 2 && p->split != 1) return p->ce ? run_cstash<true>(p, R) : run_cstash<false>(p, R);
  if (stash == 1 && p->split != 1) return p->ce ? run_pstash<true>(p, R) : run_pstash<false>(p, R);
  return p->ce ? run_async<true>(p, R) : run_async<false>(p, R);      // index stash; the five-event decomposition always
}

static int begin_run(tdr_problem *p, u64 n) {
  if (!p || n == 0) return fail(TDR_EINVAL, "bad argument");
  if (!p->ws) return fail(TDR_ESTATE, "no workspace bound (tdr_bind_workspace)");
  u64 need = layout(p, n, nullptr, false);
  if (need > p->ws_bytes) return fail(TDR_ENOMEM, "workspace too small: need %llu bytes, have %llu", need, (u64)p->ws_bytes);
  layout(p, n, p->ws, true);
  p->out.err = (int *)(p->ctr + (C_COUNT - 1));
  cudaStream_t st = p->stream;
  CK(cudaMemsetAsync(p->out.flux, 0, p->dp.n_bins * 8, st)); CK(cudaMemsetAsync(p->out.coll, 0, p->dp.n_bins * 8, st));
  CK(cudaMemsetAsync(p->out.leak, 0, 48, st)); CK(cudaMemsetAsync(p->out.totals, 0, TDR_T_COUNT * 8, st));
  p->ran = false; p->gen_n.clear(); p->gen_m.clear(); p->gen_p.clear(); p->gen_pc.clear(); p->gen_k.clear();
  p->k_mean = p->k_std = 0; p->n_hist = p->n_bank = 0;
  memset(&p->diag, 0, sizeof p->diag); p->ev_used = 0;
  drop_stack_graph(p);                         // the graph's kernel arguments are this run's pointers and options
  return 0;
}

struct RunClock {
  cudaEvent_t a, b; cudaStream_t st;
  RunClock(cudaStream_t s) : st(s) { cudaEventCreate(&a); cudaEventCreate(&b); cudaEventRecord(a, st); }
  double stop() { cudaEventRecord(b, st); cudaEventSynchronize(b); float ms = 0; cudaEventElapsedTime(&ms, a, b); return ms; }
  ~RunClock() { cudaEventDestroy(a); cudaEventDestroy(b); }
};

int tdr_run_fixed_source(tdr_problem *p, uint64_t n, uint64_t seed) {
  int rc = begin_run(p, n); if (rc) return rc;
  RunClock clk(p->stream);
  DevRun R; memset(&R, 0, sizeof R);
  R.seed = seed; R.gen = 0; R.kmode = 0; R.active = 1; R.k_prev = 1.0; R.src_sites = 0; R.sites = nullptr; R.src_total = n;
  R.id_offset = p->id_offset;
  bool keep = p->keep_history < 0 ? n <= 2000000 : p->keep_history != 0;
  R.hist_cap = keep ? p->hist_cap : 0;
  if ((rc = run_generation(p, R))) return rc;
  CK(cudaMemcpyAsync(p->h_ctr, p->ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, p->stream));
  p->diag.gpu_ms = clk.stop();
  collect_kernel_times(p);
  if (keep && p->h_ctr[C_HIST] > p->hist_cap) return fail(TDR_ECAPACITY, "history record buffer overflow");
  p->n_hist = keep ? p->h_ctr[C_HIST] : 0;
  p->ran = true;
  return TDR_OK;
}

// ---------------------------------------------------------------------------------- D2 in steps (one problem on several GPUs)
int tdr_k_begin(tdr_problem *p, uint64_t first_id, uint64_t n_local, uint32_t n_gen, uint64_t seed) {
  if (n_gen == 0 || n_gen > 65535) return fail(TDR_EINVAL, "bad generation counts");
  if (p && (p->dp.n_t > 0 || p->dp.implicit)) return fail(TDR_EINVAL, "the time mesh and implicit capture belong to fixed-source runs");
  int rc = begin_run(p, n_local ? n_local : 1); if (rc) return rc;
  p->k_first = first_id; p->k_nsrc = n_local; p->k_seed = seed; p->k_ngen = n_gen; p->k_last_bank = 0;
  p->k_keep = p->keep_history < 0 ? n_local <= 2000000 : p->keep_history != 0;
  p->k_clock_ms = 0.0;
  return TDR_OK;
}

int tdr_k_generation(tdr_problem *p, uint32_t gen, int active, double k_prev, int last, int64_t sums[4]) {
  if (!p || !sums || !p->ws) return fail(TDR_EINVAL, "bad argument");
  RunClock clk(p->stream);
  cudaStream_t st = p->stream;
  DevRun R; memset(&R, 0, sizeof R);
  R.seed = p->k_seed; R.gen = gen; R.kmode = 1; R.active = active != 0; R.k_prev = k_prev;
  R.src_sites = gen > 0; R.sites = p->srcbank; R.src_total = p->k_nsrc; R.id_offset = p->k_first;
  R.hist_cap = (p->k_keep && last) ? p->hist_cap : 0;
  int rc;
  if (p->k_nsrc > 0) { if ((rc = run_generation(p, R))) return rc; }
  else { CK(cudaMemsetAsync(p->ctr, 0, C_COUNT * 8, st)); CK(cudaMemsetAsync(p->out.PPc, 0, 16, st)); }     // a rank without a share
  CK(cudaMemcpyAsync(p->h_ctr, p->ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(p->h_ctr + 16, p->out.PPc, 16, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  const u64 M = p->h_ctr[C_BANK];
  if (M > p->bank_cap) return fail(TDR_ECAPACITY, "fission bank overflow");
  sums[0] = (i64)p->h_ctr[16]; sums[1] = (i64)p->h_ctr[17]; sums[2] = (i64)p->k_nsrc; sums[3] = (i64)M;
  p->k_last_bank = M;
  if (last) { p->n_bank = M; p->n_hist = R.hist_cap ? p->h_ctr[C_HIST] : 0; }
  p->k_clock_ms += clk.stop();
  return TDR_OK;
}

int tdr_k_population_control(tdr_problem *p, uint32_t gen_next, double pr, uint64_t *n_next) {
  if (!p || !n_next || !p->ws) return fail(TDR_EINVAL, "bad argument");
  NvtxRange nvtx("tdr population control");
  RunClock clk(p->stream);
  cudaStream_t st = p->stream;
  const u64 M = p->k_last_bank;
  CK(cudaMemsetAsync(p->ctr + C_NEXT_BANK, 0, 8, st));
  if (M) { k_popctrl<<<p->num_sms * 4, 256, 0, st>>>(p->bank, M, p->srcbank, p->src_cap, p->ctr + C_NEXT_BANK, p->k_seed, gen_next, pr, p->out.err); LAUNCH_CHECK(); p->diag.kernel_launches++; p->diag.events[6] += M; }
  CK(cudaMemcpyAsync(p->h_ctr, p->ctr, C_COUNT * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  int rc;
  if ((rc = check_dev_err(p, (int)p->h_ctr[C_COUNT - 1]))) return rc;
  p->k_nsrc = p->h_ctr[C_NEXT_BANK];
  *n_next = p->k_nsrc;
  p->k_clock_ms += clk.stop();
  return TDR_OK;
}

int tdr_k_end(tdr_problem *p, uint32_t n_gen, uint32_t n_inactive, const uint64_t *gen_n, const uint64_t *gen_m, const int64_t *gen_p,
              const int64_t *gen_pc, const double *gen_k) {
  if (!p || n_gen == 0 || n_inactive > n_gen || !gen_n || !gen_m || !gen_p || !gen_pc || !gen_k) return fail(TDR_EINVAL, "bad argument");
  p->gen_n.assign(gen_n, gen_n + n_gen); p->gen_m.assign(gen_m, gen_m + n_gen); p->gen_p.assign(gen_p, gen_p + n_gen);
  p->gen_pc.assign(gen_pc, gen_pc + n_gen); p->gen_k.assign(gen_k, gen_k + n_gen);
  p->diag.gpu_ms = p->k_clock_ms;
  collect_kernel_times(p);
  const u32 n_active = n_gen - n_inactive;
  double sum = 0.0;
  for (u32 g = n_inactive; g < n_gen; g++) sum = sum + p->gen_k[g];
  p->k_mean = n_active ? sum / (double)n_active : 0.0;
  double var = 0.0;
  for (u32 g = n_inactive; g < n_gen; g++) { double dk = p->gen_k[g] - p->k_mean; var = var + dk * dk; }
  p->k_std = n_active > 1 ? sqrt((var / (double)(n_active - 1)) / (double)n_active) : 0.0;
  p->ran = true;
  return TDR_OK;
}

// D2 on one GPU: the loop over the steps above with a single share
int tdr_run_k_eigenvalue(tdr_problem *p, uint64_t n, uint32_t n_inactive, uint32_t n_active, uint64_t seed) {
  if ((u64)n_inactive + n_active == 0 || (u64)n_inactive + n_active > 65535) return fail(TDR_EINVAL, "bad generation counts");
  if (n == 0) return fail(TDR_EINVAL, "bad argument");
  const u32 n_gen = n_inactive + n_active;
  int rc = tdr_k_begin(p, 0, n, n_gen, seed); if (rc) return rc;
  std::vector<u64> gn, gm; std::vector<i64> gp, gpc; std::vector<double> gk;
  double k_prev = 1.0;
  for (u32 g = 0; g < n_gen; g++) {
    i64 sums[4];
    const bool last = g + 1 == n_gen;
    if ((rc = tdr_k_generation(p, g, g >= n_inactive, k_prev, last, (int64_t *)sums))) return rc;
    const double k = ((double)sums[0] * (1.0 / p->dp.scale)) / (double)sums[2];                    // D2
    gn.push_back((u64)sums[2]); gm.push_back((u64)sums[3]); gp.push_back(sums[0]); gpc.push_back(sums[1]); gk.push_back(k);
    if (sums[3] == 0) return fail(TDR_ESTATE, "fission bank empty in generation %u", g);
    if (last) break;
    const double pr = (double)n / (double)sums[3];
    u64 n_next = 0;
    if ((rc = tdr_k_population_control(p, g + 1, pr, (uint64_t *)&n_next))) return rc;
    k_prev = k;
    if (n_next == 0) return fail(TDR_ESTATE, "population died out");
  }
  return tdr_k_end(p, n_gen, n_inactive, (const uint64_t *)gn.data(), (const uint64_t *)gm.data(), (const int64_t *)gp.data(), (const int64_t *)gpc.data(), gk.data());
}

int tdr_tally_sizes(const tdr_problem *p, tdr_sizes *o) {
  if (!p || !o) return fail(TDR_EINVAL, "null argument");
  o->n_bins = p->dp.n_bins; o->n_gen = p->gen_n.size(); o->n_hist = p->n_hist; o->n_bank = p->n_bank;
  return TDR_OK;
}

int tdr_read_tallies(const tdr_problem *p, tdr_tallies *t) {
  if (!p || !t) return fail(TDR_EINVAL, "null argument");
  NvtxRange nvtx("tdr read_tallies");
  if (!p->ran) return fail(TDR_ESTATE, "no completed run");
  cudaStream_t st = p->stream;
  if (t->flux) CK(cudaMemcpyAsync(t->flux, p->out.flux, p->dp.n_bins * 8, cudaMemcpyDeviceToHost, st));
  if (t->coll) CK(cudaMemcpyAsync(t->coll, p->out.coll, p->dp.n_bins * 8, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(t->leak, p->out.leak, 48, cudaMemcpyDeviceToHost, st));
  CK(cudaMemcpyAsync(t->totals, p->out.totals, TDR_T_COUNT * 8, cudaMemcpyDeviceToHost, st));
  if (t->hist_id && p->n_hist) CK(cudaMemcpyAsync(t->hist_id, p->hist_id, p->n_hist * 8, cudaMemcpyDeviceToHost, st));
  if (t->hist_nseg && p->n_hist) CK(cudaMemcpyAsync(t->hist_nseg, p->hist_nseg, p->n_hist * 4, cudaMemcpyDeviceToHost, st));
  if (t->hist_ncoll && p->n_hist) CK(cudaMemcpyAsync(t->hist_ncoll, p->hist_ncoll, p->n_hist * 4, cudaMemcpyDeviceToHost, st));
  if (t->bank && p->n_bank) CK(cudaMemcpyAsync(t->bank, p->bank, p->n_bank * sizeof(tdr_site), cudaMemcpyDeviceToHost, st));
  CK(cudaStreamSynchronize(st));
  t->k_mean = p->k_mean; t->k_std = p->k_std;
  size_t ng = p->gen_n.size();
  if (t->gen_n) memcpy(t->gen_n, p->gen_n.data(), ng * 8);
  if (t->gen_m) memcpy(t->gen_m, p->gen_m.data(), ng * 8);
  if (t->gen_p) memcpy(t->gen_p, p->gen_p.data(), ng * 8);
  if (t->gen_pc) memcpy(t->gen_pc, p->gen_pc.data(), ng * 8);
  if (t->gen_k) memcpy(t->gen_k, p->gen_k.data(), ng * 8);
  return TDR_OK;
}

int tdr_read_diagnostics(const tdr_problem *p, tdr_diag *o) {
  if (!p || !o) return fail(TDR_EINVAL, "null argument");
  *o = p->diag;
  return TDR_OK;
}

int tdr_dev_det_log(const double *x, double *out, uint64_t n, void *stream) {
  k_det_log<<<296, 256, 0, (cudaStream_t)stream>>>(x, out, n);
  CK(cudaGetLastError()); CK(cudaStreamSynchronize((cudaStream_t)stream));
  return TDR_OK;
}
int tdr_dev_draw(uint64_t seed, const uint64_t *id, uint32_t gen, uint32_t seg, uint32_t purpose, uint32_t j, double *out, uint64_t n, void *stream) {
  k_draw<<<296, 256, 0, (cudaStream_t)stream>>>(seed, (const u64 *)id, gen, seg, purpose, j, out, n);
  CK(cudaGetLastError()); CK(cudaStreamSynchronize((cudaStream_t)stream));
  return TDR_OK;
}

// what: 0 = fp64 DFMA rate in TFLOP/s, 1 = L2-resident copy bandwidth in GB/s (read + write).  Uses its own scratch memory.
int tdr_measure_peak(int what, double *value, void *stream) {
  if (!value || what < 0 || what > 1) return fail(TDR_EINVAL, "bad argument");
  cudaStream_t st = (cudaStream_t)stream;
  cudaDeviceProp prop; int dev = 0; CK(cudaGetDevice(&dev)); CK(cudaGetDeviceProperties(&prop, dev));
  const int sms = prop.multiProcessorCount;
  cudaEvent_t e0, e1; CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
  float best = 1e30f; double work = 0.0;
  if (what == 0) {
    const int grid = sms * 8, iters = 1 << 16;
    double *out = nullptr; CK(cudaMalloc(&out, (size_t)grid * 256 * 8));
    for (int r = 0; r < 4; r++) {
      CK(cudaEventRecord(e0, st));
      k_peak_dfma<<<grid, 256, 0, st>>>(out, iters, 1.0000001, 1e-9);
      CK(cudaEventRecord(e1, st)); CK(cudaEventSynchronize(e1));
      float ms = 0; CK(cudaEventElapsedTime(&ms, e0, e1)); if (r > 0 && ms < best) best = ms;
    }
    CK(cudaFree(out));
    work = 2.0 * 8.0 * iters * (double)grid * 256.0 / 1e12;                 // TFLOP
  } else {
    const size_t n = (size_t)1 << 20;                                        // 16 MB in + 16 MB out
    const int reps = 64;
    double2 *buf = nullptr; CK(cudaMalloc(&buf, 2 * n * sizeof(double2))); CK(cudaMemsetAsync(buf, 0, 2 * n * sizeof(double2), st));
    for (int r = 0; r < 4; r++) {
      CK(cudaEventRecord(e0, st));
      k_peak_copy<<<sms * 8, 256, 0, st>>>(buf, buf + n, n, reps);
      CK(cudaEventRecord(e1, st)); CK(cudaEventSynchronize(e1));
      float ms = 0; CK(cudaEventElapsedTime(&ms, e0, e1)); if (r > 0 && ms < best) best = ms;
    }
    CK(cudaFree(buf));
    work = 2.0 * (double)n * sizeof(double2) * reps / 1e9;                   // GB
  }
  CK(cudaGetLastError());
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *value = work / (best / 1e3);
  return TDR_OK;
}

// ---------------------------------------------------------------------------------- population control on caller-owned arrays
// tdr_dev_popctrl: the driver's own kernel (k_popctrl) with a counter and an error word the call allocates and frees.
int tdr_dev_popctrl(const tdr_site *bank, uint64_t n_bank, tdr_site *next, uint64_t next_cap, uint64_t *count_dev,
                    uint64_t seed, uint32_t gen_next, double pr, void *stream) {
  if ((!bank && n_bank) || !next || !count_dev) return fail(TDR_EINVAL, "null argument");
  cudaStream_t st = (cudaStream_t)stream;
  int *err = nullptr; CK(cudaMalloc(&err, 256));
  CK(cudaMemsetAsync(err, 0, 256, st)); CK(cudaMemsetAsync(count_dev, 0, 8, st));
  if (n_bank) k_popctrl<<<148 * 4, 256, 0, st>>>(bank, n_bank, next, next_cap, (u64 *)count_dev, seed, gen_next, pr, err);
  cudaError_t e = cudaGetLastError();
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(err);
  if (e != cudaSuccess) return fail(TDR_ECUDA, "tdr_dev_popctrl: %s", cudaGetErrorString(e));
  return TDR_OK;
}

// tdr_dev_popctrl_noalloc: the variant that allocates nothing.  Scratch = ONE file-scope device array (include/tdr.h):
//   [0, 256)                         header: word 0 = total number of copies
//   [256, 256 + 4 MAX)               m[i]   = copies of site i
//   [256 + 4 MAX, 256 + 8 MAX)       off[i] = exclusive prefix sum of m
// In HOST code the array's name is a host-side stand-in, not a device address: the address every kernel gets comes from
// cudaGetSymbolAddress, resolved once per device with that device current.  (Device code could name the array directly.)
#define NOALLOC_HDR 256
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_HDR + 8ull * TDR_NOALLOC_MAX_SITES];
static void *g_noalloc_ptr[64];                                // per device ordinal; nullptr = not resolved yet

__global__ void __launch_bounds__(256) k_na_count(const tdr_site *bank, u32 n, u32 *m, u64 seed, u32 gen_next, double pr) {
  for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    int c = (int)floor(pr + draw(seed, bank[i].id, gen_next, 0, PUR_POPCTRL, 0));          // D2, as k_popctrl
    m[i] = (u32)(c < 0 ? 0 : c > 2048 ? 2048 : c);
  }
}

// one CTA of 1024 threads: thread t owns the contiguous chunk [t c, (t + 1) c); chunk sums are scanned in shared memory
__global__ void __launch_bounds__(1024) k_na_scan(const u32 *m, u32 *off, u32 n, u64 *total_scratch, u64 *count_out) {
  __shared__ u32 part[1024];
  const u32 t = threadIdx.x, c = (n + 1023u) / 1024u;
  const u32 lo = min(t * c, n), hi = min(lo + c, n);
  u32 s = 0;
  for (u32 i = lo; i < hi; i++) s += m[i];
  part[t] = s;
  __syncthreads();
  for (u32 d = 1; d < 1024; d <<= 1) {                          // inclusive Hillis-Steele scan of the 1024 chunk sums
    const u32 v = t >= d ? part[t - d] : 0u;
    __syncthreads();
    part[t] += v;
    __syncthreads();
  }
  u32 run = part[t] - s;                                        // exclusive offset of this thread's chunk
  for (u32 i = lo; i < hi; i++) { off[i] = run; run += m[i]; }
  if (t == 1023) { *total_scratch = (u64)part[1023]; *count_out = (u64)part[1023]; }
}

__global__ void __launch_bounds__(256) k_na_write(const tdr_site *bank, u32 n, const u32 *m, const u32 *off, tdr_site *next, u64 next_cap,
                                                  u64 seed, u32 gen_next) {
  for (u32 i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    const u32 c = m[i]; const u64 base = off[i];
    if (c == 0) continue;
    tdr_site s = bank[i]; const u64 sid = s.id;
    for (u32 r = 0; r < c; r++) {
      s.id = derive_id(seed, sid, gen_next, 0, 2048u + r);       // R4, as k_popctrl
      if (base + r < next_cap) next[base + r] = s;
    }
  }
}

int tdr_dev_popctrl_noalloc(const tdr_site *bank, uint64_t n_bank, tdr_site *next, uint64_t next_cap, uint64_t *count_dev,
                            uint64_t seed, uint32_t gen_next, double pr, void *stream) {
  if ((!bank && n_bank) || !next || !count_dev) return fail(TDR_EINVAL, "null argument");
  if (n_bank > TDR_NOALLOC_MAX_SITES)
    return fail(TDR_EINVAL, "tdr_dev_popctrl_noalloc: %llu sites exceed the static scratch (TDR_NOALLOC_MAX_SITES = %d); use tdr_dev_popctrl or split the bank",
                (unsigned long long)n_bank, TDR_NOALLOC_MAX_SITES);
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(TDR_EINVAL, "device ordinal %d out of range", dev);
  if (!g_noalloc_ptr[dev]) {                                    // set-up, once per device, with that device current
    void *ptr = nullptr;
    CK(cudaGetSymbolAddress(&ptr, g_noalloc_scratch));
    if (!ptr) return fail(TDR_ECUDA, "cudaGetSymbolAddress returned a null address");
    g_noalloc_ptr[dev] = ptr;
  }
  unsigned char *scr = (unsigned char *)g_noalloc_ptr[dev];
  u64 *total = (u64 *)scr; u32 *m = (u32 *)(scr + NOALLOC_HDR), *off = m + TDR_NOALLOC_MAX_SITES;
  cudaStream_t st = (cudaStream_t)stream;
  const u32 n = (u32)n_bank;
  // every word a kernel reads is written by this call first (m[0..n), off[0..n), the total): nothing of the last call survives into it
  const int grid = n ? (int)((n + 255u) / 256u < 148u * 8u ? (n + 255u) / 256u : 148u * 8u) : 1;
  k_na_count<<<grid, 256, 0, st>>>(bank, n, m, seed, gen_next, pr);
  k_na_scan<<<1, 1024, 0, st>>>(m, off, n, total, (u64 *)count_dev);
  k_na_write<<<grid, 256, 0, st>>>(bank, n, m, off, next, next_cap, seed, gen_next);
  CK(cudaGetLastError());
  return TDR_OK;
}
