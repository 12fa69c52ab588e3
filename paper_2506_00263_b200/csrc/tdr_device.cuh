// tdr_device.cuh — device primitives and per-event physics (sm_100a, fp64, -fmad=false).
// Follows DESIGN.md section 3 (N numerics, R RNG keying, G geometry, X cross sections, B birth,
// T transport segment).  Shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/tdr.h"

#define TDR_INF __longlong_as_double(0x7FF0000000000000LL)
#define FULL 0xFFFFFFFFu

enum { PUR_DIST = 0, PUR_SELECT = 1, PUR_ENERGY = 2, PUR_DIR = 3, PUR_MULT = 4, PUR_POS = 5, PUR_POPCTRL = 6,
       PUR_CLOSEOUT = 7, PUR_IDDERIVE = 15 };
#define MAX_ATTEMPT 1024

typedef unsigned long long u64;
typedef long long i64;
typedef unsigned int u32;

// ---------------------------------------------------------------------------------- problem on the device
struct DevProb {
  int nx, ny, nz, n_univ, G, n_mat, n_e, by_group, n_grid, n_nuc, n_t;      // n_t: time bins (0 = time-independent)
  int bc[6], mesh_n[3];
  const double *xp, *yp, *zp, *cx, *cy, *univ_rad, *mesh[3], *e_edges, *t_edges, *speed;
  const int *cell_univ, *univ_nr, *univ_mat;
  int src_kind, src_dir_kind, src_energy_kind, src_index;
  double src_lo[3], src_hi[3], src_dir[3], src_energy, scale;
  int implicit; double w_roulette, w_survive;   // W: implicit capture + weight roulette (fixed source)
  // MG table (staged to shared memory): per (m,g) row of MGROW doubles, then chi cdf per material
  const double *mg; int mg_doubles;
  // CE
  const int *mat_nnuc, *mat_nuc; const double *mat_dens;
  const double *grid; const double4 *xs;     // xs[nuc*n_grid + i] = {sig_s, sig_c, sig_f, 0}
  const double *A, *nuc_nu, *wa, *wb;
  const u32 *hash; u32 hash_bmin, hash_n;    // X3: bucket -> first candidate grid index
  double grid_lo, grid_hi;
  // general cells (readings C1-C6): a universe with univ_nr == -1 is a list of cells, each an intersection of half-spaces
  int n_surf, n_cell; const int *surf_kind, *univ_cell0, *univ_ncell, *cell_nsurf, *cell_surf, *cell_mat; const double *surf_coef;
  u64 n_bins;
  static constexpr bool EXT = true;            // as a plain DevProb every extension is decided at run time (see ProbX)
};
// The time mesh (TD1-TD6) and implicit capture (W1-W4) are extensions most runs do not use; carried as run-time switches they
// cost the hot kernels registers (time, weight, speed, distance to the time edge).  The hot kernels therefore come in two
// builds and see the problem and the state through these tag types: with EXT = false the extensions are compiled out (the
// host launches that build only when n_t == 0 and implicit == 0), with EXT = true they are the run-time switches above.
template <bool X_> struct ProbX : DevProb { static constexpr bool EXT = X_; };
// MG row layout: [0] sig_t [1] sig_s_tot [2] sig_c [3] nu*sig_f [4] nu [5..5+G) scatter cdf
#define MGROW(G) (5 + (G))

struct DevOut {
  u64 *flux, *coll, *leak, *totals, *PPc;    // PPc[0] = P, PPc[1] = Pc
  int *err;
};

struct Soa {                                  // particle state, one array per field
  double *x, *y, *z, *u, *v, *w, *E, *t, *wgt; // t: time-dependent runs only, wgt: implicit capture only (else nullptr)
  u64 *id, *loc0, *loc1;
  u32 *seg, *ncoll;
  double *s_sigt, *s_nsf, *s_d, *s_f;        // split-decomposition scratch
  u32 *s_flags, *s_gi;
  static constexpr bool EXT = true;
};
template <bool X_> struct SoaX : Soa { static constexpr bool EXT = X_; };

struct DevRun {
  u64 seed; u32 gen; int kmode, active; double k_prev;
  int src_sites; const tdr_site *sites; u64 src_total; u64 *src_next;
  tdr_site *sec; double *sec_time, *sec_w; u64 sec_cap; u64 *sec_tail, *sec_head; u64 sec_limit, sec_head0;   // fixed-source secondaries (ring):
                                                  // records [sec_head0, sec_limit) are complete and claimable
  tdr_site *bank; u64 bank_cap; u64 *bank_count;                        // k-mode fission bank
  u64 *hist_id; u32 *hist_nseg, *hist_ncoll; u64 *hist_count; u64 hist_cap;
  // asynchronous scheme only: outstanding-particle count, bump allocator of window slots, count of starved warps, window size
  u64 *outstanding, *slot_next, *starved; u64 W;
  u64 id_offset;                              // first source id of this run (multi-GPU sharding of a fixed source)
  int defer_death;                            // deaths are booked by the SOURCE event (asynchronous scheme)
  int *err;                                   // the run's sticky error word (for the events that have no DevOut at hand)
};

struct Part {
  double x, y, z, u, v, w, E, t, wgt;
  u64 id;
  int ix, iy, iz, ring, depth, mx, my, mz, g, it;
  u32 seg, ncoll;
};

// ---------------------------------------------------------------------------------- R1 Philox4x32-10
struct Blk { u32 w0, w1, w2, w3; };

#ifdef TDR_PHILOX_CALL
#define TDR_PHILOX_ATTR __noinline__
#else
#define TDR_PHILOX_ATTR __forceinline__
#endif
#ifdef TDR_COLD_CALL
#define TDR_COLD __noinline__
#else
#define TDR_COLD __forceinline__
#endif
__device__ TDR_PHILOX_ATTR Blk philox(u32 c0, u32 c1, u32 c2, u32 c3, u32 k0, u32 k1) {
#pragma unroll
  for (int r = 0; r < 10; r++) {
    u32 h0 = __umulhi(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
    u32 h1 = __umulhi(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
    c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  Blk b; b.w0 = c0; b.w1 = c1; b.w2 = c2; b.w3 = c3;
  return b;
}

__device__ __forceinline__ Blk rng_block(u64 seed, u64 id, u32 gen, u32 seg, u32 purpose, u32 pair) {
  u32 blk = (purpose << 12) | (pair & 0xFFFu);
  return philox((u32)id, (u32)(id >> 32), (gen & 0xFFFFu) | (blk << 16), seg, (u32)seed, (u32)(seed >> 32));
}

__device__ __forceinline__ double to_unit(u32 lo, u32 hi) {          // N3
  u64 u52 = (((u64)hi << 32) | lo) >> 12;
  return (double)(i64)(2 * u52 + 1) * 0x1p-53;
}
__device__ __forceinline__ double blk_even(const Blk &b) { return to_unit(b.w0, b.w1); }
__device__ __forceinline__ double blk_odd(const Blk &b) { return to_unit(b.w2, b.w3); }

__device__ __forceinline__ double draw(u64 seed, u64 id, u32 gen, u32 seg, u32 purpose, u32 j) {
  Blk b = rng_block(seed, id, gen, seg, purpose, j >> 1);
  return (j & 1u) ? blk_odd(b) : blk_even(b);
}

__device__ __forceinline__ u64 derive_id(u64 seed, u64 id, u32 gen, u32 seg, u32 tag) {   // R4
  Blk b = rng_block(seed, id, gen, seg, PUR_IDDERIVE, tag);
  return ((u64)b.w1 << 32) | b.w0;
}

// ---------------------------------------------------------------------------------- N4 det_log
__device__ __forceinline__ double det_log(double x) {
  u64 bits = (u64)__double_as_longlong(x);
  int e = (int)((bits >> 52) & 0x7FF) - 1022;
  double m = __longlong_as_double((i64)((bits & 0x000FFFFFFFFFFFFFull) | 0x3FE0000000000000ull));
  if (m < 0x1.6a09e667f3bcdp-1) { m = 2.0 * m; e = e - 1; }
  double f = m - 1.0;
  double s = f / (2.0 + f);
  double z = s * s;
  double p = 1.0 / 21.0;
  p = __fma_rn(p, z, 1.0 / 19.0); p = __fma_rn(p, z, 1.0 / 17.0); p = __fma_rn(p, z, 1.0 / 15.0);
  p = __fma_rn(p, z, 1.0 / 13.0); p = __fma_rn(p, z, 1.0 / 11.0); p = __fma_rn(p, z, 1.0 / 9.0);
  p = __fma_rn(p, z, 1.0 / 7.0);  p = __fma_rn(p, z, 1.0 / 5.0);  p = __fma_rn(p, z, 1.0 / 3.0);
  double t = (s * z) * p;
  double r = 2.0 * (s + t);
  double de = (double)e;
  return (de * 0x1.62e42fee00000p-1) + ((de * 0x1.a39ef35793c76p-33) + r);
}

__device__ __forceinline__ i64 fixp(double v, double scale) { return __double2ll_rn(v * scale); }   // N5

// ---------------------------------------------------------------------------------- B2 / B3 / T6 samplers
__device__ __forceinline__ int iso_dir(u64 seed, u64 id, u32 gen, u32 seg, double &u, double &v, double &w) {
#pragma unroll 1
  for (u32 a = 0; a < MAX_ATTEMPT; a++) {
    Blk b = rng_block(seed, id, gen, seg, PUR_DIR, a);
    double v1 = 2.0 * blk_even(b) - 1.0, v2 = 2.0 * blk_odd(b) - 1.0;
    double s = v1 * v1 + v2 * v2;
    if (s < 1.0) {
      double t = 2.0 * sqrt(1.0 - s);
      u = v1 * t; v = v2 * t; w = 1.0 - 2.0 * s;
      return 0;
    }
  }
  u = 0.0; v = 0.0; w = 1.0;
  return 1;
}

__device__ __forceinline__ double watt(u64 seed, u64 id, u32 gen, double a, double b) {
  double cos2 = 1.0;
#pragma unroll 1
  for (u32 t = 0; t < MAX_ATTEMPT; t++) {
    Blk k = rng_block(seed, id, gen, 0, PUR_ENERGY, 4 + t);          // j = 8+2t, 9+2t
    double v1 = 2.0 * blk_even(k) - 1.0, v2 = 2.0 * blk_odd(k) - 1.0;
    double s = v1 * v1 + v2 * v2;
    if (s < 1.0 && s > 0.0) { cos2 = (v1 * v1) / s; break; }
  }
  Blk b0 = rng_block(seed, id, gen, 0, PUR_ENERGY, 0), b1 = rng_block(seed, id, gen, 0, PUR_ENERGY, 1);
  double l0 = det_log(blk_even(b0)), l1 = det_log(blk_odd(b0)), x2 = blk_even(b1);
  double W = -a * (l0 + l1 * cos2);
  double aab = (a * a) * b;
  return (W + aab / 4.0) + (2.0 * x2 - 1.0) * sqrt(aab * W);
}

__device__ __forceinline__ void scatter_ce(u64 seed, u32 gen, Part &p, double A) {
  double u = p.u, v = p.v, w = p.w;
  double mu = 2.0 * draw(seed, p.id, gen, p.seg, PUR_ENERGY, 0) - 1.0;
  double q = (A * A + (2.0 * A) * mu) + 1.0;
  p.E = p.E * (q / ((A + 1.0) * (A + 1.0)));
  double mul = (1.0 + A * mu) / sqrt(q);
  double cphi = 1.0, sphi = 0.0;
#pragma unroll 1
  for (u32 t = 0; t < MAX_ATTEMPT; t++) {
    Blk b = rng_block(seed, p.id, gen, p.seg, PUR_DIR, t);
    double v1 = 2.0 * blk_even(b) - 1.0, v2 = 2.0 * blk_odd(b) - 1.0;
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
  p.u = un / n; p.v = vn / n; p.w = wn / n;
}

// ---------------------------------------------------------------------------------- G3 / G4 distances
// Both are written without branches so that a warp issues ONE division (and one square root) whatever the signs
// of its lanes' direction components; the selected operands and hence the quotients are those of G3 / G4.
__device__ __forceinline__ double plane_dist(double lo, double hi, double x, double c) {
  const double pl = c > 0.0 ? hi : lo;
  const double num = pl - x;
  // an infinite plane or a zero direction component gives +inf (G3) without entering the division: infinite or
  // zero operands would send the whole warp through the slow path of the software fp64 division
  const bool ok = (c != 0.0) && (fabs(num) < TDR_INF);
  double ns = ok ? num : 1.0, cs = ok ? c : 1.0;
  asm volatile("" : "+d"(ns), "+d"(cs));   // opaque: otherwise the compiler sees the result unused and divides inf by c anyway
  const double d = ns / cs;
  return ok ? d : TDR_INF;
}

__device__ __forceinline__ double dist_cyl(double X, double Y, double u, double v, double R, bool inside) {
  const double a = u * u + v * v;
  const double b = X * u + Y * v;
  const double c = (X * X + Y * Y) - R * R;
  const double disc = b * b - a * c;
  double dsafe = disc > 0.0 ? disc : 1.0;             // sqrt(0) takes the square root's slow path: a non-positive
  asm volatile("" : "+d"(dsafe));                     // discriminant gives 0 without entering it
  const double sq = disc > 0.0 ? sqrt(dsafe) : 0.0;
  double d = (-b + (inside ? sq : -sq)) / a;          // x - y is x + (-y) exactly
  if (d < 0.0) d = 0.0;
  if (!inside && (b >= 0.0 || disc <= 0.0)) d = TDR_INF;
  if (a == 0.0) d = TDR_INF;
  return d;
}

// ---------------------------------------------------------------------------------- C2-C4 general cells
__device__ __forceinline__ double surf_eval(int kind, const double *co, double X, double Y, double Z) {   // C2: negative inside
  if (kind == 0) return ((co[0] * X + co[1] * Y) + co[2] * Z) - co[3];
  const double ox = X - co[0], oy = Y - co[1];
  if (kind == 1) { const double oz = Z - co[2]; return ((ox * ox + oy * oy) + oz * oz) - co[3] * co[3]; }
  return (ox * ox + oy * oy) - co[3] * co[3];
}

// C3: distance to the surface for a particle known (from its cell) to be on the given side
__device__ __forceinline__ double surf_dist(int kind, const double *co, double X, double Y, double Z, double u, double v, double w, bool negative_side) {
  double d;
  if (kind == 0) {
    const double den = (co[0] * u + co[1] * v) + co[2] * w;
    if (negative_side ? !(den > 0.0) : !(den < 0.0)) return TDR_INF;
    d = (co[3] - ((co[0] * X + co[1] * Y) + co[2] * Z)) / den;
  } else {
    const double ox = X - co[0], oy = Y - co[1], oz = kind == 1 ? Z - co[2] : 0.0, wz = kind == 1 ? w : 0.0;
    const double a = (u * u + v * v) + wz * wz;
    if (a == 0.0) return TDR_INF;
    const double b = (ox * u + oy * v) + oz * wz;
    const double c = ((ox * ox + oy * oy) + oz * oz) - co[3] * co[3];
    double disc = b * b - a * c;
    if (negative_side) {
      if (disc < 0.0) disc = 0.0;
      d = (-b + sqrt(disc)) / a;
    } else {
      if (b >= 0.0) return TDR_INF;
      if (disc <= 0.0) return TDR_INF;
      d = (-b - sqrt(disc)) / a;
    }
  }
  if (d < 0.0) d = 0.0;
  return d;
}

// C4: the first cell of the universe all of whose half-spaces hold the point; a surface flagged in `crossed` (bit j = slot j
// of cell `from`) is taken to be on the side opposite to the one `from` names.  -1: no such cell.
__device__ __forceinline__ int locate_cell(const DevProb &P, int univ, double X, double Y, double Z, int from, u32 crossed) {
  const int c0 = P.univ_cell0[univ], nc = P.univ_ncell[univ];
  for (int k = 0; k < nc; k++) {
    const int cell = c0 + k; bool ok = true;
    for (int j = 0; j < P.cell_nsurf[cell] && ok; j++) {
      const int r = P.cell_surf[cell * TDR_MAX_CSURF + j], sf = abs(r) - 1; const bool want_neg = r < 0;
      int neg = -1;
      if (from >= 0)
        for (int i = 0; i < P.cell_nsurf[from]; i++) {
          const int rf = P.cell_surf[from * TDR_MAX_CSURF + i];
          if ((crossed >> i & 1u) && abs(rf) - 1 == sf) neg = !(rf < 0);
        }
      if (neg < 0) neg = surf_eval(P.surf_kind[sf], P.surf_coef + 4 * sf, X, Y, Z) < 0.0;
      ok = (neg != 0) == want_neg;
    }
    if (ok) return k;
  }
  return -1;
}

__device__ __forceinline__ int find_bin(const double *pl, int n, double x) {   // G2
  int k = 0;
#pragma unroll 1
  for (int i = 1; i < n; i++) if (pl[i] <= x) k = i;
  return k;
}

__device__ __forceinline__ int locate_ring(const DevProb &P, int univ, double X, double Y) {
  int nr = P.univ_nr[univ];
  double r2 = X * X + Y * Y;
  for (int r = 0; r < nr; r++) { double R = P.univ_rad[univ * TDR_MAX_RINGS + r]; if (r2 < R * R) return r; }
  return nr;
}

__device__ __forceinline__ int locate_in_universe(const DevProb &P, int univ, double X, double Y, double Z) {   // G2 / C4
  if (P.univ_nr[univ] < 0) return locate_cell(P, univ, X, Y, Z, -1, 0u);
  return locate_ring(P, univ, X, Y);
}

__device__ __forceinline__ int sample_cdf(const double *cdf, int n, double xi) {   // X1
  const double t = xi * cdf[n - 1];
  int k = n - 1;                                      // first index with t < cdf[k], else the last: no early exit
  for (int j = n - 2; j >= 0; j--) if (t < cdf[j]) k = j;
  return k;
}

// ---------------------------------------------------------------------------------- SoA load / store
__device__ __forceinline__ void unpack_loc(Part &p, u64 l0, u64 l1) {
  p.ix = (int)(short)(l0 & 0xFFFF); p.iy = (int)(short)((l0 >> 16) & 0xFFFF); p.iz = (int)(short)((l0 >> 32) & 0xFFFF);
  p.ring = (int)((l0 >> 48) & 0xFF); p.depth = (int)((l0 >> 56) & 0xFF);
  p.mx = (int)(short)(l1 & 0xFFFF); p.my = (int)(short)((l1 >> 16) & 0xFFFF); p.mz = (int)(short)((l1 >> 32) & 0xFFFF);
  p.g = (int)((l1 >> 48) & 0xFF); p.it = (int)((l1 >> 56) & 0xFF);
}
__device__ __forceinline__ u64 pack_loc0(const Part &p) {
  return (u64)(p.ix & 0xFFFF) | ((u64)(p.iy & 0xFFFF) << 16) | ((u64)(p.iz & 0xFFFF) << 32) |
         ((u64)(p.ring & 0xFF) << 48) | ((u64)(p.depth & 0xFF) << 56);
}
__device__ __forceinline__ u64 pack_loc1(const Part &p) {
  return (u64)(p.mx & 0xFFFF) | ((u64)(p.my & 0xFFFF) << 16) | ((u64)(p.mz & 0xFFFF) << 32) | ((u64)(p.g & 0xFF) << 48) | ((u64)(p.it & 0xFF) << 56);
}

template <bool CE, class ST>
__device__ __forceinline__ void load_part(const ST &s, u32 i, Part &p) {
  p.x = s.x[i]; p.y = s.y[i]; p.z = s.z[i]; p.u = s.u[i]; p.v = s.v[i]; p.w = s.w[i];
  p.E = CE ? s.E[i] : 0.0; p.t = (ST::EXT && s.t) ? s.t[i] : 0.0; p.wgt = (ST::EXT && s.wgt) ? s.wgt[i] : 1.0;
  p.id = s.id[i]; p.seg = s.seg[i]; p.ncoll = s.ncoll[i];
  unpack_loc(p, s.loc0[i], s.loc1[i]);
}
template <bool CE, class ST>
__device__ __forceinline__ void store_part(const ST &s, u32 i, const Part &p) {
  s.x[i] = p.x; s.y[i] = p.y; s.z[i] = p.z; s.u[i] = p.u; s.v[i] = p.v; s.w[i] = p.w;
  if (CE) s.E[i] = p.E;
  if (ST::EXT && s.t) s.t[i] = p.t;
  if (ST::EXT && s.wgt) s.wgt[i] = p.wgt;
  s.id[i] = p.id; s.seg[i] = p.seg; s.ncoll[i] = p.ncoll;
  s.loc0[i] = pack_loc0(p); s.loc1[i] = pack_loc1(p);
}
