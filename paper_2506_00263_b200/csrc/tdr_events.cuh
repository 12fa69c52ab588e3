// tdr_events.cuh — the transport events (A1-A6 of DESIGN.md section 2) on a register-resident particle.
// LOOKUP (T1) -> MOVE (T2-T4) -> TALLY (T5) -> COLLIDE (T6) | SURFACE (T7); fused `step` = all of them
// (monolithic task scheme), split = one kernel/event each (decomposed).
#pragma once
#include "tdr_device.cuh"

// flags produced by MOVE
enum { F_COLLIDE = 1, F_DX = 2, F_DY = 4, F_DZ = 8, F_DOUT = 16, F_DIN = 32, F_MX = 64, F_MY = 128, F_MZ = 256, F_LOST = 512, F_TIME = 1024,
       F_CS0 = 2048 /* .. F_CS0 << 5: surface slot j of the current general cell was reached */ };

// per-block accumulators in shared memory, flushed once per kernel (finalize hook).  Every 64-bit sum
// is two 32-bit words updated with native shared atomics: the carry out of the low word goes to the high word, so
// the sum is exact mod 2^64 (a 64-bit shared atomicAdd would be a compare-and-swap loop).
struct BlockAcc {
  u32 lo[TDR_T_COUNT + 2], hi[TDR_T_COUNT + 2];     // totals, then P and Pc
  u32 leak[6];
};
#define ACC_P TDR_T_COUNT
#define ACC_PC (TDR_T_COUNT + 1)

__device__ __forceinline__ void add64_shared(u32 *lo, u32 *hi, u32 k, u64 val) {
  u32 vl = (u32)val, vh = (u32)(val >> 32);
  u32 old = atomicAdd(&lo[k], vl);
  vh += (u32)(((u64)old + vl) >> 32);
  if (vh) atomicAdd(&hi[k], vh);
}
__device__ __forceinline__ void acc_add(BlockAcc *a, int kind, u64 v) { add64_shared(a->lo, a->hi, (u32)kind, v); }

__device__ __forceinline__ void acc_init(BlockAcc *a) {
  for (int i = threadIdx.x; i < (int)(sizeof(BlockAcc) / 4); i += blockDim.x) ((u32 *)a)[i] = 0;
  __syncthreads();
}

__device__ __forceinline__ i64 warp_sum_i64(i64 v) {      // exact: 3 limbs of <= 24 bits via REDUX
  u64 x = (u64)v;
  u32 a = __reduce_add_sync(FULL, (u32)(x & 0xFFFFFFu));
  u32 b = __reduce_add_sync(FULL, (u32)((x >> 24) & 0xFFFFFFu));
  u32 c = __reduce_add_sync(FULL, (u32)(x >> 48));
  return (i64)((u64)a + ((u64)b << 24) + ((u64)c << 48));
}

__device__ __forceinline__ void acc_flush(BlockAcc *a, const DevOut &o, i64 P, i64 Pc) {
  i64 wp = warp_sum_i64(P), wpc = warp_sum_i64(Pc);      // two's complement limbs: exact mod 2^64
  if ((threadIdx.x & 31) == 0) { acc_add(a, ACC_P, (u64)wp); acc_add(a, ACC_PC, (u64)wpc); }
  __syncthreads();
  int t = threadIdx.x;
  if (t < TDR_T_COUNT + 2) {
    u64 v = ((u64)a->hi[t] << 32) + a->lo[t];
    if (v) {
      const u64 old = atomicAdd(t < TDR_T_COUNT ? &o.totals[t] : &o.PPc[t - TDR_T_COUNT], v);
      if (t >= TDR_T_COUNT && ((old + v) >> 63 || old + v < old)) atomicExch(o.err, TDR_EOVERFLOW);   // N5: P, Pc left int64
    }
  } else if (t < TDR_T_COUNT + 8) { if (a->leak[t - TDR_T_COUNT - 2]) atomicAdd(&o.leak[t - TDR_T_COUNT - 2], (u64)a->leak[t - TDR_T_COUNT - 2]); }
}

// Block-private tallies in shared memory (finalize hook): used when the tally has few bins, where
// every score would otherwise hit the same few global addresses.  An int64 bin is two 32-bit words updated with
// native shared atomics; the carry out of the low word is added to the high word, so the sum is exact mod 2^64.
#define PRIV_MAX_BINS 256
struct TallyPriv { u32 *flux_lo, *flux_hi, *coll_lo, *coll_hi; int n; };

__device__ __forceinline__ TallyPriv priv_init(const DevProb &P, void *mem) {
  TallyPriv t; t.n = P.n_bins <= PRIV_MAX_BINS ? (int)P.n_bins : 0;
  u32 *w = (u32 *)mem;
  t.flux_lo = w; t.flux_hi = w + t.n; t.coll_lo = w + 2 * t.n; t.coll_hi = w + 3 * t.n;
  for (int i = threadIdx.x; i < 4 * t.n; i += blockDim.x) w[i] = 0;
  return t;
}
__device__ __forceinline__ void priv_add(u32 *lo, u32 *hi, u32 bin, u64 val) { add64_shared(lo, hi, bin, val); }
__device__ __forceinline__ void priv_flush(const TallyPriv &t, const DevOut &o) {   // after __syncthreads()
  for (int i = threadIdx.x; i < t.n; i += blockDim.x) {
    u64 f = ((u64)t.flux_hi[i] << 32) | t.flux_lo[i], c = ((u64)t.coll_hi[i] << 32) | t.coll_lo[i];
    // N5: scores are non-negative, so a fixed-point sum that reaches 2^63 (or wraps) has left int64: an error, not a wrap
    if (f) { const u64 old = atomicAdd(&o.flux[i], f); if ((old + f) >> 63 || old + f < old) atomicExch(o.err, TDR_EOVERFLOW); }
    if (c) { const u64 old = atomicAdd(&o.coll[i], c); if ((old + c) >> 63 || old + c < old) atomicExch(o.err, TDR_EOVERFLOW); }
  }
}

// warp-cooperative tally: every lane of the warp calls it (valid = lane has a score)
__device__ __forceinline__ void tally_add(u64 *arr, u32 *lo, u32 *hi, bool priv, u64 bin, i64 val, bool valid) {
  u32 m = __ballot_sync(FULL, valid);
  if (m == 0) return;
  int leader = __ffs(m) - 1;
  u64 b0 = __shfl_sync(FULL, bin, leader);
  bool same = __all_sync(FULL, !valid || bin == b0);
  if (same) {
    i64 s = warp_sum_i64(valid ? val : 0);
    if ((threadIdx.x & 31) == leader) { if (priv) priv_add(lo, hi, (u32)b0, (u64)s); else atomicAdd(&arr[b0], (u64)s); }
  } else if (valid) {
    if (priv) priv_add(lo, hi, (u32)bin, (u64)val); else atomicAdd(&arr[bin], (u64)val);
  }
}

// ---------------------------------------------------------------------------------- helpers
template <class PT>
__device__ __forceinline__ int cell_material(const PT &P, const Part &p, int &univ) {
  univ = P.cell_univ[((size_t)p.iz * P.ny + p.iy) * P.nx + p.ix];
  if (PT::EXT && P.n_surf > 0 && P.univ_nr[univ] < 0) return P.cell_mat[P.univ_cell0[univ] + p.ring];
  return P.univ_mat[univ * (TDR_MAX_RINGS + 1) + p.ring];
}

__device__ __forceinline__ int grid_index(const DevProb &P, const u32 *hash, double El) {   // X3 hashed search == X2 index; hash: the staged buckets
  u32 b = (u32)((u64)__double_as_longlong(El) >> 45) - P.hash_bmin;
  u32 lo = hash[b], hi = hash[b + 1] + 1;           // grid[lo] <= El (or lo == 0), answer in [lo, hi)
  if (hi > (u32)P.n_grid) hi = (u32)P.n_grid;
  while (hi - lo > 1) {
    u32 mid = lo + ((hi - lo) >> 1);
    if (P.grid[mid] <= El) lo = mid; else hi = mid;
  }
  if (lo > (u32)P.n_grid - 2) lo = (u32)P.n_grid - 2;
  return (int)lo;
}

// ---------------------------------------------------------------------------------- T1 LOOKUP
template <bool CE, class PT>
__device__ __forceinline__ void ev_lookup(const PT &P, const double *mg, const Part &p, double &St, double &nsf,
                                          int &gi, double &f) {
  int univ; int mat = cell_material(P, p, univ);
  if (!CE) {
    const double *row = mg + (mat * P.G + p.g) * MGROW(P.G);
    St = row[0]; nsf = row[3]; gi = 0; f = 0.0;
  } else {
    double El = p.E; if (El < P.grid_lo) El = P.grid_lo; if (El > P.grid_hi) El = P.grid_hi;
    gi = grid_index(P, reinterpret_cast<const u32 *>(mg), El);
    double e0 = P.grid[gi], e1 = P.grid[gi + 1];
    f = (El - e0) / (e1 - e0);
    St = 0.0; nsf = 0.0;
    int nn = P.mat_nnuc[mat];
    for (int n = 0; n < nn; n++) {
      int nuc = P.mat_nuc[mat * TDR_MAX_NUC + n]; double N = P.mat_dens[mat * TDR_MAX_NUC + n];
      const double4 a = P.xs[(size_t)nuc * P.n_grid + gi], b = P.xs[(size_t)nuc * P.n_grid + gi + 1];
      double ss = a.x + f * (b.x - a.x), sc = a.y + f * (b.y - a.y), sf = a.z + f * (b.z - a.z);
      double st = (ss + sc) + sf;
      St = St + N * st;
      nsf = nsf + N * (P.nuc_nu[nuc] * sf);
    }
  }
}

// ---------------------------------------------------------------------------------- T2-T4 MOVE
template <class PT>
__device__ __forceinline__ void ev_move(const PT &P, u64 seed, u32 gen, Part &p, double St, double &d, u32 &flags) {
  p.seg += 1;                                                          // R3
  double dcoll = TDR_INF;
  if (St > 0.0) dcoll = -det_log(draw(seed, p.id, gen, p.seg, PUR_DIST, 0)) / St;
  const double xl = P.xp[p.ix], xh = P.xp[p.ix + 1], yl = P.yp[p.iy], yh = P.yp[p.iy + 1], zl = P.zp[p.iz], zh = P.zp[p.iz + 1];
  double dx = plane_dist(xl, xh, p.x, p.u);
  double dy = plane_dist(yl, yh, p.y, p.v);
  double dz = plane_dist(zl, zh, p.z, p.w);
  double dout = TDR_INF, din = TDR_INF;
  int univ = P.cell_univ[((size_t)p.iz * P.ny + p.iy) * P.nx + p.ix];
  int nr = P.univ_nr[univ];
  if (nr > 0) {
    double X = p.x - P.cx[p.ix], Y = p.y - P.cy[p.iy];
    // a lane needs the cylinder outside it, the one inside it, or both; the first of them is computed by every lane
    // in one instruction sequence (outward for one lane, inward for its neighbour), the second only between two rings
    const bool out1 = p.ring < nr;
    const double d1 = dist_cyl(X, Y, p.u, p.v, P.univ_rad[univ * TDR_MAX_RINGS + (out1 ? p.ring : p.ring - 1)], out1);
    if (out1) dout = d1; else din = d1;
    if (out1 && p.ring > 0) din = dist_cyl(X, Y, p.u, p.v, P.univ_rad[univ * TDR_MAX_RINGS + p.ring - 1], false);
  }
  double dcs[TDR_MAX_CSURF]; int ncs = 0;                             // C5: the surfaces of the current general cell
  if (PT::EXT && nr < 0) {
    const int gcell = P.univ_cell0[univ] + p.ring; ncs = P.cell_nsurf[gcell];
    const double X = p.x - P.cx[p.ix], Y = p.y - P.cy[p.iy];
#pragma unroll
    for (int j = 0; j < TDR_MAX_CSURF; j++) {
      dcs[j] = TDR_INF;
      if (j < ncs) { const int r = P.cell_surf[gcell * TDR_MAX_CSURF + j], sf = abs(r) - 1; dcs[j] = surf_dist(P.surf_kind[sf], P.surf_coef + 4 * sf, X, Y, p.z, p.u, p.v, p.w, r < 0); }
    }
  }
  // mesh planes: a mesh cell bounded by the very same plane values as the lattice cell gives the very same quotient
  const double mxl = P.mesh[0][p.mx], mxh = P.mesh[0][p.mx + 1], myl = P.mesh[1][p.my], myh = P.mesh[1][p.my + 1];
  const double mzl = P.mesh[2][p.mz], mzh = P.mesh[2][p.mz + 1];
  double dmx = (mxl == xl && mxh == xh) ? dx : plane_dist(mxl, mxh, p.x, p.u);
  double dmy = (myl == yl && myh == yh) ? dy : plane_dist(myl, myh, p.y, p.v);
  double dmz = (mzl == zl && mzh == zh) ? dz : plane_dist(mzl, mzh, p.z, p.w);
  double vel = 0.0, dtm = TDR_INF;                                    // TD1, TD2: speed, distance to the next time edge
  if (PT::EXT && P.n_t > 0) {
    vel = P.G > 0 ? P.speed[p.g] : 1.3831592e6 * sqrt(p.E);
    dtm = (P.t_edges[p.it + 1] - p.t) * vel;
  }
  double ds = dx;
  if (dy < ds) ds = dy;
  if (dz < ds) ds = dz;
  if (dout < ds) ds = dout;
  if (din < ds) ds = din;
  if (PT::EXT && ncs > 0) {
#pragma unroll
    for (int j = 0; j < TDR_MAX_CSURF; j++) if (dcs[j] < ds) ds = dcs[j];
  }
  if (dmx < ds) ds = dmx;
  if (dmy < ds) ds = dmy;
  if (dmz < ds) ds = dmz;
  if (dtm < ds) ds = dtm;
  bool collide = dcoll < ds;                                           // G5
  d = collide ? dcoll : ds;
  flags = 0;
  if (!(d < TDR_INF)) { flags = F_LOST; d = 0.0; return; }
  if (collide) flags = F_COLLIDE;
  else flags = (dx == d ? F_DX : 0) | (dy == d ? F_DY : 0) | (dz == d ? F_DZ : 0) | (dout == d ? F_DOUT : 0) |
               (din == d ? F_DIN : 0) | (dmx == d ? F_MX : 0) | (dmy == d ? F_MY : 0) | (dmz == d ? F_MZ : 0) | ((PT::EXT && dtm == d) ? F_TIME : 0);
  if (PT::EXT && ncs > 0 && !collide) {
#pragma unroll
    for (int j = 0; j < TDR_MAX_CSURF; j++) if (j < ncs && dcs[j] == d) flags |= F_CS0 << j;
  }
  p.x = p.x + d * p.u; p.y = p.y + d * p.v; p.z = p.z + d * p.w;       // G6
  if (PT::EXT && P.n_t > 0) p.t = p.t + d / vel;                                  // TD3
}

// ---------------------------------------------------------------------------------- T5 TALLY (warp-cooperative)
template <bool CE, class PT>
__device__ __forceinline__ void ev_tally(const PT &P, const DevOut &o, const TallyPriv &tp, const DevRun &R, const Part &p, bool valid,
                                         double d, double St, double nsf, u32 flags, i64 &accP, i64 &accPc) {
  int e = -1;
  if (valid) {
    if (!CE) e = P.by_group ? p.g : 0;
    else if (p.E >= P.e_edges[0] && p.E < P.e_edges[P.n_e]) {
      int lo = 0, hi = P.n_e;
      while (hi - lo > 1) { int mid = lo + ((hi - lo) >> 1); if (P.e_edges[mid] <= p.E) lo = mid; else hi = mid; }
      e = lo;
    }
  }
  bool collide = valid && (flags & F_COLLIDE);
  // (0/St = 0 scores nothing, and a zero numerator would take the slow path of the software division)
  if (R.kmode && valid) { accP += fixp(d * nsf, P.scale); if (collide && nsf != 0.0) accPc += fixp(nsf / St, P.scale); }
  if (R.active) {
    u64 bin = 0;
    if (e >= 0) bin = (((((u64)(PT::EXT ? p.it : 0) * P.mesh_n[2] + p.mz) * P.mesh_n[1] + p.my) * P.mesh_n[0]) + p.mx) * P.n_e + e;     // TD4
    // W2: scores carry the weight (identically 1 in analog runs)
    tally_add(o.flux, tp.flux_lo, tp.flux_hi, tp.n > 0, bin, fixp((PT::EXT && P.implicit) ? p.wgt * d : d, P.scale), e >= 0);
    tally_add(o.coll, tp.coll_lo, tp.coll_hi, tp.n > 0, bin, fixp((PT::EXT && P.implicit) ? p.wgt : 1.0, P.scale), e >= 0 && collide);
  }
}

// ---------------------------------------------------------------------------------- death bookkeeping (D3)
__device__ __forceinline__ void record_death(BlockAcc *a, const DevRun &R, const Part &p, int total_kind) {
  acc_add(a, total_kind, 1ull);
  if (R.defer_death) return;                 // asynchronous scheme: the SOURCE event books the rest, 32 lanes wide
  acc_add(a, TDR_T_NSEG, (u64)p.seg);
  acc_add(a, TDR_T_NCOLL, (u64)p.ncoll);
  acc_add(a, TDR_T_NCROSS, (u64)(p.seg - p.ncoll));
  Blk h = philox((u32)p.id, (u32)(p.id >> 32), p.ncoll, p.seg - p.ncoll, p.seg, 0x7D12u);
  acc_add(a, TDR_T_DIGEST, ((u64)h.w1 << 32) | h.w0);
  if (R.hist_cap) {
    u64 k = atomicAdd(R.hist_count, 1ull);
    if (k < R.hist_cap) { R.hist_id[k] = p.id; R.hist_nseg[k] = p.seg; R.hist_ncoll[k] = p.ncoll; }
  }
}

// the same bookkeeping for a whole link of dead particles (valid = lane holds one): warp-reduced, one atomic each
__device__ TDR_COLD void record_deaths_warp(BlockAcc *a, const DevRun &R, bool valid, u64 id, u32 seg, u32 ncoll) {
  const u32 lane = threadIdx.x & 31;
  const u32 m = __ballot_sync(FULL, valid);
  if (m == 0) return;
  const u32 sseg = __reduce_add_sync(FULL, valid ? seg : 0u), scoll = __reduce_add_sync(FULL, valid ? ncoll : 0u);
  u64 dg = 0;
  if (valid) { Blk h = philox((u32)id, (u32)(id >> 32), ncoll, seg - ncoll, seg, 0x7D12u); dg = ((u64)h.w1 << 32) | h.w0; }
  const u64 sdg = (u64)warp_sum_i64((i64)dg);
  u64 base = 0;
  if (lane == 0) {
    acc_add(a, TDR_T_NSEG, (u64)sseg); acc_add(a, TDR_T_NCOLL, (u64)scoll);
    acc_add(a, TDR_T_NCROSS, (u64)(sseg - scoll)); acc_add(a, TDR_T_DIGEST, sdg);
    if (R.hist_cap) base = atomicAdd(R.hist_count, (u64)__popc(m));
  }
  if (R.hist_cap) {
    base = __shfl_sync(FULL, base, 0);
    const u64 k = base + __popc(m & ((1u << lane) - 1u));
    if (valid && k < R.hist_cap) { R.hist_id[k] = id; R.hist_nseg[k] = seg; R.hist_ncoll[k] = ncoll; }
  }
}

// ---------------------------------------------------------------------------------- W4 CLOSEOUT
// "handles weights and weight windows for the particle's next loop iteration": weight roulette below w_roulette.  It runs
// at the tail of the COLLIDE and SURFACE events (the two that end a segment) under every decomposition; analog runs
// (weights identically 1) skip it on a uniform branch.
template <class PT>
__device__ __forceinline__ bool ev_closeout(const PT &P, const DevRun &R, BlockAcc *acc, Part &p) {
  if (!PT::EXT || !P.implicit || !(p.wgt < P.w_roulette)) return true;
  if (draw(R.seed, p.id, R.gen, p.seg, PUR_CLOSEOUT, 0) * P.w_survive < p.wgt) { p.wgt = P.w_survive; return true; }
  record_death(acc, R, p, TDR_T_NROULETTE);
  return false;
}

// ---------------------------------------------------------------------------------- T6 COLLIDE
// returns true if the particle survives; n_children / child_src set on fission
template <bool CE, class PT>
__device__ __forceinline__ bool ev_collide(const PT &P, const double *mg, const DevRun &R, BlockAcc *acc, Part &p,
                                           double St, int gi, double f, int &n_children, int &child_src) {
  const u64 seed = R.seed; const u32 gen = R.gen;
  n_children = 0; child_src = 0;
  p.ncoll += 1;
  int univ; int mat = cell_material(P, p, univ);
  int kind; double nu;
  if (!CE) {
    const double *row = mg + (mat * P.G + p.g) * MGROW(P.G);
    double r = draw(seed, p.id, gen, p.seg, PUR_SELECT, 1) * St;
    if (r < row[1]) kind = 0; else if (r < row[1] + row[2]) kind = 1; else kind = 2;
    if (PT::EXT && P.implicit) {                                       // W3: capture by weight, then scatter or fission
      const double snc = St - row[2];
      if (snc > 0.0) { p.wgt = p.wgt * (snc / St); kind = (draw(seed, p.id, gen, p.seg, PUR_SELECT, 1) * snc < row[1]) ? 0 : 2; }
      else kind = 1;
    }
    nu = row[4]; child_src = mat;
    if (kind == 0) {
      p.g = sample_cdf(row + 5, P.G, draw(seed, p.id, gen, p.seg, PUR_ENERGY, 0));
      if (iso_dir(seed, p.id, gen, p.seg, p.u, p.v, p.w)) acc_add(acc, TDR_T_NDIRFAIL, 1ull);
      return ev_closeout(P, R, acc, p);
    }
  } else {
    Blk sb = rng_block(seed, p.id, gen, p.seg, PUR_SELECT, 0);
    double r = blk_even(sb) * St;
    int nn = P.mat_nnuc[mat];
    double acc_s = 0.0, ss = 0.0, sc = 0.0, st = 0.0; int nuc = 0;
    for (int n = 0; n < nn; n++) {
      nuc = P.mat_nuc[mat * TDR_MAX_NUC + n]; double N = P.mat_dens[mat * TDR_MAX_NUC + n];
      const double4 a = P.xs[(size_t)nuc * P.n_grid + gi], b = P.xs[(size_t)nuc * P.n_grid + gi + 1];
      ss = a.x + f * (b.x - a.x); sc = a.y + f * (b.y - a.y); double sf = a.z + f * (b.z - a.z);
      st = (ss + sc) + sf;
      acc_s = acc_s + N * st;
      if (r < acc_s) break;
    }
    double r2 = blk_odd(sb) * st;
    if (r2 < ss) kind = 0; else if (r2 < ss + sc) kind = 1; else kind = 2;
    if (PT::EXT && P.implicit) {                                       // W3
      const double snc = st - sc;
      if (snc > 0.0) { p.wgt = p.wgt * (snc / st); kind = (blk_odd(sb) * snc < ss) ? 0 : 2; }
      else kind = 1;
    }
    nu = P.nuc_nu[nuc]; child_src = nuc;
    if (kind == 0) { scatter_ce(seed, gen, p, P.A[nuc]); return ev_closeout(P, R, acc, p); }
  }
  if (kind == 1) { record_death(acc, R, p, TDR_T_NABS); return false; }
  double nu_eff = R.kmode ? nu / R.k_prev : nu;
  int n = (int)floor(nu_eff + draw(seed, p.id, gen, p.seg, PUR_MULT, 0));
  if (n > 64) n = 64;
  if (!R.kmode && p.depth >= 200) { acc_add(acc, TDR_T_NDROPPED, (u64)n); n = 0; }
  n_children = n;
  record_death(acc, R, p, TDR_T_NFIS);
  return false;
}

// ---------------------------------------------------------------------------------- T7 SURFACE (G7)
template <class PT>
__device__ __forceinline__ bool ev_surface(const PT &P, const DevRun &R, BlockAcc *acc, Part &p, u32 flags) {
  bool alive = true;
  const double u0 = p.u, v0 = p.v, w0 = p.w;
  int univ = P.cell_univ[((size_t)p.iz * P.ny + p.iy) * P.nx + p.ix];
  bool moved_xy = false, moved_z = false;
  // lattice / zone planes: the lanes of a warp cross different axes in different directions, so ONE pass handles whichever
  // axis a lane crossed with selected operands (a second pass only for a lane that crossed two planes at once, G5)
  for (u32 af = flags & (F_DX | F_DY | F_DZ); af; af &= af - 1) {
    const int a = (af & F_DX) ? 0 : (af & F_DY) ? 1 : 2;
    const double c0 = a == 0 ? u0 : a == 1 ? v0 : w0;
    const double *pl = a == 0 ? P.xp : a == 1 ? P.yp : P.zp;
    const int n = a == 0 ? P.nx : a == 1 ? P.ny : P.nz;
    int idx = a == 0 ? p.ix : a == 1 ? p.iy : p.iz;
    const bool pos = c0 > 0.0;
    const double plane = pl[idx + (pos ? 1 : 0)];
    const bool edge = pos ? (idx + 1 == n) : (idx == 0);
    double cn = c0;
    if (edge) {
      const int face = 2 * a + (pos ? 1 : 0);
      if (P.bc[face]) cn = -c0; else { alive = false; atomicAdd(&acc->leak[face], 1u); }
    } else idx += pos ? 1 : -1;
    if (a == 0) { p.x = plane; p.u = cn; p.ix = idx; moved_xy = moved_xy || !edge; }
    else if (a == 1) { p.y = plane; p.v = cn; p.iy = idx; moved_xy = moved_xy || !edge; }
    else { p.z = plane; p.w = cn; p.iz = idx; moved_z = moved_z || !edge; }
  }
  if (flags & F_DOUT) p.ring += 1;
  if (flags & F_DIN) p.ring -= 1;
  if (moved_xy || moved_z) {
    int nu2 = P.cell_univ[((size_t)p.iz * P.ny + p.iy) * P.nx + p.ix];
    if (PT::EXT && P.n_surf > 0 && P.univ_nr[nu2] < 0) { if (moved_xy || nu2 != univ) p.ring = locate_in_universe(P, nu2, p.x - P.cx[p.ix], p.y - P.cy[p.iy], p.z); }
    else if (moved_xy) p.ring = P.univ_nr[nu2];
    else if (nu2 != univ) p.ring = locate_ring(P, nu2, p.x - P.cx[p.ix], p.y - P.cy[p.iy]);
    if (PT::EXT && p.ring < 0) { atomicExch(R.err, TDR_ELOST); p.ring = 0; }
  } else if (PT::EXT && (flags >> 11 & 63u)) {                         // C6: through one or more surfaces of a general cell
    p.ring = locate_cell(P, univ, p.x - P.cx[p.ix], p.y - P.cy[p.iy], p.z, P.univ_cell0[univ] + p.ring, flags >> 11 & 63u);
    if (p.ring < 0) { atomicExch(R.err, TDR_ELOST); p.ring = 0; }
  }
  for (u32 mf = flags & (F_MX | F_MY | F_MZ); mf; mf &= mf - 1) {      // mesh planes, the same way (indices clamp at the mesh box)
    const int a = (mf & F_MX) ? 0 : (mf & F_MY) ? 1 : 2;
    const double c0 = a == 0 ? u0 : a == 1 ? v0 : w0;
    int idx = a == 0 ? p.mx : a == 1 ? p.my : p.mz;
    const bool pos = c0 > 0.0;
    const double plane = P.mesh[a][idx + (pos ? 1 : 0)];
    if (pos) { if (idx + 1 < P.mesh_n[a]) idx += 1; } else if (idx > 0) idx -= 1;
    if (a == 0) { p.x = plane; p.mx = idx; } else if (a == 1) { p.y = plane; p.my = idx; } else { p.z = plane; p.mz = idx; }
  }
  if (!alive) record_death(acc, R, p, TDR_T_NLEAK);
  if (PT::EXT && (flags & F_TIME)) {                                   // TD3: a time edge; the last one is the census
    p.t = P.t_edges[p.it + 1]; p.it += 1;
    if (p.it == P.n_t && alive) { alive = false; record_death(acc, R, p, TDR_T_NCENSUS); }
  }
  return alive ? ev_closeout(P, R, acc, p) : false;
}

// ---------------------------------------------------------------------------------- B birth (A1 SOURCE)
template <bool CE>
__device__ __forceinline__ void birth_common(const DevProb &P, const double *mg, const DevRun &R, BlockAcc *acc, Part &p,
                                             int src, bool from_site) {
  p.seg = 0; p.ncoll = 0; p.E = 0.0; p.g = 0;
  if (!from_site && P.src_dir_kind == 1) { p.u = P.src_dir[0]; p.v = P.src_dir[1]; p.w = P.src_dir[2]; }
  else if (iso_dir(R.seed, p.id, R.gen, 0, p.u, p.v, p.w)) acc_add(acc, TDR_T_NDIRFAIL, 1ull);
  if (from_site) {
    if (!CE) p.g = sample_cdf(mg + P.n_mat * P.G * MGROW(P.G) + src * P.G, P.G, draw(R.seed, p.id, R.gen, 0, PUR_ENERGY, 0));
    else p.E = watt(R.seed, p.id, R.gen, P.wa[src], P.wb[src]);
  } else if (P.src_energy_kind == 0) p.g = P.src_index;
  else if (P.src_energy_kind == 1) p.E = P.src_energy;
  else p.E = watt(R.seed, p.id, R.gen, P.wa[P.src_index], P.wb[P.src_index]);
  acc_add(acc, TDR_T_NBORN, 1ull);
}

template <bool CE>
__device__ TDR_COLD void birth_primary(const DevProb &P, const double *mg, const DevRun &R, BlockAcc *acc, Part &p, u64 i) {
  p.id = i + R.id_offset; p.depth = 0;         // id_offset: this GPU's share of a source sharded by contiguous id ranges
  p.it = 0; p.t = P.n_t > 0 ? P.t_edges[0] : 0.0; p.wgt = 1.0;         // TD5, W1
  if (P.src_kind == 0) { p.x = P.src_lo[0]; p.y = P.src_lo[1]; p.z = P.src_lo[2]; }
  else {
    Blk b0 = rng_block(R.seed, p.id, R.gen, 0, PUR_POS, 0), b1 = rng_block(R.seed, p.id, R.gen, 0, PUR_POS, 1);
    p.x = P.src_lo[0] + blk_even(b0) * (P.src_hi[0] - P.src_lo[0]);
    p.y = P.src_lo[1] + blk_odd(b0) * (P.src_hi[1] - P.src_lo[1]);
    p.z = P.src_lo[2] + blk_even(b1) * (P.src_hi[2] - P.src_lo[2]);
  }
  p.ix = find_bin(P.xp, P.nx, p.x); p.iy = find_bin(P.yp, P.ny, p.y); p.iz = find_bin(P.zp, P.nz, p.z);
  p.mx = find_bin(P.mesh[0], P.mesh_n[0], p.x); p.my = find_bin(P.mesh[1], P.mesh_n[1], p.y); p.mz = find_bin(P.mesh[2], P.mesh_n[2], p.z);
  int univ = P.cell_univ[((size_t)p.iz * P.ny + p.iy) * P.nx + p.ix];
  p.ring = locate_in_universe(P, univ, p.x - P.cx[p.ix], p.y - P.cy[p.iy], p.z);
  if (p.ring < 0) { atomicExch(R.err, TDR_ELOST); p.ring = 0; }
  birth_common<CE>(P, mg, R, acc, p, 0, false);
}

template <bool CE>
__device__ TDR_COLD void birth_site(const DevProb &P, const double *mg, const DevRun &R, BlockAcc *acc, Part &p, const tdr_site &s, double t = 0.0, double wgt = 1.0) {
  p.id = s.id; p.depth = s.depth; p.x = s.x; p.y = s.y; p.z = s.z; p.t = t; p.it = s.it; p.wgt = wgt;
  p.ix = s.ix; p.iy = s.iy; p.iz = s.iz; p.mx = s.mx; p.my = s.my; p.mz = s.mz; p.ring = s.ring;
  birth_common<CE>(P, mg, R, acc, p, s.src, true);
}

__device__ __forceinline__ tdr_site make_site(const DevRun &R, const Part &p, int src, u32 c) {
  tdr_site s;
  s.x = p.x; s.y = p.y; s.z = p.z; s.id = derive_id(R.seed, p.id, R.gen, p.seg, c);
  s.ix = (short)p.ix; s.iy = (short)p.iy; s.iz = (short)p.iz; s.mx = (short)p.mx; s.my = (short)p.my; s.mz = (short)p.mz;
  s.ring = (unsigned char)p.ring; s.src = (unsigned char)src; s.depth = (unsigned char)(R.kmode ? 0 : p.depth + 1); s.it = (unsigned char)p.it;
  return s;
}
