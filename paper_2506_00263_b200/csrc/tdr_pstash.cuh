// tdr_pstash.cuh — asynchronous remapping with a WHOLE-PARTICLE stash in shared memory.
//
// The paper's stash keeps the particles themselves in shared memory ("Ideally, all particle data would be stored within
// the stash for its entire life span") and falls back to global memory only for what does not fit.  This is
// that design on a B200 SM (228 KB of shared memory):
//   * every warp owns a pool of NS particle slots in shared memory (SoA inside the pool), 80 B (multigroup) or 108 B
//     (continuous energy) per particle; a particle's state never travels through L2 between two of its events;
//   * the "partially filled work links" of PAPER.md:83-85 are three rings of slot numbers per warp — MOVE, COLLIDE and
//     BIRTH (free slots; the SOURCE event / make_work of PAPER.md:65-67) — filled by ballot/popc prefix pushes, so packing
//     is always optimal and costs no serial bookkeeping;
//   * the scheduler runs whichever ring holds a full warp of work: with NS >= 96 one of the three always does while the
//     source lasts, so every event executes 32 lanes wide (the divergence TDR exists to remove);
//   * spill / fetch: fission secondaries of a fixed-source run that the producing warp cannot take go
//     into global links of 32 site records, published whole through the queue words claimed by atomicExch (q_deposit /
//     q_pop of tdr_async.cuh); a link in a queue is complete by construction, so nobody ever waits on a writer;
//   * no barrier between warps after start-up, no grid-wide synchronisation, termination by the lazily flushed count of
//     outstanding particles (as in tdr_async.cuh).
// Task schemes: MODE 0 = monolithic step (the collision runs inside MOVE, divergent), MODE 2 = MOVE and COLLIDE as two
// events (the decomposition that pays on this machine).  The five-event decomposition stays with the index stash.
#pragma once
#include "tdr_async.cuh"

// ---------------------------------------------------------------------------------- the per-warp pool
#define PS_RING 128                       // ring capacity (slot numbers are bytes); NS <= PS_RING
enum { PF_X = 0, PF_Y, PF_Z, PF_U, PF_V, PF_W, PF_ID, PF_L0, PF_L1, PF_E, PF_ST, PF_F };

template <bool CE>
struct PsPool {
  static constexpr int N64 = CE ? 12 : 9, N32 = CE ? 3 : 2;
  double *d; u64 *q; u32 *w; int NS;
  __host__ __device__ static size_t bytes(int NS) { return (size_t)NS * (N64 * 8 + N32 * 4) + 3 * PS_RING; }
  __device__ void bind(char *mem, int ns) { NS = ns; d = (double *)mem; q = (u64 *)mem; w = (u32 *)(mem + (size_t)ns * N64 * 8); }
  __device__ unsigned char *rings() const { return (unsigned char *)(w + (size_t)NS * N32); }
  __device__ __forceinline__ void load(u32 s, Part &p) const {
    p.x = d[PF_X * NS + s]; p.y = d[PF_Y * NS + s]; p.z = d[PF_Z * NS + s];
    p.u = d[PF_U * NS + s]; p.v = d[PF_V * NS + s]; p.w = d[PF_W * NS + s];
    p.E = CE ? d[PF_E * NS + s] : 0.0;
    p.id = q[PF_ID * NS + s]; unpack_loc(p, q[PF_L0 * NS + s], q[PF_L1 * NS + s]);
    p.seg = w[s]; p.ncoll = w[NS + s];
  }
  __device__ __forceinline__ void store(u32 s, const Part &p) const {
    d[PF_X * NS + s] = p.x; d[PF_Y * NS + s] = p.y; d[PF_Z * NS + s] = p.z;
    d[PF_U * NS + s] = p.u; d[PF_V * NS + s] = p.v; d[PF_W * NS + s] = p.w;
    if (CE) d[PF_E * NS + s] = p.E;
    q[PF_ID * NS + s] = p.id; q[PF_L0 * NS + s] = pack_loc0(p); q[PF_L1 * NS + s] = pack_loc1(p);
    w[s] = p.seg; w[NS + s] = p.ncoll;
  }
};

struct PsRing {                           // warp-uniform head / count in registers, slot numbers in shared memory
  unsigned char *buf; u32 head, count;
  __device__ __forceinline__ void push(u32 slot, bool pred) {
    const u32 m = __ballot_sync(FULL, pred);
    if (m == 0) return;
    if (pred) buf[(head + count + __popc(m & lanemask_lt())) & (PS_RING - 1)] = (unsigned char)slot;
    count += __popc(m);
    __syncwarp();
  }
  __device__ __forceinline__ u32 pop(u32 n, u32 lane) {      // n <= min(32, count); lanes >= n get 0
    const u32 s = lane < n ? buf[(head + lane) & (PS_RING - 1)] : 0u;
    head = (head + n) & (PS_RING - 1); count -= n;
    return s;
  }
};

#ifndef PS_THREADS
#define PS_THREADS 256
#endif
#ifndef PS_MINB
#define PS_MINB 2
#endif

// ---------------------------------------------------------------------------------- the persistent kernel
template <bool CE, int MODE>
__global__ void __launch_bounds__(PS_THREADS, PS_MINB) k_pstash(DevProb P0, DevOut O, DevRun R, PsMem A, int NS, u64 deadline_ns) {
  const ProbX<false> &P = static_cast<const ProbX<false> &>(P0);   // the particle stashes run without the time mesh / weights (the host refuses)
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  const double *mg = stage_mg(P, smem);
  const TallyPriv tp = stage_priv(P, smem, mg);
  acc_init(&acc);
  PsWarp w;
  w.lane = threadIdx.x & 31; w.gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w.A = A; w.err = O.err;
  w.open_id = NOLINK; w.open_count = 0; w.n_spill = 0; w.n_fetch = 0;
  const u32 lane = w.lane;
  PsPool<CE> pl;
  pl.bind((char *)(smem + staged_doubles(P, false)) + 16 * tp.n + (threadIdx.x >> 5) * PsPool<CE>::bytes(NS), NS);
  PsRing mq, cq, bq;
  mq.buf = pl.rings(); cq.buf = mq.buf + PS_RING; bq.buf = cq.buf + PS_RING;
  mq.head = mq.count = cq.head = cq.count = 0; bq.head = 0; bq.count = (u32)NS;
  for (u32 i = lane; i < (u32)NS; i += 32) bq.buf[i] = (unsigned char)i;
  __syncwarp();
  i64 accP = 0, accPc = 0, delta = 0;
  bool primary_done = false, starved = false;
  u32 n_iter = 0, backoff = 250, gwork_hint = 0, starved_hint = 0;
  u32 ev_cnt[3] = { 0, 0, 0 }, ln_cnt[3] = { 0, 0, 0 };
  u64 t_idle = 0, last_out = ~0ull;
  const u64 t_start = global_ns();
  enum { E_MOVE = 0, E_COLLIDE = 1, E_BIRTH = 2 };
  for (;;) {
    if ((n_iter & 4095u) == 4095u) {           // hard watchdog: a warp that stays busy for ever ends in an error code, not in a hung device
      int ex = 0;
      if (lane == 0 && global_ns() - t_start > 4 * deadline_ns) { ex = 1; atomicExch(O.err, TDR_ELOST); }
      if (__shfl_sync(FULL, ex, 0)) break;
    }
    // periodic housekeeping of a busy warp: publish the outstanding delta; fixed source: look at the global queues
    if ((++n_iter & 31u) == 0) {
      if (delta != 0) { if (lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
      if (!R.kmode) {
        u32 g = 0, s = 0;
        if (lane == 0) { g = (u32)ld_vol(&A.ctr[PC_GWORK]); s = (u32)ld_vol(R.starved); }
        gwork_hint = __shfl_sync(FULL, g, 0); starved_hint = __shfl_sync(FULL, s, 0);
        // load balance: somebody is starved and this warp sits on secondaries -> hand them over
        if (starved_hint > 0 && w.open_count > 0 && mq.count + cq.count >= 32) ps_open_deposit(w);
      }
    }
    const bool can_birth = !primary_done || (!R.kmode && (w.open_count > 0 || gwork_hint > 0));
    int ev;
    if (cq.count >= 32) ev = E_COLLIDE;
    else if (mq.count >= 32) ev = E_MOVE;
    else if (bq.count >= 32 && can_birth) ev = E_BIRTH;
    else if (mq.count + cq.count > 0) ev = (bq.count > 0 && can_birth && bq.count > mq.count && bq.count > cq.count) ? E_BIRTH : (cq.count > mq.count ? E_COLLIDE : E_MOVE);
    else if (bq.count > 0 && can_birth) ev = E_BIRTH;
    else {
      // nothing in the pool and nothing to claim: leave (k-mode), or wait for links from busy warps (fixed source)
      if (R.kmode) break;
      if (delta != 0) { if (lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
      u64 out = 0; int er = 0; u32 g = 0;
      if (lane == 0) {
        out = ld_vol(R.outstanding); er = *(volatile int *)O.err; g = (u32)ld_vol(&A.ctr[PC_GWORK]);
        if (out != last_out) { last_out = out; t_idle = global_ns(); }
        else if (starved && global_ns() - t_idle > deadline_ns) { atomicExch(O.err, TDR_ELOST); er = 1; }
      }
      out = __shfl_sync(FULL, out, 0); er = __shfl_sync(FULL, er, 0); gwork_hint = __shfl_sync(FULL, g, 0);
      if (out == 0 || er != 0) break;
      if (gwork_hint > 0) continue;
      if (!starved) { starved = true; if (lane == 0) { atomicAdd(R.starved, 1ull); t_idle = global_ns(); } }
      __nanosleep(backoff); if (backoff < 4000) backoff += backoff;
      continue;
    }
    if (starved) { starved = false; backoff = 250; if (lane == 0) atomicAdd(R.starved, ~0ull); }

    if (ev == E_BIRTH) {
      // ------------------------------------------------------------------ SOURCE event / make_work
      const u32 n = min(32u, bq.count);
      const bool want = lane < n;
      const u32 slot = bq.pop(n, lane);
      Part p; bool born = false;
      if (!R.kmode) {                                             // (1), (2): secondaries first
        if (w.open_count < n) { u32 g = 0; if (lane == 0) g = (u32)ld_vol(&A.ctr[PC_GWORK]); gwork_hint = __shfl_sync(FULL, g, 0); }
        born = ps_birth_from_links<CE>(w, P, mg, R, &acc, p, want, gwork_hint);
      }
      const u32 m = __ballot_sync(FULL, want && !born);           // (3) the primary source: one atomic per warp
      if (m && !primary_done) {
        const int leader = __ffs(m) - 1; u64 h = ~0ull;
        if (lane == (u32)leader && ld_vol(R.src_next) < R.src_total) h = atomicAdd(R.src_next, (u64)__popc(m));
        h = __shfl_sync(FULL, h, leader);
        if (h == ~0ull || h + __popc(m) >= R.src_total) primary_done = true;
        if (want && !born && h != ~0ull) {
          const u64 idx = h + __popc(m & lanemask_lt());
          if (idx < R.src_total) {
            if (R.src_sites) { const tdr_site s = R.sites[idx]; birth_site<CE>(P, mg, R, &acc, p, s); }
            else birth_primary<CE>(P, mg, R, &acc, p, idx);
            born = true;
          }
        }
      }
      if (born) pl.store(slot, p);
      mq.push(slot, born);
      bq.push(slot, want && !born);
      ev_cnt[E_BIRTH]++; ln_cnt[E_BIRTH] += __popc(__ballot_sync(FULL, born));
      continue;
    }

    if (ev == E_MOVE) {
      // ------------------------------------------------------------------ MOVE: T1-T5, then SURFACE in place (T7)
      const u32 n = min(32u, mq.count);
      const bool valid = lane < n;
      const u32 slot = mq.pop(n, lane);
      Part p;
      double St = 0.0, nsf = 0.0, d = 0.0, f = 0.0; int gi = 0; u32 flags = 0;
      if (valid) { pl.load(slot, p); ev_lookup<CE>(P, mg, p, St, nsf, gi, f); ev_move(P, R.seed, R.gen, p, St, d, flags); }
      ev_tally<CE>(P, O, tp, R, p, valid && !(flags & F_LOST), d, St, nsf, flags, accP, accPc);
      bool alive = false, tocoll = false, died = false; int nch = 0, csrc = 0;
      if (valid) {
        if ((flags & F_LOST) || p.seg >= (1u << 24)) atomicExch(O.err, TDR_ELOST);
        else if (flags & F_COLLIDE) {
          if (MODE == 2) {
            pl.d[PF_X * NS + slot] = p.x; pl.d[PF_Y * NS + slot] = p.y; pl.d[PF_Z * NS + slot] = p.z; pl.w[slot] = p.seg;
            if (CE) { pl.d[PF_ST * NS + slot] = St; pl.d[PF_F * NS + slot] = f; pl.w[2 * NS + slot] = (u32)gi; }
            tocoll = true;
          } else { alive = ev_collide<CE>(P, mg, R, &acc, p, St, gi, f, nch, csrc); died = !alive; }
        } else { alive = ev_surface(P, R, &acc, p, flags); died = !alive; }
        if (alive) pl.store(slot, p);
      }
      if (MODE != 2) {
        const u32 ncw = __reduce_add_sync(FULL, (u32)nch);
        if (ncw) { if (R.kmode) push_children(O, R, &acc, p, nch, csrc); else { ps_push_secondaries(w, R, &acc, p, nch, csrc); delta += (i64)ncw; } }
      }
      record_deaths_warp(&acc, R, died, p.id, p.seg, p.ncoll);
      const u32 dm = __ballot_sync(FULL, valid && !alive && !tocoll);
      delta -= (i64)__popc(__ballot_sync(FULL, died));
      mq.push(slot, alive);
      if (MODE == 2) cq.push(slot, tocoll);
      if (dm) bq.push(slot, valid && !alive && !tocoll);
      ev_cnt[E_MOVE]++; ln_cnt[E_MOVE] += n;
      continue;
    }

    {
      // ------------------------------------------------------------------ COLLIDE: T6 on a full warp of colliders
      const u32 n = min(32u, cq.count);
      const bool valid = lane < n;
      const u32 slot = cq.pop(n, lane);
      Part p; bool alive = false; int nch = 0, csrc = 0;
      if (valid) {
        pl.load(slot, p);
        double St, f = 0.0; int gi = 0;
        if (CE) { St = pl.d[PF_ST * NS + slot]; f = pl.d[PF_F * NS + slot]; gi = (int)pl.w[2 * NS + slot]; }
        else { int univ; const int mat = cell_material(P, p, univ); St = mg[(mat * P.G + p.g) * MGROW(P.G)]; }
        alive = ev_collide<CE>(P, mg, R, &acc, p, St, gi, f, nch, csrc);
        if (alive) {
          pl.d[PF_U * NS + slot] = p.u; pl.d[PF_V * NS + slot] = p.v; pl.d[PF_W * NS + slot] = p.w; pl.w[NS + slot] = p.ncoll;
          if (CE) pl.d[PF_E * NS + slot] = p.E; else pl.q[PF_L1 * NS + slot] = pack_loc1(p);
        }
      }
      const u32 ncw = __reduce_add_sync(FULL, (u32)nch);
      if (ncw) { if (R.kmode) push_children(O, R, &acc, p, nch, csrc); else { ps_push_secondaries(w, R, &acc, p, nch, csrc); delta += (i64)ncw; } }
      const bool died = valid && !alive;
      record_deaths_warp(&acc, R, died, p.id, p.seg, p.ncoll);
      delta -= (i64)__popc(__ballot_sync(FULL, died));
      mq.push(slot, alive);
      bq.push(slot, died);
      ev_cnt[E_COLLIDE]++; ln_cnt[E_COLLIDE] += n;
    }
  }
  ps_open_deposit(w);                       // (cannot hold records here: a warp leaves only with an empty pool and open link)
  if (lane == 0) {
    atomicAdd(&A.ctr[PC_EV_MOVE], (u64)ev_cnt[0]); atomicAdd(&A.ctr[PC_EV_COLLIDE], (u64)ev_cnt[1]); atomicAdd(&A.ctr[PC_EV_BIRTH], (u64)ev_cnt[2]);
    atomicAdd(&A.ctr[PC_LN_MOVE], (u64)ln_cnt[0]); atomicAdd(&A.ctr[PC_LN_COLLIDE], (u64)ln_cnt[1]); atomicAdd(&A.ctr[PC_LN_BIRTH], (u64)ln_cnt[2]);
    atomicAdd(&A.ctr[PC_SPILLS], (u64)w.n_spill); atomicAdd(&A.ctr[PC_FETCHES], (u64)w.n_fetch);
  }
  __syncthreads();
  acc_flush(&acc, O, accP, accPc);
  priv_flush(tp, O);
}
