// tdr_async.cuh — asynchronous remapping (section 3.2): ONE persistent kernel per generation.
//  * work link: a warp-sized array of particle slots that all wait for the same event, with the
//    event id, the fill count and a next pointer.  Particle state stays in the SoA arrays (DESIGN.md reading
//    Q21); links carry 4-byte slot indices.
//  * stash: per warp, in shared memory: L links, a free list, a full list and a table
//    event id -> partially filled link.  Inserting fills the partial link of that event; a link that fills up
//    moves to the full list; a processed link returns to the free list.
//  * spill / fetch: global links come from one arena; two sets of AQ queues (empty links,
//    work links), each queue one 64-bit word (head << 32 | tail).  A warp claims a queue by atomicExch with the
//    null queue, edits the list privately, and swaps it back; nobody ever waits on an owner.
//  * make_work: a lane whose particle died claims a pending secondary (links of site records,
//    tdr_links.cuh) or the next source index
//    and is reborn in the same slot; a warp with no runnable link claims up to 32 fresh slots and fills them.
//  * load balance / termination: a global count of starved warps makes busy warps spill; a global count of
//    outstanding particles (source not yet dead + secondaries) tells a starved warp when to exit.  The count is
//    flushed lazily (when a warp goes idle), so a stale zero can only make an idle warp leave early; a warp that
//    holds work never leaves, and every warp re-checks the source, its open link of secondaries and the global queues
//    before it leaves, so no work is stranded.  No grid-wide synchronisation anywhere.
#pragma once
#include "tdr_links.cuh"

struct GLink { u32 idx[32]; u32 count, ev, next, pad; };
enum { AC_GWORK = 0, AC_SPILLS, AC_FETCHES, AC_MAKEWORK, AC_EVENTS, AC_DBG = 8, AC_COUNT = 16 };
struct AsyncMem { GLink *links; u64 n_links; u64 *q_empty, *q_work; u64 *actr; };

template <class C>
static void async_layout(C &c, u64 W, u64 sec_cap, u64 n_links_opt, AsyncMem &am) {
  am.n_links = n_links_opt ? n_links_opt : 2 * (W / 32) + 4096;
  am.links = c.template take<GLink>(am.n_links);
  am.q_empty = c.template take<u64>(AQ); am.q_work = c.template take<u64>(AQ);
  am.actr = c.template take<u64>(AC_COUNT);
}

// builds the empty-link queues (arena link i belongs to queue i % AQ, chained in index order) and resets the
// scheduler counters; any grid
__global__ void k_async_init(AsyncMem A, u64 *outstanding, u64 n_source, u64 *slot_next, u64 *starved, u64 starved0) {
  const u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x, nt = (u64)gridDim.x * blockDim.x;
  for (u64 i = t; i < A.n_links; i += nt) A.links[i].next = (i + AQ < A.n_links) ? (u32)(i + AQ) : NOLINK;
  if (t < AQ) {
    const u64 q = t;
    u64 last = A.n_links > q ? q + ((A.n_links - 1 - q) / AQ) * AQ : 0;
    A.q_empty[q] = A.n_links > q ? ((q << 32) | last) : NULLQ;
    A.q_work[q] = NULLQ;
  }
  if (t < AC_COUNT) A.actr[t] = 0;
  if (t == 0) { *outstanding = n_source; *slot_next = 0; *starved = starved0; }   // starved0 > 0: stress, every warp believes one is starved
}

// ---------------------------------------------------------------------------------- stash (per warp, shared memory)
struct Stash {
  u32 *idx;            // [L][32]
  int *meta;           // [0] nfree [1] nrun [2..2+EV_COUNT) partial[ev] ; then cnt[L], ev[L], freel[L], run[L]
  int L;
  __device__ __forceinline__ int &nfree() const { return meta[0]; }
  __device__ __forceinline__ int &nfull() const { return meta[1]; }
  __device__ __forceinline__ int &partial(int e) const { return meta[2 + e]; }
  __device__ __forceinline__ int &cnt(int l) const { return meta[2 + EV_COUNT + l]; }
  __device__ __forceinline__ int &ev(int l) const { return meta[2 + EV_COUNT + L + l]; }
  __device__ __forceinline__ int &freel(int i) const { return meta[2 + EV_COUNT + 2 * L + i]; }
  __device__ __forceinline__ int &full(int i) const { return meta[2 + EV_COUNT + 3 * L + i]; }
};
#define STASH_WORDS(L) (32 * (L) + 2 + EV_COUNT + 4 * (L))

struct WarpCtx {                       // warp-uniform scheduler state
  Stash s; AsyncMem A; int *err; u32 lane, gw;
};

__device__ __forceinline__ void stash_init(const Stash &s, u32 lane) {
  if (lane == 0) {
    s.nfree() = s.L; s.nfull() = 0;
    for (int e = 0; e < EV_COUNT; e++) s.partial(e) = -1;
    for (int l = 0; l < s.L; l++) { s.cnt(l) = 0; s.ev(l) = 0; s.freel(l) = s.L - 1 - l; }
  }
  __syncwarp();
}

// spill: move stash link l (run-list position fi, or fi < 0 for a partial link) to a global link
__device__ __forceinline__ void spill_link(WarpCtx &w, int l, int fi) {
  const Stash &s = w.s;
  int c = s.cnt(l), e = s.ev(l);
  u32 g = NOLINK;
  if (w.lane == 0) g = q_pop(w.A.links, w.A.q_empty, w.gw, 256);
  g = __shfl_sync(FULL, g, 0);
  if (g == NOLINK) { if (w.lane == 0) atomicExch(w.err, TDR_ECAPACITY); return; }
  if ((int)w.lane < c) w.A.links[g].idx[w.lane] = s.idx[l * 32 + w.lane];
  if (w.lane == 0) { w.A.links[g].count = (u32)c; w.A.links[g].ev = (u32)e; w.A.links[g].next = NOLINK; }
  __threadfence();
  __syncwarp();
  if (w.lane == 0) {
    q_deposit(w.A.links, w.A.q_work, w.gw % AQ, ((u64)g << 32) | g);
    atomicAdd(&w.A.actr[AC_GWORK], 1ull); atomicAdd(&w.A.actr[AC_SPILLS], 1ull);
    if (fi >= 0) { s.full(fi) = s.full(s.nfull() - 1); s.nfull() -= 1; } else s.partial(e) = -1;
    s.cnt(l) = 0; s.freel(s.nfree()) = l; s.nfree() += 1;
  }
  __syncwarp();
}

// fetch: bring one global work link into the stash's run list
__device__ __forceinline__ bool fetch_link(WarpCtx &w) {
  const Stash &s = w.s;
  if (s.nfree() == 0) return false;
  u32 g = NOLINK;
  if (w.lane == 0 && ld_vol(&w.A.actr[AC_GWORK]) > 0) g = q_pop(w.A.links, w.A.q_work, w.gw, 2);
  g = __shfl_sync(FULL, g, 0);
  if (g == NOLINK) return false;
  const int c = (int)*(volatile u32 *)&w.A.links[g].count, e = (int)*(volatile u32 *)&w.A.links[g].ev;
  const int l = s.freel(s.nfree() - 1);
  if ((int)w.lane < c) s.idx[l * 32 + w.lane] = *(volatile u32 *)&w.A.links[g].idx[w.lane];
  __syncwarp();
  if (w.lane == 0) {
    s.nfree() -= 1; s.cnt(l) = c; s.ev(l) = e; s.full(s.nfull()) = l; s.nfull() += 1;
    atomicAdd(&w.A.actr[AC_GWORK], ~0ull); atomicAdd(&w.A.actr[AC_FETCHES], 1ull);
    *(volatile u32 *)&w.A.links[g].next = NOLINK;
    __threadfence();
    q_deposit(w.A.links, w.A.q_empty, w.gw % AQ, ((u64)g << 32) | g);
  }
  __syncwarp();
  return true;
}

// make sure the free list has a link; spills a runnable link if it must ("production exceeds stash capacity")
__device__ __forceinline__ void ensure_free_link(WarpCtx &w) {
  const Stash &s = w.s;
  if (s.nfree() > 0) return;
  int fi = s.nfull() - 1;
  if (fi >= 0) spill_link(w, s.full(fi), fi);
  else if (w.lane == 0) atomicExch(w.err, TDR_ECAPACITY);        // cannot happen while L > EV_COUNT
}

// warp-collective insert of one slot per flagged lane into the partial link of event e
__device__ __forceinline__ void stash_insert(WarpCtx &w, int e, u32 value, bool pred) {
  const Stash &s = w.s;
  u32 m = __ballot_sync(FULL, pred);
  int n = __popc(m);
  if (n == 0) return;
  int rank = __popc(m & lanemask_lt()), served = 0;
  while (served < n) {
    int pl = s.partial(e);
    if (pl < 0) {
      ensure_free_link(w);
      const bool none = s.nfree() == 0;
      __syncwarp();                                               // every lane has read the free count before lane 0 edits it
      if (none) return;                                           // error already flagged
      if (w.lane == 0) { pl = s.freel(s.nfree() - 1); s.nfree() -= 1; s.partial(e) = pl; s.cnt(pl) = 0; s.ev(pl) = e; }
      __syncwarp();
      pl = s.partial(e);
    }
    int c = s.cnt(pl), take = min(32 - c, n - served);
    if (pred && rank >= served && rank < served + take) s.idx[pl * 32 + c + (rank - served)] = value;
    __syncwarp();
    if (w.lane == 0) {
      s.cnt(pl) = c + take;
      if (c + take == 32) { s.full(s.nfull()) = pl; s.nfull() += 1; s.partial(e) = -1; }
    }
    __syncwarp();
    served += take;
  }
}

// ---------------------------------------------------------------------------------- make_work
// Lanes flagged `want` hold a slot with no particle.  Fixed source: secondaries first — the warp's open link of site
// records, then a full link from the global queues (ps_birth_from_links, tdr_links.cuh: a link is published whole, so
// nobody waits on a writer) — then the primary source.  Returns true if reborn.
template <bool CE>
__device__ __forceinline__ bool make_work_async(const DevProb &P, const double *mg, const DevRun &R, PsWarp &sw, BlockAcc *acc, Part &p, bool want) {
  const u32 lane = threadIdx.x & 31;
  bool reborn = false;
  u32 m = __ballot_sync(FULL, want);
  if (m == 0) return false;
  if (!R.kmode) {
    u32 hint = 0;
    if (sw.open_count < (u32)__popc(m)) { if (lane == 0) hint = (u32)ld_vol(&sw.A.ctr[PC_GWORK]); hint = __shfl_sync(FULL, hint, 0); }
    reborn = ps_birth_from_links<CE>(sw, P, mg, R, acc, p, want, hint);
    m = __ballot_sync(FULL, want && !reborn);
    if (m == 0) return reborn;
  }
  const int leader2 = __ffs(m) - 1;
  u64 h = ~0ull;
  if (lane == (u32)leader2 && ld_vol(R.src_next) < R.src_total) h = atomicAdd(R.src_next, (u64)__popc(m));
  h = __shfl_sync(FULL, h, leader2);
  if (want && !reborn && h != ~0ull) {
    u64 idx = h + __popc(m & lanemask_lt());
    if (idx < R.src_total) {
      if (R.src_sites) { tdr_site s = R.sites[idx]; birth_site<CE>(P, mg, R, acc, p, s); }
      else birth_primary<CE>(P, mg, R, acc, p, idx);
      reborn = true;
    }
  }
  return reborn;
}

// warp-uniform; `primary_done` is this warp's sticky note that the primary source is exhausted (the cursor only grows),
// which in k-mode (no secondaries) makes every later call free of global loads
__device__ __forceinline__ bool source_has_work(const DevRun &R, const PsWarp &sw, bool &primary_done) {
  if (primary_done && R.kmode) return false;
  if (!R.kmode && sw.open_count > 0) return true;
  int yes = 0;
  if ((threadIdx.x & 31) == 0) {
    if (!primary_done) yes = ld_vol(R.src_next) < R.src_total ? 1 : 2;
    if (yes != 1 && !R.kmode && ld_vol(&sw.A.ctr[PC_GWORK]) > 0) yes |= 1;
  }
  yes = __shfl_sync(FULL, yes, 0);
  if (yes & 2) primary_done = true;
  return (yes & 1) != 0;
}

// ---------------------------------------------------------------------------------- the persistent kernel
// MODE: 0 fused (monolithic step), 1 split (five events), 2 hybrid (step with the collision as its own event)
#ifndef TDR_ASYNC_MINB
#define TDR_ASYNC_MINB 2
#endif
#ifndef TDR_ASYNC_MAXT
#define TDR_ASYNC_MAXT 512
#endif
template <bool CE, int MODE, bool EXT>
__global__ void __launch_bounds__(TDR_ASYNC_MAXT, 1) k_async(DevProb P0, DevOut O, DevRun R, Soa S0, AsyncMem A, PsMem SA, int L, u64 deadline_ns, u32 fresh_max, int lockstep, u32 seg_per_event) {
  const ProbX<EXT> &P = static_cast<const ProbX<EXT> &>(P0);
  const SoaX<EXT> &S = static_cast<const SoaX<EXT> &>(S0);
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  const double *mg = stage_mg(P, smem, true);
  const TallyPriv tp = stage_priv(P, smem, mg, true);
  acc_init(&acc);
  WarpCtx w;
  w.lane = threadIdx.x & 31; w.gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w.A = A; w.err = O.err;
  u32 *stash_mem = (u32 *)(smem + P.mg_doubles) + 4 * tp.n + (threadIdx.x >> 5) * STASH_WORDS(L);
  w.s.idx = stash_mem; w.s.meta = (int *)(stash_mem + 32 * L); w.s.L = L;
  stash_init(w.s, w.lane);
  const Stash &s = w.s;
  PsWarp sw;                                  // fixed source: the warp's open link of secondaries (site records)
  sw.A = SA; sw.err = O.err; sw.lane = w.lane; sw.gw = w.gw; sw.open_id = NOLINK; sw.open_count = 0; sw.n_spill = 0; sw.n_fetch = 0;
  constexpr bool SPLIT = MODE == 1;
  const int first_ev = SPLIT ? EV_LOOKUP : EV_STEP;
  i64 accP = 0, accPc = 0, delta = 0;         // delta: outstanding particles not yet flushed (warp-uniform)
  u32 myfree = NOSLOT;                        // a slot this lane owns that holds no particle
  bool starved = false, primary_done = false;
  u32 n_events = 0, n_makework = 0, n_iter = 0, fresh = 0, backoff = 250;
  const u64 t_start = global_ns();
  u64 t_idle = 0, last_out = ~0ull;           // watchdog: no change of the outstanding count for deadline_ns while idle -> error
  bool done = false; u32 inner_used = 0;
  for (;;) {
    // Lockstep: the warps of a CTA pass the loop top together, so that they run the same event code at the same time
    // and an instruction line fetched for one warp serves the others from the SM's instruction cache (the loop is
    // instruction-fetch bound, profiles/ncu_r01.md).  A warp with nothing to do keeps voting (and keeps looking for
    // work) until every warp of its CTA is done; the CTA then leaves as one.  Only warps of the SAME CTA meet at
    // this barrier, and each arrives after a bounded amount of its own work: no warp waits for another CTA.
    if (lockstep) {
      // Between two votes every warp of the CTA passes exactly seg_per_event - 1 further barriers: a step event meets
      // them between its segments (so the segments of all warps start together as well), every other path makes up
      // for them here.
      if (MODE == 0 && !CE) { for (u32 j = inner_used; j + 1 < seg_per_event; j++) __syncthreads_and(1); inner_used = 0; }
      // the vote: every warp is done, or (k-mode) has seen the source exhausted -> the CTA drops the lockstep for the
      // tail; a warp that is done then leaves on its own, the others drain their links without a barrier
      if (__syncthreads_and((done || (MODE == 0 && R.kmode && primary_done)) ? 1 : 0)) lockstep = 0;
      done = false;
    }
    int l = -1, fi = -1;
    if (s.nfull() > 0) { fi = s.nfull() - 1; l = s.full(fi); }
    else {
      // make_work by a starved warp: only a warp that may still grow its pool of slots, or that holds
      // spare ones, asks; the others are refilled through their SOURCE links
      if ((fresh < fresh_max || __any_sync(FULL, myfree != NOSLOT)) && source_has_work(R, sw, primary_done)) {
        // starved warp: every lane brings a slot (its own spare one, else a fresh one from the window) and claims work
        u32 need = __ballot_sync(FULL, myfree == NOSLOT);
        if (fresh >= fresh_max) need = 0;                       // this warp's pool of slots is large enough
        if (need) {
          fresh += 32;
          const int ld = __ffs(need) - 1; u64 b = ~0ull;
          if (w.lane == (u32)ld && ld_vol(R.slot_next) < R.W) b = atomicAdd(R.slot_next, (u64)__popc(need));
          b = __shfl_sync(FULL, b, ld);
          if (b != ~0ull && myfree == NOSLOT) { u64 k = b + __popc(need & lanemask_lt()); if (k < R.W) myfree = (u32)k; }
        }
        Part p;
        bool born = make_work_async<CE>(P, mg, R, sw, &acc, p, myfree != NOSLOT);
        u32 slot = myfree;
        if (born) { store_part<CE>(S, slot, p); myfree = NOSLOT; }
        n_makework++;
        if (__any_sync(FULL, born)) { stash_insert(w, first_ev, slot, born); if (s.nfull() > 0) continue; }
      }
      int bc = 0;                                                 // fullest partial link among this mode's event types
      constexpr int n_ev = MODE == 0 ? 2 : MODE == 2 ? 3 : 6;
      constexpr int evs[3][6] = { { EV_STEP, EV_SOURCE, 0, 0, 0, 0 }, { EV_LOOKUP, EV_MOVE, EV_TALLY, EV_COLLIDE, EV_SURFACE, EV_SOURCE },
                                  { EV_STEP, EV_COLLIDE, EV_SOURCE, 0, 0, 0 } };
#pragma unroll
      for (int k = 0; k < n_ev; k++) { const int pl = s.partial(evs[MODE][k]); const int pc = pl >= 0 ? s.cnt(pl) : 0; if (pc > bc) { l = pl; bc = pc; } }
      if (l < 0) {
        if (fetch_link(w)) continue;
        // nothing anywhere in reach: publish what this warp knows, then leave or wait (no other warp is waited for).
        // Secondaries this warp cannot take itself (it holds no free slot) go to the global queues for the others.
        if (!R.kmode && sw.open_count > 0) ps_open_deposit(sw);
        if (delta != 0) { if (w.lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
        u64 out = 0; int er = 0;
        if (w.lane == 0) {
          out = ld_vol(R.outstanding); er = *(volatile int *)O.err;
          if (out != last_out) { last_out = out; t_idle = global_ns(); }          // someone made progress
          else if (starved && global_ns() - t_idle > deadline_ns) { atomicExch(O.err, TDR_ELOST); er = 1; }
        }
        out = __shfl_sync(FULL, out, 0); er = __shfl_sync(FULL, er, 0);
        if (out == 0 || er != 0) { if (!lockstep) break; done = true; continue; }
        if (!starved) { starved = true; if (w.lane == 0) { atomicAdd(R.starved, 1ull); t_idle = global_ns(); } }
        if (lockstep) __nanosleep(400);                               // the CTA's busy warps wait for this one at the barrier
        else { __nanosleep(backoff); if (backoff < 8000) backoff += backoff; }   // idle warps leave the issue slots to the others
        continue;
      }
    }
    if (starved) { starved = false; backoff = 250; if (w.lane == 0) atomicAdd(R.starved, ~0ull); }
    if ((n_iter & 1023u) == 1023u) {                              // hard watchdog for a warp that stays busy
      int ex = 0;
      if (w.lane == 0 && global_ns() - t_start > 4 * deadline_ns) {
        ex = 1; atomicExch(O.err, TDR_ELOST);
        A.actr[AC_DBG] = w.gw; A.actr[AC_DBG + 1] = (u64)s.cnt(l); A.actr[AC_DBG + 2] = (u64)s.ev(l); A.actr[AC_DBG + 3] = (u64)s.nfull();
        A.actr[AC_DBG + 4] = (u64)s.nfree(); A.actr[AC_DBG + 5] = n_iter; A.actr[AC_DBG + 6] = n_events; A.actr[AC_DBG + 7] = (u64)delta;
      }
      if (__shfl_sync(FULL, ex, 0) && !lockstep) break;           // in lockstep the CTA leaves as one, once every warp sees the error
    }
    // take the link out of the stash, then run its event on all lanes
    const int c = s.cnt(l), e = s.ev(l);
    const bool valid = (int)w.lane < c;
    const u32 slot = valid ? s.idx[l * 32 + w.lane] : 0;
    __syncwarp();
    if (w.lane == 0) {
      if (fi >= 0) { s.full(fi) = s.full(s.nfull() - 1); s.nfull() -= 1; } else s.partial(e) = -1;
      s.cnt(l) = 0; s.freel(s.nfree()) = l; s.nfree() += 1;
    }
    __syncwarp();
    Part p; int nch = 0, csrc = 0, next = NEXT_DEAD;
    if (e == EV_SOURCE) {
      // SOURCE event (make_work as an event): the link holds slots whose particles died.  Book the
      // deaths 32 lanes wide, then refill the slots from the pending secondaries / the source.
      u64 id = 0; u32 sg = 0, nc = 0;
      if (valid) { id = S.id[slot]; sg = S.seg[slot]; nc = S.ncoll[slot]; }
      record_deaths_warp(&acc, R, valid, id, sg, nc);
      bool born = false;
      if (source_has_work(R, sw, primary_done)) { born = make_work_async<CE>(P, mg, R, sw, &acc, p, valid); n_makework++; }
      if (born) store_part<CE>(S, slot, p);
      else if (valid && myfree == NOSLOT) myfree = slot;
      stash_insert(w, first_ev, slot, born);
      continue;
    }
    n_events += (u32)c;
    if (MODE == 0) {
      // Monolithic scheme: the `step` event is "history-length truncation with length 1".  Here the
      // length is seg_per_event: a particle is followed for up to that many segments in registers before it goes
      // back through L2 and the stash to be regrouped; a lane whose particle dies idles until the event ends.  In the
      // tail of a generation (k-mode, source exhausted, lockstep dropped, the warp's last partial link) nothing is left
      // to regroup with and the length is unbounded.  Deaths go through the SOURCE link either way.
      const u32 kmax = (!lockstep && R.kmode && primary_done && fi < 0) ? 0xFFFFFFFFu : seg_per_event;
      if (valid) load_part<CE>(S, slot, p);
      bool live = valid; u32 nc_tot = 0;
      for (u32 k = 0; k < kmax; k++) {
        int nc1 = 0, cs1 = 0;
        const int nx = exec_event<CE, EV_STEP, false, 0>(P, mg, O, tp, R, S, &acc, slot, live, p, nc1, cs1, accP, accPc, first_ev);
        const u32 ncw = __reduce_add_sync(FULL, (u32)nc1);
        if (ncw) { if (R.kmode) push_children(O, R, &acc, p, nc1, cs1); else ps_push_secondaries(sw, R, &acc, p, nc1, cs1); nc_tot += ncw; }
        if (live && nx == NEXT_DEAD) live = false;
        const u32 lm = __ballot_sync(FULL, live);
        if (lm == 0) break;
        if (k + 1 < kmax) {
          n_events += (u32)__popc(lm);
          if (lockstep && !CE) { __syncthreads_and(1); inner_used++; }   // continuous energy: the cross-section gathers make the
                                                                        // segments' durations uneven and the extra barrier costs 5 %
        }
      }
      if (live) store_part<CE>(S, slot, p);
      const bool died = valid && !live;
      const u32 dm = __ballot_sync(FULL, died);
      delta += (R.kmode ? 0 : (i64)nc_tot) - (i64)__popc(dm);
      if (dm) stash_insert(w, EV_SOURCE, slot, died);
      stash_insert(w, EV_STEP, slot, live);
      if ((++n_iter & 63u) == 0) {
        if (delta != 0) { if (w.lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
        if (!R.kmode && sw.open_count > 0) {     // load balance: somebody is starved and this warp sits on secondaries
          u64 st = 0;
          if (w.lane == 0) st = ld_vol(R.starved);
          if (__shfl_sync(FULL, st, 0) > 0) ps_open_deposit(sw);
        }
      }
      if (!lockstep && s.nfull() >= 2) {          // no lockstep (tail, or switched off): hand a full link to a starved warp
        u64 st = 0;
        if (w.lane == 0) st = ld_vol(R.starved);
        if (__shfl_sync(FULL, st, 0) > 0) spill_link(w, s.full(0), 0);
      }
      continue;
    }
    if (MODE == 2) {
      if (e == EV_STEP) next = exec_event<CE, EV_STEP, true>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev);
      else next = exec_event<CE, EV_COLLIDE>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev);
    }
    else switch (e) {
      case EV_LOOKUP: next = exec_event<CE, EV_LOOKUP>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev); break;
      case EV_MOVE: next = exec_event<CE, EV_MOVE>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev); break;
      case EV_TALLY: next = exec_event<CE, EV_TALLY>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev); break;
      case EV_COLLIDE: next = exec_event<CE, EV_COLLIDE>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev); break;
      default: next = exec_event<CE, EV_SURFACE>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, first_ev); break;
    }
    const bool died = valid && next == NEXT_DEAD;
    const u32 dm = __ballot_sync(FULL, died);
    if (dm) {                                                   // only STEP / COLLIDE / SURFACE (or a lost particle) get here
      const u32 nc = __reduce_add_sync(FULL, (u32)nch);
      if (nc) { if (R.kmode) push_children(O, R, &acc, p, nch, csrc); else ps_push_secondaries(sw, R, &acc, p, nch, csrc); }
      delta += (R.kmode ? 0 : (i64)nc) - (i64)__popc(dm);     // k-mode children belong to the next generation
      stash_insert(w, EV_SOURCE, slot, died);                   // the slot waits for the SOURCE event
    }
    if (MODE == 2) { stash_insert(w, EV_STEP, slot, next == EV_STEP); if (e == EV_STEP) stash_insert(w, EV_COLLIDE, slot, next == EV_COLLIDE); }
    else {
      if (e == EV_LOOKUP) stash_insert(w, EV_MOVE, slot, next == EV_MOVE);
      else if (e == EV_MOVE) stash_insert(w, EV_TALLY, slot, next == EV_TALLY);
      else if (e == EV_TALLY) { stash_insert(w, EV_COLLIDE, slot, next == EV_COLLIDE); stash_insert(w, EV_SURFACE, slot, next == EV_SURFACE); }
      else stash_insert(w, EV_LOOKUP, slot, next == EV_LOOKUP);
    }
    if ((++n_iter & 63u) == 0) {
      if (delta != 0) { if (w.lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
      if (!R.kmode && sw.open_count > 0) {
        u64 st = 0;
        if (w.lane == 0) st = ld_vol(R.starved);
        if (__shfl_sync(FULL, st, 0) > 0) ps_open_deposit(sw);
      }
    }
    // load balance: a warp is starved and this one holds more than one runnable link -> hand one over
    if (s.nfull() >= 2) {
      u64 st = 0;
      if (w.lane == 0) st = ld_vol(R.starved);
      st = __shfl_sync(FULL, st, 0);
      if (st > 0) spill_link(w, s.full(0), 0);
    }
  }
  if (w.lane == 0) {
    atomicAdd(&A.actr[AC_EVENTS], (u64)n_events); atomicAdd(&A.actr[AC_MAKEWORK], (u64)n_makework);
    if (sw.n_spill) atomicAdd(&A.actr[AC_SPILLS], (u64)sw.n_spill);
    if (sw.n_fetch) atomicAdd(&A.actr[AC_FETCHES], (u64)sw.n_fetch);
  }
  __syncthreads();
  acc_flush(&acc, O, accP, accPc);
  priv_flush(tp, O);
}
