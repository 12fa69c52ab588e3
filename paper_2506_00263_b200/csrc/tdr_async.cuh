// tdr_async.cuh — asynchronous remapping (section 3.2): ONE persistent kernel per generation.
//  * work link: a warp-sized array of particle slots that all wait for the same event, with the
//    event id, the fill count and a next pointer.  Particle state stays in the SoA arrays (DESIGN.md reading
//    Q21); links carry 4-byte slot indices.  Free slots travel the same way, as links of event EV_FREE.
//  * stash: per warp, in shared memory: L links, a free list, a full list and a table
//    event id -> partially filled link.  Inserting fills the partial link of that event; a link that fills up
//    moves to the full list; a processed link returns to the free list.
//  * spill / fetch: global links come from one arena; three sets of AQ queues (empty links,
//    work links, free-slot links), each queue one 64-bit word (head << 32 | tail).  A warp claims a queue by
//    atomicExch with the null queue, edits the list privately, and swaps it back; nobody ever waits on an owner.
//  * make_work: called by a warp with no full link; claims source indices with one atomicAdd.
//  * load balance / termination: a global count of starved warps makes busy warps spill; a global count of live
//    particles tells a starved warp when to exit.  No grid-wide synchronisation anywhere.
#pragma once
#include "tdr_exec.cuh"

#define AQ 32
#define NULLQ 0xFFFFFFFFFFFFFFFFull
#define NOLINK 0xFFFFFFFFu
#define NOSLOT 0xFFFFFFFFu

struct GLink { u32 idx[32]; u32 count, ev, next, pad; };
enum { AC_GWORK = 0, AC_GFREE, AC_SPILLS, AC_FETCHES, AC_MAKEWORK, AC_COUNT = 8 };
struct AsyncMem { GLink *links; u64 n_links; u64 *q_empty, *q_work, *q_free; u64 *actr; };

template <class C>
static void async_layout(C &c, u64 W, int num_sms, AsyncMem &am) {
  am.n_links = 2 * (W / 32) + 4096;
  am.links = c.template take<GLink>(am.n_links);
  am.q_empty = c.template take<u64>(AQ); am.q_work = c.template take<u64>(AQ); am.q_free = c.template take<u64>(AQ);
  am.actr = c.template take<u64>(AC_COUNT);
  (void)num_sms;
}

__device__ __forceinline__ u64 ld_vol(const u64 *p) { return *(const volatile u64 *)p; }

// ---------------------------------------------------------------------------------- global queues (lane 0 only)
__device__ __forceinline__ void q_deposit(GLink *links, u64 *qs, u32 i, u64 mine) {
  for (;;) {
    u64 cur = atomicExch(&qs[i], NULLQ);                         // claim whatever is there
    if (cur != NULLQ) {                                          // merge privately: cur ++ mine
      *(volatile u32 *)&links[(u32)cur].next = (u32)(mine >> 32);
      mine = (cur & 0xFFFFFFFF00000000ull) | (mine & 0xFFFFFFFFull);
    }
    __threadfence();
    u64 old = atomicExch(&qs[i], mine);                          // swap it back
    if (old == NULLQ) return;
    mine = old; i = (i + 1) % AQ;                                // someone deposited meanwhile: place theirs elsewhere
  }
}

__device__ __forceinline__ u32 q_pop(GLink *links, u64 *qs, u32 start) {
  for (u32 a = 0; a < AQ; a++) {
    u32 i = (start + a) % AQ;
    if (ld_vol(&qs[i]) == NULLQ) continue;
    u64 w = atomicExch(&qs[i], NULLQ);
    if (w == NULLQ) continue;
    __threadfence();
    u32 head = (u32)(w >> 32), tail = (u32)w;
    if (head != tail) {
      u32 nxt = *(volatile u32 *)&links[head].next;
      q_deposit(links, qs, i, ((u64)nxt << 32) | tail);
    }
    return head;
  }
  return NOLINK;
}

// builds the empty-link queues: arena link i belongs to queue i % AQ
__global__ void k_async_init(AsyncMem A) {
  u32 q = threadIdx.x;
  if (q < AQ) {
    u32 last = NOLINK, first = NOLINK;
    for (u64 i = q; i < A.n_links; i += AQ) { if (first == NOLINK) first = (u32)i; A.links[i].next = (i + AQ < A.n_links) ? (u32)(i + AQ) : NOLINK; last = (u32)i; }
    A.q_empty[q] = first == NOLINK ? NULLQ : (((u64)first << 32) | last);
    A.q_work[q] = NULLQ; A.q_free[q] = NULLQ;
  }
  if (q < AC_COUNT) A.actr[q] = 0;
}

// ---------------------------------------------------------------------------------- stash (per warp, shared memory)
struct Stash {
  u32 *idx;            // [L][32]
  int *meta;           // [0] nfree [1] nfull [2..2+EV_COUNT) partial[ev] ; then cnt[L], ev[L], freel[L], full[L]
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
  int n_free_slots;                    // free slots held in this stash
};

__device__ __forceinline__ void stash_init(const Stash &s, u32 lane) {
  if (lane == 0) {
    s.nfree() = s.L; s.nfull() = 0;
    for (int e = 0; e < EV_COUNT; e++) s.partial(e) = -1;
    for (int l = 0; l < s.L; l++) { s.cnt(l) = 0; s.ev(l) = 0; s.freel(l) = s.L - 1 - l; }
  }
  __syncwarp();
}

// move stash link l (full list position fi, or fi < 0 for a partial link) to the global queues
__device__ __forceinline__ void spill_link(WarpCtx &w, int l, int fi) {
  const Stash &s = w.s;
  int c = s.cnt(l), e = s.ev(l);
  u32 g = NOLINK;
  if (w.lane == 0) g = q_pop(w.A.links, w.A.q_empty, w.gw);
  g = __shfl_sync(FULL, g, 0);
  if (g == NOLINK) { if (w.lane == 0) atomicExch(w.err, TDR_ECAPACITY); return; }
  if ((int)w.lane < c) w.A.links[g].idx[w.lane] = s.idx[l * 32 + w.lane];
  if (w.lane == 0) { w.A.links[g].count = (u32)c; w.A.links[g].ev = (u32)e; w.A.links[g].next = NOLINK; }
  __threadfence();
  __syncwarp();
  if (w.lane == 0) {
    q_deposit(w.A.links, e == EV_FREE ? w.A.q_free : w.A.q_work, w.gw % AQ, ((u64)g << 32) | g);
    atomicAdd(&w.A.actr[e == EV_FREE ? AC_GFREE : AC_GWORK], 1ull); atomicAdd(&w.A.actr[AC_SPILLS], 1ull);
    if (fi >= 0) { s.full(fi) = s.full(s.nfull() - 1); s.nfull() -= 1; } else s.partial(e) = -1;
    s.cnt(l) = 0; s.freel(s.nfree()) = l; s.nfree() += 1;
  }
  if (e == EV_FREE) w.n_free_slots -= c;
  __syncwarp();
}

// make sure the free list has a link; spills a full link if it must ("production exceeds stash capacity")
__device__ __forceinline__ void ensure_free_link(WarpCtx &w) {
  const Stash &s = w.s;
  if (s.nfree() > 0) return;
  int fi = -1;
  for (int i = 0; i < s.nfull(); i++) if (s.ev(s.full(i)) == EV_FREE) fi = i;     // prefer shedding free slots
  if (fi < 0) fi = s.nfull() - 1;
  if (fi >= 0) spill_link(w, s.full(fi), fi);
  else if (w.lane == 0) atomicExch(w.err, TDR_ECAPACITY);
}

// warp-collective insert of one slot per flagged lane into the partial link of event e
__device__ __forceinline__ void stash_insert(WarpCtx &w, int e, u32 value, bool pred) {
  const Stash &s = w.s;
  u32 m = __ballot_sync(FULL, pred);
  int n = __popc(m);
  if (n == 0) return;
  int rank = __popc(m & lanemask_lt()), served = 0;
  if (e == EV_FREE) w.n_free_slots += n;
  while (served < n) {
    int pl = s.partial(e);
    if (pl < 0) {
      ensure_free_link(w);
      if (s.nfree() == 0) return;                                 // error already flagged
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
