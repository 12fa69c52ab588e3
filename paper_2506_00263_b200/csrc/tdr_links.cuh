// tdr_links.cuh — global work links of the asynchronous scheme: the lock-free link queues (one 64-bit word
// per queue, claimed by atomicExch with the null queue, edited privately, swapped back: nobody ever waits on an owner) and the
// links of fission-site records through which the secondaries of a fixed-source run travel between warps.  A link enters a
// work queue only when every record in it is written, so a reader never waits on a writer.  Used by all three stashes.
#pragma once
#include "tdr_exec.cuh"

#define AQ 32
#define NULLQ 0xFFFFFFFFFFFFFFFFull
#define NOLINK 0xFFFFFFFFu
#define NOSLOT 0xFFFFFFFFu



__device__ __forceinline__ u64 ld_vol(const u64 *p) { return *(const volatile u64 *)p; }
__device__ __forceinline__ u64 global_ns() { u64 t; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)); return t; }

// ---------------------------------------------------------------------------------- global queues (lane 0 only)
template <class LinkT>
__device__ __noinline__ void q_deposit(LinkT *links, u64 *qs, u32 i, u64 mine) {
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

// A claimed queue looks like an empty one, so `rounds` full scans are made before the set is taken to be empty.
template <class LinkT>
__device__ __noinline__ u32 q_pop(LinkT *links, u64 *qs, u32 start, u32 rounds) {
  for (u32 a = 0; a < AQ * rounds; a++) {
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

struct SLink { tdr_site s[32]; u32 count, next, pad0, pad1; };      // a global work link of fission-site records
enum { PC_GWORK = 0, PC_SPILLS, PC_FETCHES, PC_EV_MOVE, PC_EV_COLLIDE, PC_EV_BIRTH, PC_LN_MOVE, PC_LN_COLLIDE, PC_LN_BIRTH,
       PC_DBG = 10, PC_COUNT = 16 };
// link_t / link_w: time (TD5) and weight (W1) a secondary inherits, record r of link g at [32 g + r]; nullptr in runs without
struct PsMem { SLink *links; u64 n_links; u64 *q_empty, *q_work; u64 *ctr; double *link_t, *link_w; };

template <class C>
static void pstash_layout(C &c, u64 W, u64 n_links_opt, bool with_time, bool with_weight, PsMem &pm) {
  pm.n_links = n_links_opt ? n_links_opt : W / 32 + 8192;
  pm.links = c.template take<SLink>(pm.n_links);
  pm.link_t = with_time ? c.template take<double>(32 * pm.n_links) : nullptr;
  pm.link_w = with_weight ? c.template take<double>(32 * pm.n_links) : nullptr;
  pm.q_empty = c.template take<u64>(AQ); pm.q_work = c.template take<u64>(AQ);
  pm.ctr = c.template take<u64>(PC_COUNT);
}

__global__ void k_ps_init(PsMem A, u64 *outstanding, u64 n_source, u64 *starved, u64 starved0) {
  const u64 t = (u64)blockIdx.x * blockDim.x + threadIdx.x, nt = (u64)gridDim.x * blockDim.x;
  for (u64 i = t; i < A.n_links; i += nt) A.links[i].next = (i + AQ < A.n_links) ? (u32)(i + AQ) : NOLINK;
  if (t < AQ) {
    const u64 q = t;
    u64 last = A.n_links > q ? q + ((A.n_links - 1 - q) / AQ) * AQ : 0;
    A.q_empty[q] = A.n_links > q ? ((q << 32) | last) : NULLQ;
    A.q_work[q] = NULLQ;
  }
  if (t < PC_COUNT) A.ctr[t] = 0;
  if (t == 0) { *outstanding = n_source; *starved = starved0; }
}

__device__ __forceinline__ tdr_site load_site_cg(const tdr_site *p) {       // written by another SM: bypass L1
  const ulonglong2 *q = (const ulonglong2 *)p;
  union { tdr_site s; ulonglong2 v[3]; } r;
  r.v[0] = __ldcg(q); r.v[1] = __ldcg(q + 1); r.v[2] = __ldcg(q + 2);
  return r.s;
}

struct PsWarp {                           // warp-uniform runtime state
  PsMem A; int *err; u32 lane, gw;
  u32 open_id, open_count;                // the global link this warp is filling with secondaries (private until deposited)
  u32 n_spill, n_fetch;
};

__device__ __forceinline__ bool ps_open_acquire(PsWarp &w) {
  u32 g = NOLINK;
  if (w.lane == 0) g = q_pop(w.A.links, w.A.q_empty, w.gw, 256);
  g = __shfl_sync(FULL, g, 0);
  if (g == NOLINK) { if (w.lane == 0) atomicExch(w.err, TDR_ECAPACITY); return false; }
  w.open_id = g; w.open_count = 0;
  return true;
}

// publish the open link whole: it enters a work queue only when every record in it is written
__device__ __forceinline__ void ps_open_deposit(PsWarp &w) {
  if (w.open_id == NOLINK || w.open_count == 0) return;
  __syncwarp();
  if (w.lane == 0) {
    w.A.links[w.open_id].count = w.open_count; w.A.links[w.open_id].next = NOLINK;
    __threadfence();
    q_deposit(w.A.links, w.A.q_work, w.gw % AQ, ((u64)w.open_id << 32) | w.open_id);
    atomicAdd(&w.A.ctr[PC_GWORK], 1ull);
  }
  __syncwarp();
  w.n_spill++; w.open_id = NOLINK; w.open_count = 0;
}

// fixed source: n fission secondaries per lane (T6) -> site records in the warp's open link; full links are deposited
__device__ TDR_COLD void ps_push_secondaries(PsWarp &w, const DevRun &R, BlockAcc *acc, const Part &p, int n, int src) {
  const u32 total = __reduce_add_sync(FULL, (u32)n);
  if (total == 0) return;
  u32 incl = (u32)n;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const u32 t = __shfl_up_sync(FULL, incl, o); if (w.lane >= (u32)o) incl += t; }
  const u32 excl = incl - (u32)n;
  if (w.lane == 0) acc_add(acc, TDR_T_NSITES, (u64)total);
  u32 done = 0;
  while (done < total) {
    if (w.open_id == NOLINK && !ps_open_acquire(w)) return;
    const u32 take = min(32u - w.open_count, total - done);
    for (int c = 0; c < n; c++) {
      const u32 o = excl + (u32)c;
      if (o >= done && o < done + take) {
        const u32 r = w.open_count + (o - done);
        w.A.links[w.open_id].s[r] = make_site(R, p, src, (u32)c);
        if (w.A.link_t) w.A.link_t[32ull * w.open_id + r] = p.t;
        if (w.A.link_w) w.A.link_w[32ull * w.open_id + r] = p.wgt;
      }
    }
    w.open_count += take; done += take;
    if (w.open_count == 32) ps_open_deposit(w);
  }
  __syncwarp();
}

// SOURCE event of a fixed-source run: secondaries BEFORE new source particles (depth first), so the links in flight stay
// bounded by what the resident particles produce however long the source is.  Lanes flagged `want` hold a free slot.
// (1) the warp's open link, newest record first; (2) when it runs dry and full links wait in the global queues, one of
// them becomes the open link (the fetch of PAPER.md:87, 95: claimed whole, so nobody waits on a writer) and serves the
// rest.  Returns true for a lane that was born from a site; gwork_hint is cleared when the queues in reach were empty.
template <bool CE>
__device__ __forceinline__ bool ps_birth_from_links(PsWarp &w, const DevProb &P, const double *mg, const DevRun &R, BlockAcc *acc, Part &p,
                                                    bool want, u32 &gwork_hint) {
  const u32 wm = __ballot_sync(FULL, want);
  const u32 n = (u32)__popc(wm), rank = (u32)__popc(wm & lanemask_lt());
  bool born = false; u32 served = 0;
  for (int round = 0; round < 2; round++) {
    const u32 t = min(n - served, w.open_count);
    if (t) {
      if (want && rank >= served && rank < served + t) {
        const u32 r = w.open_count - t + (rank - served);
        const tdr_site s = load_site_cg(&w.A.links[w.open_id].s[r]);
        birth_site<CE>(P, mg, R, acc, p, s, w.A.link_t ? __ldcg(&w.A.link_t[32ull * w.open_id + r]) : 0.0,
                       w.A.link_w ? __ldcg(&w.A.link_w[32ull * w.open_id + r]) : 1.0);
        born = true;
      }
      w.open_count -= t; served += t;
    }
    if (served == n || round == 1 || gwork_hint == 0) break;
    u32 g = NOLINK;                                  // the open link is empty here
    if (w.lane == 0) g = q_pop(w.A.links, w.A.q_work, w.gw, 4);
    g = __shfl_sync(FULL, g, 0);
    if (g == NOLINK) { gwork_hint = 0; break; }
    const u32 c = __ldcg(&w.A.links[g].count);
    if (w.lane == 0) {
      atomicAdd(&w.A.ctr[PC_GWORK], ~0ull);
      if (w.open_id != NOLINK) {                     // hand the old (empty) open link back
        *(volatile u32 *)&w.A.links[w.open_id].next = NOLINK;
        __threadfence();
        q_deposit(w.A.links, w.A.q_empty, w.gw % AQ, ((u64)w.open_id << 32) | w.open_id);
      }
    }
    __syncwarp();
    w.open_id = g; w.open_count = c; w.n_fetch++;
  }
  return born;
}

