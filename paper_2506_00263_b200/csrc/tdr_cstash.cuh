// tdr_cstash.cuh — asynchronous remapping with ONE STASH SHARED BY ALL WARPS OF A CTA ("With the
// introduction of lock-free stash transactions, the same stash may be used by multiple warps, allowing for higher
// occupancy"), whole particles in shared memory, and the CTA's warps running their events in rounds.
//
//   * the CTA owns NS particle slots in shared memory (SoA) and three rings of slot numbers, one per event type: MOVE,
//     COLLIDE, BIRTH (free slots = the SOURCE event / make_work).  A warp pushes with one shared-memory
//     atomicAdd on the ring's tail per push (ballot/popc prefix inside the warp) — the lock-free transaction;
//   * a ROUND: thread 0 picks the event type whose ring holds the most work (any ring with a full batch for every warp
//     wins; with NS >= 3 x 32 x warps one always does while the source lasts), fixes the range [head, head + n) that this
//     round consumes and publishes it; warp w takes entries [32 w, 32 w + 32) of that range.  All warps of the CTA therefore
//     run the SAME event code at the same time — one instruction fetch serves them all (the round-1 profile showed the
//     persistent loop bound by instruction fetch) — and every warp runs 32 lanes wide, also in the tail of a generation,
//     where the CTA-wide packing keeps batches full 16 x longer than per-warp stashes;
//   * deaths are booked when the dead particle's slot is reused (a BIRTH batch is 32 dead slots wide), and at the end;
//   * spill / fetch as in tdr_pstash.cuh: fission secondaries travel in global links of 32 site records
//     through the atomicExch queues; no wait on any other CTA, no grid-wide synchronisation; only the warps of ONE CTA meet
//     at its barriers, each after one event's worth of its own work.
#pragma once
#include "tdr_pstash.cuh"

#ifndef CS_THREADS
#define CS_THREADS 256
#endif
#ifndef CS_MINB
#define CS_MINB 2
#endif
#define CS_FRESH 0xFFFFFFFFu               // seg word of a slot that holds no unbooked death

enum { CE_MOVE = 0, CE_COLLIDE = 1, CE_BIRTH = 2, CE_IDLE = 3, CE_EXIT = 4 };

struct CsCtl {                              // CTA-wide scheduler state in shared memory
  u32 tail[3], head[3];                     // monotonically increasing counters; ring index = counter & mask
  u32 ev, base, n;                          // the round descriptor
  u32 primary_done, open_total, reaping, gwork_hint, starved, backoff, rounds;
  unsigned long long t_idle, last_out, t_start;
};

template <bool CE>
struct CsPool {                             // NS slots, SoA; then three rings of u16 slot numbers (capacity RC, power of two)
  static constexpr int N64 = CE ? 12 : 9, N32 = CE ? 3 : 2;
  double *d; u64 *q; u32 *w; unsigned short *ring[3]; int NS; u32 mask;
  // a round reads up to 32 x warps consumed entries while survivors are pushed behind the tail: capacity >= NS + that
  __host__ __device__ static u32 ring_cap(int NS) { u32 c = 64; while (c < (u32)NS + 1024u) c <<= 1; return c; }
  __host__ __device__ static size_t bytes(int NS) { return (size_t)NS * (N64 * 8 + N32 * 4) + 3 * (size_t)ring_cap(NS) * 2; }
  __device__ void bind(char *mem, int ns) {
    NS = ns; d = (double *)mem; q = (u64 *)mem; w = (u32 *)(mem + (size_t)ns * N64 * 8);
    const u32 rc = ring_cap(ns); mask = rc - 1;
    ring[0] = (unsigned short *)(w + (size_t)ns * N32); ring[1] = ring[0] + rc; ring[2] = ring[1] + rc;
  }
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
  // the lock-free stash transaction: one atomicAdd on the ring's tail per warp-wide push
  __device__ __forceinline__ void push(CsCtl *c, int r, u32 slot, bool pred) const {
    const u32 m = __ballot_sync(FULL, pred);
    if (m == 0) return;
    const int leader = __ffs(m) - 1;
    u32 base = 0;
    if ((int)(threadIdx.x & 31) == leader) base = atomicAdd(&c->tail[r], (u32)__popc(m));
    base = __shfl_sync(FULL, base, leader);
    if (pred) ring[r][(base + __popc(m & lanemask_lt())) & mask] = (unsigned short)slot;
  }
  // every lane's slot goes to at most one of the three rings: lanes 0, 1, 2 reserve the three ranges with ONE atomic
  // instruction (three addresses), instead of three dependent ballot / atomic / shuffle rounds
  __device__ __forceinline__ void push3(CsCtl *c, u32 slot, bool to_move, bool to_collide, bool to_birth) const {
    const u32 mM = __ballot_sync(FULL, to_move), mC = __ballot_sync(FULL, to_collide), mB = __ballot_sync(FULL, to_birth);
    const u32 lane = threadIdx.x & 31;
    const u32 cnt = (u32)__popc(lane == 0 ? mM : lane == 1 ? mC : mB);
    u32 base = 0;
    if (lane < 3 && cnt) base = atomicAdd(&c->tail[lane], cnt);
    const u32 bM = __shfl_sync(FULL, base, 0), bC = __shfl_sync(FULL, base, 1), bB = __shfl_sync(FULL, base, 2);
    const u32 lt = lanemask_lt();
    if (to_move) ring[CE_MOVE][(bM + __popc(mM & lt)) & mask] = (unsigned short)slot;
    else if (to_collide) ring[CE_COLLIDE][(bC + __popc(mC & lt)) & mask] = (unsigned short)slot;
    else if (to_birth) ring[CE_BIRTH][(bB + __popc(mB & lt)) & mask] = (unsigned short)slot;
  }
};

// k-mode fission sites -> bank, one child per lane (the batch's children are spread over the warp, so the id derivation
// runs once, 32 lanes wide, instead of once per child ordinal on the few lanes that fissioned)
__device__ __forceinline__ void cs_push_children_bank(const DevOut &O, const DevRun &R, BlockAcc *acc, const Part &p, int n, int src) {
  const u32 lane = threadIdx.x & 31;
  const u32 total = __reduce_add_sync(FULL, (u32)n);
  if (total == 0) return;
  u32 incl = (u32)n;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const u32 t = __shfl_up_sync(FULL, incl, o); if (lane >= (u32)o) incl += t; }
  u64 base = 0;
  if (lane == 0) { base = atomicAdd(R.bank_count, (u64)total); acc_add(acc, TDR_T_NSITES, (u64)total); }
  base = __shfl_sync(FULL, base, 0);
  const u64 l0 = pack_loc0(p), l1 = pack_loc1(p);
  for (u32 done = 0; done < total; done += 32) {
    const u32 j = done + lane;                                     // this lane's child ordinal within the batch
    // parent = the lane whose inclusive prefix first exceeds j = the number of lanes whose prefix is <= j (the prefixes
    // are non-decreasing): a 5-step search over the shuffled prefixes
    u32 lo = 0;
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) { const u32 v = __shfl_sync(FULL, incl, (int)(lo + s - 1)); if (v <= j) lo += s; }
    int par = (int)lo;
    if (par > 31) par = 31;
    const double px = __shfl_sync(FULL, p.x, par), py = __shfl_sync(FULL, p.y, par), pz = __shfl_sync(FULL, p.z, par);
    const u64 pid = __shfl_sync(FULL, p.id, par), pl0 = __shfl_sync(FULL, l0, par), pl1 = __shfl_sync(FULL, l1, par);
    const u32 pseg = __shfl_sync(FULL, p.seg, par), pincl = __shfl_sync(FULL, incl, par);
    const int pn = __shfl_sync(FULL, n, par), psrc = __shfl_sync(FULL, src, par);
    if (j < total) {
      const u32 c = j - (pincl - (u32)pn);
      Part q; q.x = px; q.y = py; q.z = pz; q.id = pid; q.seg = pseg; unpack_loc(q, pl0, pl1);
      const tdr_site s = make_site(R, q, psrc, c);
      const u64 t = base + j;
      if (t < R.bank_cap) R.bank[t] = s; else atomicExch(O.err, TDR_ECAPACITY);
    }
  }
}

template <bool CE, int MODE>
__global__ void __launch_bounds__(CS_THREADS, CS_MINB) k_cstash(DevProb P0, DevOut O, DevRun R, PsMem A, int NS, u64 deadline_ns) {
  const ProbX<false> &P = static_cast<const ProbX<false> &>(P0);   // the particle stashes run without the time mesh / weights (the host refuses)
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  __shared__ CsCtl ctl;
  const double *mg = stage_mg(P, smem);
  const TallyPriv tp = stage_priv(P, smem, mg);
  CsPool<CE> pl;
  pl.bind((char *)(smem + staged_doubles(P, false)) + 16 * tp.n, NS);
  const u32 lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5, cap = nw * 32;
  for (u32 i = threadIdx.x; i < (u32)NS; i += blockDim.x) { pl.ring[CE_BIRTH][i] = (unsigned short)i; pl.w[i] = CS_FRESH; }
  if (threadIdx.x == 0) {
    for (int r = 0; r < 3; r++) { ctl.tail[r] = 0; ctl.head[r] = 0; }
    ctl.tail[CE_BIRTH] = (u32)NS;
    ctl.primary_done = 0; ctl.open_total = 0; ctl.reaping = 0; ctl.gwork_hint = 0; ctl.starved = 0; ctl.backoff = 250;
    ctl.t_idle = 0; ctl.last_out = ~0ull; ctl.rounds = 0; ctl.t_start = global_ns();
  }
  acc_init(&acc);                             // (ends with a barrier)
  PsWarp w;
  w.lane = lane; w.gw = blockIdx.x * nw + wid; w.A = A; w.err = O.err;
  w.open_id = NOLINK; w.open_count = 0; w.n_spill = 0; w.n_fetch = 0;
  i64 accP = 0, accPc = 0, delta = 0;
  u32 ev_cnt[3] = { 0, 0, 0 }, ln_cnt[3] = { 0, 0, 0 }, open_pub = 0;
  for (;;) {
    __syncthreads();                          // A: every push of the last round is in the rings
    if (threadIdx.x == 0) {
      const u32 cM = ctl.tail[CE_MOVE] - ctl.head[CE_MOVE], cC = ctl.tail[CE_COLLIDE] - ctl.head[CE_COLLIDE], cB = ctl.tail[CE_BIRTH] - ctl.head[CE_BIRTH];
      bool can_birth = !ctl.primary_done;
      if (!R.kmode) {
        // a look at the global queues (one L2 round trip) before any round that could be a birth round: full links are taken
        // BEFORE new source particles (depth first), so the links in flight stay bounded by what the resident particles
        // produce however long the source is; once the source is exhausted, the look decides whether births are possible
        const bool birth_in_reach = can_birth ? (cB >= cap || (cB > cM && cB > cC)) : (ctl.open_total == 0 && cB >= 32 && cM + cC < cap);
        if (birth_in_reach) ctl.gwork_hint = (u32)ld_vol(&A.ctr[PC_GWORK]);
        if (!can_birth) can_birth = ctl.open_total > 0 || (cB >= 32 && ctl.gwork_hint > 0);
      }
      // hard watchdog (a scheduler that stopped making progress must end in an error code, not in a hung device)
      if ((++ctl.rounds & 4095u) == 0 && !ctl.reaping && global_ns() - ctl.t_start > 4 * deadline_ns) { atomicExch(O.err, TDR_ELOST); ctl.reaping = 1; }
      u32 ev;
      if (ctl.reaping) ev = cB > 0 ? CE_BIRTH : CE_EXIT;
      else if (cC >= cap) ev = CE_COLLIDE;
      else if (cM >= cap) ev = CE_MOVE;
      else if (cB >= cap && can_birth) ev = CE_BIRTH;
      else if (cM + cC > 0) ev = (can_birth && cB > cM && cB > cC) ? CE_BIRTH : (cC > cM ? CE_COLLIDE : CE_MOVE);
      else if (cB > 0 && can_birth) ev = CE_BIRTH;
      else if (R.kmode) { ctl.reaping = 1; ev = CE_BIRTH; }       // nothing left: book the remaining deaths, then leave
      else ev = CE_IDLE;
      if (ev <= CE_BIRTH) {
        const u32 c = ev == CE_MOVE ? cM : ev == CE_COLLIDE ? cC : cB;
        ctl.base = ctl.head[ev]; ctl.n = c < cap ? c : cap; ctl.head[ev] += ctl.n;
        if (ctl.starved) { ctl.starved = 0; ctl.backoff = 250; atomicAdd(R.starved, ~0ull); }
      }
      ctl.ev = ev;
    }
    __syncthreads();                          // B: the round descriptor is published
    const u32 ev = ctl.ev;
    if (ev == CE_EXIT) break;
    if (ev == CE_IDLE) {
      // fixed source, nothing in the stash and nothing to claim: publish this CTA's count of outstanding particles, then
      // leave if the whole run is done, else wait for links from busy CTAs (nobody in particular is waited for)
      if (delta != 0) { if (lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
      __syncthreads();
      if (threadIdx.x == 0) {
        const u64 out = ld_vol(R.outstanding); const int er = *(volatile int *)O.err;
        const u64 now = global_ns();
        if (out != ctl.last_out) { ctl.last_out = out; ctl.t_idle = now; }
        else if (now - ctl.t_idle > deadline_ns) atomicExch(O.err, TDR_ELOST);
        if (out == 0 || er != 0 || now - ctl.t_idle > deadline_ns) ctl.reaping = 1;
        else {
          if (!ctl.starved) { ctl.starved = 1; atomicAdd(R.starved, 1ull); }
          __nanosleep(ctl.backoff); if (ctl.backoff < 4000) ctl.backoff += ctl.backoff;
        }
      }
      continue;
    }
    const u32 my = wid * 32;
    const u32 n = ctl.n > my ? min(32u, ctl.n - my) : 0u;
    if (n == 0) {
      // a BIRTH round that brought this warp no free slot while it sits on secondaries and the source is exhausted: publish
      // them, so that whichever warp does get slots can take them (otherwise the round could repeat unchanged for ever)
      if (ev == CE_BIRTH && !R.kmode && w.open_count > 0 && ctl.primary_done) {
        ps_open_deposit(w);
        if (lane == 0) atomicAdd(&ctl.open_total, 0u - open_pub);
        open_pub = 0;
      }
      continue;
    }
    const bool valid = lane < n;
    const u32 slot = valid ? (u32)pl.ring[ev][(ctl.base + my + lane) & pl.mask] : 0u;

    if (ev == CE_BIRTH) {
      // ------------------------------------------------------------------ SOURCE event / make_work
      // the slots of this batch are free; those that still hold a dead particle are booked first, 32 lanes wide
      {
        const bool dead = valid && pl.w[slot] != CS_FRESH;
        u64 id = 0; u32 sg = 0, nc = 0;
        if (dead) { id = pl.q[PF_ID * NS + slot]; sg = pl.w[slot]; nc = pl.w[NS + slot]; pl.w[slot] = CS_FRESH; }
        record_deaths_warp(&acc, R, dead, id, sg, nc);
      }
      if (ctl.reaping) continue;
      Part p; bool born = false;
      if (!R.kmode) {                                             // (1), (2): secondaries first (the warp's open link, then the global queues)
        u32 hint = ctl.gwork_hint;
        born = ps_birth_from_links<CE>(w, P, mg, R, &acc, p, valid, hint);
        if (hint == 0 && lane == 0) ctl.gwork_hint = 0;           // the hint was stale: no further attempt before it is read again
      }
      const u32 m = __ballot_sync(FULL, valid && !born);          // (3) the primary source: one atomic per warp
      if (m && !*(volatile u32 *)&ctl.primary_done) {
        const int leader = __ffs(m) - 1; u64 h = ~0ull;
        if (lane == (u32)leader && ld_vol(R.src_next) < R.src_total) h = atomicAdd(R.src_next, (u64)__popc(m));
        h = __shfl_sync(FULL, h, leader);
        if ((h == ~0ull || h + __popc(m) >= R.src_total) && lane == 0) ctl.primary_done = 1;
        if (valid && !born && h != ~0ull) {
          const u64 idx = h + __popc(m & lanemask_lt());
          if (idx < R.src_total) {
            if (R.src_sites) { const tdr_site s = R.sites[idx]; birth_site<CE>(P, mg, R, &acc, p, s); }
            else birth_primary<CE>(P, mg, R, &acc, p, idx);
            born = true;
          }
        }
      }
      if (born) pl.store(slot, p);
      pl.push3(&ctl, slot, born, false, valid && !born);
      if (!R.kmode && w.open_count != open_pub) { if (lane == 0) atomicAdd(&ctl.open_total, w.open_count - open_pub); open_pub = w.open_count; }
      ev_cnt[CE_BIRTH]++; ln_cnt[CE_BIRTH] += __popc(__ballot_sync(FULL, born));
      continue;
    }

    if (ev == CE_MOVE) {
      // ------------------------------------------------------------------ MOVE: T1-T5, then SURFACE in place (T7)
      Part p;
      double St = 0.0, nsf = 0.0, d = 0.0, f = 0.0; int gi = 0; u32 flags = 0;
      if (valid) { pl.load(slot, p); ev_lookup<CE>(P, mg, p, St, nsf, gi, f); ev_move(P, R.seed, R.gen, p, St, d, flags); }
      ev_tally<CE>(P, O, tp, R, p, valid && !(flags & F_LOST), d, St, nsf, flags, accP, accPc);
      bool alive = false, tocoll = false, died = false; int nch = 0, csrc = 0;
      if (valid) {
        if ((flags & F_LOST) || p.seg >= (1u << 24)) { atomicExch(O.err, TDR_ELOST); pl.w[slot] = CS_FRESH; }
        else if (flags & F_COLLIDE) {
          if (MODE == 2) {
            pl.d[PF_X * NS + slot] = p.x; pl.d[PF_Y * NS + slot] = p.y; pl.d[PF_Z * NS + slot] = p.z; pl.w[slot] = p.seg;
            if (CE) { pl.d[PF_ST * NS + slot] = St; pl.d[PF_F * NS + slot] = f; pl.w[2 * NS + slot] = (u32)gi; }
            tocoll = true;
          } else { alive = ev_collide<CE>(P, mg, R, &acc, p, St, gi, f, nch, csrc); died = !alive; }
        } else { alive = ev_surface(P, R, &acc, p, flags); died = !alive; }
        if (alive) pl.store(slot, p);
        else if (died) { pl.w[slot] = p.seg; pl.w[NS + slot] = p.ncoll; }       // booked when the slot is reused
      }
      if (MODE != 2) {
        const u32 ncw = __reduce_add_sync(FULL, (u32)nch);
        if (ncw) { if (R.kmode) cs_push_children_bank(O, R, &acc, p, nch, csrc); else { ps_push_secondaries(w, R, &acc, p, nch, csrc); delta += (i64)ncw; } }
      }
      delta -= (i64)__popc(__ballot_sync(FULL, died));
      pl.push3(&ctl, slot, alive, tocoll, valid && !alive && !tocoll);
      ev_cnt[CE_MOVE]++; ln_cnt[CE_MOVE] += n;
    } else {
      // ------------------------------------------------------------------ COLLIDE: T6 on a full warp of colliders
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
        } else pl.w[NS + slot] = p.ncoll;
      }
      const u32 ncw = __reduce_add_sync(FULL, (u32)nch);
      if (ncw) { if (R.kmode) cs_push_children_bank(O, R, &acc, p, nch, csrc); else { ps_push_secondaries(w, R, &acc, p, nch, csrc); delta += (i64)ncw; } }
      const bool died = valid && !alive;
      delta -= (i64)__popc(__ballot_sync(FULL, died));
      pl.push3(&ctl, slot, alive, false, died);
      ev_cnt[CE_COLLIDE]++; ln_cnt[CE_COLLIDE] += n;
    }
    if (!R.kmode) {
      if (w.open_count != open_pub) { if (lane == 0) atomicAdd(&ctl.open_total, w.open_count - open_pub); open_pub = w.open_count; }
      // publish the outstanding delta now and then; hand secondaries over when some CTA is starved
      if (((ev_cnt[0] + ev_cnt[1]) & 15u) == 0) {
        if (delta != 0) { if (lane == 0) atomicAdd(R.outstanding, (u64)delta); delta = 0; }
        u32 s = 0;
        if (lane == 0) s = (u32)ld_vol(R.starved);
        if (__shfl_sync(FULL, s, 0) > 0 && w.open_count > 0) {
          ps_open_deposit(w);
          if (lane == 0) atomicAdd(&ctl.open_total, 0u - open_pub);
          open_pub = 0;
        }
      }
    }
  }
  if (delta != 0 && lane == 0) atomicAdd(R.outstanding, (u64)delta);
  if (lane == 0) {
    atomicAdd(&A.ctr[PC_EV_MOVE], (u64)ev_cnt[0]); atomicAdd(&A.ctr[PC_EV_COLLIDE], (u64)ev_cnt[1]); atomicAdd(&A.ctr[PC_EV_BIRTH], (u64)ev_cnt[2]);
    atomicAdd(&A.ctr[PC_LN_MOVE], (u64)ln_cnt[0]); atomicAdd(&A.ctr[PC_LN_COLLIDE], (u64)ln_cnt[1]); atomicAdd(&A.ctr[PC_LN_BIRTH], (u64)ln_cnt[2]);
    atomicAdd(&A.ctr[PC_SPILLS], (u64)w.n_spill); atomicAdd(&A.ctr[PC_FETCHES], (u64)w.n_fetch);
  }
  __syncthreads();
  acc_flush(&acc, O, accP, accPc);
  priv_flush(tp, O);
}
