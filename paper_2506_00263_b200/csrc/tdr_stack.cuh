// tdr_stack.cuh — stack-based remapping: per-event particle-index stacks with device counters,
// warp-collective push (one atomicAdd per warp, lanes index relative to it), pop by grid-stride over [0, count).
// make_work is folded into the event that kills a particle: the dead lane claims the next
// source index (or a pending secondary) with a warp-aggregated atomic and is reborn in the same slot.
#pragma once
#include "tdr_events.cuh"

// device counters (u64 each), one 128-byte readback per remap iteration
enum { C_SRC_NEXT = 0, C_SEC_TAIL, C_SEC_HEAD, C_BANK, C_HIST, C_NEXT_BANK, C_PENDING, C_STARVED,
       C_STACK0 = 8, /* C_STACK0..+7: stack counts */ C_COUNT = 16 };

// event ids (split decomposition; async scheme)
enum { EV_LOOKUP = 0, EV_MOVE, EV_TALLY, EV_COLLIDE, EV_SURFACE, EV_STEP, EV_SOURCE, EV_COUNT };

__device__ __forceinline__ u32 lanemask_lt() { u32 m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

// warp-collective push of one index per flagged lane
__device__ __forceinline__ void stack_push(u32 *stack, u64 *count, u32 value, bool pred) {
  u32 m = __ballot_sync(FULL, pred);
  if (m == 0) return;
  int leader = __ffs(m) - 1;
  u64 base = 0;
  if ((threadIdx.x & 31) == leader) base = atomicAdd(count, (u64)__popc(m));
  base = __shfl_sync(FULL, base, leader);
  if (pred) stack[base + __popc(m & lanemask_lt())] = value;
}

// warp-collective push of n sites per lane into the fission bank (k-mode) or the stack scheme's secondary ring (fixed source;
// the asynchronous scheme sends its secondaries through links of site records instead: tdr_links.cuh)
__device__ TDR_COLD void push_children(const DevOut &O, const DevRun &R, BlockAcc *acc, const Part &p, int n, int src) {
  u32 lane = threadIdx.x & 31;
  u32 total = __reduce_add_sync(FULL, (u32)n);
  if (total == 0) return;
  u32 incl = (u32)n;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { u32 t = __shfl_up_sync(FULL, incl, o); if (lane >= (u32)o) incl += t; }
  u32 excl = incl - (u32)n;
  u64 base = 0;
  if (lane == 0) { base = atomicAdd(R.kmode ? R.bank_count : R.sec_tail, (u64)total); acc_add(acc, TDR_T_NSITES, (u64)total); }
  base = __shfl_sync(FULL, base, 0);
  for (int c = 0; c < n; c++) {
    u64 t = base + excl + c;
    tdr_site s = make_site(R, p, src, (u32)c);
    if (R.kmode) { if (t < R.bank_cap) R.bank[t] = s; else atomicExch(O.err, TDR_ECAPACITY); }
    else if (t - R.sec_head0 < R.sec_cap) {                      // stack scheme: the ring; claimable once the loop control has seen the tail
      R.sec[t % R.sec_cap] = s; if (R.sec_time) R.sec_time[t % R.sec_cap] = p.t; if (R.sec_w) R.sec_w[t % R.sec_cap] = p.wgt;
    } else atomicExch(O.err, TDR_ECAPACITY);
  }
}

// make_work for dead lanes: pending secondaries first, then the primary source.  Returns true if reborn.
template <bool CE>
__device__ __forceinline__ bool make_work(const DevProb &P, const double *mg, const DevRun &R, BlockAcc *acc, Part &p, bool dead) {
  u32 lane = threadIdx.x & 31;
  bool reborn = false;
  if (!R.kmode && R.sec_limit > R.sec_head0) {
    u32 m = __ballot_sync(FULL, dead);
    if (m) {
      int leader = __ffs(m) - 1; u64 h = ~0ull;
      if (lane == (u32)leader && *(volatile u64 *)R.sec_head < R.sec_limit) h = atomicAdd(R.sec_head, (u64)__popc(m));
      h = __shfl_sync(FULL, h, leader);
      if (dead && h != ~0ull) {
        u64 idx = h + __popc(m & lanemask_lt());
        if (idx < R.sec_limit) { tdr_site s = R.sec[idx % R.sec_cap]; birth_site<CE>(P, mg, R, acc, p, s, R.sec_time ? R.sec_time[idx % R.sec_cap] : 0.0, R.sec_w ? R.sec_w[idx % R.sec_cap] : 1.0); reborn = true; }
      }
    }
  }
  u32 m = __ballot_sync(FULL, dead && !reborn);
  if (m) {
    int leader = __ffs(m) - 1; u64 h = ~0ull;
    if (lane == (u32)leader && *(volatile u64 *)R.src_next < R.src_total) h = atomicAdd(R.src_next, (u64)__popc(m));
    h = __shfl_sync(FULL, h, leader);
    if (dead && !reborn && h != ~0ull) {
      u64 idx = h + __popc(m & lanemask_lt());
      if (idx < R.src_total) {
        if (R.src_sites) { tdr_site s = R.sites[idx]; birth_site<CE>(P, mg, R, acc, p, s); }
        else birth_primary<CE>(P, mg, R, acc, p, idx);
        reborn = true;
      }
    }
  }
  return reborn;
}

// The table every lookup of the run reads, staged to shared memory by each CTA: the multigroup rows (X1), or, in continuous
// energy, the hash buckets of the energy grid (X3; BASELINE.json north_star: "hashed binary search staged through shared
// memory") — the events receive the block as `mg` either way.
// stage_ce = false: a continuous-energy kernel that would not win the copy back (one event per thread and launch, or a
// stash that needs the shared memory as L1: measured, profiles/ncu_r02.md) reads the same block from global memory.
__device__ __forceinline__ const double *stage_mg(const DevProb &P, double *smem, bool stage_ce = false) {
  if (P.mg_doubles == 0) return nullptr;
  if (P.G == 0 && !stage_ce) return P.mg;
  for (int i = threadIdx.x; i < P.mg_doubles; i += blockDim.x) smem[i] = P.mg[i];
  return smem;
}
// dynamic shared memory = [MG table | private tally words]; host side: smem_bytes()
__device__ __forceinline__ int staged_doubles(const DevProb &P, bool stage_ce) { return (P.G == 0 && !stage_ce) ? 0 : P.mg_doubles; }
__device__ __forceinline__ TallyPriv stage_priv(const DevProb &P, double *smem, const double *mg, bool stage_ce = false) {
  return priv_init(P, smem + staged_doubles(P, stage_ce));
}

// ---------------------------------------------------------------------------------- A1 SOURCE: fill slots [0, n)
template <bool CE>
__global__ void __launch_bounds__(256) k_source(DevProb P, DevOut O, DevRun R, Soa S, u32 *stack, u64 *count,
                                                u64 sec_start, u64 n_sec, u64 src_start, u64 n) {
  // the host knows both cursors exactly here (it just synchronised): publish them for make_work
  if (blockIdx.x == 0 && threadIdx.x == 0) { *R.src_next = src_start + (n - n_sec); *R.sec_head = sec_start + n_sec; }
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  const double *mg = stage_mg(P, smem);
  acc_init(&acc);
  for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) {
    Part p;
    if (i < n_sec) { tdr_site s = R.sec[(sec_start + i) % R.sec_cap]; birth_site<CE>(P, mg, R, &acc, p, s, R.sec_time ? R.sec_time[(sec_start + i) % R.sec_cap] : 0.0, R.sec_w ? R.sec_w[(sec_start + i) % R.sec_cap] : 1.0); }
    else {
      u64 idx = src_start + (i - n_sec);
      if (R.src_sites) { tdr_site s = R.sites[idx]; birth_site<CE>(P, mg, R, &acc, p, s); }
      else birth_primary<CE>(P, mg, R, &acc, p, idx);
    }
    store_part<CE>(S, (u32)i, p);
    stack[i] = (u32)i;
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) *count = n;
  acc_flush(&acc, O, 0, 0);
}

// ---------------------------------------------------------------------------------- where a remap kernel finds its DevRun
// DEV = false: by value, the host drives the remap loop and reads the counters back between batches.  DEV = true: from
// device memory, copied to shared memory at kernel start — the remap loop then runs as a CUDA-graph WHILE node whose last
// kernel (k_loop_ctl) updates the claimable range of the secondary ring and decides whether another pass is needed, so the
// host is out of the loop ("fixed costs": the launch and read-back latency of every remap iteration).
#define TDR_BIND_RUN(DEV, Rv, Rp)                                                                                               \
  __shared__ DevRun Rs_;                                                                                                        \
  if (DEV) { for (u32 i_ = threadIdx.x; i_ < (u32)(sizeof(DevRun) / 8); i_ += blockDim.x) ((u64 *)&Rs_)[i_] = ((const u64 *)(Rp))[i_]; } \
  const DevRun &R = DEV ? Rs_ : Rv;        /* visible after the barrier that ends acc_init */

// ---------------------------------------------------------------------------------- fused STEP (monolithic scheme)
// HYBRID: a particle that collides is not processed here; it is pushed onto the collide stack (cstack) and the
// collision runs as its own event in k_collide, where every lane of a warp takes the same path.
// The step stacks alternate and their counters rotate by three (in, out, the one to clear) with the remap iteration `it`.
// The host-driven loop passes the pointers of its iteration; the device-driven loop passes the bases (stack_in = stack 0,
// stack_out = stack 1, count_in = the counter block `ctr`) and every kernel derives its own from the iteration counter that
// k_loop_ctl keeps in ctr[C_PENDING] — so the WHILE body is ONE iteration and the loop condition is tested after each.
template <bool CE, bool HYBRID, bool DEV, bool EXT>
__global__ void __launch_bounds__(256, 2) k_step(DevProb P0, DevOut O, DevRun Rv, const DevRun *Rp, Soa S0, const u32 *stack_in, const u64 *count_in,
                                              u32 *stack_out, u64 *count_out, u64 *count_zero,
                                              u32 *cstack, u64 *ccount, u64 *ccount_zero, u32 seg_per_launch, int sync_seg) {
  const ProbX<EXT> &P = static_cast<const ProbX<EXT> &>(P0);
  const SoaX<EXT> &S = static_cast<const SoaX<EXT> &>(S0);
  if (DEV) {
    u64 *ctr = const_cast<u64 *>(count_in);
    const u64 it = ctr[C_PENDING];
    u32 *s0 = const_cast<u32 *>(stack_in), *s1 = stack_out;
    stack_in = (it & 1) ? s1 : s0; stack_out = (it & 1) ? s0 : s1;
    count_in = ctr + C_STACK0 + it % 3; count_out = ctr + C_STACK0 + (it + 1) % 3; count_zero = ctr + C_STACK0 + (it + 2) % 3;
    if (HYBRID) { ccount = ctr + C_STACK0 + 3 + (it & 1); ccount_zero = ctr + C_STACK0 + 3 + ((it + 1) & 1); }
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {       // the stacks the previous launches drained (rotating counters)
    *count_zero = 0;
    if (HYBRID) *ccount_zero = 0;
  }
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  TDR_BIND_RUN(DEV, Rv, Rp)
  const double *mg = stage_mg(P, smem, true);
  const TallyPriv tp = stage_priv(P, smem, mg, true);
  acc_init(&acc);
  const u64 n_in = *count_in;
  i64 accP = 0, accPc = 0;
  for (u64 i0 = (u64)blockIdx.x * blockDim.x; i0 < n_in; i0 += (u64)gridDim.x * blockDim.x) {
    __syncthreads();       // the CTA's warps start each tile together: they share the instruction lines they fetch
    u64 i = i0 + threadIdx.x;
    bool valid = i < n_in;
    Part p; u32 slot = 0;
    if (valid) { slot = stack_in[i]; load_part<CE>(S, slot, p); }
    // sync_seg: the CTA's warps also start every SEGMENT of the tile together and leave the loop together (the vote below), so the
    // lines one warp fetches serve the others for the whole tile, as in the persistent kernel's lockstep (+7 ... +19 % in
    // multigroup, -5 ... -7 % in continuous energy where the cross-section gathers make segments uneven: profiles/ncu_r02.md)
    // up to seg_per_launch segments per particle in registers before it is pushed again ("history-length truncation",
    // PAPER.md:119, with a length > 1): fewer launches and state round trips; a lane whose particle died idles
    bool alive = valid, to_collide = false;
    for (u32 k = 0; k < seg_per_launch; k++) {
      double St = 0.0, nsf = 0.0, d = 0.0, f = 0.0; int gi = 0; u32 flags = 0;
      if (alive) { ev_lookup<CE>(P, mg, p, St, nsf, gi, f); ev_move(P, R.seed, R.gen, p, St, d, flags); }
      ev_tally<CE>(P, O, tp, R, p, alive && !(flags & F_LOST), d, St, nsf, flags, accP, accPc);
      int nch = 0, csrc = 0;
      if (alive) {
        if ((flags & F_LOST) || p.seg >= (1u << 24)) { atomicExch(O.err, TDR_ELOST); alive = false; }
        else if (flags & F_COLLIDE) {
          if (HYBRID) {
            if (k > 0) store_part<CE>(S, slot, p);       // an earlier crossing of this launch changed direction / indices too
            else { S.x[slot] = p.x; S.y[slot] = p.y; S.z[slot] = p.z; S.seg[slot] = p.seg; if (EXT && S.t) S.t[slot] = p.t; }
            S.s_sigt[slot] = St;
            if (CE) { S.s_gi[slot] = (u32)gi; S.s_f[slot] = f; }
            to_collide = true; alive = false;
          } else alive = ev_collide<CE>(P, mg, R, &acc, p, St, gi, f, nch, csrc);
        }
        else alive = ev_surface(P, R, &acc, p, flags);
      }
      if (!HYBRID) push_children(O, R, &acc, p, nch, csrc);
      if (sync_seg ? !__syncthreads_or(alive) : !__any_sync(FULL, alive)) break;
    }
    if (make_work<CE>(P, mg, R, &acc, p, valid && !alive && !to_collide)) alive = true;
    if (alive) store_part<CE>(S, slot, p);
    stack_push(stack_out, count_out, slot, alive);
    if (HYBRID) stack_push(cstack, ccount, slot, to_collide);
  }
  acc_flush(&acc, O, accP, accPc);
  priv_flush(tp, O);
}

// ---------------------------------------------------------------------------------- tail drain (stack scheme, k-mode)
// Once the source is exhausted and only a few thousand particles are left, a remap iteration is a kernel launch
// that lasts one segment's latency (the "fixed costs" of PAPER.md:153).  This kernel pops the step stack once and
// follows each remaining particle to its death in registers: one launch instead of ~100.  No make_work (nothing is
// left to claim), children go to the fission bank as usual; a warp keeps calling the warp-cooperative tally until
// its last lane is done.
template <bool CE, bool EXT>
__global__ void __launch_bounds__(256) k_drain(DevProb P0, DevOut O, DevRun R, Soa S0, const u32 *stack_in, const u64 *count_in) {
  const ProbX<EXT> &P = static_cast<const ProbX<EXT> &>(P0);
  const SoaX<EXT> &S = static_cast<const SoaX<EXT> &>(S0);
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  const double *mg = stage_mg(P, smem, true);
  const TallyPriv tp = stage_priv(P, smem, mg, true);
  acc_init(&acc);
  const u64 n_in = *count_in;
  i64 accP = 0, accPc = 0;
  for (u64 i0 = (u64)blockIdx.x * blockDim.x; i0 < n_in; i0 += (u64)gridDim.x * blockDim.x) {
    const u64 i = i0 + threadIdx.x;
    bool live = i < n_in;
    Part p;
    if (live) load_part<CE>(S, stack_in[i], p);
    while (__any_sync(FULL, live)) {
      double St = 0.0, nsf = 0.0, d = 0.0, f = 0.0; int gi = 0; u32 flags = 0;
      if (live) { ev_lookup<CE>(P, mg, p, St, nsf, gi, f); ev_move(P, R.seed, R.gen, p, St, d, flags); }
      ev_tally<CE>(P, O, tp, R, p, live && !(flags & F_LOST), d, St, nsf, flags, accP, accPc);
      int nch = 0, csrc = 0;
      if (live) {
        if ((flags & F_LOST) || p.seg >= (1u << 24)) { atomicExch(O.err, TDR_ELOST); live = false; }
        else if (flags & F_COLLIDE) live = ev_collide<CE>(P, mg, R, &acc, p, St, gi, f, nch, csrc);
        else live = ev_surface(P, R, &acc, p, flags);
      }
      push_children(O, R, &acc, p, nch, csrc);
    }
  }
  acc_flush(&acc, O, accP, accPc);
  priv_flush(tp, O);
}

// ---------------------------------------------------------------------------------- device-driven remap loop: the WHILE condition
// Last kernel of a pass of the graph's body (one thread).  It does what the host does between two batches of the host-driven
// loop: every kernel of the pass has completed, so every secondary below the ring's tail is whole and claimable; claims past
// the old limit got nothing and are given back.  Another pass follows while particles are alive, no error is flagged and the
// k-mode tail has not become short enough for k_drain.
struct LoopCtl { u64 *ctr; DevRun *R; int split; u64 drain_below; };
__global__ void k_loop_ctl(LoopCtl c, cudaGraphConditionalHandle h) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  u64 *ctr = c.ctr; DevRun *R = c.R;
  const u64 it = ctr[C_PENDING] + 1;               // iterations made (the stack scheme has no other use for this counter)
  ctr[C_PENDING] = it;
  const u64 alive = ctr[C_STACK0 + (c.split ? (u64)EV_LOOKUP : it % 3)];
  const int err = *(const int *)(ctr + (C_COUNT - 1));
  u64 head = ctr[C_SEC_HEAD];
  if (head > R->sec_limit) { head = R->sec_limit; ctr[C_SEC_HEAD] = head; }
  R->sec_limit = ctr[C_SEC_TAIL]; R->sec_head0 = head;
  const bool exhausted = ctr[C_SRC_NEXT] >= R->src_total;
  const bool drain = R->kmode && exhausted && alive <= c.drain_below;
  cudaGraphSetConditional(h, (alive > 0 && err == 0 && !drain) ? 1u : 0u);
}

// ---------------------------------------------------------------------------------- A9 population control (D2)
__global__ void __launch_bounds__(256) k_popctrl(const tdr_site *bank, u64 n_bank, tdr_site *next, u64 next_cap, u64 *next_count,
                                                 u64 seed, u32 gen_next, double pr, int *err) {
  u32 lane = threadIdx.x & 31;
  for (u64 i0 = (u64)blockIdx.x * blockDim.x; i0 < n_bank; i0 += (u64)gridDim.x * blockDim.x) {
    u64 i = i0 + threadIdx.x;
    int m = 0; tdr_site s;
    if (i < n_bank) {
      s = bank[i];
      m = (int)floor(pr + draw(seed, s.id, gen_next, 0, PUR_POPCTRL, 0));
      if (m > 2048) m = 2048;
    }
    u32 total = __reduce_add_sync(FULL, (u32)m);
    if (total == 0) continue;
    u32 incl = (u32)m;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { u32 t = __shfl_up_sync(FULL, incl, o); if (lane >= (u32)o) incl += t; }
    u64 base = 0;
    if (lane == 0) base = atomicAdd(next_count, (u64)total);
    base = __shfl_sync(FULL, base, 0) + (incl - (u32)m);
    u64 sid = s.id;
    for (int r = 0; r < m; r++) {
      s.id = derive_id(seed, sid, gen_next, 0, 2048u + (u32)r);
      if (base + r < next_cap) next[base + r] = s; else atomicExch(err, TDR_ECAPACITY);
    }
  }
}

// N5 for tallies too large to be block-private (global `red`): after every generation / run, a bin whose top bit is set
// has left int64 (scores are non-negative; one generation cannot add 2^63 to a bin)
__global__ void k_overflow_check(const u64 *flux, const u64 *coll, u64 n_bins, int *err) {
  for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n_bins; i += (u64)gridDim.x * blockDim.x)
    if ((flux[i] | coll[i]) >> 63) atomicExch(err, TDR_EOVERFLOW);
}

// ---------------------------------------------------------------------------------- unit kernels
__global__ void k_det_log(const double *x, double *out, u64 n) {
  for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x) out[i] = det_log(x[i]);
}
__global__ void k_draw(u64 seed, const u64 *id, u32 gen, u32 seg, u32 purpose, u32 j, double *out, u64 n) {
  for (u64 i = (u64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (u64)gridDim.x * blockDim.x)
    out[i] = draw(seed, id[i], gen, seg, purpose, j);
}
