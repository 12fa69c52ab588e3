// tdr_split.cuh — decomposed task scheme under stack-based remapping:
// five event types (LOOKUP, MOVE, TALLY, COLLIDE, SURFACE), one index stack and one kernel per event.
// One remap iteration launches the five kernels in flow order, each popping its own stack (count read on
// the device) and pushing every particle onto the stack of its next event; a kernel whose stack is empty
// returns at once.  Dead lanes call make_work in place (COLLIDE / SURFACE) and re-enter at LOOKUP.
#pragma once
#include "tdr_exec.cuh"

struct StackSet { u32 *s[EV_COUNT]; u64 *cnt; };      // cnt[e] = device counter of stack e

template <bool CE, int EV, bool DEV, bool EXT>
__global__ void __launch_bounds__(256) k_event(DevProb P0, DevOut O, DevRun Rv, const DevRun *Rp, Soa S0, StackSet K, int zero_ev) {
  const ProbX<EXT> &P = static_cast<const ProbX<EXT> &>(P0);
  const SoaX<EXT> &S = static_cast<const SoaX<EXT> &>(S0);
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  TDR_BIND_RUN(DEV, Rv, Rp)
  const double *mg = stage_mg(P, smem);
  const TallyPriv tp = stage_priv(P, smem, mg);
  acc_init(&acc);
  if (blockIdx.x == 0 && threadIdx.x == 0 && zero_ev >= 0) K.cnt[zero_ev] = 0;   // the stack the previous kernel drained
  const u64 n_in = K.cnt[EV];
  i64 accP = 0, accPc = 0;
  for (u64 i0 = (u64)blockIdx.x * blockDim.x; i0 < n_in; i0 += (u64)gridDim.x * blockDim.x) {
    u64 i = i0 + threadIdx.x;
    bool valid = i < n_in;
    u32 slot = valid ? K.s[EV][i] : 0;
    Part p; int nch, csrc;
    int next = exec_event<CE, EV>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, EV_LOOKUP);
    if (EV == EV_COLLIDE || EV == EV_SURFACE) {
      if (EV == EV_COLLIDE) push_children(O, R, &acc, p, nch, csrc);
      bool dead = valid && next == NEXT_DEAD;
      if (make_work<CE>(P, mg, R, &acc, p, dead)) { store_part<CE>(S, slot, p); next = EV_LOOKUP; }
      stack_push(K.s[EV_LOOKUP], &K.cnt[EV_LOOKUP], slot, next == EV_LOOKUP);
    } else if (EV == EV_TALLY) {
      stack_push(K.s[EV_COLLIDE], &K.cnt[EV_COLLIDE], slot, next == EV_COLLIDE);
      stack_push(K.s[EV_SURFACE], &K.cnt[EV_SURFACE], slot, next == EV_SURFACE);
    } else {
      const int nx = EV == EV_LOOKUP ? EV_MOVE : EV_TALLY;
      stack_push(K.s[nx], &K.cnt[nx], slot, next == nx);
    }
  }
  acc_flush(&acc, O, accP, accPc);
  if (EV == EV_TALLY) priv_flush(tp, O);
}

// hybrid scheme, second kernel of a remap iteration: the COLLIDE event on the collide stack; survivors (and lanes
// reborn by make_work) join the step stack the preceding k_step<CE, true> launch was pushing to.
template <bool CE, bool DEV, bool EXT>
__global__ void __launch_bounds__(256) k_collide(DevProb P0, DevOut O, DevRun Rv, const DevRun *Rp, Soa S0, const u32 *cstack, const u64 *ccount,
                                                 u32 *stack_out, u64 *count_out) {
  const ProbX<EXT> &P = static_cast<const ProbX<EXT> &>(P0);
  const SoaX<EXT> &S = static_cast<const SoaX<EXT> &>(S0);
  if (DEV) {                                       // bases in, this iteration's pointers out (see k_step)
    u64 *ctr = const_cast<u64 *>(ccount);
    const u64 it = ctr[C_PENDING];
    ccount = ctr + C_STACK0 + 3 + (it & 1);
    u32 *s0 = stack_out, *s1 = reinterpret_cast<u32 *>(count_out);
    stack_out = (it & 1) ? s0 : s1; count_out = ctr + C_STACK0 + (it + 1) % 3;
  }
  extern __shared__ double smem[];
  __shared__ BlockAcc acc;
  TDR_BIND_RUN(DEV, Rv, Rp)
  const double *mg = stage_mg(P, smem);
  const TallyPriv tp = stage_priv(P, smem, mg);
  acc_init(&acc);
  const u64 n_in = *ccount;
  i64 accP = 0, accPc = 0;
  for (u64 i0 = (u64)blockIdx.x * blockDim.x; i0 < n_in; i0 += (u64)gridDim.x * blockDim.x) {
    u64 i = i0 + threadIdx.x;
    bool valid = i < n_in;
    u32 slot = valid ? cstack[i] : 0;
    Part p; int nch, csrc;
    int next = exec_event<CE, EV_COLLIDE>(P, mg, O, tp, R, S, &acc, slot, valid, p, nch, csrc, accP, accPc, EV_STEP);
    push_children(O, R, &acc, p, nch, csrc);
    if (make_work<CE>(P, mg, R, &acc, p, valid && next == NEXT_DEAD)) { store_part<CE>(S, slot, p); next = EV_STEP; }
    stack_push(stack_out, count_out, slot, next == EV_STEP);
  }
  acc_flush(&acc, O, accP, accPc);
}

