// tdr_exec.cuh — one executor per event type, shared by the stack scheme's per-event kernels (decomposed task
// scheme) and by the asynchronous scheme's persistent kernel.  An executor loads
// the fields its event needs from the SoA state, runs the event, stores what changed and names the next event.
// Between split events the segment's intermediate values travel in scratch arrays (s_sigt, s_nsf, s_d, s_f,
// s_gi, s_flags).  All lanes of a warp call the same executor (valid = lane holds a particle).
#pragma once
#include "tdr_stack.cuh"

#define NEXT_DEAD (-1)

template <bool CE>
__device__ __forceinline__ void load_loc_energy(const Soa &S, u32 i, Part &p) {
  unpack_loc(p, S.loc0[i], S.loc1[i]);
  p.E = CE ? S.E[i] : 0.0;
}

// returns the next event of this lane's particle (NEXT_DEAD if it died or the lane is idle)
// IO (EV_STEP only): bit 0 = load the particle from the SoA state first, bit 1 = store a survivor back
template <bool CE, int EV, bool HYBRID = false, int IO = 3, class PT, class ST>
__device__ __forceinline__ int exec_event(const PT &P, const double *mg, const DevOut &O, const TallyPriv &tp, const DevRun &R, const ST &S,
                                          BlockAcc *acc, u32 slot, bool valid, Part &p, int &nch, int &csrc,
                                          i64 &accP, i64 &accPc, int first_ev) {
  nch = 0; csrc = 0;
  if (EV == EV_STEP) {                                   // monolithic step: T1..T8 in one event
    double St = 0.0, nsf = 0.0, d = 0.0, f = 0.0; int gi = 0; u32 flags = 0;
    if (valid) {
      if (IO & 1) load_part<CE>(S, slot, p);
      ev_lookup<CE>(P, mg, p, St, nsf, gi, f);
      ev_move(P, R.seed, R.gen, p, St, d, flags);
    }
    ev_tally<CE>(P, O, tp, R, p, valid && !(flags & F_LOST), d, St, nsf, flags, accP, accPc);
    bool alive = false;
    if (valid) {
      if ((flags & F_LOST) || p.seg >= (1u << 24)) atomicExch(O.err, TDR_ELOST);
      else if (flags & F_COLLIDE) {
        if (HYBRID) {                                     // hybrid scheme: collisions are their own event (uniform warps)
          S.x[slot] = p.x; S.y[slot] = p.y; S.z[slot] = p.z; S.seg[slot] = p.seg; S.s_sigt[slot] = St; if (ST::EXT && S.t) S.t[slot] = p.t;
          if (CE) { S.s_gi[slot] = (u32)gi; S.s_f[slot] = f; }
          return EV_COLLIDE;
        }
        alive = ev_collide<CE>(P, mg, R, acc, p, St, gi, f, nch, csrc);
      }
      else alive = ev_surface(P, R, acc, p, flags);
      if (alive) { if (IO & 2) store_part<CE>(S, slot, p); }
      else if (R.defer_death) { S.seg[slot] = p.seg; S.ncoll[slot] = p.ncoll; }
    }
    return alive ? EV_STEP : NEXT_DEAD;
  }
  if (EV == EV_LOOKUP) {
    if (!valid) return NEXT_DEAD;
    load_loc_energy<CE>(S, slot, p);
    double St, nsf, f; int gi;
    ev_lookup<CE>(P, mg, p, St, nsf, gi, f);
    S.s_sigt[slot] = St; S.s_nsf[slot] = nsf;
    if (CE) { S.s_gi[slot] = (u32)gi; S.s_f[slot] = f; }
    return EV_MOVE;
  }
  if (EV == EV_MOVE) {
    if (!valid) return NEXT_DEAD;
    load_part<CE>(S, slot, p);
    double d; u32 flags;
    ev_move(P, R.seed, R.gen, p, S.s_sigt[slot], d, flags);
    if ((flags & F_LOST) || p.seg >= (1u << 24)) { atomicExch(O.err, TDR_ELOST); return NEXT_DEAD; }
    S.x[slot] = p.x; S.y[slot] = p.y; S.z[slot] = p.z; S.seg[slot] = p.seg; if (ST::EXT && S.t) S.t[slot] = p.t;
    S.s_d[slot] = d; S.s_flags[slot] = flags;
    return EV_TALLY;
  }
  if (EV == EV_TALLY) {
    double d = 0.0, St = 0.0, nsf = 0.0; u32 flags = 0;
    if (valid) {
      load_loc_energy<CE>(S, slot, p);
      p.wgt = (ST::EXT && S.wgt) ? S.wgt[slot] : 1.0;
      d = S.s_d[slot]; St = S.s_sigt[slot]; nsf = S.s_nsf[slot]; flags = S.s_flags[slot];
    }
    ev_tally<CE>(P, O, tp, R, p, valid, d, St, nsf, flags, accP, accPc);
    if (!valid) return NEXT_DEAD;
    return (flags & F_COLLIDE) ? EV_COLLIDE : EV_SURFACE;
  }
  if (EV == EV_COLLIDE) {
    if (!valid) return NEXT_DEAD;
    load_part<CE>(S, slot, p);
    int gi = CE ? (int)S.s_gi[slot] : 0; double f = CE ? S.s_f[slot] : 0.0;
    bool alive = ev_collide<CE>(P, mg, R, acc, p, S.s_sigt[slot], gi, f, nch, csrc);
    if (alive) {
      S.u[slot] = p.u; S.v[slot] = p.v; S.w[slot] = p.w; S.ncoll[slot] = p.ncoll; S.loc1[slot] = pack_loc1(p);
      if (CE) S.E[slot] = p.E;
      if (ST::EXT && S.wgt) S.wgt[slot] = p.wgt;
    } else if (R.defer_death) S.ncoll[slot] = p.ncoll;
    return alive ? first_ev : NEXT_DEAD;
  }
  if (EV == EV_SURFACE) {
    if (!valid) return NEXT_DEAD;
    load_part<CE>(S, slot, p);
    bool alive = ev_surface(P, R, acc, p, S.s_flags[slot]);
    if (alive) {
      S.x[slot] = p.x; S.y[slot] = p.y; S.z[slot] = p.z; S.u[slot] = p.u; S.v[slot] = p.v; S.w[slot] = p.w;
      S.loc0[slot] = pack_loc0(p); S.loc1[slot] = pack_loc1(p); if (ST::EXT && S.t) S.t[slot] = p.t; if (ST::EXT && S.wgt) S.wgt[slot] = p.wgt;
    }
    return alive ? first_ev : NEXT_DEAD;
  }
  return NEXT_DEAD;
}
