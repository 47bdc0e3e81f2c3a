// One particle, one timestep: gather E, Boris push, move, boundary (+ re-injection / pair source),
// null-collision Monte Carlo.  SURVEY.md 8(c) "G, B, M, W, C, A"; PAPER.md:33 steps (i),(iv) and the
// "MC routines", PAPER.md:111 mover move0/moveb, PAPER.md:95 wall absorption.
//
// SINK says what becomes of the step's side effects (same arithmetic in every case):
//   SinkList   mover pass A: counters and diagnostics are updated, births go to the side list;
//   SinkNone   arranger pass B (the recompute pass): no side effects;
//   SinkStore  general path (general_kernels.cu): counters are left alone (pass A has already counted this step),
//              births are handed back to the caller, which ranks them itself.
#pragma once
#include <cooperative_groups.h>

#include "device_math.cuh"
#include "pipeline.cuh"

namespace bit1 {

namespace cg_adv = cooperative_groups;

__device__ __forceinline__ unsigned long long make_key(const Params& P, int cell, unsigned cls,
                                                       unsigned long long ord) {
  return ((unsigned long long)(unsigned)cell << P.cell_shift) | ((unsigned long long)cls << P.ord_bits) | ord;
}

// Append one record (far mover or birth) to the side list.  Order of arrival is irrelevant: k_mid sorts by key.
// Warp-aggregated (BASELINE.json north_star, "warp-aggregated append of newborn particles"): the lanes of a warp that
// arrive here together take their slots with ONE atomic on the list's counter -- the lowest of them adds their number,
// everybody gets the base by shuffle and adds its rank among them -- instead of one atomic per record on a single
// address, which is what serialises a step with many far movers (profiles/r2_far_mover_sweep.md).
static __device__ __noinline__ void emit_record(const Params& P, unsigned long long key, double x, double vx, double vy,
                                         double vz, unsigned pid, int sp) {
  const cg_adv::coalesced_group together = cg_adv::coalesced_threads();
  unsigned base = 0;
  if (together.thread_rank() == 0) base = atomicAdd(&P.st->ovf_count, (unsigned)together.size());
  const unsigned slot = together.shfl(base, 0) + together.thread_rank();
  if (slot >= P.ovf_cap) return;   // k_mid sees ovf_count > ovf_cap and stalls the step: the general path takes it
  P.ovf_key[BIT1_CHECK(P.st, slot, P.ovf_cap)] = key;
  OvfRec r;
  r.x = x; r.vx = vx; r.vy = vy; r.vz = vz; r.pid = pid; r.sp = (unsigned)sp;
  P.ovf_rec[slot] = r;
}

struct PairBirth {
  int on;
  double vx, vy, vz;
};

// kind of a birth = its place among its parent's births (SURVEY 8(c) "A"): 0 source partner, 1 ionisation
// electron, 2 ionisation ion, 3 recycled neutral (reading N2-a)
struct SinkNone {
  static constexpr bool kCounters = false, kBirths = false;
  __device__ __forceinline__ void birth(const Params&, int, int, double, double, double, double, int) {}
};
struct SinkList {
  static constexpr bool kCounters = true, kBirths = true;
  unsigned gidx;   // array index of the parent: births are ordered by (parent index, kind)
  __device__ __forceinline__ void birth(const Params& P, int kind, int cell, double x, double vx, double vy,
                                        double vz, int sp) {
    emit_record(P, make_key(P, cell, 2u, (unsigned long long)gidx * 4ull + (unsigned long long)kind), x, vx, vy, vz,
                0u, sp);
  }
};
struct BirthRec {
  double x, vx, vy, vz;
  int cell, sp;
};
struct SinkStore {
  static constexpr bool kCounters = false, kBirths = true;
  unsigned mask;
  BirthRec rec[4];
  __device__ __forceinline__ void birth(const Params&, int kind, int cell, double x, double vx, double vy, double vz,
                                        int sp) {
    mask |= 1u << kind;
    BirthRec& r = rec[kind];
    r.x = x; r.vx = vx; r.vy = vy; r.vz = vz; r.cell = cell; r.sp = sp;
  }
};

// W: wall hit on an absorbing boundary.  Returns alive.
template <class SINK>
__device__ __noinline__ bool wall_event(const Params& P, const SpeciesP* S, unsigned long long step, int sp,
                                        unsigned pid, SINK& sink, int side, bool escaped, double& x, double& vx,
                                        double& vy, double& vz, PairBirth& pb) {
  const SpeciesP& s = S[sp];
  if (SINK::kCounters) {
    if (escaped) {
      atomicOr(&P.st->flags, kFlagEscape);
      atomicAdd(&P.st->escape, 1ull);
    }
    atomicAdd(&P.st->wall_count[side][sp], 1ull);
    atomicAdd((unsigned long long*)&P.st->wall_charge[side], (unsigned long long)((long long)s.sign * s.Q));
  }
  if (SINK::kBirths) {
    if (s.recycle_to >= 0) {
      // NEXT-2 wall recycling (reading N2-a): one particle of species recycle_to is born at
      // the wall, half-Maxwellian into the plasma, from slot 14 of the parent's stream; the parent's fourth birth
      const uint4 wr = draw(P, pid, step, 14u);
      double z0 = normal_from_word(P, wr.x);
      if (z0 < 0.0) z0 = -z0;
      const double vz0 = s.recycle_vth * z0;
      const double rvx = side == 0 ? vz0 : -vz0;
      const double rvy = s.recycle_vth * normal_from_word(P, wr.y);
      const double rvz = s.recycle_vth * normal_from_word(P, wr.z);
      const double rx = side == 0 ? 0.0 : P.L - P.dx * 9.5367431640625e-07;
      const int rc = side == 0 ? 0 : P.nc - 1;
      sink.birth(P, 3, rc, rx, rvx, rvy, rvz, s.recycle_to);
      if (SINK::kCounters) atomicAdd(&P.st->recycled, 1ull);
    }
  }
  if (s.src_mode == kSrcNone) return false;
  const uint4 w = draw(P, pid, step, 2u);  // slot RJ
  const double u0 = u32(w.x);
  x = P.src_lo + u0 * P.src_span;
  vx = s.src_vth * normal_from_word(P, w.y);
  vy = s.src_vth * normal_from_word(P, w.z);
  vz = s.src_vth * normal_from_word(P, w.w);
  if (SINK::kCounters) atomicAdd(&P.st->reinject, 1ull);
  if (s.src_mode == kSrcPair) {
    const double pv = S[s.src_partner].src_vth;
    const uint4 wp = draw(P, pid, step, 13u);  // slot PB
    pb.on = 1;
    pb.vx = pv * normal_from_word(P, wp.x);
    pb.vy = pv * normal_from_word(P, wp.y);
    pb.vz = pv * normal_from_word(P, wp.z);
  }
  return true;
}

// C: a null-collision candidate (u0 < pnull).  Rewrites v; ionisation emits two births.
template <class SINK>
__device__ __noinline__ void collide(const Params& P, const SpeciesP* S, unsigned long long step, int sp,
                                     unsigned pid, SINK& sink, double u1, double x, int cn, double& vx,
                                     double& vy, double& vz) {
  static_assert(SINK::kBirths || !SINK::kCounters, "the direction-fallback counter needs the births' second draw");
  const SpeciesP& s = S[sp];
  const unsigned fl = s.flags;
  if (SINK::kCounters) atomicAdd(&P.st->candidates[sp], 1ull);
  double vnx = 0.0, vny = 0.0, vnz = 0.0;
  if (fl & kTargetMaxwellian) {
    const uint4 wn = draw(P, pid, step, 1u);  // slot NV
    vnx = P.vth_n * normal_from_word(P, wn.x);
    vny = P.vth_n * normal_from_word(P, wn.y);
    vnz = P.vth_n * normal_from_word(P, wn.z);
  }
  const double gx = vx - vnx, gy = vy - vny, gz = vz - vnz;
  const double g2 = (gx * gx + gy * gy) + gz * gz;
  const double g = sqrt(g2);
  const double EeV = s.kin_eV * g2;
  const double r = u1 * s.numax;
  // NEXT-2 (reading N2-b): the target density is the neutral particles' own, in the candidate's new cell, from the
  // previous step's deposit (mean of the cell's two nodes)
  double nloc = P.n0;
  if (P.target_species >= 0) {
    int j1 = cn + 1;
    if (!P.bc && j1 == P.nc) j1 = 0;
    const long long* D = P.dens_old + (size_t)P.target_species * (size_t)P.ng;
    nloc = (double)(D[cn] + D[j1]) * P.kn;
  }
  double cum = 0.0;
  int chosen = -1;
  if (fl & kElastic) {
    cum = cum + (nloc * sigma_lookup(P, P.sig_el, EeV)) * g;
    if (chosen < 0 && r < cum) chosen = 0;
  }
  if (fl & kIonise) {
    // reading R-thr: zero at or below the threshold, whatever the table interpolates to there
    const double sig_i = EeV > P.E_ion ? sigma_lookup(P, P.sig_ion, EeV) : 0.0;
    cum = cum + (nloc * sig_i) * g;
    if (chosen < 0 && r < cum) chosen = 1;
  }
  if (fl & kCx) {
    cum = cum + (nloc * sigma_lookup(P, P.sig_cx, EeV)) * g;
    if (chosen < 0 && r < cum) chosen = 2;
  }
  if (SINK::kCounters && cum > s.numax) atomicAdd(&P.st->nu_overflow, 1ull);
  if (chosen == 0) {
    double nn[3];
    const int fb = direction(P, pid, step, 4u, nn);
    const double dot = (vx * nn[0] + vy * nn[1]) + vz * nn[2];
    const double cosx = dot / g;
    const double gn = g * sqrt(1.0 - s.el_loss * (1.0 - cosx));
    vx = gn * nn[0]; vy = gn * nn[1]; vz = gn * nn[2];
    if (SINK::kCounters) {
      if (fb) atomicAdd(&P.st->dir_fallback, 1ull);
      atomicAdd(&P.st->events[sp][0], 1ull);
    }
  } else if (chosen == 1) {
    const double Er = EeV - P.E_ion;
    const uint4 ws = draw(P, pid, step, 3u);  // slot SP
    const double u = u52(ws.x, ws.y);
    const double E1 = u * Er;
    const double E2 = Er - E1;
    double n1[3], n2[3];
    const int fb1 = direction(P, pid, step, 4u, n1);
    const double sp1 = sqrt(E1 * s.two_e_over_m);
    vx = sp1 * n1[0]; vy = sp1 * n1[1]; vz = sp1 * n1[2];
    if (SINK::kBirths) {
      const int fb2 = direction(P, pid, step, 8u, n2);
      const double sp2 = sqrt(E2 * S[P.sp_ep].two_e_over_m);
      const uint4 wb = draw(P, pid, step, 12u);  // slot BI
      const double ivx = P.vth_n * normal_from_word(P, wb.x);
      const double ivy = P.vth_n * normal_from_word(P, wb.y);
      const double ivz = P.vth_n * normal_from_word(P, wb.z);
      sink.birth(P, 1, cn, x, sp2 * n2[0], sp2 * n2[1], sp2 * n2[2], P.sp_ep);
      sink.birth(P, 2, cn, x, ivx, ivy, ivz, P.sp_ip);
      if (SINK::kCounters) {
        if (fb1 + fb2) atomicAdd(&P.st->dir_fallback, (unsigned long long)(fb1 + fb2));
        atomicAdd(&P.st->events[sp][1], 1ull);
      }
    }
  } else if (chosen == 2) {
    vx = vnx; vy = vny; vz = vnz;
    if (SINK::kCounters) atomicAdd(&P.st->events[sp][2], 1ull);
  }
}

// The whole per-particle step.  In: state at step k (c = current cell).  Out: state at k+1, c = new cell
// or -1 when the particle died.  Eptr[c], Eptr[c+1] must be readable (global E or a shared-memory window).
template <class SINK>
__device__ __forceinline__ void advance(const Params& P, const SpeciesP* S, unsigned long long step,
                                        const double* Eptr, int sp, unsigned pid, SINK& sink, double& x,
                                        double& vx, double& vy, double& vz, int& c) {
  const SpeciesP& s = S[sp];
  // G
  const double f = x * P.inv_dx - (double)c;
  const double e0 = Eptr[c], e1 = Eptr[c + 1];
  const double Ex = e0 + f * (e1 - e0);
  // B
  const double a = s.h * Ex;
  const double ux = vx + a, uy = vy, uz = vz;
  const double px = ux + (uy * s.tz - uz * s.ty);
  const double py = uy + (uz * s.tx - ux * s.tz);
  const double pz = uz + (ux * s.ty - uy * s.tx);
  const double wx = ux + (py * s.sz - pz * s.sy);
  const double wy = uy + (pz * s.sx - px * s.sz);
  const double wz = uz + (px * s.sy - py * s.sx);
  vx = wx + a; vy = wy; vz = wz;
  // M
  x = x + vx * P.dt;
  // W
  bool alive = true;
  PairBirth pb;
  pb.on = 0;
  if (!P.bc) {
    if (x < 0.0) x = x + P.L;
    if (x >= P.L) x = x - P.L;
    if (!(x >= 0.0 && x < P.L)) {
      if (SINK::kCounters) {
        atomicOr(&P.st->flags, kFlagEscape);
        atomicAdd(&P.st->escape, 1ull);
      }
      x = 0.0;
    }
  } else if (!(x >= 0.0 && x < P.L)) {
    const int side = (x >= P.L) ? 1 : 0;
    const bool escaped = !(x < 0.0) && !(x >= P.L);  // NaN
    alive = wall_event<SINK>(P, S, step, sp, pid, sink, side, escaped, x, vx, vy, vz, pb);
  }
  const int cn = alive ? cell_of(P, x) : -1;
  // C
  if (alive && (s.flags & (kElastic | kIonise | kCx))) {
    const uint4 w = draw(P, pid, step, 0u);  // slot C0
    const double u0 = u52(w.x, w.y);
    if (u0 < s.pnull) collide<SINK>(P, S, step, sp, pid, sink, u52(w.z, w.w), x, cn, vx, vy, vz);
  }
  // A: the pair-source partner is the parent's first birth (kind 0)
  if (SINK::kBirths && pb.on) sink.birth(P, 0, cn, x, pb.vx, pb.vy, pb.vz, s.src_partner);
  c = cn;
}

// G, B, M only: the part of the step that every particle takes.  Same expressions, same order as advance().
// Returns true when the moved particle is inside [0, L) -- no wall hit, no periodic wrap.
__device__ __forceinline__ bool push_fast(const Params& P, const SpeciesP& s, const double* Eptr, int c, double& x,
                                          double& vx, double& vy, double& vz) {
  const double f = x * P.inv_dx - (double)c;
  const double e0 = Eptr[c], e1 = Eptr[c + 1];
  const double Ex = e0 + f * (e1 - e0);
  const double a = s.h * Ex;
  const double ux = vx + a, uy = vy, uz = vz;
  const double px = ux + (uy * s.tz - uz * s.ty);
  const double py = uy + (uz * s.tx - ux * s.tz);
  const double pz = uz + (ux * s.ty - uy * s.tx);
  const double wx = ux + (py * s.sz - pz * s.sy);
  const double wy = uy + (pz * s.sx - px * s.sz);
  const double wz = uz + (px * s.sy - py * s.sx);
  vx = wx + a; vy = wy; vz = wz;
  x = x + vx * P.dt;
  return x >= 0.0 && x < P.L;
}

// The rare path (wall hit, periodic wrap, null-collision candidate): redo the whole step of particle `off` of
// the staged tile from its stored state, write the new state back into the stage and return the new cell
// (-1: dead).  Taking the state from shared memory keeps every by-reference argument of the rare code out of
// the callers' registers and stack.
template <class SINK>
static __device__ __noinline__ int slow_advance(const Params& P, const SpeciesP* S, unsigned long long step,
                                                const double* Eptr, Stage* st, int off, unsigned gidx) {
  double x = st->x[off], vx = st->vx[off], vy = st->vy[off], vz = st->vz[off];
  int c = cell_of(P, x);   // the particle's current cell (the staged tile does not carry the cell array)
  SINK sink;
  if constexpr (SINK::kCounters) sink.gidx = gidx;
  advance<SINK>(P, S, step, Eptr, (int)st->sp[off], st->pid[off], sink, x, vx, vy, vz, c);
  st->x[off] = x; st->vx[off] = vx; st->vy[off] = vy; st->vz[off] = vz;
  return c;
}

}  // namespace bit1
