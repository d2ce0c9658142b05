// avm_forms.cuh — the step forms of the persistent transport kernel, as device functions.
//
// A warp iteration of transport_kernel advances its electrons in one of three forms.  Each form is a
// function here, called by the kernel AND by the parity hook avm_step_batch_form (avm.cu), so that the per-step 1e-12
// test runs the instruction sequences that earn the bench number — not a re-statement of them.  The two call sites differ
// only in the functors they pass: what happens to a pending real collision (kernel: collide + append the secondary to the
// run's arrays; hook: collide + record the child) and what happens to the result of a committed step (kernel: nothing;
// hook: record it).
#pragma once
#include "avm_device.cuh"

namespace avm {

// Per-thread tallies of the hot loop (warp-reduced at the end of the launch); null counts are derived (finalize_kernel).
struct Tally { uint32_t real = 0u, l0 = 0u, over = 0u, pen = 0u; double loss = 0.0; };

// Per-warp exchange area (shared memory).
struct WarpBuf {
  union {
    struct {                       // cooperative batches: draws of entry j = electron (j mod k') at its step (j div k')
      double dt[32];
      uint2 u2w[32];
      double ct[32], st[32], cphi[32], sphi[32];
    };
    struct {                       // time-parallel batches: base state of electron e, owner lane <-> group
      double2 bsv[16][4];          // (x, y), (z, t), (vx, vy), (vz, sum of dt up to the base)
      uint2 bnf[16];               // (n, finishing status)
      unsigned int bslot[16];
    };
  };
  unsigned long long id[32];
  unsigned int n[32];
  int last_tet[32];                // NEXT-2: the element each lane's electron was last found in (-1: none)
};
static_assert(sizeof(WarpBuf) == 2048, "WarpBuf");

// ---- full-warp form: ONE free flight of a lane's electron and its null/real decision ---------------------------------
// S3-S7 with this flight's pre-drawn (dt, u2w); the draws of the lane's NEXT flight are issued behind the threshold-record
// load.  On return: fin = finishing status (or 0), pend / pc = a real collision is pending (collision_step follows, in
// the warp's one collision phase), (dt, u2w) = the next flight's draws.
// BANDED (NEXT-1): dt carries -ln(u1); the flight's rate comes from the band of the electron's energy and
// the class of the field at its position (jcls = the class when the field is one uniform slab), a flight longer than the
// band's dtmax is cut there and ends in a null collision, and the decision compares u2 nu with the flight's own nu.
// SIGNAL (the extras variant; NEXT-4 when sig->out is set): the flight's induced charge -E_w(r) . (r' - r) goes to the bin
// of its start time.
template <int FK, bool HASB, bool TALLY, bool BANDED = false, bool SIGNAL = false>
__device__ __forceinline__ void fw_flight(const DevGas& g, const DevField& f, const PhiloxKeys& K,
                                          const ushort4* __restrict__ tab, const double2* __restrict__ logtab,
                                          const double t_max, const uint64_t id, uint32_t& n, double& x, double& y,
                                          double& z, double& t, double& vx, double& vy, double& vz, double& Ex, double& Ey,
                                          double& Ez, double& dt, uint2& u2w, int& fin, bool& pend, Pending& pc, Tally& tl,
                                          const int jcls = 0, const DevSignal* sig = nullptr, SigAcc* sacc = nullptr,
                                          int* tet_cache = nullptr) {
  bool over = false, cut = false;
  double dtf = dt, nu = g.nu_hat;
  uint32_t rho = 0u;
  if (BANDED) {
    const BandRate br = band_rate(g, vx * vx + vy * vy + vz * vz, FK == 1 ? jcls : accel_class(g, Ex, Ey, Ez));
    dtf = banded_dt(br, dt, cut);
    nu = br.nu; rho = br.rho;
  }
  double sx0 = 0.0, sy0 = 0.0, sz0 = 0.0, st0 = 0.0, swx = 0.0, swy = 0.0, swz = 0.0;
  if (SIGNAL && sig->out) { sx0 = x; sy0 = y; sz0 = z; st0 = t; weighting_at(*sig, x, y, z, swx, swy, swz); }
  const int b = advance<FK, HASB>(g, f, t_max, n, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, dtf, over, tet_cache);
  if (SIGNAL && sig->out) sig_add(*sig, *sacc, -(swx * (x - sx0) + swy * (y - sy0) + swz * (z - sz0)), st0);
  if (b < 0) { fin = -b; return; }
  AVM_CHECK(b < g.nb);
  const ushort4 rec = tab[b];
  const uint2 u2c = u2w;
  draw_flight<BANDED>(g, K, logtab, id, n, dt, u2w);  // next flight's draws: independent of the record load
  int r = decide_filter<BANDED>(rec, u2c, rho);       // branch-free; the rare outcomes below
  if (BANDED && cut) r = -1;
  if (r == -2 || r == 2) {
    pc.xr = to_unit(u2c.x, u2c.y) * nu;
    if (r == -2) r = decide_exact(g, b, pc.xr);
    if (r == 2) prefetch_row(g, b);
  }
  if (r >= 0) { pend = true; pc.lsel = r; pc.bin = b; }
  if (TALLY && over) ++tl.over;
}

// ---- time-parallel batch (one uniform slab; optional B) --------------------------------------------------------------
// In a constant field, consecutive null flights compose exactly: the state after flights dt_1 .. dt_j is the ballistic /
// helical flight of duration T_j = dt_1 + .. + dt_j from the base state.  The warp's k <= 16 electrons (lanes with `have`)
// get g = 32 / k' lanes each (k' = k rounded up to a power of two); lane s of electron e's group evaluates the END of step
// s (position, energy, bounds, bin, null/real decision with its own u2) in parallel; the first lane whose step is not null
// (real collision or termination) is the electron's next event, every step before it was null, and the draws after it
// stay valid for the next pass from the new base state.  The draws depend on (id, n) only, so this is the sequence of
// steps S0-S9 the oracle takes, evaluated out of order; T_j differs from the sequential sum by rounding only.
//
// collide(mask, pend, pc, have_d, d, fin) -> level: the collision phase for lanes with a pending real collision that is not the
//   pre-evaluated elastic one (acts on the caller's x .. vz, id, n, which are the same objects as the arguments here).
// commit(on, e, sidx, ev, bin, fin): called once per pass by every lane; on = this lane's step was taken in this pass,
//   its result is in x .. vz, n; ev = -1 null, level, or -2 ended before the decision.
// Returns the finishing status of the lane's own electron (0 = still active); its state is back in x .. vz, id, n, slot.
template <int FK, bool HASB, bool TALLY, bool SIGNAL, class Collide, class Commit>
__device__ __forceinline__ int tp_batch(const DevGas& g, const DevField& f, const PhiloxKeys& K,
                                        const ushort4* __restrict__ tab, const LevelPar* __restrict__ s_lv,
                                        const double2* __restrict__ s_logtab, WarpBuf* __restrict__ wb, const double t_max,
                                        const unsigned lane, const unsigned act, const bool have, double& x, double& y,
                                        double& z, double& t, double& vx, double& vy, double& vz, uint64_t& id, uint32_t& n,
                                        uint32_t& slot, Tally& tl, Collide&& collide, Commit&& commit,
                                        const DevSignal* sig = nullptr, SigAcc* sacc = nullptr) {
  static_assert(FK == 1, "time-parallel batches need a constant field: one uniform slab");
  const unsigned lt_mask = (1u << lane) - 1u;
  const int k = __popc(act);
  const int lg = 32 - __clz(k - 1);             // k' = 2^lg >= k  (k = 1: __clz(0) = 32)
  const int kp = 1 << lg, gl = 32 >> lg;        // gl = lanes (steps per batch) of one electron
  const int rank = __popc(act & lt_mask);
  const int e = (int)lane & (kp - 1), sidx = (int)lane >> lg;
  AVM_CHECK(k >= 1 && k <= 16 && (!have || rank < 16));
  if (have) {
    wb->bsv[rank][0] = make_double2(x, y); wb->bsv[rank][1] = make_double2(z, t);
    wb->bsv[rank][2] = make_double2(vx, vy); wb->bsv[rank][3] = make_double2(vz, 0.0);
    wb->id[rank] = id; wb->bnf[rank] = make_uint2(n, 0u); wb->bslot[rank] = slot;
  }
  __syncwarp();
  bool alive = e < k;
  double bx = 0, by = 0, bz = 0, bt = 0, bvx = 0, bvy = 0, bvz = 0;
  uint32_t bn = 0;
  if (alive) {
    const double2 q0 = wb->bsv[e][0], q1 = wb->bsv[e][1], q2 = wb->bsv[e][2], q3 = wb->bsv[e][3];
    bx = q0.x; by = q0.y; bz = q1.x; bt = q1.y; bvx = q2.x; bvy = q2.y; bvz = q3.x;
    id = wb->id[e]; bn = wb->bnf[e].x; slot = wb->bslot[e];
  }
  __syncwarp();
  // draws of step bn + sidx, and the inclusive sums P of dt over the group's steps 0 .. sidx
  double P = 0.0;
  uint2 u2j = make_uint2(0u, 0u);
  Deflection dj;
  dj.ct = 1.0; dj.st = 0.0; dj.cphi = 1.0; dj.sphi = 0.0;
  if (alive) {
    draw_flight(g, K, s_logtab, id, bn + (uint32_t)sidx, P, u2j);
    dj = deflection_draws(K, id, bn + (uint32_t)sidx);
  }
  for (int d = kp; d < 32; d <<= 1) {
    const double up = __shfl_up_sync(0xFFFFFFFFu, P, d);
    if ((int)lane >= d) P += up;
  }
  const unsigned gmask = (lg == 0 ? 0xFFFFFFFFu : lg == 1 ? 0x55555555u : lg == 2 ? 0x11111111u
                          : lg == 3 ? 0x01010101u : 0x00010001u) << e;
  const int last = ((gl - 1) << lg) | e;
  double Pb = 0.0;
  int cur = 0, gfin = 0;
#pragma unroll 1
  for (;;) {
    const bool valid = alive && sidx >= cur;
    x = bx; y = by; z = bz; t = bt; vx = bvx; vy = bvy; vz = bvz;
    n = bn + (uint32_t)(sidx - cur);
    bool over = false, ev = false, fast = false;
    int b = 0, r = -1;
    Pending pc;
    pc.lsel = 0; pc.bin = 0; pc.xr = 0.0;
    double fvx = 0.0, fvy = 0.0, fvz = 0.0, floss = 0.0;
    if (valid) {
      // One straight-line block, so that the independent chains overlap: the flight (S3-S4), the S5 predicate, the bin,
      // the threshold record and its 16-bit decision — and the ELASTIC collision this step would be, evaluated ahead
      // of the decision from the post-flight velocity (levels 0 / 1 are 97 % of the real collisions).  The rare
      // outcomes (termination, a band of the filter, another level or type) are decoded after the block.
      flight<FK, HASB>(f, 0.0, 0.0, 0.0, P - Pb, x, y, z, vx, vy, vz);
      const double s2 = vx * vx + vy * vy + vz * vz;
      t = t + (P - Pb);
      n = n + 1u;
      const bool ok = uniform_continues(f, t_max, n, x, y, z, t);
      b = energy_bin(g, s2, over);
      AVM_CHECK(b >= 0 && b < g.nb);
      r = decide_filter(tab[b], u2j);
      const LevelPar par = s_lv[r == 1 ? 1 : 0];
      fvx = vx; fvy = vy; fvz = vz;
      floss = elastic_collision(par.recoil, dj, s2, fvx, fvy, fvz);
      fast = ok & ((r == 0) | (r == 1)) & (par.type == AVM_ELASTIC) & (s2 >= 1e-280) & ((g.ext & 3) == 0);
      if (!ok) {
        b = uniform_exit_status(f, t_max, x, y, z, t);
      } else if (r == -2 || r == 2) {
        pc.xr = to_unit(u2j.x, u2j.y) * g.nu_hat;
        if (r == -2) r = decide_exact(g, b, pc.xr);
        if (r == 2) prefetch_row(g, b);
      }
      ev = b < 0 || r >= 0;
    }
    const unsigned evm = __ballot_sync(0xFFFFFFFFu, ev) & gmask;
    const int fl = __ffs(evm) - 1;                       // the group's first step that is not null, or -1
    const bool taken = valid && (fl < 0 || (int)lane <= fl);   // this lane's step is one the electron really takes
    if (SIGNAL && sig->out) {
      // the flight of step s starts where step s - 1 ended: the lane kp below (same electron), or the base state
      const double px = __shfl_up_sync(0xFFFFFFFFu, x, kp), py = __shfl_up_sync(0xFFFFFFFFu, y, kp);
      const double pz = __shfl_up_sync(0xFFFFFFFFu, z, kp), pt = __shfl_up_sync(0xFFFFFFFFu, t, kp);
      if (taken) {
        const bool first = sidx == cur;
        const double sx0 = first ? bx : px, sy0 = first ? by : py, sz0 = first ? bz : pz, st0 = first ? bt : pt;
        double swx, swy, swz;
        weighting_at(*sig, sx0, sy0, sz0, swx, swy, swz);
        sig_add(*sig, *sacc, -(swx * (x - sx0) + swy * (y - sy0) + swz * (z - sz0)), st0);
      }
    }
    // S6 counts an energy overflow only for a step that passes S5 (reaches the bin lookup)
    if (TALLY && taken && over && b >= 0) ++tl.over;
    int fin = 0, evc = -1;
    bool pend = false;
    if ((int)lane == fl) {
      if (b < 0) { fin = -b; evc = -2; }
      else if (fast) {                                   // the collision is already there
        vx = fvx; vy = fvy; vz = fvz;
        evc = r;
        if (TALLY) { ++tl.real; if (r == 0) ++tl.l0; tl.loss += floss; }
      } else { pend = true; pc.lsel = r; pc.bin = b; }
    }
    if (__any_sync(0xFFFFFFFFu, pend)) {
      const int lvl = collide(0xFFFFFFFFu, pend, pc, true, dj, fin);
      if (pend) evc = lvl;
    }
    commit(taken, e, sidx, evc, b, fin);
    // the group's new base: the state after its first event, or after its last step when all were null
    // (through the warp's exchange area: four 16-byte stores by one lane, four broadcast loads by its group)
    const int src = fl >= 0 ? fl : last;
    if (alive && (int)lane == src) {
      wb->bsv[e][0] = make_double2(x, y); wb->bsv[e][1] = make_double2(z, t);
      wb->bsv[e][2] = make_double2(vx, vy); wb->bsv[e][3] = make_double2(vz, P);
      wb->bnf[e] = make_uint2(n, (unsigned)fin);
    }
    __syncwarp();
    if (alive) {
      const double2 q0 = wb->bsv[e][0], q1 = wb->bsv[e][1], q2 = wb->bsv[e][2], q3 = wb->bsv[e][3];
      const uint2 nf = wb->bnf[e];
      bx = q0.x; by = q0.y; bz = q1.x; bt = q1.y; bvx = q2.x; bvy = q2.y; bvz = q3.x; Pb = q3.y;
      bn = nf.x; gfin = (int)nf.y;
      cur = (src >> lg) + 1;
      if (gfin != 0 || cur >= gl) alive = false;
    }
    __syncwarp();
    if (!__any_sync(0xFFFFFFFFu, alive)) break;
  }
  // the electrons go back to their owner lanes: the exchange area holds each group's final base state
  int fin = 0;
  if (have) {
    const double2 q0 = wb->bsv[rank][0], q1 = wb->bsv[rank][1], q2 = wb->bsv[rank][2], q3 = wb->bsv[rank][3];
    const uint2 nf = wb->bnf[rank];
    x = q0.x; y = q0.y; z = q1.x; t = q1.y; vx = q2.x; vy = q2.y; vz = q3.x;
    id = wb->id[rank]; n = nf.x; slot = wb->bslot[rank]; fin = (int)nf.y;
  }
  __syncwarp();
  return fin;
}

// ---- serial batch (any field) ----------------------------------------------------------------------------------------
// For a warp that holds k <= 16 electrons.  All 32 lanes first prepare the draws (Philox block 0 + logarithm, block 1 +
// deflection angles) of the next B = 32 / k' steps of the k electrons, lane j serving electron j mod k' at step j div k',
// through the warp's WarpBuf — the draws depend on (id, n) alone, so this is the same as drawing them in place, and draws
// of steps an electron does not reach are discarded.  Then every owner lane walks through ITS electron's B steps on its
// own: one straight-line block per step — flight (S3-S4), energy bin and threshold record (S6, S7), the S5 predicate with
// the field lookup at the new position (= S0 of the next step) — and, only when the step was not a null collision, one
// divergent side branch: the collision (with the append of a secondary) or the retirement of the electron.  There is no
// warp vote, ballot or shuffle on the path of a null step, and a lane never waits for another lane's electron to reach an
// event: lanes whose step was null wait only while the side branch of the others runs (reconvergence at its end), so a
// step costs the warp one flight plus, with probability 1 - (null fraction)^k, one collision.
//
// collide(mask, pend, pc, have_d, d, fin) -> level and retire(mask, fin) are called by the lanes with an event only, with
// mask = the lanes converged at the call (the warp-aggregated atomics inside them run over that mask); retire clears
// `have`.  commit(e, s, ev, bin, fin): step s of the batch of the warp's e-th electron is done, its result is in x .. vz, n.
// BANDED: as fw_flight — the exchange area holds -ln(u1) per step, the rate is looked up when the step starts.
template <int FK, bool HASB, bool TALLY, bool BANDED, bool SIGNAL, class Collide, class Retire, class Commit>
__device__ __forceinline__ void sb_batch(const DevGas& g, const DevField& f, const PhiloxKeys& K,
                                         const ushort4* __restrict__ tab, const double2* __restrict__ s_logtab,
                                         WarpBuf* __restrict__ wb, const double t_max, const unsigned lane, const unsigned act,
                                         bool& have, double& x, double& y, double& z, double& t, double& vx, double& vy,
                                         double& vz, double& Ex, double& Ey, double& Ez, const uint64_t& id, uint32_t& n,
                                         Tally& tl, Collide&& collide, Retire&& retire, Commit&& commit, const int jcls = 0,
                                         const DevSignal* sig = nullptr, SigAcc* sacc = nullptr, int* tet_cache = nullptr) {
  const unsigned lt_mask = (1u << lane) - 1u;
  const int k = __popc(act);
  const int lg = 32 - __clz(k - 1);             // k' = 2^lg >= k  (k = 1: __clz(0) = 32)
  const int kp = 1 << lg, nb_steps = 32 >> lg;
  const int rank = __popc(act & lt_mask);
  if (have) { wb->id[rank] = id; wb->n[rank] = n; }
  __syncwarp();
  {
    const int e = (int)lane & (kp - 1), s = (int)lane >> lg;
    if (e < k) {
      const uint64_t hid = wb->id[e];
      const uint32_t hn = wb->n[e] + (uint32_t)s;
      double ddt;
      uint2 du2;
      draw_flight<BANDED>(g, K, s_logtab, hid, hn, ddt, du2);
      const Deflection d = deflection_draws(K, hid, hn);
      wb->dt[lane] = ddt; wb->u2w[lane] = du2;
      wb->ct[lane] = d.ct; wb->st[lane] = d.st; wb->cphi[lane] = d.cphi; wb->sphi[lane] = d.sphi;
    }
  }
  __syncwarp();
  int s = 0;                                    // this lane's next step of the batch
#pragma unroll 1
  while (have && s < nb_steps) {
    const int idx = s * kp + rank;
    AVM_CHECK(idx >= 0 && idx < 32 && rank < 16);
    double dtj = wb->dt[idx];
    const uint2 u2 = wb->u2w[idx];
    bool cut = false;
    double nu = g.nu_hat;
    uint32_t rho = 0u;
    if (BANDED) {
      const BandRate br = band_rate(g, vx * vx + vy * vy + vz * vz, FK == 1 ? jcls : accel_class(g, Ex, Ey, Ez));
      dtj = banded_dt(br, dtj, cut);
      nu = br.nu; rho = br.rho;
    }
    double sx0 = 0.0, sy0 = 0.0, sz0 = 0.0, st0 = 0.0, swx = 0.0, swy = 0.0, swz = 0.0;
    if (SIGNAL && sig->out) { sx0 = x; sy0 = y; sz0 = z; st0 = t; weighting_at(*sig, x, y, z, swx, swy, swz); }
    const double s2 = advance_move<FK, HASB>(f, n, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, dtj);   // S3, S4
    if (SIGNAL && sig->out) sig_add(*sig, *sacc, -(swx * (x - sx0) + swy * (y - sy0) + swz * (z - sz0)), st0);
    bool over;
    const int b = energy_bin(g, s2, over);                                                     // S6 (counts only when S5 passes)
    AVM_CHECK(b >= 0 && b < g.nb);
    int r = decide_filter<BANDED>(tab[b], u2, rho);                                            // S7 and the head of S8
    if (BANDED && cut) r = -1;
    const int st = s5_status<FK>(f, t_max, n, x, y, z, t, Ex, Ey, Ez, tet_cache);              // S5; the field at r' = S0 of the next step
    if (TALLY && over && st == 0) ++tl.over;
    int ev = -1, fin = 0;
    if (st != 0 || r != -1) {                                                                  // not a plain null collision
      if (st < 0) { fin = -st; ev = -2; }
      else {
        Pending pc;
        pc.lsel = 0; pc.bin = b; pc.xr = 0.0;
        if (r == -2 || r == 2) {
          pc.xr = to_unit(u2.x, u2.y) * nu;
          if (r == -2) r = decide_exact(g, b, pc.xr);
          if (r == 2) prefetch_row(g, b);
        }
        if (r >= 0) {
          pc.lsel = r;
          Deflection dd;
          dd.ct = wb->ct[idx]; dd.st = wb->st[idx]; dd.cphi = wb->cphi[idx]; dd.sphi = wb->sphi[idx];
          ev = collide(__activemask(), true, pc, true, dd, fin);
        }
      }
      if (fin != 0) { commit(rank, s, ev, st < 0 ? -1 : b, fin); retire(__activemask(), fin); }
    }
    if (fin == 0) commit(rank, s, ev, b, 0);
    ++s;
  }
  __syncwarp();
}

}  // namespace avm
