// avm_transport.cuh — the persistent transport kernel (a-2 .. a-11) and the run's control block.
//
// Design: one persistent transport kernel.  Every electron owns a slot of the caller's SoA output arrays
// for the whole run (live state while active, endpoint afterwards), so "stack processing" moves no data: a
// finished electron frees its lane, a new one is appended by a warp-aggregated atomic on the packed counter (total << 32 |
// done), and idle lanes pick up work through tickets (lane holding ticket s runs the electron in slot s as soon as its
// status flag is published).  The run ends when done == total.  State stays in registers between collisions.
//
// The kernel template is instantiated in avm_transport_inst.cu, compiled once per (field kind, B) pair so that the
// translation units build in parallel (build.py); avm.cu picks an instantiation through pick_transport_inst<>.
#pragma once
#include "avm_forms.cuh"

namespace avm {

#ifndef AVM_THREADS
#define AVM_THREADS 512
#endif
#ifndef AVM_BACKOFF_MAX
#define AVM_BACKOFF_MAX 2000
#endif
#ifndef AVM_THREADS_WIDE
#define AVM_THREADS_WIDE 768
#endif
#ifndef AVM_FLIGHTS
#define AVM_FLIGHTS 2
#endif
#ifndef AVM_TICKET_PACK
#define AVM_TICKET_PACK 1
#endif
#ifndef AVM_COOP_MAX
#define AVM_COOP_MAX 8
#endif
// Two launch shapes of the transport kernel, one CTA per SM either way (the threshold table takes 160 KB of shared
// memory).  Latency shape: 512 threads, up to 128 registers, with the time-parallel batches — for runs whose electrons
// are fewer than the lanes for most of their duration.  Wide shape: 768 threads, 80 registers, cooperative batches only —
// chosen when the primaries alone outnumber the lanes of the latency shape (or by flag).
constexpr int kThreads = AVM_THREADS;
constexpr int kThreadsWide = AVM_THREADS_WIDE;
constexpr uint32_t kMaxIdlePolls = 1u << 23;
constexpr uint32_t kDefaultMaxIters = 1u << 22;   // working iterations per warp and launch (seconds of work): a safety net
constexpr int64_t kStageElectrons = 1 << 18;   // primaries staged per H2D chunk (16 MiB)
constexpr int kMaxGrid = 1024;                 // done flags, one 32-byte sector per CTA
constexpr size_t kDoneOffset = 4096;
constexpr size_t kCtlBytes = kDoneOffset + (size_t)kMaxGrid * 32;
constexpr size_t kMaxDynSmem = 227 * 1024 - 6144;   // static shared memory (level parameters, logarithm table: 5.4 KB) comes on top

struct RunArrays {
  uint32_t cap;
  uint64_t* id;
  uint32_t* aval;
  int32_t* status;
  uint32_t* nsteps;
  double* birth;   // [5][cap] or null
  double* end;     // [8][cap]
};

struct RunCtl {
  unsigned long long counters;   // (electrons created << 32) | electrons finished; spawn / retire atomics only
  unsigned char pad0[120];
  unsigned int q_head;           // tickets handed out beyond the static ones (own 128-byte line)
  unsigned int dropped;          // children that did not fit in `capacity`
  unsigned char pad1[120];
  unsigned long long n_real, n_overflow, n_penning;
  unsigned long long n_steps;    // sum over electrons of their collision index n (finalize_kernel)
  unsigned long long n_term;     // electrons whose last step ended before the null/real decision (status 1-4, 6, 7)
  unsigned long long level[AVM_MAX_LEVELS];
  double sum_loss;
  double sum_d[4];               // sum over electrons of (end - birth): dx, dy, dz, dt
};
static_assert(sizeof(RunCtl) <= kDoneOffset, "ctl block");

__device__ __forceinline__ int ld_relaxed_s32(const int* p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// Acquire load: pairs with st_release_s32 of the producer, so that the slot's payload, read after it, is the published
// one under the PTX memory model (not only by in-order issue behind the branch).  Costs one CCTL.IVALL: used once per
// electron pick-up, never for polling.
__device__ __forceinline__ int ld_acquire_s32(const int* p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
// Release store: earlier writes of this thread are visible at gpu scope before the flag is.  Unlike __threadfence()
// this does not invalidate the SM's L1 (no CCTL.IVALL), which the gas-table and field-map loads live in.
__device__ __forceinline__ void st_release_s32(int* p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void idle_wait(uint32_t ns) {
  unsigned long long t0, t1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
  do {
    __nanosleep(ns);
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
  } while (t1 - t0 < (unsigned long long)ns);
}

// ---- persistent transport kernel -------------------------------------------------------------------------
// One warp iteration advances the warp's k electrons (lanes with `have`) in one of three forms:
//  * k <= kCoopMax, one uniform slab, latency shape (TPB) — time-parallel batch: consecutive null flights in a constant
//    field compose exactly, so the 32 / k' lanes of an electron (k' = k rounded up to a power of two) evaluate its next
//    32 / k' steps at once from pre-drawn flight times; the first step that is not null is the electron's event.
//  * k <= kCoopMax otherwise (grid maps, wide shape) — cooperative batch: all 32 lanes first prepare the draws (Philox
//    block 0 + logarithm, block 1 + deflection angles) of the next B = 32 / k' steps of the k electrons, lane j serving
//    electron j mod k' at step j div k', through the warp's WarpBuf; then the owners take up to B steps whose dependent
//    chain is only flight -> field -> energy -> bin -> threshold record -> branch.
//    In both, the draws depend on (id, n) alone, so the result is the same as drawing them in place; draws of steps an
//    electron does not reach are discarded.
//  * k > kCoopMax — full warp: up to kFlights free flights per lane (a lane stops flying when it draws a real
//    collision), the draws of a lane's next flight issued behind its threshold-record load, then ONE collision phase.
// Then the rare warp-uniform branches: append secondaries, retire finished electrons, refill idle lanes.
constexpr int kFlights = AVM_FLIGHTS;
constexpr int kCoopMax = AVM_COOP_MAX;

#ifndef AVM_SB_UNIFORM
#define AVM_SB_UNIFORM 0     // 1: serial batches instead of time-parallel ones in one uniform slab without B
#endif
// SIGNAL = the "extras" variant: NEXT-3 (collision extensions of the gas, DevGas.ext) and NEXT-4 (induced signal, when
// sig.out is set) are compiled in and selected at run time; the base variant has neither, and its register budget.
template <int FK, bool HASB, bool TALLY, bool SMEMTAB, int THREADS, bool TPB, bool BANDED, bool SIGNAL>
__global__ void __launch_bounds__(THREADS, 1)
transport_kernel(const __grid_constant__ DevGas g, const __grid_constant__ DevField f, const RunArrays a,
                 RunCtl* __restrict__ ctl, const __grid_constant__ PhiloxKeys K, const double t_max,
                 const uint32_t max_iters, const uint32_t n_static_tickets, const __grid_constant__ DevSignal sig) {
  extern __shared__ __align__(16) unsigned char s_dyn[];
  __shared__ LevelPar s_lv[AVM_MAX_LEVELS];
  __shared__ double2 s_logtab[128];
  __shared__ unsigned int s_hist[AVM_MAX_LEVELS];
  stage_levels(g, s_lv);
  for (int l = threadIdx.x; l < AVM_MAX_LEVELS; l += blockDim.x) s_hist[l] = 0u;
  for (int i = threadIdx.x; i < 128; i += blockDim.x)
    s_logtab[i] = make_double2(__longlong_as_double((long long)kLogTab[i].rc), __longlong_as_double((long long)kLogTab[i].L));
  const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const ushort4* tab = g.tab;
  // banded rates (NEXT-1): in one uniform slab the acceleration class is a constant of the run
  const int jcls = (BANDED && FK == 1) ? accel_class(g, f.slab[0].E[0], f.slab[0].E[1], f.slab[0].E[2]) : 0;
  size_t dyn_off = 0;
  if (SMEMTAB) {                                   // threshold table: 8 bytes per bin, resident in shared memory
    uint2* dst = reinterpret_cast<uint2*>(s_dyn);
    const uint2* src = reinterpret_cast<const uint2*>(g.tab);
    for (int b = threadIdx.x; b < g.nb; b += blockDim.x) dst[b] = __ldg(src + b);
    tab = reinterpret_cast<const ushort4*>(s_dyn);
    dyn_off = ((size_t)g.nb * sizeof(ushort4) + 15) & ~(size_t)15;
  }
  WarpBuf* const wb = reinterpret_cast<WarpBuf*>(s_dyn + dyn_off) + warp;
  int* const tet_cache = FK == 0 ? &wb->last_tet[lane] : nullptr;   // NEXT-2: only slab stacks can hold a tetrahedral map
  if (FK == 0) *tet_cache = -1;
  int* const done = reinterpret_cast<int*>(reinterpret_cast<unsigned char*>(ctl) + kDoneOffset) + 8 * blockIdx.x;
  __syncthreads();

  const uint32_t cap = a.cap;
  const size_t ld = cap;
  // static tickets, CTA-major then warp then lane: the first electrons go one per warp, spread over all SMs (packing them
  // into one warp per scheduler instead was measured slower on the map configs: DESIGN.md §7)
  constexpr int kWarpsPerCta = THREADS / 32;
  constexpr uint32_t kPack = AVM_TICKET_PACK;
  uint32_t ticket = (((lane / kPack) * kWarpsPerCta + warp) * kPack + lane % kPack) * gridDim.x + blockIdx.x;
  bool have = false, dvalid = false;
  double x = 0, y = 0, z = 0, t = 0, vx = 0, vy = 0, vz = 0, Ex = 0, Ey = 0, Ez = 0, dt = 0;
  uint2 u2w = make_uint2(0u, 0u);
  uint64_t id = 0;
  uint32_t n = 0, slot = 0;
  Tally tl;                                       // tallies kept per thread; null counts are derived (finalize_kernel)
  SigAcc sacc;                                    // NEXT-4: this thread's pending contribution to one time bin of the signal
  uint32_t backoff = 250u;
  const unsigned lt_mask = (1u << lane) - 1u;

  // idle lanes poll their own ticket: pick the electron up when its slot is published (a-10)
  auto refill = [&]() {
    if (!have) {
#pragma unroll 1
      for (int tries = 0; tries < 2 && ticket < cap; ++tries) {
        int st = ld_relaxed_s32(a.status + ticket);  // polling probe
        if (st == 0) st = ld_acquire_s32(a.status + ticket);   // consumed: order the payload loads after the flag
        if (st == 0) {                              // published and unfinished: this lane runs it
          slot = ticket;
          AVM_CHECK(slot < cap);
          x = __ldcg(a.end + slot); y = __ldcg(a.end + ld + slot); z = __ldcg(a.end + 2 * ld + slot);
          t = __ldcg(a.end + 3 * ld + slot);
          const double e = __ldcg(a.end + 4 * ld + slot);
          const double sp = kC2 * sqrt(e);
          vx = sp * __ldcg(a.end + 5 * ld + slot); vy = sp * __ldcg(a.end + 6 * ld + slot);
          vz = sp * __ldcg(a.end + 7 * ld + slot);
          id = __ldcg(a.id + slot);
          n = __ldcg(a.nsteps + slot);
          double m;
          if (FK == 0) *tet_cache = -1;
          field_at<FK>(f, x, y, z, Ex, Ey, Ez, m, tet_cache);   // S0 of its first step (in-domain by construction)
          have = true; dvalid = false;
          break;
        }
        if (st < 0) break;                          // not created yet: keep the ticket
        ticket = n_static_tickets + atomicAdd(&ctl->q_head, 1u);   // finished in an earlier launch: next ticket
      }
    }
  };
  // one collision phase for the lanes with a pending real collision, then append their secondaries (a-8, a-9)
  auto collide_and_append = [&](const unsigned mask, bool pend, const Pending& pc, bool have_d, const Deflection& dd, int& fin) -> int {
    bool spawn = false;
    Child ch;
    ch.e = 0.0; ch.u6 = 0.5; ch.u7 = 0.0;
    int l = -1;
    if (pend) {
      double loss;
      int st;
      l = collision_step<SIGNAL>(g, s_lv, K, id, n, pc, have_d, dd, vx, vy, vz, st, spawn, ch, loss);
      if (st) fin = st;
      if (TALLY) {
        ++tl.real;
        if (l == 0) ++tl.l0;
        else if (l > 1) atomicAdd(&s_hist[l], 1u);
        tl.loss += loss;
        if (SIGNAL && spawn && s_lv[l].type == AVM_EXCITATION) ++tl.pen;       // X2: a Penning transfer (extras variant only)
      }
    }
    const unsigned sm = __ballot_sync(mask, spawn);
    if (sm) {                                       // one atomic per warp (per group of converged lanes)
      const int leader = __ffs(sm) - 1;
      unsigned long long old = 0ull;
      if ((int)lane == leader) old = atomicAdd(&ctl->counters, (unsigned long long)__popc(sm) << 32);
      old = __shfl_sync(mask, old, leader);
      if (spawn) {
        const uint64_t cs = (old >> 32) + (uint64_t)__popc(sm & lt_mask);
        if (cs < (uint64_t)cap) {
          const uint32_t c = (uint32_t)cs;
          AVM_CHECK(c < cap && slot < cap && __ldcg(a.status + c) == -1);
          double ckx, cky, ckz;
          child_direction(ch.u6, ch.u7, ckx, cky, ckz);
          __stcg(a.end + c, x); __stcg(a.end + ld + c, y); __stcg(a.end + 2 * ld + c, z); __stcg(a.end + 3 * ld + c, t);
          __stcg(a.end + 4 * ld + c, ch.e);
          __stcg(a.end + 5 * ld + c, ckx); __stcg(a.end + 6 * ld + c, cky); __stcg(a.end + 7 * ld + c, ckz);
          __stcg(a.id + c, child_id_of(K, id, n - 1u));
          __stcg(a.aval + c, __ldcg(a.aval + slot));
          __stcg(a.nsteps + c, 0u);
          if (a.birth) {
            __stcg(a.birth + c, x); __stcg(a.birth + ld + c, y); __stcg(a.birth + 2 * ld + c, z);
            __stcg(a.birth + 3 * ld + c, t); __stcg(a.birth + 4 * ld + c, ch.e);
          }
          st_release_s32(a.status + c, 0);          // publish
        } else {                                    // no room: drop the child, count it as created and finished
          atomicAdd(&ctl->dropped, 1u);
          atomicAdd(&ctl->counters, 1ull);
        }
      }
    }
    return l;
  };
  // retire finished electrons: endpoint write, one atomic per warp for `finished`, one for new tickets; the lane that
  // finishes the last electron raises every CTA's done flag (a-11)
  auto retire = [&](const unsigned mask, int fin) {
    const unsigned fm = __ballot_sync(mask, fin != 0);
    if (fm) {
      const int leader = __ffs(fm) - 1;
      unsigned int base = 0u;
      if ((int)lane == leader) base = atomicAdd(&ctl->q_head, (unsigned int)__popc(fm));
      base = __shfl_sync(mask, base, leader);
      if (fin != 0) {
        AVM_CHECK(slot < cap && have && a.status[slot] == 0);
        const double s2 = vx * vx + vy * vy + vz * vz;
        double kx = 0.0, ky = 0.0, kz = 1.0;
        if (s2 > 0.0) { const double inv = rsqrt(s2); kx = vx * inv; ky = vy * inv; kz = vz * inv; }
        a.end[slot] = x; a.end[ld + slot] = y; a.end[2 * ld + slot] = z; a.end[3 * ld + slot] = t;
        a.end[4 * ld + slot] = fmax(s2 * kInvC2Sq, kEpsFloor);
        a.end[5 * ld + slot] = kx; a.end[6 * ld + slot] = ky; a.end[7 * ld + slot] = kz;
        a.nsteps[slot] = n;
        a.status[slot] = fin;
        have = false;
        ticket = n_static_tickets + base + (uint32_t)__popc(fm & lt_mask);
      }
      if ((int)lane == leader) {
        const unsigned long long add = (unsigned long long)__popc(fm);
        const unsigned long long now = atomicAdd(&ctl->counters, add) + add;
        if ((uint32_t)(now >> 32) == (uint32_t)now) {          // created == finished: nothing can be created any more
          int* d0 = reinterpret_cast<int*>(reinterpret_cast<unsigned char*>(ctl) + kDoneOffset);
          for (unsigned b = 0; b < gridDim.x; ++b) *(volatile int*)(d0 + 8 * b) = 1;
        }
      }
    }
  };

  // `it` counts the iterations in which the warp advanced electrons; idle polling does not use up the guard (an idle
  // warp that left early would strand the electrons later published to its tickets until the next launch).  The warp
  // whose guard expires raises the stop flag (done = 2) of every CTA: idle warps leave, working warps park their
  // electrons at their next check, and the host relaunches.
  uint32_t it = 0, idle_polls = 0;
  bool stopped = false;
  while (it < max_iters) {
    unsigned act = __ballot_sync(0xFFFFFFFFu, have);
    // ---- probe the warp's lowest pending ticket (one sector per warp); consumed after the iteration's work ----
    uint32_t tmin = 0xFFFFFFFFu;
    int probe = -1;
    if (act != 0xFFFFFFFFu) {
      tmin = __reduce_min_sync(0xFFFFFFFFu, have ? 0xFFFFFFFFu : ticket);
      if (tmin < cap) probe = ld_relaxed_s32(a.status + tmin);
    }
    if (act == 0u) {                                // whole warp idle
      if (probe == -1) {                            // nothing to pick up: check for the end, back off
        if (ld_relaxed_s32(done) != 0) { stopped = true; break; }
        if (++idle_polls >= kMaxIdlePolls) { it = max_iters; break; }   // safety net: ~15 s without work ends the launch
        idle_wait(backoff);
        backoff = min(backoff * 2u, (uint32_t)AVM_BACKOFF_MAX);
        continue;
      }
      refill();
      backoff = 250u;
      idle_polls = 0;
      act = __ballot_sync(0xFFFFFFFFu, have);
      if (act == 0u) continue;
      probe = -1;
    }
    ++it;
    if ((it & 15u) == 0u && ld_relaxed_s32(done) == 2) { stopped = true; break; }
    const int k = __popc(act);

    if (TPB && !BANDED && FK == 1 && (HASB || !AVM_SB_UNIFORM) && k <= kCoopMax) {
      // ---- time-parallel batch (uniform E, optional B): g = 32 / k' lanes per electron (avm_forms.cuh) ----
      if constexpr (FK == 1) {
        const int fin = tp_batch<FK, HASB, TALLY, SIGNAL>(g, f, K, tab, s_lv, s_logtab, wb, t_max, lane, act, have, x, y, z, t, vx, vy, vz,
                                                          id, n, slot, tl, collide_and_append, [](bool, int, int, int, int, int) {}, &sig, &sacc);
        dvalid = false;
        retire(0xFFFFFFFFu, fin);
      }
    } else if (k <= kCoopMax) {
      // ---- serial batch: cooperative draws, then every owner lane walks its electron's steps alone (avm_forms.cuh) ----
      sb_batch<FK, HASB, TALLY, BANDED, SIGNAL>(g, f, K, tab, s_logtab, wb, t_max, lane, act, have, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, id, n, tl,
                                                collide_and_append, retire, [](int, int, int, int, int) {}, jcls, &sig, &sacc, tet_cache);
      dvalid = false;
    } else {
      // ---- full warp ----
      if (have && !dvalid) { draw_flight<BANDED>(g, K, s_logtab, id, n, dt, u2w); dvalid = true; }
      int fin = 0;
      bool pend = false;
      Pending pc;
      pc.lsel = 0; pc.bin = 0; pc.xr = 0.0;
#pragma unroll
      for (int fl = 0; fl < kFlights; ++fl) {
        if (have && !pend && fin == 0)
          fw_flight<FK, HASB, TALLY, BANDED, SIGNAL>(g, f, K, tab, s_logtab, t_max, id, n, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, dt, u2w, fin,
                                                     pend, pc, tl, jcls, &sig, &sacc, tet_cache);
      }
      Deflection dd;
      dd.ct = 1.0; dd.st = 0.0; dd.cphi = 1.0; dd.sphi = 0.0;
      collide_and_append(0xFFFFFFFFu, pend, pc, false, dd, fin);
      retire(0xFFFFFFFFu, fin);
    }
    // ---- refill idle lanes when the probed ticket has been published ----
    if (probe != -1) refill();
  }

  if (it >= max_iters && !stopped) {                // guard expired here: stop the launch everywhere
    int* d0 = reinterpret_cast<int*>(reinterpret_cast<unsigned char*>(ctl) + kDoneOffset);
    for (unsigned b = lane; b < gridDim.x; b += 32u)
      if (ld_relaxed_s32(d0 + 8 * b) == 0) *(volatile int*)(d0 + 8 * b) = 2;
  }
  // guard expired or launch stopped with the electron still active: park its state in its slot (status stays 0);
  // the next launch picks it up through the tickets.
  if (have) {
    const double s2 = vx * vx + vy * vy + vz * vz;
    double kx = 0.0, ky = 0.0, kz = 1.0;
    if (s2 > 0.0) { const double inv = rsqrt(s2); kx = vx * inv; ky = vy * inv; kz = vz * inv; }
    a.end[slot] = x; a.end[ld + slot] = y; a.end[2 * ld + slot] = z; a.end[3 * ld + slot] = t;
    a.end[4 * ld + slot] = fmax(s2 * kInvC2Sq, kEpsFloor);
    a.end[5 * ld + slot] = kx; a.end[6 * ld + slot] = ky; a.end[7 * ld + slot] = kz;
    a.nsteps[slot] = n;
  }
  if (SIGNAL && sig.out) sig_flush(sig, sacc);
  if (TALLY) {
    // warp reduce the per-thread counters, one atomic per warp; rare-level histogram per CTA
    unsigned long long v0 = tl.real, v1 = tl.l0, v3 = tl.over, v5 = tl.pen;
    double v4 = tl.loss;
#pragma unroll
    for (int o2 = 16; o2 > 0; o2 >>= 1) {
      v0 += __shfl_down_sync(0xFFFFFFFFu, v0, o2); v1 += __shfl_down_sync(0xFFFFFFFFu, v1, o2);
      v3 += __shfl_down_sync(0xFFFFFFFFu, v3, o2); v4 += __shfl_down_sync(0xFFFFFFFFu, v4, o2);
      v5 += __shfl_down_sync(0xFFFFFFFFu, v5, o2);
    }
    if (lane == 0u) {
      if (v0) atomicAdd(&ctl->n_real, v0);
      if (v1) atomicAdd(&ctl->level[0], v1);
      if (v3) atomicAdd(&ctl->n_overflow, v3);
      if (v5) atomicAdd(&ctl->n_penning, v5);
      if (v4 != 0.0) atomicAdd(&ctl->sum_loss, v4);
    }
    __syncthreads();
    for (int l = 2 + threadIdx.x; l < g.L; l += blockDim.x)
      if (s_hist[l]) atomicAdd(&ctl->level[l], (unsigned long long)s_hist[l]);
  }
}

typedef void (*TransportFn)(const DevGas, const DevField, const RunArrays, RunCtl*, const PhiloxKeys, const double,
                            const uint32_t, const uint32_t, const DevSignal);
// Defined (explicit specialisation) in avm_transport_inst.cu, one translation unit per (FK, B).  extras = the variant with
// NEXT-3 / NEXT-4 compiled in; with the threshold table outside shared memory (more than ~24000 energy bins) it is not
// instantiated: nullptr.
template <int FK, bool B>
TransportFn pick_transport_inst(bool smemtab, bool wide, bool banded, bool extras);

}  // namespace avm
