// avm.cu — kernels and the C ABI of libavm (include/avm.h) for sm_100a.
//
// Design: one persistent transport kernel.  Every electron owns a slot of the caller's SoA
// output arrays for the whole run (live state while active, endpoint afterwards), so "stack processing"
// moves no data: a finished electron frees its lane, a new one is appended by a
// warp-aggregated atomic on the packed counter (total << 32 | done), and idle lanes pick up work through
// tickets (lane holding ticket s runs the electron in slot s as soon as its status flag is published).
// The run ends when done == total.  State stays in registers between collisions.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "avm_transport.cuh"

using namespace avm;

namespace {

thread_local std::string g_err;

int32_t fail(int32_t code, const std::string& msg) { g_err = msg; return code; }
#define AVM_CUDA(call)                                                                                  \
  do {                                                                                                  \
    cudaError_t e_ = (call);                                                                            \
    if (e_ != cudaSuccess) return fail(AVM_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

// ---- primary injection (a-1) -----------------------------------------------------------------------------
template <int FK>
__global__ void inject_kernel(const __grid_constant__ DevField f, const RunArrays a, RunCtl* ctl,
                              const double* __restrict__ prim, const uint32_t p0, const uint32_t count,
                              const uint64_t id_offset, const double t_max) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long add = 0ull;
  if (i < count) {
    const uint32_t p = p0 + i;
    const double* q = prim + (size_t)i * 8;
    const double x = q[0], y = q[1], z = q[2], t = q[3];
    const double e = fmax(q[4], kEpsFloor);
    double kx = q[5], ky = q[6], kz = q[7];
    const double nk = sqrt(kx * kx + ky * ky + kz * kz);
    if (!(nk > 0.0)) { kx = 0.0; ky = 0.0; kz = 1.0; } else { kx /= nk; ky /= nk; kz /= nk; }
    double Ex, Ey, Ez, m = 1.0;
    const int si = field_at<FK>(f, x, y, z, Ex, Ey, Ez, m);
    int st = 0;
    if (si < 0) st = -si;
    else if (m < 0.5) st = AVM_MATERIAL;
    else if (t > t_max) st = AVM_TIME_LIMIT;
    const size_t ld = a.cap;
    a.end[p] = x; a.end[ld + p] = y; a.end[2 * ld + p] = z; a.end[3 * ld + p] = t; a.end[4 * ld + p] = e;
    a.end[5 * ld + p] = kx; a.end[6 * ld + p] = ky; a.end[7 * ld + p] = kz;
    if (a.birth) {
      a.birth[p] = x; a.birth[ld + p] = y; a.birth[2 * ld + p] = z; a.birth[3 * ld + p] = t; a.birth[4 * ld + p] = e;
    }
    a.id[p] = id_offset + (uint64_t)p;
    a.aval[p] = p;
    a.nsteps[p] = 0u;
    a.status[p] = st;
    add = (1ull << 32) | (st != 0 ? 1ull : 0ull);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) add += __shfl_down_sync(0xFFFFFFFFu, add, o);
  if ((threadIdx.x & 31u) == 0u && add) atomicAdd(&ctl->counters, add);
}

// ---- tallies derived from the endpoints (a-12) -----------------------------------------------------------
// Per-avalanche counts, flight sums (sum over electrons of end - birth) and the step bookkeeping the hot loop does
// not count: steps = sum of n; every step is null, real or the electron's last one (ended before the decision), so
// null = steps - real - #{electrons finished by status 1-4, 6, 7 after at least one step}.
__global__ void finalize_kernel(const RunArrays a, RunCtl* ctl, const uint32_t n, unsigned long long* per_aval,
                                const uint32_t n_prim, const bool want_sums) {
  double d[4] = {0.0, 0.0, 0.0, 0.0};
  unsigned long long steps = 0ull, term = 0ull;
  const size_t ld = a.cap;
  for (uint32_t s = blockIdx.x * blockDim.x + threadIdx.x; s < n; s += gridDim.x * blockDim.x) {
    const int st = a.status[s];
    const uint32_t ns = a.nsteps[s];
    steps += ns;
    if (ns > 0u && st != AVM_ATTACHED && st != AVM_ACTIVE) ++term;
    if (per_aval) {
      const uint32_t av = a.aval[s];
      if (av < n_prim) {
        atomicAdd(per_aval + 3 * (size_t)av, 1ull);
        if (st == AVM_ATTACHED) atomicAdd(per_aval + 3 * (size_t)av + 2, 1ull);
      }
    }
    if (want_sums) {
#pragma unroll
      for (int c = 0; c < 4; ++c) d[c] += a.end[c * ld + s] - a.birth[c * ld + s];
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    steps += __shfl_down_sync(0xFFFFFFFFu, steps, o);
    term += __shfl_down_sync(0xFFFFFFFFu, term, o);
  }
  if ((threadIdx.x & 31u) == 0u) {
    if (steps) atomicAdd(&ctl->n_steps, steps);
    if (term) atomicAdd(&ctl->n_term, term);
  }
  if (want_sums) {
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      double v = d[c];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xFFFFFFFFu, v, o);
      if ((threadIdx.x & 31u) == 0u && v != 0.0) atomicAdd(&ctl->sum_d[c], v);
    }
  }
}

__global__ void publish_kernel(const RunCtl* ctl, const int L, unsigned long long* per_aval, const uint32_t n_prim,
                               unsigned long long* tallies_u64, double* tallies_f64) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (per_aval && i < n_prim) {
    const unsigned long long e = per_aval[3 * (size_t)i];
    per_aval[3 * (size_t)i + 1] = e > 0ull ? e - 1ull : 0ull;     // ions = ionisations = endpoints - 1 (C11)
  }
  if (i == 0u) {
    if (tallies_u64) {
      unsigned long long others = ctl->level[0];
      for (int l = 2; l < L; ++l) others += ctl->level[l];
      for (int l = 0; l < L; ++l) tallies_u64[l] = ctl->level[l];
      if (L > 1) tallies_u64[1] = ctl->n_real - others;           // level 1 is the complement (not counted in the loop)
      tallies_u64[L] = ctl->n_steps - ctl->n_real - ctl->n_term;  // null collisions
      tallies_u64[L + 1] = ctl->n_real;
      tallies_u64[L + 2] = ctl->n_overflow; tallies_u64[L + 3] = ctl->n_steps;
      tallies_u64[L + 4] = ctl->n_penning;
    }
    if (tallies_f64) {
      for (int c = 0; c < 4; ++c) tallies_f64[c] = ctl->sum_d[c];
      tallies_f64[4] = ctl->sum_loss;
    }
  }
}

// ---- parity hooks ----------------------------------------------------------------------------------------
// FORM 0: the general sequence draw_flight -> advance -> decide -> collision_step.  FORM 1: the full-warp form of the
// transport kernel — fw_flight (avm_forms.cuh: advance, decide_filter / decide_exact, the next flight's draws hoisted
// behind the record load) and the collision phase with the deflection drawn there.
template <int FK, bool HASB, int FORM, bool BANDED>
__global__ void step_batch_kernel(const __grid_constant__ DevGas g, const __grid_constant__ DevField f,
                                  const uint64_t seed, const double t_max, const int64_t n,
                                  const double* __restrict__ in, const uint64_t* __restrict__ ids,
                                  const uint32_t* __restrict__ n_idx, double* __restrict__ out,
                                  int32_t* __restrict__ event, int32_t* __restrict__ status, int32_t* __restrict__ bin,
                                  double* __restrict__ child, uint64_t* __restrict__ child_id) {
  __shared__ LevelPar s_lv[AVM_MAX_LEVELS];
  __shared__ double2 s_logtab[128];
  stage_levels(g, s_lv);
  for (int j = threadIdx.x; j < 128; j += blockDim.x)
    s_logtab[j] = make_double2(__longlong_as_double((long long)kLogTab[j].rc), __longlong_as_double((long long)kLogTab[j].L));
  __syncthreads();
  const PhiloxKeys K = philox_keys(seed);
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double x = in[i], y = in[n + i], z = in[2 * n + i], t = in[3 * n + i];
  const double e = in[4 * n + i];
  double kx = in[5 * n + i], ky = in[6 * n + i], kz = in[7 * n + i];
  const uint64_t id = ids[i];
  uint32_t nn = n_idx[i];
  for (int c = 0; c < 8; ++c) child[c * n + i] = 0.0;
  child_id[i] = 0ull;
  double Ex, Ey, Ez, m;
  const int si = field_at<FK>(f, x, y, z, Ex, Ey, Ez, m);     // S0
  if (si < 0) {                                                     // caller error: reported as a status
    for (int c = 0; c < 8; ++c) out[c * n + i] = in[c * n + i];
    event[i] = -2; status[i] = -si; bin[i] = -1;
    return;
  }
  const double sp = kC2 * sqrt(e);
  double vx = sp * kx, vy = sp * ky, vz = sp * kz, dt;
  uint2 u2;
  draw_flight<BANDED>(g, K, s_logtab, id, nn, dt, u2);
  Pending pc;
  pc.lsel = 0; pc.bin = -1; pc.xr = 0.0;
  bool over = false, spawn = false;
  Child ch;
  ch.e = 0.0; ch.u6 = 0.5; ch.u7 = 0.0;
  int ev = -2, st = 0;
  Deflection dd;
  dd.ct = 1.0; dd.st = 0.0; dd.cphi = 1.0; dd.sphi = 0.0;
  if (FORM == 1) {
    bool pend = false;
    Tally tl;
    const int jcls = (BANDED && FK == 1) ? accel_class(g, f.slab[0].E[0], f.slab[0].E[1], f.slab[0].E[2]) : 0;
    fw_flight<FK, HASB, true, BANDED>(g, f, K, g.tab, s_logtab, t_max, id, nn, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, dt, u2, st, pend,
                                      pc, tl, jcls);
    over = tl.over != 0u;
    if (st == 0) {
      ev = -1;
      if (pend) {
        double loss;
        ev = collision_step(g, s_lv, K, id, nn, pc, false, dd, vx, vy, vz, st, spawn, ch, loss);
      } else {
        bool o2;
        pc.bin = energy_bin(g, vx * vx + vy * vy + vz * vz, o2);     // a null step leaves the velocity alone: its bin, for the report
      }
    }
  } else {
    const int b = advance<FK, HASB>(g, f, t_max, nn, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, dt, over);
    if (b < 0) st = -b;
    else {
      pc.bin = b;
      const int r = decide(g, __ldg(g.tab + b), b, u2, pc.xr);
      if (r < 0) ev = -1;
      else {
        double loss;
        pc.lsel = r;
        ev = collision_step(g, s_lv, K, id, nn, pc, false, dd, vx, vy, vz, st, spawn, ch, loss);
      }
    }
  }
  // state after the step in (energy, direction) form
  const double s2 = vx * vx + vy * vy + vz * vz;
  if (s2 > 0.0) { const double inv = rsqrt(s2); kx = vx * inv; ky = vy * inv; kz = vz * inv; }
  out[i] = x; out[n + i] = y; out[2 * n + i] = z; out[3 * n + i] = t; out[4 * n + i] = fmax(s2 * kInvC2Sq, kEpsFloor);
  out[5 * n + i] = kx; out[6 * n + i] = ky; out[7 * n + i] = kz;
  event[i] = ev; status[i] = st;
  bin[i] = pc.bin;
  if (spawn) {
    double ckx, cky, ckz;
    child_direction(ch.u6, ch.u7, ckx, cky, ckz);
    child[i] = x; child[n + i] = y; child[2 * n + i] = z; child[3 * n + i] = t; child[4 * n + i] = ch.e;
    child[5 * n + i] = ckx; child[6 * n + i] = cky; child[7 * n + i] = ckz;
    child_id[i] = child_id_of(K, id, nn - 1u);
  }
}

// FORMS 2 and 3: one batch per warp — a time-parallel batch (tp_batch) or a serial batch (sb_batch) of avm_forms.cuh — with
// k electrons per warp on scattered lanes.  Entry i * gl + s of the outputs = step s of electron i, gl = 32 / k' steps per
// batch; entries the batch does not reach (the electron finished earlier) keep what the caller put there.
template <int FK, bool HASB, int FORM, bool BANDED>
__global__ void __launch_bounds__(128)
step_form_batch_kernel(const __grid_constant__ DevGas g, const __grid_constant__ DevField f, const uint64_t seed,
                       const double t_max, const int64_t n, const int k, const double* __restrict__ in,
                       const uint64_t* __restrict__ ids, const uint32_t* __restrict__ n_idx, double* __restrict__ out,
                       int32_t* __restrict__ event, int32_t* __restrict__ status, int32_t* __restrict__ bin,
                       double* __restrict__ child, uint64_t* __restrict__ child_id) {
  __shared__ LevelPar s_lv[AVM_MAX_LEVELS];
  __shared__ double2 s_logtab[128];
  __shared__ WarpBuf s_wb[4];
  __shared__ long long s_gidx[4][16];
  stage_levels(g, s_lv);
  for (int j = threadIdx.x; j < 128; j += blockDim.x)
    s_logtab[j] = make_double2(__longlong_as_double((long long)kLogTab[j].rc), __longlong_as_double((long long)kLogTab[j].L));
  __syncthreads();
  const PhiloxKeys K = philox_keys(seed);
  const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const int64_t w = (int64_t)blockIdx.x * 4 + warp;
  int j = -1;
  for (int q = 0; q < k; ++q) if ((unsigned)((37 * q + 5) & 31) == lane) j = q;   // electron q of the warp sits on lane (37 q + 5) mod 32
  const int64_t i = w * k + j;
  bool have = j >= 0 && i < n;
  double x = 0, y = 0, z = 0, t = 0, vx = 0, vy = 0, vz = 0, Ex = 0, Ey = 0, Ez = 0;
  uint64_t id = 0;
  uint32_t nn = 0, slot = 0;
  if (have) {
    x = in[i]; y = in[n + i]; z = in[2 * n + i]; t = in[3 * n + i];
    const double sp = kC2 * sqrt(in[4 * n + i]);
    vx = sp * in[5 * n + i]; vy = sp * in[6 * n + i]; vz = sp * in[7 * n + i];
    id = ids[i]; nn = n_idx[i];
    double m;
    field_at<FK>(f, x, y, z, Ex, Ey, Ez, m);                                       // S0 of the first step (in-domain: caller's duty)
  }
  const unsigned act = __ballot_sync(0xFFFFFFFFu, have);
  if (act == 0u) return;
  const int lg = 32 - __clz(__popc(act) - 1), gl = 32 >> lg;
  const int64_t N = n * gl;
  const int rank = __popc(act & ((1u << lane) - 1u));
  if (have) s_gidx[warp][rank] = i;
  __syncwarp();
  Tally tl;
  // the output entry a lane is working on: tp_batch gives lane (e, sidx) one step; sb_batch gives the owner lane all steps
  int64_t o_cur = 0;
  auto collide = [&](const unsigned, bool pend, const Pending& pc, bool have_d, const Deflection& dd, int& fin) -> int {
    int l = -1;
    if (pend) {
      double loss;
      int st;
      bool spawn;
      Child ch;
      ch.e = 0.0; ch.u6 = 0.5; ch.u7 = 0.0;
      l = collision_step(g, s_lv, K, id, nn, pc, have_d, dd, vx, vy, vz, st, spawn, ch, loss);
      if (st) fin = st;
      if (spawn) {
        const int64_t o = FORM == 2 ? s_gidx[warp][lane & ((1u << lg) - 1u)] * gl + (lane >> lg) : o_cur;
        double ckx, cky, ckz;
        child_direction(ch.u6, ch.u7, ckx, cky, ckz);
        child[o] = x; child[N + o] = y; child[2 * N + o] = z; child[3 * N + o] = t; child[4 * N + o] = ch.e;
        child[5 * N + o] = ckx; child[6 * N + o] = cky; child[7 * N + o] = ckz;
        child_id[o] = child_id_of(K, id, nn - 1u);
      }
    }
    return l;
  };
  auto record = [&](int e, int sidx, int ev, int b, int fin) {
    const int64_t o = s_gidx[warp][e] * gl + sidx;
    const double s2 = vx * vx + vy * vy + vz * vz;
    double kx = 0.0, ky = 0.0, kz = 1.0;
    if (s2 > 0.0) { const double inv = rsqrt(s2); kx = vx * inv; ky = vy * inv; kz = vz * inv; }
    out[o] = x; out[N + o] = y; out[2 * N + o] = z; out[3 * N + o] = t; out[4 * N + o] = fmax(s2 * kInvC2Sq, kEpsFloor);
    out[5 * N + o] = kx; out[6 * N + o] = ky; out[7 * N + o] = kz;
    event[o] = ev; status[o] = fin; bin[o] = b < 0 ? -1 : b;
  };
  if constexpr (FORM == 2) {
    tp_batch<FK, HASB, true, false>(g, f, K, g.tab, s_lv, s_logtab, &s_wb[warp], t_max, lane, act, have, x, y, z, t, vx, vy, vz, id, nn,
                             slot, tl, collide, [&](bool on, int e, int sidx, int ev, int b, int fin) { if (on) record(e, sidx, ev, b, fin); });
  } else {
    // sb_batch calls commit AFTER a step; the child of a collision is recorded inside collide, before the commit of the
    // same step: o_cur is kept one step ahead (the owner lane's next output entry)
    o_cur = have ? i * gl : 0;
    const int jcls = (BANDED && FK == 1) ? accel_class(g, f.slab[0].E[0], f.slab[0].E[1], f.slab[0].E[2]) : 0;
    sb_batch<FK, HASB, true, BANDED, false>(g, f, K, g.tab, s_logtab, &s_wb[warp], t_max, lane, act, have, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, id,
                                     nn, tl, collide, [&](const unsigned, int fin) { if (fin != 0) have = false; },
                                     [&](int e, int sidx, int ev, int b, int fin) { record(e, sidx, ev, b, fin); o_cur = s_gidx[warp][e] * gl + sidx + 1; },
                                     jcls);
  }
}

// ---- NEXT-4: ion drift (W3-W4) ---------------------------------------------------------------------------
// One thread per possible ion: i < n = the positive ion left where electron i was born (none for the primaries), i >= n =
// the negative ion of electron i - n if it was attached.  Explicit midpoint along q mu E in steps of fixed length.
struct IonOpts { double mu_pos, mu_neg, step, t_max; int max_steps; };
template <bool SIGNAL>
__global__ void __launch_bounds__(256)
ion_drift_kernel(const __grid_constant__ DevField f, const __grid_constant__ DevSignal sig, const IonOpts io, const RunArrays a,
                 const uint32_t n, const uint32_t n_prim, double* __restrict__ ion_end, int32_t* __restrict__ ion_status,
                 uint32_t* __restrict__ ion_steps) {
  const size_t N = 2 * (size_t)n, ld = a.cap;
  SigAcc sacc;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (size_t)gridDim.x * blockDim.x) {
    const uint32_t s = i < n ? (uint32_t)i : (uint32_t)(i - n);
    const bool pos = i < n;
    int st = -1;
    uint32_t ns = 0u;
    double x = 0.0, y = 0.0, z = 0.0, t = 0.0;
    const int32_t est = a.status[s];                                         // <= 0: the slot holds no finished electron
    if (est > 0 && (pos ? s >= n_prim : est == AVM_ATTACHED)) {              // W3: which ions exist
      const double* src = pos ? a.birth : a.end;
      x = src[s]; y = src[ld + s]; z = src[2 * ld + s]; t = src[3 * ld + s];
      const double q = pos ? 1.0 : -1.0, qmu = q * (pos ? io.mu_pos : io.mu_neg);
      double Ex, Ey, Ez, m;
      int si = field_at<0>(f, x, y, z, Ex, Ey, Ez, m);
      st = si < 0 ? -si : (m < 0.5 ? AVM_MATERIAL : AVM_ACTIVE);
      while (st == AVM_ACTIVE) {
        if (ns >= (uint32_t)io.max_steps) { st = AVM_STEP_LIMIT; break; }
        const double k1x = qmu * Ex, k1y = qmu * Ey, k1z = qmu * Ez;
        const double n1 = sqrt(k1x * k1x + k1y * k1y + k1z * k1z);
        if (!(n1 > 0.0)) { st = AVM_STEP_LIMIT; break; }
        const double hh = 0.5 * io.step / n1;
        const double mx = x + hh * k1x, my = y + hh * k1y, mz = z + hh * k1z;
        double Emx, Emy, Emz, mm;
        if (field_at<0>(f, mx, my, mz, Emx, Emy, Emz, mm) < 0) { Emx = Ex; Emy = Ey; Emz = Ez; }   // midpoint outside: Euler step
        const double k2x = qmu * Emx, k2y = qmu * Emy, k2z = qmu * Emz;
        const double n2 = sqrt(k2x * k2x + k2y * k2y + k2z * k2z);
        if (!(n2 > 0.0)) { st = AVM_STEP_LIMIT; break; }
        const double h2 = io.step / n2;
        const double nx = x + h2 * k2x, ny = y + h2 * k2y, nz = z + h2 * k2z;
        if (SIGNAL) {
          double wx, wy, wz;
          weighting_at(sig, mx, my, mz, wx, wy, wz);
          sig_add(sig, sacc, q * (wx * (nx - x) + wy * (ny - y) + wz * (nz - z)), t);
        }
        x = nx; y = ny; z = nz;
        t = t + h2;
        ++ns;
        si = field_at<0>(f, x, y, z, Ex, Ey, Ez, m);
        if (si < 0) st = -si;
        else if (m < 0.5) st = AVM_MATERIAL;
        else if (t > io.t_max) st = AVM_TIME_LIMIT;
      }
    }
    ion_end[i] = x; ion_end[N + i] = y; ion_end[2 * N + i] = z; ion_end[3 * N + i] = t;
    ion_status[i] = st; ion_steps[i] = ns;
  }
  if (SIGNAL) sig_flush(sig, sacc);
}

// Widened copy of a grid map: node i's float4 (Ex, Ey, Ez, mask) -> four doubles, exactly (avm_slab.nodes_f64_dev).
__global__ void widen_map_kernel(const float4* __restrict__ in, double2* __restrict__ out, const size_t n_nodes) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_nodes; i += (size_t)gridDim.x * blockDim.x) {
    const float4 v = __ldg(in + i);
    out[2 * i] = make_double2((double)v.x, (double)v.y);
    out[2 * i + 1] = make_double2((double)v.z, (double)v.w);
  }
}

__global__ void field_eval_kernel(const __grid_constant__ DevField f, const int64_t n, const double* __restrict__ r,
                                  double* __restrict__ E, double* __restrict__ mask, int32_t* __restrict__ slab) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double ex = 0.0, ey = 0.0, ez = 0.0, m = 0.0;
  const int si = field_at<false>(f, r[i], r[n + i], r[2 * n + i], ex, ey, ez, m);
  E[i] = ex; E[n + i] = ey; E[2 * n + i] = ez; mask[i] = m; slab[i] = si < 0 ? -1 : si;
}

__global__ void philox_batch_kernel(const uint64_t seed, const int64_t n, const uint64_t* __restrict__ id,
                                    const uint32_t* __restrict__ n_idx, const uint32_t* __restrict__ block,
                                    uint32_t* __restrict__ words, double* __restrict__ u) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const U4 w = philox(philox_keys(seed), id[i], n_idx[i], block[i]);
  words[4 * i] = w.w0; words[4 * i + 1] = w.w1; words[4 * i + 2] = w.w2; words[4 * i + 3] = w.w3;
  u[2 * i] = to_unit(w.w0, w.w1); u[2 * i + 1] = to_unit(w.w2, w.w3);
}

// FP64 issue-rate probe: 8 independent DFMA chains per thread.
__global__ void __launch_bounds__(256) fp64_probe_kernel(const long long iters, double* sink) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3, a4 = a0 + 4e-3,
         a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.9999999, c = 1e-7;
  for (long long i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// Random-gather probes: the denominators of the map configs' roofline (SURVEY.md §7 stage 0, §8(d)).
// Every thread issues `iters` independent 32-byte loads (one sector, two 16-byte halves) at xorshift-random sector
// indices of the working set, bypassing L1 (ld.global.cg): the sustained random-sector rate of L2 (working set inside
// the 126 MB L2) or of HBM (working set far beyond it).
__global__ void __launch_bounds__(256) gather_probe_kernel(const uint4* __restrict__ buf, const unsigned long long n_sectors,
                                                          const long long iters, unsigned long long* sink) {
  unsigned long long s = 0x9E3779B97F4A7C15ull * ((unsigned long long)blockIdx.x * blockDim.x + threadIdx.x + 1ull);
  unsigned int acc = 0u;
  for (long long i = 0; i < iters; ++i) {
    s ^= s << 13; s ^= s >> 7; s ^= s << 17;
    const unsigned long long j = __umul64hi(s, n_sectors);          // uniform in [0, n_sectors)
    const uint4 a = __ldcg(buf + 2 * j), b = __ldcg(buf + 2 * j + 1);
    acc ^= a.x ^ a.w ^ b.y ^ b.z;
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}
// Shared-memory random 8-byte loads per second (the 160 KB threshold table's access pattern: one record per step).
__global__ void __launch_bounds__(512) smem_probe_kernel(const int n_entries, const long long iters, unsigned long long* sink) {
  extern __shared__ __align__(16) unsigned char s_probe[];
  unsigned long long* tab = reinterpret_cast<unsigned long long*>(s_probe);
  for (int i = threadIdx.x; i < n_entries; i += blockDim.x) tab[i] = 0x100000001ull * (unsigned)i;
  __syncthreads();
  unsigned int s = 2654435761u * (blockIdx.x * blockDim.x + threadIdx.x + 1u);
  unsigned long long acc = 0ull;
  for (long long i = 0; i < iters; ++i) {
    s ^= s << 13; s ^= s >> 17; s ^= s << 5;
    acc += tab[__umulhi(s, (unsigned)n_entries)];
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

}  // namespace

// =================================================================================================================
// Host side: handles and the C ABI
// =================================================================================================================
struct avm_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  int sm_count = 0;
  unsigned long long* h_counters = nullptr;   // pinned: the one word the host reads per launch
  int64_t n_kernel_launches = 0, n_transport_launches = 0;
  cudaEvent_t ev_t0 = nullptr, ev_t1 = nullptr;  // bracket the transport launches of the last avm_run
  float transport_ms = 0.0f;
};
struct BandTable {               // NEXT-1: host copy of the banded rates, [K][J + 1] as the readings state them
  int shift = 0, K = 0, J = 0;
  std::vector<double> a2, nu, dtmax;
};
struct avm_gas {
  DevGas d{};
  double nu_hat = 0.0;
  BandTable bands;
};
struct avm_field {
  DevField d{};
  int fk = 0;                 // 1 = one uniform slab, 2 = one grid slab, 0 = any other stack (template parameter FK)
  bool uniform1 = false;
};

namespace {

bool valid_gas(const avm_gas_desc* d, double* max_rate) {
  if (!d || d->n_bins < 1 || d->n_levels < 1 || d->n_levels > AVM_MAX_LEVELS || !(d->e_max_eV > 0) || !d->cum_rate ||
      !d->level_type || !d->level_loss_eV || !d->level_recoil || !d->level_ob_w_eV) {
    g_err = "gas: null pointer, empty table or n_levels > AVM_MAX_LEVELS";
    return false;
  }
  double mx = 0.0;
  const int L = d->n_levels;
  for (int b = 0; b < d->n_bins; ++b) {
    double prev = 0.0;
    for (int l = 0; l < L; ++l) {
      const double c = d->cum_rate[(size_t)b * L + l];
      if (!(c >= prev)) { g_err = "gas: cum_rate decreases along levels (or is NaN / negative)"; return false; }
      prev = c;
    }
    if (prev > mx) mx = prev;
  }
  for (int l = 0; l < L; ++l) {
    if (d->level_type[l] > 3) { g_err = "gas: bad level type"; return false; }
    if (d->level_type[l] == AVM_IONISATION && !(d->level_ob_w_eV[l] > 0)) { g_err = "gas: ionisation level needs w > 0"; return false; }
  }
  if (d->scat_xi)
    for (size_t i = 0; i < (size_t)d->n_bins * L; ++i)
      if (!(d->scat_xi[i] > -1.0 && d->scat_xi[i] < 1.0)) { g_err = "gas: scat_xi outside (-1, 1)"; return false; }
  if ((d->level_penning_prob != nullptr) != (d->level_penning_eV != nullptr)) { g_err = "gas: Penning probability and energy come together"; return false; }
  if (d->level_penning_prob)
    for (int l = 0; l < L; ++l)
      if (!(d->level_penning_prob[l] >= 0.0 && d->level_penning_prob[l] <= 1.0) || !(d->level_penning_eV[l] >= 0.0)) { g_err = "gas: Penning parameters"; return false; }
  if (!(d->kT_eV >= 0.0)) { g_err = "gas: kT < 0"; return false; }
  if (!(mx > 0.0) && !(d->nu_hat > 0.0)) { g_err = "gas: all rates are zero"; return false; }
  if (d->nu_hat > 0.0 && d->nu_hat < mx) { g_err = "gas: nu_hat below the maximum total rate"; return false; }
  if (max_rate) *max_rate = mx;
  return true;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

struct GasLayout { size_t nu_tot, head, tab, cum, loss, recoil, w, type, band, pen_p, pen_e, xi, total; };
constexpr int kBandClasses = 25;                 // N2: class edges 250 V/cm x 2^(j/2), j = 0 .. 24
int band_shift(int nb) { int s = 0; while ((nb >> (s + 1)) >= 256) ++s; return s; }   // N1: the most bins per band that leaves >= 256 bands
int band_count(int nb) { const int s = band_shift(nb); return (nb + (1 << s) - 1) >> s; }
int padded_levels(int L) { return (L + 1) & ~1; }
GasLayout gas_layout(int nb, int L, bool with_xi) {
  GasLayout g;
  const int Lp = padded_levels(L);
  size_t off = 0;
  g.nu_tot = off; off = align_up(off + sizeof(double) * nb, 256);
  g.head = off;   off = align_up(off + 4 * sizeof(double) * (size_t)nb, 256);
  g.tab = off;    off = align_up(off + sizeof(ushort4) * (size_t)nb, 256);
  g.cum = off;    off = align_up(off + sizeof(double) * (size_t)nb * Lp, 256);
  g.loss = off;   off += sizeof(double) * AVM_MAX_LEVELS;
  g.recoil = off; off += sizeof(double) * AVM_MAX_LEVELS;
  g.w = off;      off += sizeof(double) * AVM_MAX_LEVELS;
  g.type = off;   off = align_up(off + AVM_MAX_LEVELS, 256);
  g.band = off;   off = align_up(off + 32 * (size_t)(kBandClasses + 1) * band_count(nb), 256);
  g.pen_p = off;  off += sizeof(double) * AVM_MAX_LEVELS;
  g.pen_e = off;  off = align_up(off + sizeof(double) * AVM_MAX_LEVELS, 256);
  g.xi = off;     if (with_xi) off = align_up(off + sizeof(double) * (size_t)nb * L, 256);
  g.total = off;
  return g;
}


// NEXT-2: device form of a kind-2 slab — per element a 24-double record (vertex 3, the rows of the inverse
// edge matrix, the ten node potentials, the gas flag) and a bucket grid over the mesh's bounding box whose cells list, in
// ascending order, the elements whose bounding boxes touch them.  Layout in the caller's buffer: records | offsets | list.
struct MeshLayout { size_t rec, off, list, total; int n[3]; double lo[3], inv[3]; std::vector<int> counts; };
bool mesh_plan(const avm_slab& s, MeshLayout& L, std::vector<std::vector<int>>* buckets) {
  if (s.n_tets < 1 || s.n_tets > 0x7FFFFFFFll / 24 || s.n_mesh_nodes < 4 || !s.node_xyz || !s.node_V || !s.tet_nodes || !s.tet_gas) { g_err = "field: mesh arrays"; return false; }
  const int64_t nt = s.n_tets;
  for (int64_t i = 0; i < nt * 10; ++i) if (s.tet_nodes[i] < 0 || s.tet_nodes[i] >= s.n_mesh_nodes) { g_err = "field: mesh node index out of range"; return false; }
  double hi[3];
  for (int a = 0; a < 3; ++a) { L.lo[a] = std::numeric_limits<double>::infinity(); hi[a] = -L.lo[a]; }
  for (int64_t e = 0; e < nt; ++e)
    for (int v = 0; v < 4; ++v)
      for (int a = 0; a < 3; ++a) {
        const double x = s.node_xyz[3 * (size_t)s.tet_nodes[10 * e + v] + a];
        if (x < L.lo[a]) L.lo[a] = x;
        if (x > hi[a]) hi[a] = x;
      }
  // about two elements per cell on average, cells as cubic as the box allows
  double ext[3], vol = 1.0;
  for (int a = 0; a < 3; ++a) { ext[a] = hi[a] - L.lo[a]; if (!(ext[a] > 0.0)) { g_err = "field: degenerate mesh"; return false; } vol *= ext[a]; }
  const double cell = std::cbrt(vol / (0.5 * (double)nt));
  size_t nc = 1;
  for (int a = 0; a < 3; ++a) {
    int n = (int)std::ceil(ext[a] / cell);
    L.n[a] = n < 1 ? 1 : (n > 1024 ? 1024 : n);
    L.inv[a] = (double)L.n[a] / ext[a];
    nc *= (size_t)L.n[a];
  }
  L.counts.assign(nc, 0);
  if (buckets) buckets->assign(nc, {});
  size_t total = 0;
  for (int64_t e = 0; e < nt; ++e) {
    int c0[3], c1[3];
    for (int a = 0; a < 3; ++a) {
      double mn = std::numeric_limits<double>::infinity(), mx = -mn;
      for (int v = 0; v < 4; ++v) { const double x = s.node_xyz[3 * (size_t)s.tet_nodes[10 * e + v] + a]; if (x < mn) mn = x; if (x > mx) mx = x; }
      const double pad = 1e-9 * (mx - mn);
      const int i0 = (int)std::floor((mn - pad - L.lo[a]) * L.inv[a]), i1 = (int)std::floor((mx + pad - L.lo[a]) * L.inv[a]);
      c0[a] = i0 < 0 ? 0 : (i0 > L.n[a] - 1 ? L.n[a] - 1 : i0);
      c1[a] = i1 < 0 ? 0 : (i1 > L.n[a] - 1 ? L.n[a] - 1 : i1);
    }
    for (int k = c0[2]; k <= c1[2]; ++k) for (int j = c0[1]; j <= c1[1]; ++j) for (int i = c0[0]; i <= c1[0]; ++i) {
      const size_t c = ((size_t)k * L.n[1] + j) * L.n[0] + i;
      ++L.counts[c]; ++total;
      if (buckets) (*buckets)[c].push_back((int)e);
    }
  }
  if (total > 0x7FFFFFFFull) { g_err = "field: mesh index too large"; return false; }
  L.rec = 0;
  L.off = align_up(sizeof(double) * 24 * (size_t)nt, 256);
  L.list = align_up(L.off + sizeof(int) * (nc + 1), 256);
  L.total = align_up(L.list + sizeof(int) * total, 256);
  return true;
}
// Fills `h` (L.total bytes) with the device image of the mesh.
bool mesh_image(const avm_slab& s, const MeshLayout& L, const std::vector<std::vector<int>>& buckets, unsigned char* h) {
  double* rec = (double*)(h + L.rec);
  // Largest element extent of the mesh (bounding-box diagonal over the four vertices): scales the per-element margin of the
  // device's last-element shortcut below.
  double d_max = 0.0;
  for (int64_t e = 0; e < s.n_tets; ++e) {
    double d2 = 0.0;
    for (int a = 0; a < 3; ++a) {
      double mn = std::numeric_limits<double>::infinity(), mx = -mn;
      for (int v = 0; v < 4; ++v) { const double x = s.node_xyz[3 * (size_t)s.tet_nodes[10 * e + v] + a]; if (x < mn) mn = x; if (x > mx) mx = x; }
      d2 += (mx - mn) * (mx - mn);
    }
    if (d2 > d_max * d_max) d_max = std::sqrt(d2);
  }
  for (int64_t e = 0; e < s.n_tets; ++e) {
    const int32_t* nd = s.tet_nodes + 10 * e;
    const double* p[4];
    for (int v = 0; v < 4; ++v) p[v] = s.node_xyz + 3 * (size_t)nd[v];
    // edge matrix T = [p0 - p3 | p1 - p3 | p2 - p3] (columns); lambda_{0,1,2} = T^-1 (r - p3): rows of the inverse by cofactors
    double T[3][3];
    for (int r = 0; r < 3; ++r) for (int c = 0; c < 3; ++c) T[r][c] = p[c][r] - p[3][r];
    const double c00 = T[1][1] * T[2][2] - T[1][2] * T[2][1], c01 = T[1][2] * T[2][0] - T[1][0] * T[2][2], c02 = T[1][0] * T[2][1] - T[1][1] * T[2][0];
    const double det = T[0][0] * c00 + T[0][1] * c01 + T[0][2] * c02;
    if (!(std::fabs(det) > 0.0)) { g_err = "field: degenerate tetrahedron " + std::to_string(e); return false; }
    const double id = 1.0 / det;
    double G[3][3];
    G[0][0] = c00 * id; G[0][1] = (T[0][2] * T[2][1] - T[0][1] * T[2][2]) * id; G[0][2] = (T[0][1] * T[1][2] - T[0][2] * T[1][1]) * id;
    G[1][0] = c01 * id; G[1][1] = (T[0][0] * T[2][2] - T[0][2] * T[2][0]) * id; G[1][2] = (T[0][2] * T[1][0] - T[0][0] * T[1][2]) * id;
    G[2][0] = c02 * id; G[2][1] = (T[0][1] * T[2][0] - T[0][0] * T[2][1]) * id; G[2][2] = (T[0][0] * T[1][1] - T[0][1] * T[1][0]) * id;
    double* q = rec + 24 * (size_t)e;
    q[0] = p[3][0]; q[1] = p[3][1]; q[2] = p[3][2];
    for (int a = 0; a < 3; ++a) for (int c = 0; c < 3; ++c) q[3 + 3 * a + c] = G[a][c];
    for (int i = 0; i < 10; ++i) q[12 + i] = s.node_V[nd[i]];
    q[22] = s.tet_gas[e] ? 1.0 : 0.0;
    // Margin of the last-element shortcut (tet_at): a point whose barycentrics in THIS element are all >= q[23] lies at least
    // q[23] h_min inside it (h_min = its smallest height = 1 / max |grad lambda_i|).  Another element e' of a valid mesh does
    // not overlap it, so the point is at least that far outside e'; a point with all barycentrics of e' >= -eps is within
    // 8 eps D' of e' (D' = its extent: clip the negative coordinates and renormalise), so e' fails F2's test (eps = 1e-10)
    // whenever q[23] h_min > 8e-10 D'.  With D' <= d_max: q[23] = 1e-9 max(1, d_max / h_min) holds for ANY grading of the mesh.
    double g_max = 0.0;
    for (int a = 0; a < 4; ++a) {
      double gx, gy, gz;
      if (a < 3) { gx = G[a][0]; gy = G[a][1]; gz = G[a][2]; }
      else { gx = -(G[0][0] + G[1][0] + G[2][0]); gy = -(G[0][1] + G[1][1] + G[2][1]); gz = -(G[0][2] + G[1][2] + G[2][2]); }
      const double gn = std::sqrt(gx * gx + gy * gy + gz * gz);
      if (gn > g_max) g_max = gn;
    }
    const double ratio = d_max * g_max;                       // d_max / h_min
    q[23] = 1e-9 * (ratio > 1.0 ? ratio : 1.0);
  }
  int* off = (int*)(h + L.off);
  int* list = (int*)(h + L.list);
  int run = 0;
  for (size_t c = 0; c < buckets.size(); ++c) {
    off[c] = run;
    for (int e : buckets[c]) list[run++] = e;
  }
  off[buckets.size()] = run;
  return true;
}

// NEXT-1, readings N1-N4 of DESIGN.md §3.5: the table of banded null-collision rates.
//  N1 bands: 2^shift consecutive energy bins each (band_shift), K = ceil(nb / 2^shift) of them.
//  N2 acceleration classes: squared upper edges A_j^2 = (kappa 250 V/cm)^2 2^j, j = 0 .. J-1, J = 25; column J = any
//     stronger field.
//  N3 reach: an electron that starts a flight with energy below the band's upper edge e_hi under an acceleration <= A_j
//     has, after a time <= dt, a speed <= c2 sqrt(e_hi) + A_j dt, hence (one bin of slack) an energy bin <= reach(dt); with
//     M[b] = the largest total rate of bins 0 .. b, the rate of (k, j) for a validity time dt = m / nu is a solution of
//     nu >= M[reach(m / nu)], found by iterating from M[last bin of the band] and tightened while the next iterate still
//     bounds its own reach.
//  N4 m is the one of {1/2, 1, 2, 4, 8, 16} with the smallest nu / (1 - exp(-m)) (steps per unit time, cut flights
//     included; the last one on ties); the last band (it also holds the energies beyond the table) and column J use the
//     table's largest rate with no cut.
void build_bands(const avm_gas_desc* d, double nu_hat, BandTable& T) {
  const int nb = d->n_bins, L = d->n_levels;
  const double inf = std::numeric_limits<double>::infinity();
  const double inv_de = (double)nb / d->e_max_eV, de = d->e_max_eV / (double)nb;
  std::vector<double> M(nb);
  for (int b = 0; b < nb; ++b) {
    const double tot = d->cum_rate[(size_t)b * L + L - 1];
    M[b] = b == 0 ? (tot > 0.0 ? tot : 0.0) : (tot > M[b - 1] ? tot : M[b - 1]);
  }
  T.shift = band_shift(nb); T.K = band_count(nb); T.J = kBandClasses;
  const int W = T.J + 1;
  T.a2.resize(T.J);
  const double a0 = kKappa * 250.0;
  for (int j = 0; j < T.J; ++j) T.a2[j] = std::ldexp(a0 * a0, j);
  T.nu.assign((size_t)T.K * W, M[nb - 1]);
  T.dtmax.assign((size_t)T.K * W, inf);
  auto reach_rate = [&](double e_hi, double A, double m, double nu) {
    const double dt = m / nu;
    const double speed = kC2 * std::sqrt(e_hi) + A * dt;
    const double sb = (speed * speed * kInvC2Sq) * inv_de + 1.0;
    return M[sb >= (double)(nb - 1) ? nb - 1 : (int)sb];
  };
  static const double m_of[6] = {0.5, 1.0, 2.0, 4.0, 8.0, 16.0};
  for (int k = 0; k + 1 < T.K; ++k) {
    int last = ((k + 1) << T.shift) - 1;
    if (last > nb - 1) last = nb - 1;
    const double e_hi = (double)(last + 1) * de;
    for (int j = 0; j < T.J; ++j) {
      const double A = std::sqrt(T.a2[j]);
      double best_cost = inf, best_nu = M[nb - 1], best_dt = inf;
      for (int c = 0; c < 6; ++c) {
        const double m = m_of[c];
        double nu = reach_rate(e_hi, A, m, M[last]);
        for (int it = 0; it < 4; ++it) {
          const double next = reach_rate(e_hi, A, m, nu);
          if (!(next < nu && reach_rate(e_hi, A, m, next) <= next)) break;
          nu = next;
        }
        const double cost = nu / (1.0 - std::exp(-m));
        if (nu > 0.0 && cost <= best_cost) { best_cost = cost; best_nu = nu; best_dt = m / nu; }
      }
      T.nu[(size_t)k * W + j] = best_nu;
      T.dtmax[(size_t)k * W + j] = best_dt;
    }
  }
  for (size_t i = 0; i < T.nu.size(); ++i)
    if (!(T.nu[i] > 0.0)) { T.nu[i] = nu_hat; T.dtmax[i] = inf; }
}

template <typename K, typename... Args>
cudaError_t launch(avm_ctx* ctx, K kernel, dim3 grid, dim3 block, Args... args) {
  kernel<<<grid, block, 0, ctx->stream>>>(args...);
  ctx->n_kernel_launches++;
  return cudaGetLastError();
}

}  // namespace

extern "C" {

const char* avm_last_error(void) { return g_err.c_str(); }

int32_t avm_ctx_create(int32_t device, void* cuda_stream, avm_ctx** out) {
  if (!out) return fail(AVM_ERR_INVALID_ARG, "ctx_create: out is null");
  *out = nullptr;
  int n_dev = 0;
  AVM_CUDA(cudaGetDeviceCount(&n_dev));
  if (device < 0 || device >= n_dev) return fail(AVM_ERR_CUDA, "ctx_create: no such CUDA device");
  AVM_CUDA(cudaSetDevice(device));
  cudaDeviceProp prop;
  AVM_CUDA(cudaGetDeviceProperties(&prop, device));
  if (prop.major != 10) return fail(AVM_ERR_CUDA, "ctx_create: device is not compute capability 10.x (built for sm_100a only)");
  avm_ctx* c = new (std::nothrow) avm_ctx();
  if (!c) return fail(AVM_ERR_STATE, "ctx_create: out of host memory");
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  c->sm_count = prop.multiProcessorCount;
  cudaError_t e = cudaHostAlloc((void**)&c->h_counters, 64, cudaHostAllocDefault);
  if (e != cudaSuccess) { delete c; return fail(AVM_ERR_CUDA, std::string("ctx_create: cudaHostAlloc: ") + cudaGetErrorString(e)); }
  if (cudaEventCreate(&c->ev_t0) != cudaSuccess || cudaEventCreate(&c->ev_t1) != cudaSuccess) {
    cudaFreeHost(c->h_counters); delete c; return fail(AVM_ERR_CUDA, "ctx_create: cudaEventCreate");
  }
  *out = c;
  return AVM_OK;
}

int32_t avm_ctx_destroy(avm_ctx* c) {
  if (!c) return AVM_OK;
  if (c->h_counters) cudaFreeHost(c->h_counters);
  if (c->ev_t0) cudaEventDestroy(c->ev_t0);
  if (c->ev_t1) cudaEventDestroy(c->ev_t1);
  delete c;
  return AVM_OK;
}

int32_t avm_ctx_sm_count(const avm_ctx* c) { return c ? c->sm_count : 0; }

size_t avm_gas_bytes(const avm_gas_desc* d) {
  if (!d || d->n_bins < 1 || d->n_levels < 1 || d->n_levels > AVM_MAX_LEVELS) return 0;
  return gas_layout(d->n_bins, d->n_levels, d->scat_xi != nullptr).total;
}

int32_t avm_gas_create(avm_ctx* ctx, const avm_gas_desc* d, void* dev_buf, size_t dev_bytes, avm_gas** out) {
  if (!ctx || !out) return fail(AVM_ERR_INVALID_ARG, "gas_create: null ctx/out");
  *out = nullptr;
  double mx = 0.0;
  if (!valid_gas(d, &mx)) return AVM_ERR_INVALID_ARG;
  const int nb = d->n_bins, L = d->n_levels;
  const GasLayout lay = gas_layout(nb, L, d->scat_xi != nullptr);
  if (!dev_buf || dev_bytes < lay.total || ((uintptr_t)dev_buf & 255u)) return fail(AVM_ERR_INVALID_ARG, "gas_create: device buffer null, too small or not 256-byte aligned");
  std::vector<unsigned char> h(lay.total, 0);
  double* nu_tot = (double*)(h.data() + lay.nu_tot);
  double* head = (double*)(h.data() + lay.head);
  unsigned short* tab = (unsigned short*)(h.data() + lay.tab);
  const double nu_hat_r = d->nu_hat > 0.0 ? d->nu_hat : mx;
  auto q16 = [&](double c) {                       // floor(c / nu_hat * 2^16) clamped to 16 bits (decide())
    const double v = std::floor(c / nu_hat_r * 65536.0);
    return (unsigned short)(v < 0.0 ? 0.0 : (v > 65535.0 ? 65535.0 : v));
  };
  for (int b = 0; b < nb; ++b) {
    const double* row = d->cum_rate + (size_t)b * L;
    nu_tot[b] = row[L - 1];
    head[4 * (size_t)b + 0] = row[L - 1];               // decision record: one 32-byte sector per step
    head[4 * (size_t)b + 1] = row[0];
    head[4 * (size_t)b + 2] = row[L > 1 ? 1 : 0];
    head[4 * (size_t)b + 3] = 0.0;
    tab[4 * (size_t)b + 0] = q16(row[L - 1]);
    tab[4 * (size_t)b + 1] = q16(row[0]);
    tab[4 * (size_t)b + 2] = q16(row[L > 1 ? 1 : 0]);
    tab[4 * (size_t)b + 3] = 0;
  }
  {
    const int Lp = padded_levels(L);
    double* cum = (double*)(h.data() + lay.cum);
    for (int b = 0; b < nb; ++b) {
      for (int l = 0; l < L; ++l) cum[(size_t)b * Lp + l] = d->cum_rate[(size_t)b * L + l];
      for (int l = L; l < Lp; ++l) cum[(size_t)b * Lp + l] = std::numeric_limits<double>::infinity();
    }
  }
  BandTable bands;
  build_bands(d, nu_hat_r, bands);
  {
    // device layout [J + 1][K][2 x 16 B]: (1 / nu, dtmax), (nu, rho) with rho = floor(nu / nu_hat 2^32) in the low word
    unsigned char* bt = h.data() + lay.band;
    const int W = bands.J + 1;
    for (int j = 0; j < W; ++j)
      for (int k = 0; k < bands.K; ++k) {
        const double nu = bands.nu[(size_t)k * W + j], dtm = bands.dtmax[(size_t)k * W + j];
        const double inv = 1.0 / nu;
        double rr = std::floor(nu / nu_hat_r * 4294967296.0);
        if (rr > 4294967295.0) rr = 4294967295.0;
        if (rr < 0.0) rr = 0.0;
        const unsigned long long rho = (unsigned long long)rr;
        unsigned char* e = bt + 32 * ((size_t)j * bands.K + k);
        std::memcpy(e, &inv, 8); std::memcpy(e + 8, &dtm, 8); std::memcpy(e + 16, &nu, 8); std::memcpy(e + 24, &rho, 8);
      }
  }
  std::memcpy(h.data() + lay.loss, d->level_loss_eV, sizeof(double) * L);
  std::memcpy(h.data() + lay.recoil, d->level_recoil, sizeof(double) * L);
  std::memcpy(h.data() + lay.w, d->level_ob_w_eV, sizeof(double) * L);
  std::memcpy(h.data() + lay.type, d->level_type, L);
  if (d->level_penning_prob) {
    std::memcpy(h.data() + lay.pen_p, d->level_penning_prob, sizeof(double) * L);
    std::memcpy(h.data() + lay.pen_e, d->level_penning_eV, sizeof(double) * L);
  }
  if (d->scat_xi) std::memcpy(h.data() + lay.xi, d->scat_xi, sizeof(double) * (size_t)nb * L);
  AVM_CUDA(cudaSetDevice(ctx->device));
  AVM_CUDA(cudaMemcpyAsync(dev_buf, h.data(), lay.total, cudaMemcpyHostToDevice, ctx->stream));
  AVM_CUDA(cudaStreamSynchronize(ctx->stream));
  avm_gas* g = new (std::nothrow) avm_gas();
  if (!g) return fail(AVM_ERR_STATE, "gas_create: out of host memory");
  unsigned char* base = (unsigned char*)dev_buf;
  g->nu_hat = d->nu_hat > 0.0 ? d->nu_hat : mx;
  g->d.nb = nb; g->d.L = L; g->d.Lp = padded_levels(L);
  g->d.inv_de = (double)nb / d->e_max_eV;
  {
    const double fb = kEpsFloor * g->d.inv_de;
    g->d.bin_floor = fb >= (double)(nb - 1) ? nb - 1 : (int)fb;
  }
  g->d.nu_hat = g->nu_hat;
  g->d.inv_nu_hat = 1.0 / g->nu_hat;
  g->d.nu_tot = (const double*)(base + lay.nu_tot);
  g->d.head = (const double2*)(base + lay.head);
  g->d.tab = (const ushort4*)(base + lay.tab);
  g->d.cum = (const double*)(base + lay.cum);
  g->d.loss = (const double*)(base + lay.loss);
  g->d.recoil = (const double*)(base + lay.recoil);
  g->d.w = (const double*)(base + lay.w);
  g->d.type = (const uint8_t*)(base + lay.type);
  g->d.pen_p = (const double*)(base + lay.pen_p);
  g->d.pen_e = (const double*)(base + lay.pen_e);
  g->d.xi = d->scat_xi ? (const double*)(base + lay.xi) : nullptr;
  g->d.kT = d->kT_eV;
  g->d.ext = (d->scat_xi ? 1 : 0) | (d->kT_eV > 0.0 ? 2 : 0);
  if (d->level_penning_prob)
    for (int l = 0; l < L; ++l) if (d->level_penning_prob[l] > 0.0) g->d.ext |= 4;
  g->d.bshift = bands.shift; g->d.bK = bands.K; g->d.bJ = bands.J;
  g->d.a0sq = bands.a2[0]; g->d.inv_a0sq = 1.0 / bands.a2[0];
  g->d.band = (const double2*)(base + lay.band);
  g->bands = std::move(bands);
  *out = g;
  return AVM_OK;
}

int32_t avm_gas_destroy(avm_gas* g) { delete g; return AVM_OK; }
double avm_gas_nu_hat(const avm_gas* g) { return g ? g->nu_hat : 0.0; }

int32_t avm_gas_bands(const avm_gas* g, int32_t* shape3, double* a2, double* nu, double* dtmax) {
  if (!g || !shape3) return fail(AVM_ERR_INVALID_ARG, "gas_bands: null argument");
  const BandTable& T = g->bands;
  shape3[0] = T.K; shape3[1] = T.J; shape3[2] = T.shift;
  if (a2) std::memcpy(a2, T.a2.data(), sizeof(double) * T.a2.size());
  if (nu) std::memcpy(nu, T.nu.data(), sizeof(double) * T.nu.size());
  if (dtmax) std::memcpy(dtmax, T.dtmax.data(), sizeof(double) * T.dtmax.size());
  return AVM_OK;
}

int32_t avm_field_create(avm_ctx* ctx, const avm_field_desc* d, avm_field** out) {
  if (!ctx || !out) return fail(AVM_ERR_INVALID_ARG, "field_create: null ctx/out");
  *out = nullptr;
  if (!d || !d->slabs || d->n_slabs < 1 || d->n_slabs > AVM_MAX_SLABS) return fail(AVM_ERR_INVALID_ARG, "field_create: need 1..AVM_MAX_SLABS slabs");
  const double inf = std::numeric_limits<double>::infinity();
  avm_field* f = new (std::nothrow) avm_field();
  if (!f) return fail(AVM_ERR_STATE, "field_create: out of host memory");
  DevField& F = f->d;
  F.n_slabs = d->n_slabs;
  for (int i = 0; i < d->n_slabs; ++i) {
    const avm_slab& s = d->slabs[i];
    DevSlab& S = F.slab[i];
    const char* bad = nullptr;
    if (!(s.z_hi > s.z_lo)) bad = "field: slab z_hi <= z_lo";
    else if (i > 0 && s.z_lo != d->slabs[i - 1].z_hi) bad = "field: slabs not contiguous/ascending";
    else if (s.kind != 0 && s.kind != 1 && s.kind != 2) bad = "field: kind";
    if (!bad && s.kind == 0 && !(std::isfinite(s.E[0]) && std::isfinite(s.E[1]) && std::isfinite(s.E[2]))) bad = "field: uniform E is not finite";
    S.z_lo = s.z_lo; S.z_hi = s.z_hi; S.kind = s.kind;
    for (int a = 0; a < 3; ++a) S.E[a] = s.E[a];
    if (!bad && s.kind == 1) {
      if (!s.nodes_dev || s.nx < 2 || s.ny < 2 || s.nz < 2) bad = "field: grid needs device nodes and >= 2 nodes per axis";
      else if ((uintptr_t)s.nodes_dev & 15u) bad = "field: nodes not 16-byte aligned";
      else if (!(s.spacing[0] > 0 && s.spacing[1] > 0 && s.spacing[2] > 0)) bad = "field: spacing";
      else if (s.bc_x < 0 || s.bc_x > 2 || s.bc_y < 0 || s.bc_y > 2) bad = "field: bc";
      else {
        const double ztop = s.origin[2] + (s.nz - 1) * s.spacing[2], tol = 1e-9 * s.spacing[2];
        if (s.z_lo < s.origin[2] - tol || s.z_hi > ztop + tol) bad = "field: slab z-range outside its grid";
        if (s.bc_x && !(s.period_x > 0 && s.period_x <= (s.nx - 1) * s.spacing[0] * (1 + 1e-12))) bad = "field: period_x";
        if (s.bc_y && !(s.period_y > 0 && s.period_y <= (s.ny - 1) * s.spacing[1] * (1 + 1e-12))) bad = "field: period_y";
      }
      S.nodes = (const float4*)s.nodes_dev;
      S.nodes64 = s.nodes_f64_dev;
      if (!bad && s.nodes_f64_dev && ((uintptr_t)s.nodes_f64_dev & 15u)) bad = "field: nodes_f64_dev not 16-byte aligned";
      S.nx = s.nx; S.ny = s.ny; S.nz = s.nz;
      const int bc[2] = {s.bc_x, s.bc_y};
      const double per[2] = {s.period_x, s.period_y};
      const int nn[2] = {s.nx, s.ny};
      for (int a = 0; a < 3; ++a) { S.org[a] = s.origin[a]; S.inv_h[a] = 1.0 / s.spacing[a]; }
      for (int a = 0; a < 2; ++a) {
        S.bc[a] = bc[a];
        S.span[a] = bc[a] ? inf : (nn[a] - 1) * s.spacing[a];
        S.P[a] = bc[a] == 2 ? 2.0 * per[a] : (bc[a] == 1 ? per[a] : 1.0);
        S.inv_P[a] = bc[a] ? 1.0 / S.P[a] : 0.0;
        S.Pc[a] = bc[a] ? S.P[a] : inf;
        S.lo[a] = bc[a] ? 0.0 : -inf;
        S.half[a] = bc[a] == 2 ? per[a] : inf;
      }
    }
    if (!bad && s.kind == 2) {
      // NEXT-2: x / y fold constants as for a grid (no extent: a point in no element is solid), the mesh image uploaded
      if (s.bc_x < 0 || s.bc_x > 2 || s.bc_y < 0 || s.bc_y > 2) bad = "field: bc";
      else if ((s.bc_x && !(s.period_x > 0)) || (s.bc_y && !(s.period_y > 0))) bad = "field: period";
      const int bc[2] = {s.bc_x, s.bc_y};
      const double per[2] = {s.period_x, s.period_y};
      for (int a = 0; a < 3; ++a) { S.org[a] = s.origin[a]; S.inv_h[a] = 1.0; }
      for (int a = 0; a < 2; ++a) {
        S.bc[a] = bc[a];
        S.span[a] = inf;
        S.P[a] = bc[a] == 2 ? 2.0 * per[a] : (bc[a] == 1 ? per[a] : 1.0);
        S.inv_P[a] = bc[a] ? 1.0 / S.P[a] : 0.0;
        S.Pc[a] = bc[a] ? S.P[a] : inf;
        S.lo[a] = bc[a] ? 0.0 : -inf;
        S.half[a] = bc[a] == 2 ? per[a] : inf;
      }
      MeshLayout L;
      std::vector<std::vector<int>> buckets;
      if (!bad && !mesh_plan(s, L, &buckets)) { delete f; return AVM_ERR_INVALID_ARG; }
      if (!bad && (!s.mesh_dev || s.mesh_dev_bytes < L.total || ((uintptr_t)s.mesh_dev & 255u))) bad = "field: mesh_dev null, smaller than avm_tetmesh_bytes or not 256-byte aligned";
      if (!bad) {
        std::vector<unsigned char> img(L.total, 0);
        if (!mesh_image(s, L, buckets, img.data())) { delete f; return AVM_ERR_INVALID_ARG; }
        cudaError_t e = cudaSetDevice(ctx->device);
        if (e == cudaSuccess) e = cudaMemcpyAsync(s.mesh_dev, img.data(), L.total, cudaMemcpyHostToDevice, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) { delete f; return fail(AVM_ERR_CUDA, std::string("field_create: mesh upload: ") + cudaGetErrorString(e)); }
        unsigned char* base = (unsigned char*)s.mesh_dev;
        S.tet_rec = (const double*)(base + L.rec); S.tet_off = (const int*)(base + L.off); S.tet_list = (const int*)(base + L.list);
        for (int a = 0; a < 3; ++a) { S.tlo[a] = L.lo[a]; S.tinv[a] = L.inv[a]; S.tn[a] = L.n[a]; }
        S.n_tets = (int)s.n_tets;
      }
    }
    if (bad) { delete f; return fail(AVM_ERR_INVALID_ARG, bad); }
  }
  F.z_lo = d->slabs[0].z_lo;
  F.z_hi = d->slabs[d->n_slabs - 1].z_hi;
  for (int a = 0; a < 2; ++a) { F.xy_lo[a] = d->xy_lo[a]; F.xy_hi[a] = d->xy_hi[a]; }
  if (!(std::isfinite(d->B[0]) && std::isfinite(d->B[1]) && std::isfinite(d->B[2]))) { delete f; return fail(AVM_ERR_INVALID_ARG, "field: B is not finite"); }
  const double Bn2 = d->B[0] * d->B[0] + d->B[1] * d->B[1] + d->B[2] * d->B[2];
  F.has_B = Bn2 != 0.0;
  F.Bn2 = Bn2;
  for (int a = 0; a < 3; ++a) F.B[a] = d->B[a];
  if (F.has_B) {
    const double Bn = std::sqrt(Bn2);
    for (int a = 0; a < 3; ++a) F.bh[a] = d->B[a] / Bn;
    F.omega = kOmega1 * Bn;
    F.inv_omega = 1.0 / F.omega;
  }
  for (int i = 0; i < d->n_slabs; ++i) {           // widen the grid maps once (the one-off field transfer)
    const DevSlab& S = F.slab[i];
    if (S.kind != 1 || !S.nodes64) continue;
    const size_t nn = (size_t)S.nx * S.ny * S.nz;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) {
      widen_map_kernel<<<(unsigned)ctx->sm_count * 8u, 256, 0, ctx->stream>>>(S.nodes, (double2*)S.nodes64, nn);
      e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { delete f; return fail(AVM_ERR_CUDA, std::string("field_create: widening the map: ") + cudaGetErrorString(e)); }
  }
  f->uniform1 = d->n_slabs == 1 && d->slabs[0].kind == 0;
  f->fk = f->uniform1 ? 1 : ((d->n_slabs == 1 && d->slabs[0].kind == 1) ? 2 : 0);   // a lone tetrahedral map takes the general path
  F.xy_bounded = 0;
  for (int a = 0; a < 2; ++a)
    if (std::isfinite(F.xy_lo[a]) || std::isfinite(F.xy_hi[a]) || F.xy_lo[a] != F.xy_lo[a] || F.xy_hi[a] != F.xy_hi[a]) F.xy_bounded = 1;
  {
    // constants of the flight in slab 0 (used when the field is one uniform slab), same formulas as flight<>
    const double* E = F.slab[0].E;
    for (int a = 0; a < 3; ++a) { F.ua[a] = -kKappa * E[a]; F.uvd[a] = 0.0; F.uap[a] = 0.0; }
    if (F.has_B) {
      const double a_b = F.ua[0] * F.bh[0] + F.ua[1] * F.bh[1] + F.ua[2] * F.bh[2];
      const double sc = kExBUnit / F.Bn2;
      F.uvd[0] = sc * (E[1] * F.B[2] - E[2] * F.B[1]);
      F.uvd[1] = sc * (E[2] * F.B[0] - E[0] * F.B[2]);
      F.uvd[2] = sc * (E[0] * F.B[1] - E[1] * F.B[0]);
      for (int a = 0; a < 3; ++a) F.uap[a] = a_b * F.bh[a];
    }
  }
  *out = f;
  return AVM_OK;
}

int32_t avm_field_destroy(avm_field* f) { delete f; return AVM_OK; }

size_t avm_tetmesh_bytes(const avm_slab* s) {
  if (!s || s->kind != 2) return 0;
  MeshLayout L;
  return mesh_plan(*s, L, nullptr) ? L.total : 0;
}

int32_t avm_field_eval(avm_ctx* ctx, const avm_field* f, int64_t n, const double* r, double* E, double* mask, int32_t* slab) {
  if (!ctx || !f || n < 0 || (n > 0 && (!r || !E || !mask || !slab))) return fail(AVM_ERR_INVALID_ARG, "field_eval: null argument");
  if (n == 0) return AVM_OK;
  AVM_CUDA(cudaSetDevice(ctx->device));
  AVM_CUDA(launch(ctx, field_eval_kernel, dim3((unsigned)((n + 255) / 256)), dim3(256), f->d, n, r, E, mask, slab));
  return AVM_OK;
}

size_t avm_run_workspace_bytes(const avm_ctx*, int64_t capacity) {
  if (capacity < 0) return 0;
  const int64_t stage = capacity < kStageElectrons ? capacity : kStageElectrons;
  return kCtlBytes + (size_t)stage * 8 * sizeof(double);
}

int32_t avm_run_stats(const avm_ctx* c, int64_t* n_kernel_launches, int64_t* n_transport_launches) {
  if (!c) return fail(AVM_ERR_INVALID_ARG, "run_stats: null ctx");
  if (n_kernel_launches) *n_kernel_launches = c->n_kernel_launches;
  if (n_transport_launches) *n_transport_launches = c->n_transport_launches;
  return AVM_OK;
}

int32_t avm_run_transport_ms(const avm_ctx* c, float* ms_out) {
  if (!c || !ms_out) return fail(AVM_ERR_INVALID_ARG, "run_transport_ms: null argument");
  *ms_out = c->transport_ms;
  return AVM_OK;
}

}  // extern "C"

namespace {
TransportFn pick_transport(int fk, bool has_b, bool smemtab, bool wide, bool banded, bool signal) {
  if (fk == 1) return has_b ? pick_transport_inst<1, true>(smemtab, wide, banded, signal) : pick_transport_inst<1, false>(smemtab, wide, banded, signal);
  if (fk == 2) return has_b ? pick_transport_inst<2, true>(smemtab, wide, banded, signal) : pick_transport_inst<2, false>(smemtab, wide, banded, signal);
  return has_b ? pick_transport_inst<0, true>(smemtab, wide, banded, signal) : pick_transport_inst<0, false>(smemtab, wide, banded, signal);
}
// W1: the device form of a signal description (validated); false with g_err set when it is unusable.
bool make_signal(const avm_signal* s, DevSignal& D) {
  std::memset(&D, 0, sizeof(D));
  if (!s) return true;
  if (!s->weighting || !(s->dt_bin > 0.0) || s->n_bins < 1 || !s->signal_dev || !std::isfinite(s->t0)) { g_err = "signal: weighting field, dt_bin > 0, n_bins >= 1 and a device array are required"; return false; }
  for (int i = 0; i < s->weighting->d.n_slabs; ++i)
    if (s->weighting->d.slab[i].kind == 2) { g_err = "signal: the weighting field must consist of uniform slabs and grid maps (a tetrahedral slab, kind 2, is not accepted here)"; return false; }
  D.wf = s->weighting->d;
  D.t0 = s->t0; D.inv_dt = 1.0 / s->dt_bin; D.n_bins = s->n_bins; D.uniform1 = s->weighting->uniform1 ? 1 : 0;
  D.out = s->signal_dev;
  return true;
}
}  // namespace

extern "C" {

int32_t avm_run(avm_ctx* ctx, const avm_gas* gas, const avm_field* field, const double* primaries, int64_t np,
                const avm_run_opts* opts, const avm_outputs* o, int64_t* n_out) {
  if (!ctx || !gas || !field || !opts || !o || !n_out) return fail(AVM_ERR_INVALID_ARG, "run: null argument");
  *n_out = 0;
  if (np < 0 || (np > 0 && !primaries)) return fail(AVM_ERR_INVALID_ARG, "run: primaries");
  if (o->capacity < np || o->capacity < 1 || o->capacity > 0x7FFFFFFFll) return fail(AVM_ERR_INVALID_ARG, "run: capacity must be in [max(1, n_primaries), 2^31)");
  if (!o->id || !o->avalanche || !o->status || !o->n_steps || !o->end) return fail(AVM_ERR_INVALID_ARG, "run: id, avalanche, status, n_steps and end are required");
  if (o->tallies_f64 && !o->birth) return fail(AVM_ERR_INVALID_ARG, "run: tallies_f64 needs birth");
  if (!o->workspace || o->workspace_bytes < avm_run_workspace_bytes(ctx, o->capacity) || ((uintptr_t)o->workspace & 255u))
    return fail(AVM_ERR_INVALID_ARG, "run: workspace null, too small or not 256-byte aligned");
  // Launch shape and kernel variant first: a combination without a variant is refused before any work is queued.
  bool wide = np > (int64_t)ctx->sm_count * kThreads;            // the primaries alone outnumber the latency shape's lanes
  if (opts->flags & AVM_RUN_SHAPE_WIDE) wide = true;
  if (opts->flags & AVM_RUN_SHAPE_LATENCY) wide = false;
  const int threads = wide ? kThreadsWide : kThreads;
  const size_t buf_bytes = sizeof(WarpBuf) * (size_t)(threads / 32);
  const size_t tab_bytes = align_up(sizeof(ushort4) * (size_t)gas->d.nb, 16);
  const bool smemtab = tab_bytes + buf_bytes <= kMaxDynSmem;       // else the threshold table is read through L1
  const size_t dyn_smem = (smemtab ? tab_bytes : 0) + buf_bytes;
  DevSignal dsig;
  if (!make_signal(opts->signal, dsig)) return AVM_ERR_INVALID_ARG;
  const bool extras = opts->signal != nullptr || gas->d.ext != 0;     // NEXT-3 / NEXT-4: the kernel variant that has them
  TransportFn fn = pick_transport(field->fk, field->d.has_B != 0, smemtab, wide, (opts->flags & AVM_RUN_BANDED) != 0, extras);
  if (!fn) return fail(AVM_ERR_INVALID_ARG, "run: a signal or a gas with NEXT-3 extensions needs the threshold table in shared memory (at most ~24000 energy bins)");
  AVM_CUDA(cudaSetDevice(ctx->device));
  ctx->n_kernel_launches = 0; ctx->n_transport_launches = 0; ctx->transport_ms = 0.0f;
  cudaStream_t st = ctx->stream;
  RunCtl* ctl = (RunCtl*)o->workspace;
  double* stage = (double*)((unsigned char*)o->workspace + kCtlBytes);
  RunArrays a;
  a.cap = (uint32_t)o->capacity; a.id = o->id; a.aval = o->avalanche; a.status = o->status; a.nsteps = o->n_steps;
  a.birth = o->birth; a.end = o->end;
  const bool on_dev = opts->flags & AVM_RUN_PRIMARIES_ON_DEVICE;

  AVM_CUDA(cudaMemsetAsync(ctl, 0, kCtlBytes, st));
  AVM_CUDA(cudaMemsetAsync(o->status, 0xFF, sizeof(int32_t) * (size_t)o->capacity, st));   // -1 = slot not created yet
  if (o->per_avalanche && np > 0) AVM_CUDA(cudaMemsetAsync(o->per_avalanche, 0, sizeof(uint64_t) * 3 * (size_t)np, st));
  // a-1: primaries in (H2D inside the call), chunked through the staging area
  for (int64_t p0 = 0; p0 < np; p0 += kStageElectrons) {
    const int64_t cnt = (np - p0) < kStageElectrons ? (np - p0) : kStageElectrons;
    const double* src = primaries + p0 * 8;
    if (!on_dev) {
      AVM_CUDA(cudaMemcpyAsync(stage, src, sizeof(double) * 8 * (size_t)cnt, cudaMemcpyHostToDevice, st));
      src = stage;
    }
    const dim3 grid((unsigned)((cnt + 255) / 256));
    if (field->uniform1) AVM_CUDA(launch(ctx, inject_kernel<1>, grid, dim3(256), field->d, a, ctl, src, (uint32_t)p0, (uint32_t)cnt, opts->id_offset, opts->t_max));
    else AVM_CUDA(launch(ctx, inject_kernel<0>, grid, dim3(256), field->d, a, ctl, src, (uint32_t)p0, (uint32_t)cnt, opts->id_offset, opts->t_max));
  }
  // persistent transport (a-2 .. a-11)
  AVM_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn_smem));
  int occ = 0;
  AVM_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, dyn_smem));
  if (occ < 1) return fail(AVM_ERR_CUDA, "run: transport kernel does not fit on an SM");
  unsigned grid = (unsigned)(ctx->sm_count * occ);
  if (grid > (unsigned)kMaxGrid) grid = kMaxGrid;
  if (opts->max_ctas > 0 && (unsigned)opts->max_ctas < grid) grid = (unsigned)opts->max_ctas;
  const uint32_t n_static = grid * (uint32_t)threads;
  const uint32_t max_iters = opts->max_iters_per_launch ? opts->max_iters_per_launch : kDefaultMaxIters;
  unsigned long long c = 0ull;
  const int64_t max_launches = 1ll << 20;
  int64_t launches = 0;
  for (;;) {
    AVM_CUDA(cudaMemcpyAsync(ctx->h_counters, &ctl->counters, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    AVM_CUDA(cudaStreamSynchronize(st));
    c = *ctx->h_counters;
    if ((uint32_t)(c >> 32) == (uint32_t)c) break;              // a-11: every electron has a non-zero status
    if (++launches > max_launches) return fail(AVM_ERR_STATE, "run: launch limit reached without termination");
    AVM_CUDA(cudaMemsetAsync(&ctl->q_head, 0, sizeof(unsigned int), st));
    if (launches > 1) AVM_CUDA(cudaMemsetAsync((unsigned char*)ctl + kDoneOffset, 0, (size_t)kMaxGrid * 32, st));   // stop flags
    if (launches > 1) {                                          // close the previous launch's bracket
      float ms = 0.0f;
      AVM_CUDA(cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1));
      ctx->transport_ms += ms;
    }
    AVM_CUDA(cudaEventRecord(ctx->ev_t0, st));
    fn<<<grid, threads, dyn_smem, st>>>(gas->d, field->d, a, ctl, philox_keys(opts->seed), opts->t_max, max_iters, n_static, dsig);
    AVM_CUDA(cudaGetLastError());
    AVM_CUDA(cudaEventRecord(ctx->ev_t1, st));
    ctx->n_kernel_launches++; ctx->n_transport_launches++;
  }
  if (launches > 0) {
    float ms = 0.0f;
    AVM_CUDA(cudaEventElapsedTime(&ms, ctx->ev_t0, ctx->ev_t1));
    ctx->transport_ms += ms;
  }
  const uint64_t total = c >> 32;
  const uint32_t n_end = (uint32_t)(total < (uint64_t)a.cap ? total : (uint64_t)a.cap);
  // a-12: tallies from the endpoints
  const bool want_sums = o->tallies_f64 != nullptr;
  if ((o->per_avalanche || want_sums || o->tallies_u64) && n_end > 0) {
    unsigned blocks = (n_end + 255u) / 256u;
    const unsigned maxb = (unsigned)ctx->sm_count * 8u;
    if (blocks > maxb) blocks = maxb;
    AVM_CUDA(launch(ctx, finalize_kernel, dim3(blocks), dim3(256), a, ctl, n_end, (unsigned long long*)o->per_avalanche, (uint32_t)np, want_sums));
  }
  if (o->per_avalanche || o->tallies_u64 || o->tallies_f64) {
    const unsigned blocks = (unsigned)((np > 0 ? np : 1) + 255) / 256;
    AVM_CUDA(launch(ctx, publish_kernel, dim3(blocks), dim3(256), (const RunCtl*)ctl, gas->d.L, (unsigned long long*)o->per_avalanche, (uint32_t)np,
                    (unsigned long long*)o->tallies_u64, o->tallies_f64));
  }
  unsigned int dropped = 0;
  AVM_CUDA(cudaMemcpyAsync(ctx->h_counters + 1, &ctl->dropped, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
  AVM_CUDA(cudaStreamSynchronize(st));
  dropped = *(unsigned int*)(ctx->h_counters + 1);
  *n_out = n_end;
  if (dropped) return fail(AVM_ERR_CAPACITY, "run: capacity exceeded, " + std::to_string(dropped) + " secondaries dropped");
  return AVM_OK;
}

int32_t avm_ion_drift(avm_ctx* ctx, const avm_field* field, const avm_signal* signal, const avm_ion_opts* io, const avm_outputs* run,
                      int64_t n, int64_t n_primaries, double* ion_end, int32_t* ion_status, uint32_t* ion_steps) {
  if (!ctx || !field || !io || !run || n < 0 || n_primaries < 0) return fail(AVM_ERR_INVALID_ARG, "ion_drift: null argument");
  if (!(io->step_cm > 0.0) || !(io->mobility_pos > 0.0) || !(io->mobility_neg > 0.0) || io->max_steps < 1) return fail(AVM_ERR_INVALID_ARG, "ion_drift: step, mobilities and max_steps must be positive");
  if (n_primaries > n) return fail(AVM_ERR_INVALID_ARG, "ion_drift: n_primaries exceeds n (n = the endpoint count avm_run returned, primaries included)");
  if (n == 0) return AVM_OK;
  if (n > run->capacity || !run->birth || !run->end || !run->status || !ion_end || !ion_status || !ion_steps) return fail(AVM_ERR_INVALID_ARG, "ion_drift: run outputs (birth, end, status) and the ion arrays are required");
  DevSignal dsig;
  if (!make_signal(signal, dsig)) return AVM_ERR_INVALID_ARG;
  AVM_CUDA(cudaSetDevice(ctx->device));
  RunArrays a;
  a.cap = (uint32_t)run->capacity; a.id = run->id; a.aval = run->avalanche; a.status = run->status; a.nsteps = run->n_steps;
  a.birth = run->birth; a.end = run->end;
  IonOpts o;
  o.mu_pos = io->mobility_pos; o.mu_neg = io->mobility_neg; o.step = io->step_cm; o.t_max = io->t_max; o.max_steps = io->max_steps;
  unsigned blocks = (unsigned)((2 * n + 255) / 256);
  const unsigned maxb = (unsigned)ctx->sm_count * 8u;
  if (blocks > maxb) blocks = maxb;
  if (signal) AVM_CUDA(launch(ctx, ion_drift_kernel<true>, dim3(blocks), dim3(256), field->d, dsig, o, a, (uint32_t)n, (uint32_t)n_primaries, ion_end, ion_status, ion_steps));
  else AVM_CUDA(launch(ctx, ion_drift_kernel<false>, dim3(blocks), dim3(256), field->d, dsig, o, a, (uint32_t)n, (uint32_t)n_primaries, ion_end, ion_status, ion_steps));
  return AVM_OK;
}

int32_t avm_fetch(avm_ctx* ctx, const avm_outputs* dev, int64_t n, int64_t np, int32_t n_levels, const avm_outputs* host) {
  if (!ctx || !dev || !host || n < 0 || n > dev->capacity || n > host->capacity) return fail(AVM_ERR_INVALID_ARG, "fetch: null argument or n beyond a capacity");
  AVM_CUDA(cudaSetDevice(ctx->device));
  cudaStream_t st = ctx->stream;
#define AVM_D2H(dst, src, bytes) AVM_CUDA(cudaMemcpyAsync((dst), (src), (bytes), cudaMemcpyDeviceToHost, st))
  if (n > 0) {
    if (host->id && dev->id) AVM_D2H(host->id, dev->id, sizeof(uint64_t) * n);
    if (host->avalanche && dev->avalanche) AVM_D2H(host->avalanche, dev->avalanche, sizeof(uint32_t) * n);
    if (host->status && dev->status) AVM_D2H(host->status, dev->status, sizeof(int32_t) * n);
    if (host->n_steps && dev->n_steps) AVM_D2H(host->n_steps, dev->n_steps, sizeof(uint32_t) * n);
    if (host->birth && dev->birth)
      AVM_CUDA(cudaMemcpy2DAsync(host->birth, sizeof(double) * host->capacity, dev->birth, sizeof(double) * dev->capacity, sizeof(double) * n, 5, cudaMemcpyDeviceToHost, st));
    if (host->end && dev->end)
      AVM_CUDA(cudaMemcpy2DAsync(host->end, sizeof(double) * host->capacity, dev->end, sizeof(double) * dev->capacity, sizeof(double) * n, 8, cudaMemcpyDeviceToHost, st));
  }
  if (host->per_avalanche && dev->per_avalanche && np > 0) AVM_D2H(host->per_avalanche, dev->per_avalanche, sizeof(uint64_t) * 3 * np);
  if (host->tallies_u64 && dev->tallies_u64 && n_levels > 0) AVM_D2H(host->tallies_u64, dev->tallies_u64, sizeof(uint64_t) * (n_levels + 5));
  if (host->tallies_f64 && dev->tallies_f64) AVM_D2H(host->tallies_f64, dev->tallies_f64, sizeof(double) * 5);
#undef AVM_D2H
  AVM_CUDA(cudaStreamSynchronize(st));
  return AVM_OK;
}

int32_t avm_step_batch_form(avm_ctx* ctx, const avm_gas* gas, const avm_field* field, uint64_t seed, double t_max, int32_t form,
                            int32_t k, int64_t n, const double* in, const uint64_t* id, const uint32_t* n_idx, double* out,
                            int32_t* event, int32_t* status, int32_t* bin, double* child, uint64_t* child_id, uint32_t flags) {
  if (!ctx || !gas || !field || n < 0) return fail(AVM_ERR_INVALID_ARG, "step_batch: null argument");
  if (form < 0 || form > 3) return fail(AVM_ERR_INVALID_ARG, "step_batch: form must be 0, 1, 2 or 3");
  const bool banded = (flags & AVM_RUN_BANDED) != 0;
  if (banded && form != 1 && form != 3) return fail(AVM_ERR_INVALID_ARG, "step_batch: banded rates run in forms 1 and 3 only (the forms a banded run takes)");
  if (form >= 2 && (k < 1 || k > 16 || n % k != 0)) return fail(AVM_ERR_INVALID_ARG, "step_batch: forms 2 and 3 need 1 <= k <= 16 electrons per warp and n a multiple of k");
  if (form == 2 && !field->uniform1) return fail(AVM_ERR_INVALID_ARG, "step_batch: form 2 (time-parallel batch) needs a field of one uniform slab");
  if (n == 0) return AVM_OK;
  if (!in || !id || !n_idx || !out || !event || !status || !bin || !child || !child_id) return fail(AVM_ERR_INVALID_ARG, "step_batch: null array");
  AVM_CUDA(cudaSetDevice(ctx->device));
  const int fk = field->fk;
  const bool b = field->d.has_B != 0;
#define AVM_ARGS gas->d, field->d, seed, t_max, n, in, id, n_idx, out, event, status, bin, child, child_id
#define AVM_BARGS gas->d, field->d, seed, t_max, n, (int)k, in, id, n_idx, out, event, status, bin, child, child_id
  if (form == 2) {
    const dim3 grid((unsigned)((n / k + 3) / 4)), block(128);
    if (b) AVM_CUDA(launch(ctx, step_form_batch_kernel<1, true, 2, false>, grid, block, AVM_BARGS));
    else AVM_CUDA(launch(ctx, step_form_batch_kernel<1, false, 2, false>, grid, block, AVM_BARGS));
  } else if (form == 3) {
    const dim3 grid((unsigned)((n / k + 3) / 4)), block(128);
#define AVM_F3B(FK, B) do { if (banded) AVM_CUDA(launch(ctx, step_form_batch_kernel<FK, B, 3, true>, grid, block, AVM_BARGS)); \
                            else AVM_CUDA(launch(ctx, step_form_batch_kernel<FK, B, 3, false>, grid, block, AVM_BARGS)); } while (0)
#define AVM_F3(FK) do { if (b) AVM_F3B(FK, true); else AVM_F3B(FK, false); } while (0)
    if (fk == 1) AVM_F3(1); else if (fk == 2) AVM_F3(2); else AVM_F3(0);
#undef AVM_F3
#undef AVM_F3B
  } else {
    const dim3 grid((unsigned)((n + 127) / 128)), block(128);
#define AVM_SB(FK, B) do { if (form == 1 && banded) AVM_CUDA(launch(ctx, step_batch_kernel<FK, B, 1, true>, grid, block, AVM_ARGS)); \
                           else if (form == 1) AVM_CUDA(launch(ctx, step_batch_kernel<FK, B, 1, false>, grid, block, AVM_ARGS)); \
                           else AVM_CUDA(launch(ctx, step_batch_kernel<FK, B, 0, false>, grid, block, AVM_ARGS)); } while (0)
#define AVM_SBK(FK) do { if (b) AVM_SB(FK, true); else AVM_SB(FK, false); } while (0)
    if (fk == 1) AVM_SBK(1); else if (fk == 2) AVM_SBK(2); else AVM_SBK(0);
#undef AVM_SBK
#undef AVM_SB
  }
#undef AVM_ARGS
#undef AVM_BARGS
  return AVM_OK;
}

int32_t avm_step_batch(avm_ctx* ctx, const avm_gas* gas, const avm_field* field, uint64_t seed, double t_max, int64_t n,
                       const double* in, const uint64_t* id, const uint32_t* n_idx, double* out, int32_t* event,
                       int32_t* status, int32_t* bin, double* child, uint64_t* child_id) {
  return avm_step_batch_form(ctx, gas, field, seed, t_max, 0, 1, n, in, id, n_idx, out, event, status, bin, child, child_id, 0u);
}

int32_t avm_philox_batch(avm_ctx* ctx, uint64_t seed, int64_t n, const uint64_t* id, const uint32_t* n_idx,
                         const uint32_t* block, uint32_t* words, double* u) {
  if (!ctx || n < 0 || (n > 0 && (!id || !n_idx || !block || !words || !u))) return fail(AVM_ERR_INVALID_ARG, "philox_batch: null argument");
  if (n == 0) return AVM_OK;
  AVM_CUDA(cudaSetDevice(ctx->device));
  AVM_CUDA(launch(ctx, philox_batch_kernel, dim3((unsigned)((n + 255) / 256)), dim3(256), seed, n, id, n_idx, block, words, u));
  return AVM_OK;
}

int32_t avm_gather_probe(avm_ctx* ctx, const void* buf, size_t bytes, int32_t n_blocks, int32_t n_threads, int64_t iters,
                         uint64_t* sink, float* ms_out) {
  if (!ctx || !buf || bytes < 64 || ((uintptr_t)buf & 31u) || n_blocks < 1 || n_threads < 32 || n_threads > 256 || iters < 1 || !sink || !ms_out)
    return fail(AVM_ERR_INVALID_ARG, "gather_probe: bad argument");
  AVM_CUDA(cudaSetDevice(ctx->device));
  cudaEvent_t e0, e1;
  AVM_CUDA(cudaEventCreate(&e0));
  AVM_CUDA(cudaEventCreate(&e1));
  const unsigned long long n_sectors = bytes / 32;
  gather_probe_kernel<<<n_blocks, n_threads, 0, ctx->stream>>>((const uint4*)buf, n_sectors, iters / 8 > 0 ? iters / 8 : 1, (unsigned long long*)sink);   // warm-up
  AVM_CUDA(cudaEventRecord(e0, ctx->stream));
  gather_probe_kernel<<<n_blocks, n_threads, 0, ctx->stream>>>((const uint4*)buf, n_sectors, iters, (unsigned long long*)sink);
  AVM_CUDA(cudaEventRecord(e1, ctx->stream));
  AVM_CUDA(cudaGetLastError());
  AVM_CUDA(cudaEventSynchronize(e1));
  AVM_CUDA(cudaEventElapsedTime(ms_out, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return AVM_OK;
}

int32_t avm_smem_probe(avm_ctx* ctx, int32_t table_bytes, int32_t n_blocks, int32_t n_threads, int64_t iters, uint64_t* sink,
                       float* ms_out) {
  if (!ctx || table_bytes < 64 || table_bytes > (int32_t)kMaxDynSmem || n_blocks < 1 || n_threads < 32 || n_threads > 512 || iters < 1 || !sink || !ms_out)
    return fail(AVM_ERR_INVALID_ARG, "smem_probe: bad argument");
  AVM_CUDA(cudaSetDevice(ctx->device));
  AVM_CUDA(cudaFuncSetAttribute(smem_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, table_bytes));
  cudaEvent_t e0, e1;
  AVM_CUDA(cudaEventCreate(&e0));
  AVM_CUDA(cudaEventCreate(&e1));
  smem_probe_kernel<<<n_blocks, n_threads, table_bytes, ctx->stream>>>(table_bytes / 8, iters / 8 > 0 ? iters / 8 : 1, (unsigned long long*)sink);
  AVM_CUDA(cudaEventRecord(e0, ctx->stream));
  smem_probe_kernel<<<n_blocks, n_threads, table_bytes, ctx->stream>>>(table_bytes / 8, iters, (unsigned long long*)sink);
  AVM_CUDA(cudaEventRecord(e1, ctx->stream));
  AVM_CUDA(cudaGetLastError());
  AVM_CUDA(cudaEventSynchronize(e1));
  AVM_CUDA(cudaEventElapsedTime(ms_out, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return AVM_OK;
}

int32_t avm_fp64_probe(avm_ctx* ctx, int32_t n_blocks, int32_t n_threads, int64_t iters, double* sink, float* ms_out) {
  if (!ctx || n_blocks < 1 || n_threads < 32 || n_threads > 256 || iters < 1 || !sink || !ms_out) return fail(AVM_ERR_INVALID_ARG, "fp64_probe: bad argument");
  AVM_CUDA(cudaSetDevice(ctx->device));
  cudaEvent_t e0, e1;
  AVM_CUDA(cudaEventCreate(&e0));
  AVM_CUDA(cudaEventCreate(&e1));
  fp64_probe_kernel<<<n_blocks, n_threads, 0, ctx->stream>>>(iters / 8 > 0 ? iters / 8 : 1, sink);   // warm-up
  AVM_CUDA(cudaEventRecord(e0, ctx->stream));
  fp64_probe_kernel<<<n_blocks, n_threads, 0, ctx->stream>>>(iters, sink);
  AVM_CUDA(cudaEventRecord(e1, ctx->stream));
  AVM_CUDA(cudaGetLastError());
  AVM_CUDA(cudaEventSynchronize(e1));
  AVM_CUDA(cudaEventElapsedTime(ms_out, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return AVM_OK;
}

}  // extern "C"

// ---- avm_run_static: avm_run on the library's own scratch block (include/avm.h) -----------------------------------------
// For callers that may not allocate device memory (plug-ins given their buffers by a host framework, services with a pool
// frozen at start-up): the workspace avm_run asks for — run-control block of the persistent transport kernel + staging
// area of the primaries — lives in the array below instead of a caller buffer.  It is part of the library image, so every
// GPU that loads libavm holds these bytes until the process exits.
namespace {
constexpr int64_t kStaticMaxCapacity = AVM_RUN_STATIC_MAX_CAPACITY;
constexpr size_t kStaticWsBytes = kCtlBytes + (size_t)kStaticMaxCapacity * 8 * sizeof(double);   // 36 KiB + 4 MiB
static_assert(kStaticMaxCapacity <= kStageElectrons, "the staging part is sized per electron only up to kStageElectrons");
static __device__ __align__(256) unsigned char g_static_ws[kStaticWsBytes];

// In host code `g_static_ws` is only a handle for the runtime, not memory a kernel can use: the device address has to be
// asked for, once per device, with that device current.  Device code could name the array directly; the kernels here get
// it as the `ctl` / `stage` pointers avm_run derives from the workspace, so only the host needs the address.
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ws_addr[kStaticMaxDevices] = {};   // guarded by g_static_mu
}  // namespace

extern "C" {

size_t avm_run_static_bytes(void) { return kStaticWsBytes; }

int32_t avm_run_static(avm_ctx* ctx, const avm_gas* gas, const avm_field* field, const double* primaries, int64_t np,
                       const avm_run_opts* opts, const avm_outputs* o, int64_t* n_out) {
  if (!ctx || !gas || !field || !opts || !o || !n_out) return fail(AVM_ERR_INVALID_ARG, "run_static: null argument");
  *n_out = 0;
  if (o->capacity > kStaticMaxCapacity)
    return fail(AVM_ERR_INVALID_ARG, "run_static: capacity " + std::to_string(o->capacity) + " exceeds AVM_RUN_STATIC_MAX_CAPACITY (" +
                                     std::to_string(kStaticMaxCapacity) + " electrons, the size of the built-in scratch block); use avm_run with a caller-provided workspace");
  if (ctx->device < 0 || ctx->device >= kStaticMaxDevices) return fail(AVM_ERR_INVALID_ARG, "run_static: device ordinal beyond the 64 this entry point keeps an address for");
  AVM_CUDA(cudaSetDevice(ctx->device));
  void* ws = nullptr;
  {
    // First call on this device: resolve the array's address there (not inside a stream capture — see avm.h).
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ws_addr[ctx->device]) {
      void* p = nullptr;
      AVM_CUDA(cudaGetSymbolAddress(&p, g_static_ws));
      if (!p || ((uintptr_t)p & 255u)) return fail(AVM_ERR_CUDA, "run_static: the scratch block has no usable device address");
      g_static_ws_addr[ctx->device] = p;
    }
    ws = g_static_ws_addr[ctx->device];
  }
  // The block still holds the previous call's counters, flags and staged primaries.  avm_run zeroes the run-control part
  // on the stream before its first kernel and writes the staging part before reading it, so nothing else is cleared here.
  avm_outputs w = *o;
  w.workspace = ws;
  w.workspace_bytes = kStaticWsBytes;
  return avm_run(ctx, gas, field, primaries, np, opts, &w, n_out);
}

}  // extern "C"
