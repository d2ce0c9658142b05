// avm_device.cuh — device-side arithmetic of one transport step (S0-S9) for sm_100a.
// Shared by the persistent transport kernel and the avm_step_batch parity hook, so the hook tests the
// same code the run executes.  Shares nothing with oracle/ (the oracle has its own Philox, field and step).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/avm.h"

// -DAVM_DEBUG (python -m paper_2509_15377_b200.build -DAVM_DEBUG -> libavm_debug.so): every table, map, slot, ticket and
// exchange-area index of the device code is range-checked and the kernel traps on a violation; compute-sanitizer is not
// available on the GPU pool, so the edge-case and relaunch tests are run once per round against this build.
#ifdef AVM_DEBUG
#include <cstdio>
#define AVM_CHECK(cond)                                                              \
  do {                                                                               \
    if (!(cond)) { printf("AVM_CHECK failed: %s (%s:%d)\n", #cond, __FILE__, __LINE__); __trap(); } \
  } while (0)
#else
#define AVM_CHECK(cond) do { } while (0)
#endif

namespace avm {

// ---- constants (DESIGN.md §3 "Constants"; CODATA-2018 c = 29.9792458 cm/ns, mc^2 = 510998.95 eV) ------------
constexpr double kC2 = 0.05930969584745753;        // speed [cm/ns] = kC2 * sqrt(energy [eV])
constexpr double kInvC2Sq = 284.28150518042008;    // energy = |v|^2 * kInvC2Sq
constexpr double kKappa = 0.0017588200107589609;   // a = -kKappa * E  [cm/ns^2 per V/cm]
constexpr double kOmega1 = 175.88200107589608;     // rad/ns/T
constexpr double kExBUnit = 1.0e-5;                // v_d [cm/ns] = 1e-5 (E x B)/|B|^2
constexpr double kEpsFloor = 1.0e-10;              // eV
constexpr uint32_t kBlockChildId = 0xFFFFFFFFu;
constexpr uint32_t kStepLimit = 0xFFFFFFF0u;

// ---- device-resident descriptions (passed by value as __grid_constant__ kernel parameters) -------------
struct DevGas {
  int nb, L;
  int Lp;                 // row stride of `cum`: L rounded up to an even count, pad entries = +inf
  int bin_floor;          // (int)(eps_floor * inv_de): the bin of the energy floor (0 for any sensible table)
  double inv_de, nu_hat, inv_nu_hat;
  const double* nu_tot;   // [nb]      total real-collision rate per bin (= cum[b][L-1])
  const double2* head;    // [nb][2]   exact decision record, 32 B: (nu_tot, cum[b][0]), (cum[b][min(1,L-1)], 0)
  const ushort4* tab;     // [nb]      16-bit thresholds floor(c 2^16), c = (nu_tot, cum0, cum1)/nu_hat: the filter of decide()
  const double* cum;      // [nb][Lp]  cumulative rates, row-major by bin, rows 16-byte aligned
  const double* loss;     // [L]
  const double* recoil;   // [L]
  const double* w;        // [L]
  const uint8_t* type;    // [L]
  // NEXT-1, energy-banded null-collision rate: per acceleration class j and energy band k (2^bshift bins)
  // the rate nu that bounds the total rate wherever a flight from that band can end within dtmax.
  int bshift, bK, bJ;
  double a0sq, inv_a0sq;  // squared edge of class 0, (kappa 250 V/cm)^2; the edge of class j is a0sq 2^j
  const double2* band;    // [bJ + 1][bK][2]: (1 / nu, dtmax), (nu, floor(nu / nu_hat 2^32) as the low word's bits)
  // NEXT-3: X1 forward-scattering table, X2 Penning parameters per level, X3 gas temperature
  const double* xi;       // [nb][L] or null (isotropic)
  const double* pen_p;    // [AVM_MAX_LEVELS] transfer probability (0 where none)
  const double* pen_e;    // [AVM_MAX_LEVELS] energy available to the Penning electron
  double kT;              // 0 = cold gas
  int ext;                // bit 0: xi given, bit 1: kT > 0, bit 2: some level has a Penning probability.  Non-zero: collisions
                          // go through collision_step_ext (kept out of line, so that the base model's register budget is
                          // untouched) and the speculative elastic collision of the time-parallel batches is off
};

struct DevSlab {
  double z_lo, z_hi;
  double E[3];
  double org[3], inv_h[3], span[2];   // span = (n-1)*h in x, y for bc none, +inf otherwise
  // fold per axis, one branch-free formula for the three boundary conditions (fold_axis):
  double P[2], inv_P[2];              // fold period (periodic: P; mirror: 2P; none: 1) and its inverse (none: 0)
  double Pc[2], lo[2];                // rounding guard q >= Pc || q < lo -> 0 (none: +inf, -inf; else P, 0)
  double half[2];                     // mirror: P (reflect when q > half); else +inf
  const float4* nodes;
  const double* nodes64;              // optional widened copy [nz][ny][nx][4] (same values as doubles): no conversions per lookup
  int kind, nx, ny, nz, bc[2];
  // kind 2 (NEXT-2): unstructured map of 10-node tetrahedra.  tet_rec[e] = 24 doubles: vertex 3 (3), the
  // rows G_a of the inverse edge matrix, lambda_a = G_a . (r - p3), a = 0..2 (9), the ten node potentials (10), gas flag, pad.
  // Bucket grid over the mesh's bounding box: tet_off[cell] .. tet_off[cell + 1] index tet_list (ascending element numbers).
  const double* tet_rec;
  const int* tet_off;
  const int* tet_list;
  double tlo[3], tinv[3];
  int tn[3], n_tets;
};

struct DevField {
  DevSlab slab[AVM_MAX_SLABS];
  int n_slabs;
  int has_B;
  double z_lo, z_hi;
  double xy_lo[2], xy_hi[2];
  double B[3], bh[3], Bn2, omega, inv_omega;
  // one uniform slab (configs 1-3): constants of the flight, computed once by avm_field_create
  double ua[3];     // a = -kappa E
  double uvd[3];    // E x B drift velocity
  double uap[3];    // (a . b) b
  int xy_bounded;   // any of xy_lo / xy_hi finite
};

// Philox round keys of the run's seed: k0 + r 0x9E3779B9, k1 + r 0xBB67AE85, r = 0..9.  Passed as a kernel parameter so
// that they enter the rounds' LOP3 as constant-bank operands.
struct PhiloxKeys { uint32_t k0[10], k1[10]; };

__host__ __device__ inline PhiloxKeys philox_keys(uint64_t seed) {
  PhiloxKeys K;
  uint32_t a = (uint32_t)seed, b = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) { K.k0[r] = a; K.k1[r] = b; a += 0x9E3779B9u; b += 0xBB67AE85u; }
  return K;
}

// ---- Philox4x32-10 (Salmon et al., SC'11) — DESIGN.md §3 "Uniforms" --------------------------------------
struct U4 { uint32_t w0, w1, w2, w3; };

__device__ __forceinline__ U4 philox(const PhiloxKeys& K, uint64_t id, uint32_t n, uint32_t block) {
  uint32_t c0 = n, c1 = block, c2 = (uint32_t)id, c3 = (uint32_t)(id >> 32);
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ K.k0[r]; c1 = lo1; c2 = hi0 ^ c3 ^ K.k1[r]; c3 = lo0;
  }
  return U4{c0, c1, c2, c3};
}

// u = ((x >> 12) + 0.5) * 2^-52 with x = hi:lo — strictly inside (0,1), exactly representable.
__device__ __forceinline__ double to_unit(uint32_t hi, uint32_t lo) {
  // Build the double 1.m directly: mantissa = top 52 bits of x, value 1 + k 2^-52 in [1,2); subtracting 1 - 2^-53
  // gives (2k + 1) 2^-53, which has at most 53 significant bits: the subtraction is exact.
  const uint32_t mh = hi >> 12, ml = (hi << 20) | (lo >> 12);
  const double one_m = __hiloint2double((int)(0x3FF00000u | mh), (int)ml);
  return one_m - 0.99999999999999988898;                                     // 1 - 2^-53
}

// ---- elementary functions specialised to this path's argument ranges ------------------------------------------
// Coefficients live in constant memory so that they enter DFMA as constant-bank operands (an fp64 immediate costs
// two UMOVs).  Accuracy: a few ulp, far inside the 1e-12 parity tolerance.
// log1p(r) = r + r^2 (kLog1pC[0] + kLog1pC[1] r + ...), |r| < 2^-7: the first dropped term is r^9/9 < 2e-18 |r|
static __constant__ double kLog1pC[7] = {-1.0 / 2.0, 1.0 / 3.0, -1.0 / 4.0, 1.0 / 5.0, -1.0 / 6.0, 1.0 / 7.0, -1.0 / 8.0};
// (rc, L) per 1/128 of the mantissa range — see gen_logtab.py.  Kernels stage it in shared memory.
struct LogEntry { unsigned long long rc, L; };
static __device__ const LogEntry kLogTab[128] = {
#include "avm_logtab.inc"
};
// sin(r pi/2) = r sum_k kSinC[k] r^2k, cos(r pi/2) = sum_k kCosC[k] r^2k (Taylor; |r| <= 1/2: truncation < 5e-17)
static __constant__ double kSinC[8] = {1.5707963267948966, -0.6459640975062463, 0.07969262624616705, -0.004681754135318688,
                                0.00016044118478735983, -3.598843235212085e-06, 5.692172921967927e-08,
                                -6.688035109811468e-10};
static __constant__ double kCosC[9] = {1.0, -1.2337005501361697, 0.25366950790104803, -0.02086348076335296,
                                0.0009192602748394266, -2.5202042373060607e-05, 4.710874778818172e-07,
                                -6.386603083791852e-09, 6.565963114979473e-11};

// 1/d for normal d well inside the exponent range (MUFU.RCP64H seed, cubic Newton step): ~1 ulp.
__device__ __forceinline__ double rcp_fast(double d) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
  double e = fma(-d, r, 1.0);
  e = fma(e, e, e);
  return fma(r, e, r);
}

// log(u) for u strictly inside (0, 1) and normal (the uniforms of to_unit are >= 2^-53): no special cases.
// u = m 2^e, m in [1,2); i = top 7 mantissa bits; reduced argument m' = m (i < 53) or m/2 (e bumped) in [0.707, 1.414);
// r = m' rc' - 1 by one fma (|r| < 2^-7); log u = e' ln2 + L_i + log1p(r).  ~1 ulp, full relative accuracy as u -> 1.
// `tab` = kLogTab or its shared-memory copy.
__device__ __forceinline__ double log_unit(double u, const double2* __restrict__ tab) {
  const int hi = __double2hiint(u), lo = __double2loint(u);
  const int e = ((hi + 0x96000) >> 20) - 1023;          // mantissa >= 53/128 carries into the exponent
  const double m = __hiloint2double((hi & 0x000FFFFF) | 0x3FF00000, lo);
  const double2 en = tab[(hi >> 13) & 127];
  const double r = fma(m, en.x, -1.0);
  double p = kLog1pC[6];
#pragma unroll
  for (int k = 5; k >= 0; --k) p = fma(p, r, kLog1pC[k]);
  const double de = (double)e;
  const double l1 = fma(r * r, p, r);
  return fma(de, 0.693147180369123816490, fma(de, 1.90821492927058770002e-10, en.y + l1));
}

// (sin, cos)(2 pi u) for u in [0, 1]: quadrant q = rint(4u), r = 4u - q in [-1/2, 1/2] (exact).
__device__ __forceinline__ void sincos_2pi(double u, double& s, double& c) {
  const double a = 4.0 * u;
  const int q = __double2int_rn(a);
  const double r = a - (double)q;
  const double w = r * r;
  double ps = kSinC[7], pc = kCosC[8];
#pragma unroll
  for (int k = 6; k >= 0; --k) ps = fma(ps, w, kSinC[k]);
#pragma unroll
  for (int k = 7; k >= 0; --k) pc = fma(pc, w, kCosC[k]);
  ps *= r;
  const double ss = (q & 1) ? pc : ps, cc = (q & 1) ? ps : pc;
  s = (q & 2) ? -ss : ss;
  c = ((q + 1) & 2) ? -cc : cc;
}

// (sin, cos)(a) for the half rotation angle of a helical flight: |a| <= pi/4 (the common case: omega dt / 2 ~ 1e-2)
// through the same polynomials, anything larger through the library routine.
__device__ __forceinline__ void sincos_half_angle(double a, double& s, double& c) {
  const double r = a * 0.63661977236758134308;      // a / (pi/2)
  if (fabs(r) <= 0.5) {
    const double w = r * r;
    double ps = kSinC[7], pc = kCosC[8];
#pragma unroll
    for (int k = 6; k >= 0; --k) ps = fma(ps, w, kSinC[k]);
#pragma unroll
    for (int k = 7; k >= 0; --k) pc = fma(pc, w, kCosC[k]);
    s = ps * r; c = pc;
  } else {
    sincos(a, &s, &c);
  }
}

// ---- field (S0, R14, R15) -------------------------------------------------------------------------------
__device__ __forceinline__ double f2d(float v) { return (double)v; }

// Fold coordinate `q = x - org` of axis ax into the stored cell (R15).  Returns false when outside with bc none.
// Branch-free: the three boundary conditions differ only in the slab's constants (none: P = 1, inv_P = 0, no guard, no
// reflection, span = grid extent; periodic / mirror: span = +inf).
__device__ __forceinline__ bool fold_axis(const DevSlab& s, int ax, double x, double& q, bool& flip) {
  const double q0 = x - s.org[ax];
  const double P = s.P[ax];
  double qq = q0 - P * floor(q0 * s.inv_P[ax]);
  qq = (qq >= s.Pc[ax] || qq < s.lo[ax]) ? 0.0 : qq;
  flip = qq > s.half[ax];
  q = flip ? P - qq : qq;
  return (q >= 0.0) & (q <= s.span[ax]);
}

__device__ __forceinline__ void cell_of(double s, int n, int& i, double& w) {
  i = (int)floor(s);
  i = min(i, n - 2);
  i = max(i, 0);
  w = s - (double)i;
}

__device__ __forceinline__ double lerp3(double c000, double c100, double c010, double c110, double c001,
                                        double c101, double c011, double c111, double wx, double wy, double wz) {
  const double c00 = c000 + wx * (c100 - c000);
  const double c10 = c010 + wx * (c110 - c010);
  const double c01 = c001 + wx * (c101 - c001);
  const double c11 = c011 + wx * (c111 - c011);
  const double c0 = c00 + wy * (c10 - c00);
  const double c1 = c01 + wy * (c11 - c01);
  return c0 + wz * (c1 - c0);
}

// Grid lookup inside slab s (z already known to lie in the slab).  Returns false when x/y leave a bc-none grid.
// Nodes come from the widened fp64 copy of the map when the caller gave one (avm_slab.nodes_f64_dev): two 16-byte loads
// per node and no float-to-double conversions (32 per lookup otherwise, 8 cycles of the conversion pipe each); the values
// are the same doubles either way.
__device__ __forceinline__ bool grid_at(const DevSlab& s, double x, double y, double z, double& Ex, double& Ey,
                                        double& Ez, double& mask) {
  double qx, qy;
  bool fx, fy;
  const bool okx = fold_axis(s, 0, x, qx, fx);
  const bool oky = fold_axis(s, 1, y, qy, fy);      // outside a bc-none grid: the cell index is clamped, the result unused
  int i, j, k;
  double wx, wy, wz;
  cell_of(qx * s.inv_h[0], s.nx, i, wx);
  cell_of(qy * s.inv_h[1], s.ny, j, wy);
  cell_of((z - s.org[2]) * s.inv_h[2], s.nz, k, wz);
  const size_t sy = (size_t)s.nx, sz = (size_t)s.nx * s.ny;
  const size_t o = ((size_t)k * s.ny + j) * s.nx + i;
  AVM_CHECK(i >= 0 && j >= 0 && k >= 0 && o + sz + sy + 1 < (size_t)s.nx * s.ny * s.nz);
  double ex, ey;
  if (s.nodes64) {
    const double2* p = reinterpret_cast<const double2*>(s.nodes64) + 2 * o;
    const double2 a000 = __ldg(p), b000 = __ldg(p + 1), a100 = __ldg(p + 2), b100 = __ldg(p + 3);
    const double2 a010 = __ldg(p + 2 * sy), b010 = __ldg(p + 2 * sy + 1), a110 = __ldg(p + 2 * sy + 2), b110 = __ldg(p + 2 * sy + 3);
    const double2 a001 = __ldg(p + 2 * sz), b001 = __ldg(p + 2 * sz + 1), a101 = __ldg(p + 2 * sz + 2), b101 = __ldg(p + 2 * sz + 3);
    const double2 a011 = __ldg(p + 2 * (sz + sy)), b011 = __ldg(p + 2 * (sz + sy) + 1), a111 = __ldg(p + 2 * (sz + sy) + 2),
                  b111 = __ldg(p + 2 * (sz + sy) + 3);
    ex = lerp3(a000.x, a100.x, a010.x, a110.x, a001.x, a101.x, a011.x, a111.x, wx, wy, wz);
    ey = lerp3(a000.y, a100.y, a010.y, a110.y, a001.y, a101.y, a011.y, a111.y, wx, wy, wz);
    Ez = lerp3(b000.x, b100.x, b010.x, b110.x, b001.x, b101.x, b011.x, b111.x, wx, wy, wz);
    mask = lerp3(b000.y, b100.y, b010.y, b110.y, b001.y, b101.y, b011.y, b111.y, wx, wy, wz);
  } else {
    const float4* p = s.nodes + o;
    const float4 n000 = __ldg(p), n100 = __ldg(p + 1);
    const float4 n010 = __ldg(p + sy), n110 = __ldg(p + sy + 1);
    const float4 n001 = __ldg(p + sz), n101 = __ldg(p + sz + 1);
    const float4 n011 = __ldg(p + sz + sy), n111 = __ldg(p + sz + sy + 1);
    ex = lerp3(f2d(n000.x), f2d(n100.x), f2d(n010.x), f2d(n110.x), f2d(n001.x), f2d(n101.x), f2d(n011.x), f2d(n111.x), wx, wy, wz);
    ey = lerp3(f2d(n000.y), f2d(n100.y), f2d(n010.y), f2d(n110.y), f2d(n001.y), f2d(n101.y), f2d(n011.y), f2d(n111.y), wx, wy, wz);
    Ez = lerp3(f2d(n000.z), f2d(n100.z), f2d(n010.z), f2d(n110.z), f2d(n001.z), f2d(n101.z), f2d(n011.z), f2d(n111.z), wx, wy, wz);
    mask = lerp3(f2d(n000.w), f2d(n100.w), f2d(n010.w), f2d(n110.w), f2d(n001.w), f2d(n101.w), f2d(n011.w), f2d(n111.w), wx, wy, wz);
  }
  Ex = fx ? -ex : ex;
  Ey = fy ? -ey : ey;
  return okx & oky;
}

// ---- NEXT-2: 10-node tetrahedra (F1-F2) -------------------------------------------------------------
// Element e at r (coordinates relative to the slab's origin): false when r is not inside (some barycentric < tol); else the
// field E = -grad V from the quadratic shape functions (N_vertex = l(2l - 1), N_edge = 4 l_a l_b) and the element's flag.
// OWN_MARGIN: `tol` is ignored and the element's own shortcut margin (record word 23, written by mesh_image) is used.
template <bool OWN_MARGIN = false>
__device__ __forceinline__ bool tet_try(const DevSlab& s, int e, double tol, double x, double y, double z, double& Ex, double& Ey,
                                        double& Ez, double& mask) {
  const double2* p = reinterpret_cast<const double2*>(s.tet_rec + 24 * (size_t)e);
  if (OWN_MARGIN) tol = __ldg(p + 11).y;
  const double2 a0 = __ldg(p), a1 = __ldg(p + 1), a2 = __ldg(p + 2), a3 = __ldg(p + 3), a4 = __ldg(p + 4), a5 = __ldg(p + 5);
  const double qx = x - a0.x, qy = y - a0.y, qz = z - a1.x;
  const double g0x = a1.y, g0y = a2.x, g0z = a2.y, g1x = a3.x, g1y = a3.y, g1z = a4.x, g2x = a4.y, g2y = a5.x, g2z = a5.y;
  const double l0 = g0x * qx + g0y * qy + g0z * qz, l1 = g1x * qx + g1y * qy + g1z * qz, l2 = g2x * qx + g2y * qy + g2z * qz;
  const double l3 = 1.0 - l0 - l1 - l2;
  if (!((l0 >= tol) & (l1 >= tol) & (l2 >= tol) & (l3 >= tol))) return false;
  const double2 v01 = __ldg(p + 6), v23 = __ldg(p + 7), m01 = __ldg(p + 8), m23 = __ldg(p + 9), m45 = __ldg(p + 10), fl = __ldg(p + 11);
  const double g3x = -(g0x + g1x + g2x), g3y = -(g0y + g1y + g2y), g3z = -(g0z + g1z + g2z);
  // dV/dlambda_a: vertex terms V_a (4 l_a - 1), edge terms 4 V_ab l_b; edges (0,1) (0,2) (0,3) (1,2) (1,3) (2,3)
  const double d0 = v01.x * (4.0 * l0 - 1.0) + 4.0 * (m01.x * l1 + m01.y * l2 + m23.x * l3);
  const double d1 = v01.y * (4.0 * l1 - 1.0) + 4.0 * (m01.x * l0 + m23.y * l2 + m45.x * l3);
  const double d2 = v23.x * (4.0 * l2 - 1.0) + 4.0 * (m01.y * l0 + m23.y * l1 + m45.y * l3);
  const double d3 = v23.y * (4.0 * l3 - 1.0) + 4.0 * (m23.x * l0 + m45.x * l1 + m45.y * l2);
  Ex = -(d0 * g0x + d1 * g1x + d2 * g2x + d3 * g3x);
  Ey = -(d0 * g0y + d1 * g1y + d2 * g2y + d3 * g3y);
  Ez = -(d0 * g0z + d1 * g1z + d2 * g2z + d3 * g3z);
  mask = fl.x;
  return true;
}
// Field and flag at (x, y, z) of a kind-2 slab (z inside the slab).  The element that contains the point is the lowest-
// numbered one with all barycentrics >= -1e-10 (F2); `cache` (may be null) holds the electron's last element: it is taken
// without a search only when the point is strictly inside it: all barycentrics >= the element's own margin, 1e-9 scaled by
// (largest element extent of the mesh) / (this element's smallest height) — then no other element passes F2's test, however
// strongly the mesh is graded (derivation at mesh_image in avm.cu).
__device__ __forceinline__ void tet_at(const DevSlab& s, double x, double y, double z, int* cache, double& Ex, double& Ey,
                                       double& Ez, double& mask) {
  double qx, qy;
  bool fx, fy;
  fold_axis(s, 0, x, qx, fx);
  fold_axis(s, 1, y, qy, fy);
  const double qz = z - s.org[2];
  double ex = 0.0, ey = 0.0, ez = 0.0, m = 0.0;
  bool found = false;
  // The cached index is a hint and may stem from ANOTHER kind-2 slab of the stack (the electron crossed a slab plane since):
  // strictly inside element e of this slab the answer is e whatever made us try it first, so a foreign hint is harmless —
  // provided it indexes this slab's records at all (slabs differ in n_tets; checked in every build, not only AVM_DEBUG).
  if (cache && *cache >= 0 && *cache < s.n_tets) found = tet_try<true>(s, *cache, 0.0, qx, qy, qz, ex, ey, ez, m);
  if (!found) {
    const double ux = (qx - s.tlo[0]) * s.tinv[0], uy = (qy - s.tlo[1]) * s.tinv[1], uz = (qz - s.tlo[2]) * s.tinv[2];
    int cx = (int)floor(ux), cy = (int)floor(uy), cz = (int)floor(uz);
    if (cx == s.tn[0] && ux <= (double)s.tn[0] * (1.0 + 1e-12)) cx = s.tn[0] - 1;
    if (cy == s.tn[1] && uy <= (double)s.tn[1] * (1.0 + 1e-12)) cy = s.tn[1] - 1;
    if (cz == s.tn[2] && uz <= (double)s.tn[2] * (1.0 + 1e-12)) cz = s.tn[2] - 1;
    if (cx >= 0 && cx < s.tn[0] && cy >= 0 && cy < s.tn[1] && cz >= 0 && cz < s.tn[2]) {
      const size_t cell = ((size_t)cz * s.tn[1] + cy) * s.tn[0] + cx;
      const int q1 = __ldg(s.tet_off + cell + 1);
      for (int q = __ldg(s.tet_off + cell); q < q1; ++q) {
        const int e = __ldg(s.tet_list + q);
        AVM_CHECK(e >= 0 && e < s.n_tets);
        if (tet_try(s, e, -1e-10, qx, qy, qz, ex, ey, ez, m)) { if (cache) *cache = e; found = true; break; }
      }
    }
    if (!found) { ex = 0.0; ey = 0.0; ez = 0.0; m = 0.0; }                      // in no element: solid (an unmeshed electrode)
  }
  Ex = fx ? -ex : ex; Ey = fy ? -ey : ey; Ez = ez; mask = m;
}

// Field and mask at r.  Returns the slab index (>= 0) or -status when r is outside the domain.
// FK = field kind the kernel is compiled for: 1 = the field is one uniform slab (configs 1-3: no dispatch, no loads), 2 = one
// grid slab (config 4: the slab's constants are read at fixed constant-bank offsets instead of through a dynamic slab
// index), 0 = any slab stack (config 5).
// Slow path of the bounds test: which face was crossed (S5 order: z_lo, z_hi, then x/y; NaN coordinates -> 3).
__device__ __forceinline__ int outside_status(const DevField& f, double x, double y, double z) {
  if (z < f.z_lo) return -AVM_LEFT_ZLO;
  if (z > f.z_hi) return -AVM_LEFT_ZHI;
  return -AVM_LEFT_XY;
}

template <int FK>
__device__ __forceinline__ int field_at(const DevField& f, double x, double y, double z, double& Ex, double& Ey,
                                        double& Ez, double& mask, int* tet_cache = nullptr) {
  // written so that NaN coordinates fail the test, like the oracle
  bool in = (z >= f.z_lo) & (z <= f.z_hi);
  if (f.xy_bounded) in = in & (x >= f.xy_lo[0]) & (x <= f.xy_hi[0]) & (y >= f.xy_lo[1]) & (y <= f.xy_hi[1]);
  else in = in & ((x + y) == (x + y));
  if (!in) return outside_status(f, x, y, z);
  if (FK == 1) {
    Ex = f.slab[0].E[0]; Ey = f.slab[0].E[1]; Ez = f.slab[0].E[2]; mask = 1.0;
    return 0;
  }
  int si = 0;
  if (FK == 0) {
    si = f.n_slabs - 1;
    for (int i = f.n_slabs - 2; i >= 0; --i) if (z < f.slab[i].z_hi) si = i;
  }
  const DevSlab& s = f.slab[si];
  if (FK == 0 && s.kind == 0) { Ex = s.E[0]; Ey = s.E[1]; Ez = s.E[2]; mask = 1.0; return si; }
  if (FK == 0 && s.kind == 2) { tet_at(s, x, y, z, tet_cache, Ex, Ey, Ez, mask); return si; }
  if (!grid_at(s, x, y, z, Ex, Ey, Ez, mask)) return -AVM_LEFT_XY;
  return si;
}

// ---- NEXT-4: induced signal (W1-W2) ----------------------------------------------------------------------
// wf = the weighting field E_w [1/cm] of the read-out electrode as a field description (mask and B ignored; E_w = 0 outside
// it).  A step r -> r' of a charge q that starts at time t adds q E_w(at) . (r' - r) to out[floor((t - t0) / dt_bin)].
struct DevSignal {
  DevField wf;
  double t0, inv_dt;
  int n_bins, uniform1;     // uniform1: wf is one uniform slab
  double* out;              // [n_bins]
};
__device__ __forceinline__ void weighting_at(const DevSignal& s, double x, double y, double z, double& wx, double& wy, double& wz) {
  double ex = 0.0, ey = 0.0, ez = 0.0, m;
  const int si = s.uniform1 ? field_at<1>(s.wf, x, y, z, ex, ey, ez, m) : field_at<0>(s.wf, x, y, z, ex, ey, ez, m);
  const bool in = si >= 0;
  wx = in ? ex : 0.0; wy = in ? ey : 0.0; wz = in ? ez : 0.0;
}
// Per-thread accumulator: contributions to one time bin are summed in a register and flushed with one atomicAdd when the
// bin changes (a bin holds ~100 flights) and at the end of the launch.  Any thread may hold any electron's contributions:
// the signal is a plain sum.
struct SigAcc { int bin = -1; double q = 0.0; };
__device__ __forceinline__ void sig_flush(const DevSignal& s, SigAcc& a) {
  if (a.bin >= 0 && a.q != 0.0) atomicAdd(s.out + a.bin, a.q);
  a.q = 0.0;
}
__device__ __forceinline__ void sig_add(const DevSignal& s, SigAcc& a, double dq, double t) {
  const double sb = floor((t - s.t0) * s.inv_dt);
  const int b = (sb >= 0.0 && sb < (double)s.n_bins) ? (int)sb : -1;
  if (b != a.bin) { sig_flush(s, a); a.bin = b; }
  if (b >= 0) a.q += dq;
}

// ---- S2-S3: free flight of duration dt in constant E (and B) from (r, v) ---------------------------------
// UNIFORM1: E is the run constant of slab 0 and the arguments Ex, Ey, Ez are ignored (a, E x B drift and a-parallel
// come precomputed from DevField).
template <int FK, bool HASB>
__device__ __forceinline__ void flight(const DevField& f, double Ex, double Ey, double Ez, double dt, double& x,
                                       double& y, double& z, double& vx, double& vy, double& vz) {
  constexpr bool UNIFORM1 = FK == 1;
  const double ax = UNIFORM1 ? f.ua[0] : -kKappa * Ex, ay = UNIFORM1 ? f.ua[1] : -kKappa * Ey,
               az = UNIFORM1 ? f.ua[2] : -kKappa * Ez;
  if (!HASB) {
    const double h = 0.5 * dt * dt;
    x = (x + vx * dt) + ax * h; y = (y + vy * dt) + ay * h; z = (z + vz * dt) + az * h;
    vx = vx + ax * dt; vy = vy + ay * dt; vz = vz + az * dt;
  } else {
    const double bx = f.bh[0], by = f.bh[1], bz = f.bh[2];
    const double v_b = vx * bx + vy * by + vz * bz;
    double dx_, dy_, dz_, qx, qy, qz;
    if (UNIFORM1) {
      dx_ = f.uvd[0]; dy_ = f.uvd[1]; dz_ = f.uvd[2]; qx = f.uap[0]; qy = f.uap[1]; qz = f.uap[2];
    } else {
      const double a_b = ax * bx + ay * by + az * bz;
      const double sc = kExBUnit / f.Bn2;
      dx_ = sc * (Ey * f.B[2] - Ez * f.B[1]);                  // E x B drift velocity
      dy_ = sc * (Ez * f.B[0] - Ex * f.B[2]);
      dz_ = sc * (Ex * f.B[1] - Ey * f.B[0]);
      qx = a_b * bx; qy = a_b * by; qz = a_b * bz;             // a parallel
    }
    const double px = v_b * bx, py = v_b * by, pz = v_b * bz;  // v parallel
    const double wx = vx - px - dx_, wy = vy - py - dy_, wz = vz - pz - dz_;
    const double cx = by * wz - bz * wy, cy = bz * wx - bx * wz, cz = bx * wy - by * wx;   // b x w0
    const double th = f.omega * dt;
    double sh, ch;
    sincos_half_angle(0.5 * th, sh, ch);
    const double sn = 2.0 * sh * ch, vers = 2.0 * sh * sh, cs = 1.0 - vers;
    const double h = 0.5 * dt * dt, io = f.inv_omega;
    x = x + px * dt + qx * h + dx_ * dt + (wx * sn + cx * vers) * io;
    y = y + py * dt + qy * h + dy_ * dt + (wy * sn + cy * vers) * io;
    z = z + pz * dt + qz * h + dz_ * dt + (wz * sn + cz * vers) * io;
    vx = px + qx * dt + dx_ + wx * cs + cx * sn;
    vy = py + qy * dt + dy_ + wy * cs + cy * sn;
    vz = pz + qz * dt + dz_ + wz * cs + cz * sn;
  }
}

// ---- S9: collision outcome ------------------------------------------------------------------------------
struct Child { double e, u6, u7; };   // secondary: energy and the two uniforms of its isotropic direction

// Level parameters as the kernels keep them in shared memory: two 16-byte loads per collision.
struct __align__(16) LevelPar { double loss, recoil, w; int type, pad; };

__device__ __forceinline__ void stage_levels(const DevGas& g, LevelPar* s_lv) {
  for (int l = threadIdx.x; l < AVM_MAX_LEVELS; l += blockDim.x) {
    const bool in = l < g.L;
    LevelPar p;
    p.loss = in ? g.loss[l] : 0.0; p.recoil = in ? g.recoil[l] : 0.0; p.w = in ? g.w[l] : 1.0;
    p.type = in ? g.type[l] : 0; p.pad = 0;
    s_lv[l] = p;
  }
}

// 1/sqrt(a) for normal a > 0 (MUFU.RSQ64H seed, one third-order step): ~1 ulp.
__device__ __forceinline__ double rsqrt_fast(double a) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
  const double e = fma(-a, y * y, 1.0);
  return fma(fma(e, 0.375, 0.5), y * e, y);
}
// sqrt(a) for normal a > 0: a / sqrt(a) with one correction step.
__device__ __forceinline__ double sqrt_fast(double a) {
  const double y = rsqrt_fast(a);
  const double r = a * y;
  return fma(fma(-r, r, a), 0.5 * y, r);
}
// x with its sign flipped when sbit = 0x80000000 (sbit = 0: unchanged): the product x * (+-1) on the integer pipe.
__device__ __forceinline__ double xor_sign(double x, int sbit) {
  return __hiloint2double(__double2hiint(x) ^ sbit, __double2loint(x));
}

__device__ __forceinline__ void child_direction(double u6, double u7, double& kx, double& ky, double& kz) {
  const double sc = 2.0 * sqrt_fast(u6 * (1.0 - u6));
  double s, c;
  sincos_2pi(u7, s, c);
  kx = sc * c; ky = sc * s; kz = 1.0 - 2.0 * u6;
}

__device__ __forceinline__ uint64_t child_id_of(const PhiloxKeys& K, uint64_t id, uint32_t n_s) {
  const U4 w = philox(K, id, n_s, kBlockChildId);
  return (uint64_t)w.w0 | ((uint64_t)w.w1 << 32);
}

// S9b: the deflection draws of step n_s — block 1 -> (cos theta, sin theta, cos phi, sin phi).  They depend on
// (id, n_s) only, so idle lanes can prepare them ahead of the decision (transport kernel, batches).
struct Deflection { double ct, st, cphi, sphi; };

__device__ __forceinline__ Deflection deflection_draws(const PhiloxKeys& K, uint64_t id, uint32_t n_s) {
  const U4 r1 = philox(K, id, n_s, 1u);
  const double u3 = to_unit(r1.w0, r1.w1), u4 = to_unit(r1.w2, r1.w3);
  Deflection d;
  d.ct = 1.0 - 2.0 * u3;
  d.st = 2.0 * sqrt_fast(u3 * (1.0 - u3));        // u3 (1 - u3) >= 2^-54: normal
  sincos_2pi(u4, d.sphi, d.cphi);
  return d;
}

// S8 for the rare levels: smallest l >= 2 with cum[b][l] > x (x < cum[b][L-1] is known; levels 0 and 1 are decided
// from the head record).  The row is non-decreasing, so l = 2 + #{2 <= j < L-1 : cum[b][j] <= x}: independent loads,
// one memory round trip instead of a dependent scan (rows padded with +inf to an even count: 16-byte loads).
__device__ __forceinline__ int select_level_from2(const DevGas& g, int b, double xr) {
  const double2* row = reinterpret_cast<const double2*>(g.cum + (size_t)b * g.Lp) + 1;   // entries 2, 3, ...
  const int np = (g.Lp - 2) >> 1;
  int l = 2;
#pragma unroll 4
  for (int j = 0; j < np; ++j) {
    const double2 v = __ldg(row + j);
    l += ((v.x <= xr) ? 1 : 0) + ((v.y <= xr) ? 1 : 0);
  }
  return l;
}
// Issued when the decision record says "a level >= 2": the row is in L1 by the time the collision phase scans it.
__device__ __forceinline__ void prefetch_row(const DevGas& g, int b) {
  const char* row = reinterpret_cast<const char*>(g.cum + (size_t)b * g.Lp);
  asm volatile("prefetch.global.L1 [%0];" ::"l"(row + 16));
  asm volatile("prefetch.global.L1 [%0];" ::"l"(row + (size_t)g.Lp * 8 - 8));
}

// ---- one step, split at the null/real decision ----------------------------------------------------------------
// Electron state is kept in velocity form (r, t, v, id, n).  The draws of a flight depend on (id, n) only and are
// prepared ahead of the flight that uses them — by the lane itself one step ahead, or by the idle lanes of its warp a
// whole batch ahead (transport kernel).  u2 travels as its raw Philox words (w2, w3): the decision needs only their
// top 16 bits, the double is built in the rare exact path.
struct Pending { int lsel, bin; double xr; };   // lsel: 0 / 1 = level decided from the head record, 2 = scan the row

// BANDED: dt returns -ln(u1); the flight's rate is known only when the flight starts (band_rate).
template <bool BANDED = false>
__device__ __forceinline__ void draw_flight(const DevGas& g, const PhiloxKeys& K, const double2* __restrict__ logtab,
                                            uint64_t id, uint32_t n, double& dt, uint2& u2w) {
  const U4 r0 = philox(K, id, n, 0u);                                           // S1
  const double ml = -log_unit(to_unit(r0.w0, r0.w1), logtab);
  dt = BANDED ? ml : ml * g.inv_nu_hat;                                         // S2
  u2w = make_uint2(r0.w2, r0.w3);
}

// ---- NEXT-1: the rate of one flight under the energy-banded null-collision method (N5) ---------------
// Acceleration class of the field E: the number of class edges A_j^2 = a0sq 2^j, j = 0 .. J-1, strictly below |kappa E|^2
// (J = above every class).  |kappa E|^2 is formed with the oracle's roundings (no contraction), the class from the exponent
// of a2 / a0sq, corrected by one exact comparison against the neighbouring edge (an edge is a0sq with j added to its exponent).
__device__ __forceinline__ int accel_class(const DevGas& g, double Ex, double Ey, double Ez) {
  const double ax = kKappa * Ex, ay = kKappa * Ey, az = kKappa * Ez;
  const double a2 = __dadd_rn(__dadd_rn(__dmul_rn(ax, ax), __dmul_rn(ay, ay)), __dmul_rn(az, az));
  const int e = ((__double2hiint(a2 * g.inv_a0sq) >> 20) & 0x7FF) - 1023;
  int j = min(max(e + 1, 0), g.bJ);
  const int h0 = __double2hiint(g.a0sq), l0 = __double2loint(g.a0sq);
  const double below = __hiloint2double(h0 + ((j - 1) << 20), l0), at = __hiloint2double(h0 + (j << 20), l0);
  if (j > 0 && !(a2 > below)) --j;
  else if (j < g.bJ && a2 > at) ++j;
  return j;
}
struct BandRate { double inv_nu, dtmax, nu; uint32_t rho; };
// s2 = |v|^2 at the start of the flight; its energy bin (as energy_bin) >> bshift = the band.
__device__ __forceinline__ BandRate band_rate(const DevGas& g, double s2, int jcls) {
  const int braw = __double2int_rz((s2 * kInvC2Sq) * g.inv_de);
  const int b0 = max(min(braw, g.nb - 1), g.bin_floor);
  AVM_CHECK(jcls >= 0 && jcls <= g.bJ && b0 >= 0 && (b0 >> g.bshift) < g.bK);
  const double2* p = g.band + 2 * ((size_t)jcls * g.bK + (b0 >> g.bshift));
  const double2 q0 = __ldg(p), q1 = __ldg(p + 1);
  BandRate r;
  r.inv_nu = q0.x; r.dtmax = q0.y; r.nu = q1.x; r.rho = (uint32_t)__double2loint(q1.y);
  return r;
}
// The flight time of a banded flight from its -ln(u1): cut at dtmax (a cut flight ends in a null collision, N6).
__device__ __forceinline__ double banded_dt(const BandRate& br, double mlog, bool& cut) {
  const double dt = mlog * br.inv_nu;
  cut = dt > br.dtmax;
  return cut ? br.dtmax : dt;
}

// S7 + the common part of S8 for bin b and uniform u2 = to_unit(u2w): -1 = null collision, 0 / 1 = level 0 / 1, 2 = a
// level >= 2 (xr = u2 nu_hat is then set for the row scan).  `rec` = tab[b] holds q = floor(c 2^16) for c = (nu_tot,
// cum0, cum1)/nu_hat; h = floor(u2 2^16) = w2 >> 16 exactly (u2 = ((x >> 12) + 1/2) 2^-52, x = w2:w3).  h >= q + 2 implies
// u2 nu_hat >= cum and h <= q - 2 implies u2 nu_hat < cum with a margin of nu_hat 2^-16, far above the rounding of the
// fp64 product — so the 16-bit filter takes the oracle's decision exactly, and the 2e-4 of the steps that fall inside a
// band are decided from the exact fp64 record.
// The 16-bit filter alone, branch-free: -1 / 0 / 1 / 2 as decide(), or -2 when h lies in a band (exact record needed).
// BANDED: the comparison is u2 nu >= cum with the flight's own rate nu = rho nu_hat, rho <= 1: h = floor(u2 rho 2^16) up to
// [0, 1 + 2^-14) (umulhi of the top words of u2 and rho 2^32), which the +-2 band of the filter still covers.
template <bool BANDED = false>
__device__ __forceinline__ int decide_filter(const ushort4 rec, uint2 u2w, uint32_t rho = 0u) {
  const uint32_t h = BANDED ? (__umulhi(u2w.x, rho) >> 16) : (u2w.x >> 16);
  const uint32_t qt = rec.x, q0 = rec.y, q1 = rec.z;
  const bool null = h >= qt + 2u, l0 = h + 2u <= q0;
  const bool l1 = (h >= q0 + 2u) & (h + 2u <= q1), l2 = (h >= q1 + 2u) & (h + 2u <= qt);
  return null ? -1 : (l0 ? 0 : (l1 ? 1 : (l2 ? 2 : -2)));
}
// The exact decision from the fp64 record (inside a band of the filter).
__device__ __forceinline__ int decide_exact(const DevGas& g, int b, double xr) {
  const double2 h0 = __ldg(g.head + 2 * (size_t)b), h1 = __ldg(g.head + 2 * (size_t)b + 1);
  if (xr >= h0.x) return -1;
  if (xr < h0.y) return 0;
  return xr < h1.x ? 1 : 2;
}
__device__ __forceinline__ int decide(const DevGas& g, const ushort4 rec, int b, uint2 u2w, double& xr) {
  const uint32_t h = u2w.x >> 16;
  const uint32_t qt = rec.x, q0 = rec.y, q1 = rec.z;
  if (h >= qt + 2u) return -1;
  if (h + 2u <= q0) return 0;
  if (h >= q0 + 2u && h + 2u <= q1) return 1;
  xr = to_unit(u2w.x, u2w.y) * g.nu_hat;
  int r = 2;
  if (!(h >= q1 + 2u && h + 2u <= qt)) r = decide_exact(g, b, xr);
  if (r == 2) prefetch_row(g, b);
  return r;
}

// S6.  eps' = max(s2 inv_c2sq, eps_floor) and b = min(nb - 1, (int)(eps' inv_de)); the floor is applied to the bin
// (monotone: (int)(max(e, fl) c) = max((int)(e c), (int)(fl c))), the clamp after a saturating conversion.
__device__ __forceinline__ int energy_bin(const DevGas& g, double s2, bool& overflow) {
  const int braw = __double2int_rz((s2 * kInvC2Sq) * g.inv_de);
  overflow = braw >= g.nb;
  return max(min(braw, g.nb - 1), g.bin_floor);
}

// S5 in one uniform slab: every condition under which the electron goes on, as one predicate; and, when it fails, the
// status in S5's order (z faces, x/y bounds or NaN, time limit, step limit), negated.
__device__ __forceinline__ bool uniform_continues(const DevField& f, double t_max, uint32_t n, double x, double y,
                                                  double z, double t) {
  bool ok = (z >= f.z_lo) & (z <= f.z_hi) & (t <= t_max) & (n < kStepLimit);
  if (f.xy_bounded) ok = ok & (x >= f.xy_lo[0]) & (x <= f.xy_hi[0]) & (y >= f.xy_lo[1]) & (y <= f.xy_hi[1]);
  else ok = ok & ((x + y) == (x + y));
  return ok;
}
__device__ __forceinline__ int uniform_exit_status(const DevField& f, double t_max, double x, double y, double z,
                                                   double t) {
  const bool in = (z >= f.z_lo) & (z <= f.z_hi) & (x >= f.xy_lo[0]) & (x <= f.xy_hi[0]) & (y >= f.xy_lo[1]) &
                  (y <= f.xy_hi[1]);
  if (!in) return outside_status(f, x, y, z);
  return t > t_max ? -AVM_TIME_LIMIT : -AVM_STEP_LIMIT;
}

// S5 at r' (and S0 of the next step: the field there): 0 when the electron goes on — Ex, Ey, Ez then hold the field at
// r' — or -(finishing status).  One uniform slab: one predicate.  Maps: the lookup runs unconditionally (indices are
// clamped, so any r' is safe to look up), every condition joins one predicate, and the status is decoded, in S5's
// order, only when it fails.
template <int FK>
__device__ __forceinline__ int s5_status(const DevField& f, double t_max, uint32_t n, double x, double y, double z,
                                         double t, double& Ex, double& Ey, double& Ez, int* tet_cache = nullptr) {
  if (FK == 1) {
    if (!uniform_continues(f, t_max, n, x, y, z, t)) return uniform_exit_status(f, t_max, x, y, z, t);
    return 0;
  }
  bool inb = (z >= f.z_lo) & (z <= f.z_hi);
  if (f.xy_bounded) inb = inb & (x >= f.xy_lo[0]) & (x <= f.xy_hi[0]) & (y >= f.xy_lo[1]) & (y <= f.xy_hi[1]);
  else inb = inb & ((x + y) == (x + y));
  int si = 0;
  if (FK == 0) {
    si = f.n_slabs - 1;
    for (int i = f.n_slabs - 2; i >= 0; --i) if (z < f.slab[i].z_hi) si = i;
  }
  const DevSlab& s = f.slab[si];
  double nEx, nEy, nEz, mask = 1.0;
  bool fold_ok = true;
  if (FK == 0 && s.kind == 0) { nEx = s.E[0]; nEy = s.E[1]; nEz = s.E[2]; }
  else if (FK == 0 && s.kind == 2) {
    if (inb) tet_at(s, x, y, z, tet_cache, nEx, nEy, nEz, mask);              // a search outside the domain is wasted work
    else { nEx = 0.0; nEy = 0.0; nEz = 0.0; }
  }
  else fold_ok = grid_at(s, x, y, z, nEx, nEy, nEz, mask);
  const bool ok = inb & fold_ok & !(mask < 0.5) & !(t > t_max) & (n < kStepLimit);
  if (!ok) {
    if (!inb) return outside_status(f, x, y, z);
    if (!fold_ok) return -AVM_LEFT_XY;
    if (mask < 0.5) return -AVM_MATERIAL;
    return t > t_max ? -AVM_TIME_LIMIT : -AVM_STEP_LIMIT;
  }
  Ex = nEx; Ey = nEy; Ez = nEz;
  return 0;
}

// S3-S4: the flight itself; t and n advance.  Returns |v'|^2.
template <int FK, bool HASB>
__device__ __forceinline__ double advance_move(const DevField& f, uint32_t& n, double& x, double& y, double& z, double& t,
                                               double& vx, double& vy, double& vz, double Ex, double Ey, double Ez,
                                               double dt) {
  flight<FK, HASB>(f, Ex, Ey, Ez, dt, x, y, z, vx, vy, vz);
  t = t + dt;
  n = n + 1u;
  return vx * vx + vy * vy + vz * vz;
}

// S3-S6 for one electron with this flight's dt.  Returns the energy bin (>= 0) or -(finishing status).
template <int FK, bool HASB>
__device__ __forceinline__ int advance(const DevGas& g, const DevField& f, double t_max, uint32_t& n, double& x,
                                       double& y, double& z, double& t, double& vx, double& vy, double& vz, double& Ex,
                                       double& Ey, double& Ez, double dt, bool& overflow, int* tet_cache = nullptr) {
  const double s2 = advance_move<FK, HASB>(f, n, x, y, z, t, vx, vy, vz, Ex, Ey, Ez, dt);   // S3, S4
  const int st = s5_status<FK>(f, t_max, n, x, y, z, t, Ex, Ey, Ez, tet_cache);             // S5
  if (st < 0) return st;
  return energy_bin(g, s2, overflow);                                                            // S6
}

// S9d in velocity form (see collision_step): v'' = (c2 sqrt(e2) / s) R(v') for |v'|^2 = s2 >= 1e-280.
__device__ __forceinline__ void rotate_scale(const Deflection& d, double s2, double e2, double& vx, double& vy,
                                             double& vz) {
  const double rs = rsqrt_fast(s2), s = s2 * rs;
  const int sb = __double2hiint(vz) & 0x80000000;                              // sg = copysign(1, v'z)
  const double sgs = xor_sign(s, sb);
  const double A = -rcp_fast(sgs + vz);
  const double Bq = vx * vy * A;
  const double b1x = fma(xor_sign(vx * vx, sb), A, s), b1y = xor_sign(Bq, sb), b1z = xor_sign(vx, sb ^ 0x80000000);
  const double b2x = Bq, b2y = fma(vy * vy, A, sgs), b2z = -vy;
  const double rx = fma(d.ct, vx, d.st * fma(d.cphi, b1x, d.sphi * b2x));
  const double ry = fma(d.ct, vy, d.st * fma(d.cphi, b1y, d.sphi * b2y));
  const double rz = fma(d.ct, vz, d.st * fma(d.cphi, b1z, d.sphi * b2z));
  const double ratio = (kC2 * sqrt_fast(e2)) * rs;                             // speed'' / s
  vx = rx * ratio; vy = ry * ratio; vz = rz * ratio;
}

// S9c + S9d of an ELASTIC collision with recoil factor r_l from the post-flight velocity (s2 = |v'|^2 >= 1e-280).
// Returns the energy loss.  Branch-free: the time-parallel batches evaluate it for every step ahead of the decision.
__device__ __forceinline__ double elastic_collision(double recoil, const Deflection& d, double s2, double& vx, double& vy,
                                                    double& vz) {
  double e1 = s2 * kInvC2Sq;
  e1 = e1 < kEpsFloor ? kEpsFloor : e1;
  const double e2 = e1 * (1.0 - recoil * (1.0 - d.ct));
  rotate_scale(d, s2, e2, vx, vy, vz);
  return e1 - e2;
}

// S8-S9 for an electron with a pending real collision (n already incremented by the flight).  Returns the level;
// status = AVM_ATTACHED for an attachment, else 0 and v is the velocity after the collision.  d = deflection_draws of
// step n - 1 when `have_d`, else drawn here.
// S9d in velocity form: with s = |v'|, sg = sign(v'z), A = -1/(sg s + v'z), the Duff et al. basis about k' = v'/s scaled
// by s is  s e1 = (s + sg v'x^2 A, sg v'x v'y A, -sg v'x),  s e2 = (v'x v'y A, sg s + v'y^2 A, -v'y),  so that
// v'' = (speed''/s) [cos(theta) v' + sin(theta) (cos(phi) s e1 + sin(phi) s e2)] without normalising k' first.
//
// NEXT-3: with any extension on (g.ext != 0) the whole collision is computed by collision_step_ext, a
// __noinline__ function that takes and returns everything by value — the base model's code below stays what it was.
struct CollisionOut { double vx, vy, vz, loss, che, chu6, chu7; int l, status, spawn; };

static __device__ __noinline__ CollisionOut collision_step_ext(const DevGas& g, const LevelPar* __restrict__ lv, const PhiloxKeys& K,
                                                        uint64_t id, uint32_t n, int lsel, int bin, double xr, bool have_d,
                                                        Deflection d, double vx, double vy, double vz) {
  CollisionOut o;
  o.l = lsel < 2 ? lsel : select_level_from2(g, bin, xr);                     // S8
  AVM_CHECK(o.l >= 0 && o.l < g.L && bin >= 0 && bin < g.nb);
  const int l = o.l;
  const LevelPar par = lv[l];
  o.status = 0; o.spawn = 0; o.loss = 0.0; o.che = 0.0; o.chu6 = 0.5; o.chu7 = 0.0;
  o.vx = vx; o.vy = vy; o.vz = vz;
  if (par.type == AVM_ATTACHMENT) { o.status = AVM_ATTACHED; return o; }       // S9a
  if (!have_d) d = deflection_draws(K, id, n - 1u);                            // S9b
  if (g.xi) {                                     // X1: cos(theta) = (c0 + xi) / (1 + xi c0), sin(theta) cancellation-free
    const double xi = __ldg(g.xi + (size_t)bin * g.L + l);
    const double den = 1.0 + xi * d.ct;
    d.st = d.st * sqrt(1.0 - xi * xi) / den;
    d.ct = (d.ct + xi) / den;
  }
  double s2 = vx * vx + vy * vy + vz * vz;
  if (!(s2 >= 1e-280)) { vx = 0.0; vy = 0.0; vz = kC2 * 1e-5; s2 = vz * vz; }
  double e1 = s2 * kInvC2Sq;
  if (e1 < kEpsFloor) e1 = kEpsFloor;
  double e2;                                                                    // S9c
  if (par.type == AVM_ELASTIC && g.kT > 0.0 && par.recoil > 0.0) {
    // X3: the atom moves with velocity V (normal components, sigma = c2 sqrt(kT r / 4), Box-Muller from blocks 2 and 3);
    // the cold-gas collision acts on the relative velocity w = v' - V, then V is added back.  Library math.
    const U4 r2 = philox(K, id, n - 1u, 2u);
    const U4 r3 = philox(K, id, n - 1u, 3u);
    const double u5 = to_unit(r2.w0, r2.w1), u6 = to_unit(r2.w2, r2.w3), u7 = to_unit(r3.w0, r3.w1), u8 = to_unit(r3.w2, r3.w3);
    const double sigma = kC2 * sqrt(g.kT * par.recoil * 0.25);
    const double ra = sqrt(-2.0 * log(u5)), rb = sqrt(-2.0 * log(u7));
    double s6, c6, s8, c8;
    sincos_2pi(u6, s6, c6);
    sincos_2pi(u8, s8, c8);
    const double Vx = sigma * ra * c6, Vy = sigma * ra * s6, Vz = sigma * rb * c8;
    double wx = vx - Vx, wy = vy - Vy, wz = vz - Vz;
    double w2 = wx * wx + wy * wy + wz * wz;
    if (!(w2 >= 1e-280)) { wx = 0.0; wy = 0.0; wz = kC2 * 1e-5; w2 = wz * wz; }
    double ew = w2 * kInvC2Sq;
    if (ew < kEpsFloor) ew = kEpsFloor;
    const double e2w = ew * (1.0 - par.recoil * (1.0 - d.ct));
    rotate_scale(d, w2, e2w, wx, wy, wz);
    o.vx = wx + Vx; o.vy = wy + Vy; o.vz = wz + Vz;
    o.loss = e1 - fmax((o.vx * o.vx + o.vy * o.vy + o.vz * o.vz) * kInvC2Sq, kEpsFloor);
    return o;
  }
  if (par.type == AVM_ELASTIC) {
    e2 = e1 * (1.0 - par.recoil * (1.0 - d.ct));
    o.loss = e1 - e2;
  } else if (par.type == AVM_EXCITATION) {
    e2 = e1 - par.loss;
    if (!(e2 > kEpsFloor)) e2 = kEpsFloor;
    o.loss = e1 - e2;
    const double pen_p = __ldg(g.pen_p + l);
    if (pen_p > 0.0) {                            // X2: Penning transfer — one more electron with probability pen_p
      const U4 r2 = philox(K, id, n - 1u, 2u);
      if (to_unit(r2.w0, r2.w1) < pen_p) {
        const U4 r3 = philox(K, id, n - 1u, 3u);
        o.chu6 = to_unit(r2.w2, r2.w3);
        o.chu7 = to_unit(r3.w0, r3.w1);
        o.che = fmax(to_unit(r3.w2, r3.w3) * __ldg(g.pen_e + l), kEpsFloor);
        o.spawn = 1;
      }
    }
  } else {   // ionisation: Opal-Peterson-Beaty sharing (R10)
    const U4 r2 = philox(K, id, n - 1u, 2u);
    const U4 r3 = philox(K, id, n - 1u, 3u);
    const double u5 = to_unit(r2.w0, r2.w1);
    o.chu6 = to_unit(r2.w2, r2.w3);
    o.chu7 = to_unit(r3.w0, r3.w1);
    const double ea = fmax(e1 - par.loss, 0.0);
    const double es = par.w * tan(u5 * atan(ea / (2.0 * par.w)));
    e2 = fmax(ea - es, kEpsFloor);
    o.che = fmax(es, kEpsFloor);
    o.spawn = 1;
    o.loss = e1 - e2 - o.che;
  }
  rotate_scale(d, s2, e2, vx, vy, vz);                                         // S9d
  o.vx = vx; o.vy = vy; o.vz = vz;
  return o;
}

// EXT = the kernel variant that supports the extensions (transport_kernel<.., XTR>; the parity hooks always do): the call
// is compiled only there — even untaken, it costs the base kernels ~180 bytes of spills in the 80-register launch shape
// (config 3s: 414 -> 576 ms).
template <bool EXT = true>
__device__ __forceinline__ int collision_step(const DevGas& g, const LevelPar* __restrict__ lv, const PhiloxKeys& K,
                                              uint64_t id, uint32_t n, const Pending& p, bool have_d, Deflection d,
                                              double& vx, double& vy, double& vz, int& status, bool& spawn, Child& ch,
                                              double& loss) {
  if (EXT && g.ext != 0) {
    const CollisionOut o = collision_step_ext(g, lv, K, id, n, p.lsel, p.bin, p.xr, have_d, d, vx, vy, vz);
    vx = o.vx; vy = o.vy; vz = o.vz; status = o.status; spawn = o.spawn != 0; loss = o.loss;
    ch.e = o.che; ch.u6 = o.chu6; ch.u7 = o.chu7;
    return o.l;
  }
  const int l = p.lsel < 2 ? p.lsel : select_level_from2(g, p.bin, p.xr);     // S8
  AVM_CHECK(l >= 0 && l < g.L && p.bin >= 0 && p.bin < g.nb);
  const LevelPar par = lv[l];
  status = 0; spawn = false; loss = 0.0;
  if (par.type == AVM_ATTACHMENT) { status = AVM_ATTACHED; return l; }         // S9a
  if (!have_d) d = deflection_draws(K, id, n - 1u);                            // S9b
  double s2 = vx * vx + vy * vy + vz * vz;
  if (!(s2 >= 1e-280)) {                          // v' = 0 (never in practice): direction +z, energy at the floor
    vx = 0.0; vy = 0.0; vz = kC2 * 1e-5; s2 = vz * vz;
  }
  double e1 = s2 * kInvC2Sq;
  if (e1 < kEpsFloor) e1 = kEpsFloor;
  double e2;                                                                    // S9c
  if (par.type == AVM_ELASTIC) {
    e2 = e1 * (1.0 - par.recoil * (1.0 - d.ct));
    loss = e1 - e2;
  } else if (par.type == AVM_EXCITATION) {
    e2 = e1 - par.loss;
    if (!(e2 > kEpsFloor)) e2 = kEpsFloor;
    loss = e1 - e2;
  } else {   // ionisation: Opal-Peterson-Beaty sharing (R10)
    const U4 r2 = philox(K, id, n - 1u, 2u);
    const U4 r3 = philox(K, id, n - 1u, 3u);
    const double u5 = to_unit(r2.w0, r2.w1);
    ch.u6 = to_unit(r2.w2, r2.w3);
    ch.u7 = to_unit(r3.w0, r3.w1);
    const double ea = fmax(e1 - par.loss, 0.0);
    const double es = par.w * tan(u5 * atan(ea / (2.0 * par.w)));
    e2 = fmax(ea - es, kEpsFloor);
    ch.e = fmax(es, kEpsFloor);
    spawn = true;
    loss = e1 - e2 - ch.e;
  }
  rotate_scale(d, s2, e2, vx, vy, vz);                                         // S9d
  return l;
}

}  // namespace avm
