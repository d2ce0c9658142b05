// avmo.cpp — ORACLE (test infrastructure; see avmo.h).  Plain serial C++17, fp64, one electron at a time,
// written in the order and notation of SURVEY.md §8(c) steps S0-S9 (restated in DESIGN.md §3).
// Compile: g++ -O2 -ffp-contract=off -std=c++17 -shared -fPIC (no fused multiply-add, no fast-math).
// Shares nothing with paper_2509_15377_b200/csrc/.
#include "avmo.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <memory>
#include <string>
#include <thread>
#include <vector>

namespace {

// ---- constants (SURVEY.md §8(c) "Constants"; CODATA-2018: c = 29.9792458 cm/ns, mc^2 = 510998.95 eV) ----
const double C2 = 0.05930969584745753;        // speed [cm/ns] = C2 * sqrt(energy [eV])
const double INV_C2SQ = 284.28150518042008;   // energy = |v|^2 * INV_C2SQ
const double KAPPA = 0.0017588200107589609;   // acceleration a = -KAPPA * E  [cm/ns^2 per V/cm]
const double OMEGA1 = 175.88200107589608;     // cyclotron angular frequency per tesla [rad/ns/T]
const double EXB_UNIT = 1.0e-5;               // v_d [cm/ns] = 1e-5 (E x B)/|B|^2, E in V/cm, B in T
const double EPS_FLOOR = 1.0e-10;             // eV
const double TWO_PI = 6.283185307179586;
const uint32_t BLOCK_CHILD_ID = 0xFFFFFFFFu;
const uint32_t N_STEP_LIMIT = 0xFFFFFFF0u;

thread_local std::string g_err;

// ---- Philox4x32-10 (Salmon et al., SC'11), SURVEY.md §8(c) "Uniforms" ------------------------------------
void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1) {
  const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = M0 * (uint64_t)c[0];
    uint64_t p1 = M1 * (uint64_t)c[2];
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c[1] ^ k0, n1 = lo1, n2 = hi0 ^ c[3] ^ k1, n3 = lo0;
    c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
    if (round < 9) { k0 += 0x9E3779B9u; k1 += 0xBB67AE85u; }
  }
}

void philox_block(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, uint32_t w[4]) {
  w[0] = n; w[1] = block; w[2] = (uint32_t)id; w[3] = (uint32_t)(id >> 32);
  philox4x32_10(w, (uint32_t)seed, (uint32_t)(seed >> 32));
}

double to_unit(uint32_t hi, uint32_t lo) {           // ((x >> 12) + 0.5) * 2^-52, strictly inside (0,1)
  uint64_t x = ((uint64_t)hi << 32) | (uint64_t)lo;
  return ((double)(x >> 12) + 0.5) * 2.220446049250313e-16;
}

void uniform_pair(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, double& ua, double& ub) {
  uint32_t w[4];
  philox_block(seed, id, n, block, w);
  ua = to_unit(w[0], w[1]);
  ub = to_unit(w[2], w[3]);
}

// ---- data ---------------------------------------------------------------------------------------------
// NEXT-1: the energy-banded null-collision rate, DESIGN.md §3.5 readings N1-N6.  nu[k][j] bounds the
// total collision rate over every energy an electron that starts a flight in energy band k, under an acceleration of
// class j, can reach within dtmax[k][j]; a flight drawn longer than dtmax is cut there and counted as a null collision
// (the exponential is memoryless: thinning with a piecewise-constant majorant is exact).
struct Majorant {
  int shift = 0, K = 0, J = 0;
  std::vector<double> a2;                       // [J]: squared upper edge of acceleration class j
  std::vector<double> nu, inv_nu, dtmax;        // [K][J+1]; column J = accelerations above every class: global rate, no cut
};

struct Gas {
  int nb = 0, L = 0;
  double e_max = 0, inv_de = 0, nu_hat = 0, inv_nu_hat = 0;
  const double* cum = nullptr;
  const uint8_t* type = nullptr;
  const double *loss = nullptr, *recoil = nullptr, *w = nullptr;
  const double *xi = nullptr, *pen_p = nullptr, *pen_e = nullptr;   // NEXT-3: X1, X2
  double kT = 0.0;                                                  // X3
  Majorant M;
};

struct Electron {
  double x, y, z, t, e, kx, ky, kz;
  uint64_t id;
  uint32_t n, aval;
  int32_t status;
  double birth[5];
  bool primary = false;
};

struct Tally {
  std::vector<uint64_t> level;
  uint64_t n_null = 0, n_real = 0, n_overflow = 0, n_steps = 0, n_viol = 0, n_penning = 0;
  double sdx = 0, sdy = 0, sdz = 0, sdt = 0, sloss = 0;
};

// N1-N4: the table of banded rates.  Bands: 2^shift energy bins each, shift the largest with nb >> shift >= 256 (else 0).
// Acceleration classes: upper edges A_j = a0 2^(j/2), a0 = kappa x 250 V/cm, j = 0 .. 24 (250 V/cm .. 1.02 MV/cm).
// For band k (upper energy edge e_hi) and class j: a flight of at most dt = m / nu from an energy <= e_hi ends with speed
// <= c2 sqrt(e_hi) + A_j dt, i.e. (one bin of slack) in an energy bin <= b_r(nu); with P[b] = max of the total rate over
// bins 0 .. b and f(nu) = P[b_r(nu)] (non-increasing in nu), nu1 = f(P[last bin of the band]) satisfies nu1 >= f(nu1): a
// valid bound; it is tightened while f(f(nu)) stays below.  m is the candidate of {1/2, 1, 2, 4, 8, 16} with the fewest
// expected steps per unit time, nu / (1 - exp(-m)).  The last band also holds the energies above the table (R5), which
// only the global maximum bounds.
void build_majorant(Gas& g) {
  Majorant& M = g.M;
  const int nb = g.nb;
  std::vector<double> P(nb);
  double run = 0.0;
  for (int b = 0; b < nb; ++b) { run = std::max(run, g.cum[(size_t)b * g.L + g.L - 1]); P[b] = run; }
  M.shift = 0;
  while ((nb >> (M.shift + 1)) >= 256) ++M.shift;
  M.K = (nb + (1 << M.shift) - 1) >> M.shift;
  M.J = 25;
  const double a0 = KAPPA * 250.0, de = g.e_max / (double)nb;
  M.a2.resize(M.J);
  for (int j = 0; j < M.J; ++j) {
    M.a2[j] = std::ldexp(a0 * a0, j);             // A_j^2 = a0^2 2^j, exact scaling
  }
  const double INF = std::numeric_limits<double>::infinity();
  const double mc[6] = {0.5, 1.0, 2.0, 4.0, 8.0, 16.0};
  M.nu.assign((size_t)M.K * (M.J + 1), 0.0); M.inv_nu = M.nu; M.dtmax = M.nu;
  for (int k = 0; k < M.K; ++k) {
    const int b_hi = std::min((k + 1) << M.shift, nb) - 1;
    const double e_hi = (double)(b_hi + 1) * de;
    for (int j = 0; j <= M.J; ++j) {
      double nu = P[nb - 1], dtm = INF;
      if (k < M.K - 1 && j < M.J) {
        const double A = std::sqrt(M.a2[j]);
        double best = INF;
        for (int c = 0; c < 6; ++c) {
          const double m = mc[c];
          auto f = [&](double v) {
            const double dt = m / v;
            const double sp = C2 * std::sqrt(e_hi) + A * dt;
            const double sb = (sp * sp * INV_C2SQ) * g.inv_de + 1.0;
            return P[sb >= (double)(nb - 1) ? nb - 1 : (int)sb];
          };
          double v = f(P[b_hi]);
          for (int it = 0; it < 4; ++it) {
            const double v2 = f(v);
            if (v2 < v && f(v2) <= v2) v = v2; else break;
          }
          const double cost = v / (1.0 - std::exp(-m));
          if (v > 0.0 && cost <= best) { best = cost; nu = v; dtm = m / v; }
        }
      }
      if (!(nu > 0.0)) { nu = g.nu_hat; dtm = INF; }
      const size_t o = (size_t)k * (M.J + 1) + j;
      M.nu[o] = nu; M.inv_nu[o] = 1.0 / nu; M.dtmax[o] = dtm;
    }
  }
}

bool load_gas(const avmo_gas_desc* d, Gas& g) {
  if (!d || d->n_bins < 1 || d->n_levels < 1 || !(d->e_max_eV > 0) || !d->cum_rate || !d->level_type ||
      !d->level_loss_eV || !d->level_recoil || !d->level_ob_w_eV) { g_err = "gas: null or empty field"; return false; }
  g.nb = d->n_bins; g.L = d->n_levels; g.e_max = d->e_max_eV;
  g.inv_de = (double)g.nb / g.e_max;
  g.cum = d->cum_rate; g.type = d->level_type; g.loss = d->level_loss_eV; g.recoil = d->level_recoil; g.w = d->level_ob_w_eV;
  double mx = 0;
  for (int b = 0; b < g.nb; ++b) {
    double prev = 0;
    for (int l = 0; l < g.L; ++l) {
      double c = g.cum[(size_t)b * g.L + l];
      if (!(c >= prev)) { g_err = "gas: cum_rate decreases along levels"; return false; }
      prev = c;
    }
    mx = std::max(mx, prev);
  }
  for (int l = 0; l < g.L; ++l) if (g.type[l] > 3) { g_err = "gas: bad level type"; return false; }
  g.xi = d->scat_xi; g.pen_p = d->level_penning_prob; g.pen_e = d->level_penning_eV; g.kT = d->kT_eV;
  if (g.xi)
    for (size_t i = 0; i < (size_t)g.nb * g.L; ++i) if (!(g.xi[i] > -1.0 && g.xi[i] < 1.0)) { g_err = "gas: scat_xi outside (-1, 1)"; return false; }
  if ((g.pen_p != nullptr) != (g.pen_e != nullptr)) { g_err = "gas: Penning probability and energy come together"; return false; }
  if (g.pen_p)
    for (int l = 0; l < g.L; ++l) if (!(g.pen_p[l] >= 0.0 && g.pen_p[l] <= 1.0) || !(g.pen_e[l] >= 0.0)) { g_err = "gas: Penning parameters"; return false; }
  if (!(g.kT >= 0.0)) { g_err = "gas: kT < 0"; return false; }
  g.nu_hat = d->nu_hat > 0 ? d->nu_hat : mx;      // R4: one global null-collision rate
  if (!(g.nu_hat > 0) || g.nu_hat < mx) { g_err = "gas: nu_hat must be >= max total rate and > 0"; return false; }
  g.inv_nu_hat = 1.0 / g.nu_hat;
  build_majorant(g);
  return true;
}

bool check_field(const avmo_field_desc* f) {
  if (!f || !f->slabs || f->n_slabs < 1) { g_err = "field: no slabs"; return false; }
  for (int i = 0; i < f->n_slabs; ++i) {
    const avmo_slab& s = f->slabs[i];
    if (!(s.z_hi > s.z_lo)) { g_err = "field: slab z_hi <= z_lo"; return false; }
    if (i > 0 && s.z_lo != f->slabs[i - 1].z_hi) { g_err = "field: slabs not contiguous/ascending"; return false; }
    if (s.kind == 1) {
      if (!s.nodes || s.nx < 2 || s.ny < 2 || s.nz < 2) { g_err = "field: grid needs nodes and >=2 per axis"; return false; }
      for (int a = 0; a < 3; ++a) if (!(s.spacing[a] > 0)) { g_err = "field: spacing"; return false; }
      double ztop = s.origin[2] + (s.nz - 1) * s.spacing[2];
      double tol = 1e-9 * s.spacing[2];
      if (s.z_lo < s.origin[2] - tol || s.z_hi > ztop + tol) { g_err = "field: slab z-range outside its grid"; return false; }
      if (s.bc_x < 0 || s.bc_x > 2 || s.bc_y < 0 || s.bc_y > 2) { g_err = "field: bc"; return false; }
      if (s.bc_x && !(s.period_x > 0 && s.period_x <= (s.nx - 1) * s.spacing[0] * (1 + 1e-12))) { g_err = "field: period_x"; return false; }
      if (s.bc_y && !(s.period_y > 0 && s.period_y <= (s.ny - 1) * s.spacing[1] * (1 + 1e-12))) { g_err = "field: period_y"; return false; }
    } else if (s.kind == 2) {
      if (s.n_tets < 1 || s.n_mesh_nodes < 4 || !s.node_xyz || !s.node_V || !s.tet_nodes || !s.tet_gas) { g_err = "field: mesh arrays"; return false; }
      for (int64_t i = 0; i < s.n_tets * 10; ++i) if (s.tet_nodes[i] < 0 || s.tet_nodes[i] >= s.n_mesh_nodes) { g_err = "field: mesh node index"; return false; }
      if (s.bc_x < 0 || s.bc_x > 2 || s.bc_y < 0 || s.bc_y > 2) { g_err = "field: bc"; return false; }
      if ((s.bc_x && !(s.period_x > 0)) || (s.bc_y && !(s.period_y > 0))) { g_err = "field: period"; return false; }
    } else if (s.kind != 0) { g_err = "field: kind"; return false; }
  }
  return true;
}

// ---- NEXT-2: unstructured tetrahedral maps ----------------------------------------------------------
// F2: the element that contains a point.  Definition: element e contains r when its four barycentric coordinates are all
// >= -1e-10 (interior points belong to exactly one element; on a shared face, the lowest index wins).  Brute force over
// all elements is that definition; the bucket grid below only skips elements whose bounding box cannot contain r, and
// keeps each bucket's candidates in ascending order, so it returns the same element (pinned against brute force).
const double TET_TOL = 1e-10;

// barycentric coordinates of r in the tetrahedron with vertices p[0..3] (Cramer's rule on the edge matrix)
bool barycentric(const double* p0, const double* p1, const double* p2, const double* p3, const double r[3], double lam[4]) {
  const double a[3] = {p0[0] - p3[0], p0[1] - p3[1], p0[2] - p3[2]};
  const double b[3] = {p1[0] - p3[0], p1[1] - p3[1], p1[2] - p3[2]};
  const double c[3] = {p2[0] - p3[0], p2[1] - p3[1], p2[2] - p3[2]};
  const double q[3] = {r[0] - p3[0], r[1] - p3[1], r[2] - p3[2]};
  auto det3 = [](const double* u, const double* v, const double* w) {
    return u[0] * (v[1] * w[2] - v[2] * w[1]) - u[1] * (v[0] * w[2] - v[2] * w[0]) + u[2] * (v[0] * w[1] - v[1] * w[0]);
  };
  const double D = det3(a, b, c);
  if (D == 0.0) return false;
  lam[0] = det3(q, b, c) / D;
  lam[1] = det3(a, q, c) / D;
  lam[2] = det3(a, b, q) / D;
  lam[3] = 1.0 - lam[0] - lam[1] - lam[2];
  return true;
}

struct MeshIndex {
  double lo[3], inv[3];
  int n[3];
  std::vector<int64_t> off;
  std::vector<int32_t> list;
};

std::unique_ptr<MeshIndex> build_mesh_index(const avmo_slab& s) {
  auto M = std::make_unique<MeshIndex>();
  double hi[3];
  for (int a = 0; a < 3; ++a) { M->lo[a] = 1e300; hi[a] = -1e300; }
  for (int64_t e = 0; e < s.n_tets; ++e)
    for (int v = 0; v < 4; ++v)
      for (int a = 0; a < 3; ++a) {
        const double x = s.node_xyz[3 * (size_t)s.tet_nodes[10 * e + v] + a];
        M->lo[a] = std::min(M->lo[a], x); hi[a] = std::max(hi[a], x);
      }
  const double per_axis = std::cbrt((double)s.n_tets / 4.0);
  for (int a = 0; a < 3; ++a) {
    const double ext = std::max(hi[a] - M->lo[a], 1e-300);
    const double vol_share = ext / std::cbrt(std::max((hi[0] - M->lo[0]) * (hi[1] - M->lo[1]) * (hi[2] - M->lo[2]), 1e-300));
    M->n[a] = std::max(1, std::min(512, (int)(per_axis * vol_share)));
    M->inv[a] = M->n[a] / ext;
  }
  const size_t nc = (size_t)M->n[0] * M->n[1] * M->n[2];
  std::vector<std::vector<int32_t>> buckets(nc);
  for (int64_t e = 0; e < s.n_tets; ++e) {                     // ascending e: every bucket's list is ascending
    int c0[3], c1[3];
    for (int a = 0; a < 3; ++a) {
      double mn = 1e300, mx = -1e300;
      for (int v = 0; v < 4; ++v) { const double x = s.node_xyz[3 * (size_t)s.tet_nodes[10 * e + v] + a]; mn = std::min(mn, x); mx = std::max(mx, x); }
      const double pad = 1e-9 * (mx - mn) + 1e-300;
      c0[a] = std::max(0, std::min(M->n[a] - 1, (int)std::floor((mn - pad - M->lo[a]) * M->inv[a])));
      c1[a] = std::max(0, std::min(M->n[a] - 1, (int)std::floor((mx + pad - M->lo[a]) * M->inv[a])));
    }
    for (int k = c0[2]; k <= c1[2]; ++k) for (int j = c0[1]; j <= c1[1]; ++j) for (int i = c0[0]; i <= c1[0]; ++i)
      buckets[((size_t)k * M->n[1] + j) * M->n[0] + i].push_back((int32_t)e);
  }
  M->off.assign(nc + 1, 0);
  for (size_t c = 0; c < nc; ++c) M->off[c + 1] = M->off[c] + (int64_t)buckets[c].size();
  M->list.reserve((size_t)M->off[nc]);
  for (auto& b : buckets) M->list.insert(M->list.end(), b.begin(), b.end());
  return M;
}

// An avmo_field_desc with the mesh indices of its kind-2 slabs (built once per entry call).
struct PreparedField : avmo_field_desc {
  std::vector<std::unique_ptr<MeshIndex>> mesh;
  bool prepared = true;
  explicit PreparedField(const avmo_field_desc* f) : avmo_field_desc(*f) {
    mesh.resize(f->n_slabs);
    for (int i = 0; i < f->n_slabs; ++i) if (f->slabs[i].kind == 2) mesh[i] = build_mesh_index(f->slabs[i]);
  }
};

// F1: potential gradient of a 10-node tetrahedron at barycentric point lam; element test and evaluation in one.
// Returns true when the element contains r.
bool tet_eval(const avmo_slab& s, int64_t e, const double r[3], double E[3], double& mask) {
  const int32_t* nd = s.tet_nodes + 10 * e;
  const double* p[4];
  for (int v = 0; v < 4; ++v) p[v] = s.node_xyz + 3 * (size_t)nd[v];
  double lam[4];
  if (!barycentric(p[0], p[1], p[2], p[3], r, lam)) return false;
  for (int v = 0; v < 4; ++v) if (!(lam[v] >= -TET_TOL)) return false;
  // grad lambda_a: lambda is affine; recover its gradient from unit displacements
  double g[4][3];
  for (int a = 0; a < 3; ++a) {
    double rp[3] = {r[0], r[1], r[2]}, lp[4];
    rp[a] += 1.0;
    barycentric(p[0], p[1], p[2], p[3], rp, lp);
    for (int v = 0; v < 4; ++v) g[v][a] = lp[v] - lam[v];
  }
  static const int EA[6] = {0, 0, 0, 1, 1, 2}, EB[6] = {1, 2, 3, 2, 3, 3};
  double grad[3] = {0.0, 0.0, 0.0};
  for (int v = 0; v < 4; ++v) {
    const double c = s.node_V[nd[v]] * (4.0 * lam[v] - 1.0);                    // d/dl [l (2l - 1)] = 4l - 1
    for (int a = 0; a < 3; ++a) grad[a] += c * g[v][a];
  }
  for (int k = 0; k < 6; ++k) {
    const double V = 4.0 * s.node_V[nd[4 + k]];                                 // N = 4 l_a l_b
    for (int a = 0; a < 3; ++a) grad[a] += V * (lam[EB[k]] * g[EA[k]][a] + lam[EA[k]] * g[EB[k]][a]);
  }
  E[0] = -grad[0]; E[1] = -grad[1]; E[2] = -grad[2];
  mask = s.tet_gas[e] ? 1.0 : 0.0;
  return true;
}

// R15: fold one coordinate into the stored cell.  Returns false when outside with bc none.
// q = (x - origin) mod period (periodic) or mod 2P with reflection (mirror); flip = normal component changes sign.
bool fold(double x, double origin, double h, int n, int bc, double P, double& q, bool& flip) {
  flip = false;
  q = x - origin;
  if (bc == 0) return q >= 0.0 && q <= (n - 1) * h;
  if (bc == 1) { q = q - P * std::floor(q / P); if (q >= P) q = 0.0; return true; }
  double two_p = 2.0 * P;
  q = q - two_p * std::floor(q / two_p);
  if (q >= two_p) q = 0.0;
  if (q > P) { q = two_p - q; flip = true; }
  return true;
}

void cell(double q, double h, int n, int& i, double& w) {   // i = min(floor(q/h), n-2), w = q/h - i
  double s = q / h;
  i = (int)std::floor(s);
  if (i > n - 2) i = n - 2;
  if (i < 0) i = 0;
  w = s - (double)i;
}

// S0 / R14 / R15: field and gas-mask at r.  Returns the slab index, or a negative status code
// (-AVMO_LEFT_*) when r is outside the domain.
int field_at(const avmo_field_desc* f, double x, double y, double z, double E[3], double& mask) {
  const avmo_slab* S = f->slabs;
  int ns = f->n_slabs;
  if (z < S[0].z_lo) return -AVMO_LEFT_ZLO;
  if (z > S[ns - 1].z_hi) return -AVMO_LEFT_ZHI;
  if (x < f->xy_lo[0] || x > f->xy_hi[0] || y < f->xy_lo[1] || y > f->xy_hi[1]) return -AVMO_LEFT_XY;
  if (!(z == z) || !(x == x) || !(y == y)) return -AVMO_LEFT_XY;
  int si = ns - 1;
  for (int i = 0; i < ns; ++i) if (z < S[i].z_hi) { si = i; break; }
  const avmo_slab& s = S[si];
  if (s.kind == 0) { E[0] = s.E[0]; E[1] = s.E[1]; E[2] = s.E[2]; mask = 1.0; return si; }
  if (s.kind == 2) {
    // F3: fold x, y as for a grid (bc none: no fold and no range: a point in no element is solid), look the element up
    double qx = x - s.origin[0], qy = y - s.origin[1];
    bool fx = false, fy = false;
    if (s.bc_x) fold(x, s.origin[0], 1.0, 2, s.bc_x, s.period_x, qx, fx);
    if (s.bc_y) fold(y, s.origin[1], 1.0, 2, s.bc_y, s.period_y, qy, fy);
    const double r[3] = {qx, qy, z - s.origin[2]};
    const MeshIndex& M = *static_cast<const PreparedField*>(f)->mesh[si];
    E[0] = E[1] = E[2] = 0.0; mask = 0.0;
    int c[3];
    bool inside = true;
    for (int a = 0; a < 3; ++a) {
      const double u = (r[a] - M.lo[a]) * M.inv[a];
      c[a] = (int)std::floor(u);
      if (c[a] == M.n[a] && u <= (double)M.n[a] * (1.0 + 1e-12)) c[a] = M.n[a] - 1;
      if (c[a] < 0 || c[a] >= M.n[a]) inside = false;
    }
    if (inside) {
      const size_t cell = ((size_t)c[2] * M.n[1] + c[1]) * M.n[0] + c[0];
      for (int64_t q = M.off[cell]; q < M.off[cell + 1]; ++q)
        if (tet_eval(s, M.list[q], r, E, mask)) break;
    }
    if (fx) E[0] = -E[0];
    if (fy) E[1] = -E[1];
    return si;
  }
  double qx, qy; bool fx, fy;
  if (!fold(x, s.origin[0], s.spacing[0], s.nx, s.bc_x, s.period_x, qx, fx)) return -AVMO_LEFT_XY;
  if (!fold(y, s.origin[1], s.spacing[1], s.ny, s.bc_y, s.period_y, qy, fy)) return -AVMO_LEFT_XY;
  int i, j, k; double wx, wy, wz;
  cell(qx, s.spacing[0], s.nx, i, wx);
  cell(qy, s.spacing[1], s.ny, j, wy);
  cell(z - s.origin[2], s.spacing[2], s.nz, k, wz);
  double out[4];
  for (int c = 0; c < 4; ++c) {
    auto N = [&](int kk, int jj, int ii) { return (double)s.nodes[(((size_t)kk * s.ny + jj) * s.nx + ii) * 4 + c]; };
    // lerp a + w (b - a): x, then y, then z
    double c00 = N(k, j, i) + wx * (N(k, j, i + 1) - N(k, j, i));
    double c10 = N(k, j + 1, i) + wx * (N(k, j + 1, i + 1) - N(k, j + 1, i));
    double c01 = N(k + 1, j, i) + wx * (N(k + 1, j, i + 1) - N(k + 1, j, i));
    double c11 = N(k + 1, j + 1, i) + wx * (N(k + 1, j + 1, i + 1) - N(k + 1, j + 1, i));
    double c0 = c00 + wy * (c10 - c00);
    double c1 = c01 + wy * (c11 - c01);
    out[c] = c0 + wz * (c1 - c0);
  }
  E[0] = fx ? -out[0] : out[0];
  E[1] = fy ? -out[1] : out[1];
  E[2] = out[2];
  mask = out[3];
  return si;
}

struct StepOut {
  int event = -2;      // -1 null, l >= 0 level, -2 terminated before the decision
  int bin = -1;
  bool child = false;
  Electron c;
};

// One step S0-S9 for an in-domain, active electron.
// W1: the weighting field at r: E_w, zero outside its description (mask and B ignored).
void weighting_at(const avmo_field_desc* wf, double x, double y, double z, double Ew[3]) {
  double m;
  Ew[0] = Ew[1] = Ew[2] = 0.0;
  double e[3];
  if (field_at(wf, x, y, z, e, m) >= 0) { Ew[0] = e[0]; Ew[1] = e[1]; Ew[2] = e[2]; }
}
// W2: charge q moved from r0 to r1 in a step that starts at time t: q E_w(at) . (r1 - r0) into the bin of t.
void induce(const avmo_signal* sg, double* acc, double q, const double at[3], const double r0[3], const double r1[3], double t) {
  double Ew[3];
  weighting_at(sg->weighting, at[0], at[1], at[2], Ew);
  const double dq = q * (Ew[0] * (r1[0] - r0[0]) + Ew[1] * (r1[1] - r0[1]) + Ew[2] * (r1[2] - r0[2]));
  const double sb = std::floor((t - sg->t0) / sg->dt_bin);
  if (sb >= 0.0 && sb < (double)sg->n_bins) acc[(int)sb] += dq;
}

void step(const Gas& g, const avmo_field_desc* f, uint64_t seed, double t_max, bool banded, Electron& el, StepOut& so, Tally* tl,
          const avmo_signal* sgn = nullptr, double* sig_acc = nullptr) {
  so.event = -2; so.bin = -1; so.child = false;
  // S0: field at r (held constant during the flight); B is a run constant.  R3: re-evaluated every step.
  double E[3], m;
  int si = field_at(f, el.x, el.y, el.z, E, m);
  if (si < 0) { el.status = -si; return; }      // not in domain: caller error, reported as a status
  // S1: the step's counter n_s; block 0 -> (u1, u2)
  const uint32_t n_s = el.n;
  double u1, u2;
  uniform_pair(seed, el.id, n_s, 0, u1, u2);
  // S2: free-flight time under the null-collision rate nu_hat (R4: one global rate) — or, banded (N5), under the rate of
  // the electron's energy band and this flight's acceleration class, cut at dtmax
  double nu_hat = g.nu_hat, inv_nu_hat = g.inv_nu_hat, dt_cut = std::numeric_limits<double>::infinity();
  if (banded) {
    const Majorant& M = g.M;
    const double sb0 = el.e * g.inv_de;
    const int b0 = sb0 >= (double)g.nb ? g.nb - 1 : (int)sb0;
    const double ax = KAPPA * E[0], ay = KAPPA * E[1], az = KAPPA * E[2];
    const double a2 = ax * ax + ay * ay + az * az;
    int j = 0;
    while (j < M.J && a2 > M.a2[j]) ++j;           // smallest class whose edge covers |a| (J = above all)
    const size_t o = (size_t)(b0 >> M.shift) * (M.J + 1) + j;
    nu_hat = M.nu[o]; inv_nu_hat = M.inv_nu[o]; dt_cut = M.dtmax[o];
  }
  double dt = -std::log(u1) * inv_nu_hat;
  const bool cut = dt > dt_cut;
  if (cut) dt = dt_cut;
  // S3: flight in constant E (and B)
  const double sp = C2 * std::sqrt(el.e);
  const double v0[3] = {sp * el.kx, sp * el.ky, sp * el.kz};
  const double a[3] = {-KAPPA * E[0], -KAPPA * E[1], -KAPPA * E[2]};
  const double r0[3] = {el.x, el.y, el.z};
  double r1[3], v1[3];
  const double Bn2 = f->B[0] * f->B[0] + f->B[1] * f->B[1] + f->B[2] * f->B[2];
  if (Bn2 == 0.0) {
    for (int i = 0; i < 3; ++i) {
      r1[i] = r0[i] + v0[i] * dt + 0.5 * a[i] * dt * dt;
      v1[i] = v0[i] + a[i] * dt;
    }
  } else {
    const double Bn = std::sqrt(Bn2);
    const double bh[3] = {f->B[0] / Bn, f->B[1] / Bn, f->B[2] / Bn};
    const double omega = OMEGA1 * Bn;
    const double a_b = a[0] * bh[0] + a[1] * bh[1] + a[2] * bh[2];
    const double v_b = v0[0] * bh[0] + v0[1] * bh[1] + v0[2] * bh[2];
    const double ExB[3] = {E[1] * f->B[2] - E[2] * f->B[1], E[2] * f->B[0] - E[0] * f->B[2], E[0] * f->B[1] - E[1] * f->B[0]};
    double apar[3], vpar[3], vd[3], w0[3], bxw[3];
    for (int i = 0; i < 3; ++i) {
      apar[i] = a_b * bh[i];
      vpar[i] = v_b * bh[i];
      vd[i] = EXB_UNIT * ExB[i] / Bn2;
      w0[i] = v0[i] - vpar[i] - vd[i];
    }
    bxw[0] = bh[1] * w0[2] - bh[2] * w0[1];
    bxw[1] = bh[2] * w0[0] - bh[0] * w0[2];
    bxw[2] = bh[0] * w0[1] - bh[1] * w0[0];
    const double th = omega * dt;
    const double sn = std::sin(th), cs = std::cos(th);
    const double sh = std::sin(0.5 * th);
    const double vers = 2.0 * sh * sh;               // 1 - cos(theta), cancellation-free
    for (int i = 0; i < 3; ++i) {
      v1[i] = vpar[i] + apar[i] * dt + vd[i] + w0[i] * cs + bxw[i] * sn;
      r1[i] = r0[i] + vpar[i] * dt + 0.5 * apar[i] * dt * dt + vd[i] * dt + (w0[i] * sn + bxw[i] * vers) / omega;
    }
  }
  if (sgn) induce(sgn, sig_acc, -1.0, r0, r0, r1, el.t);   // W2: every flight, the last one of an electron included
  // S4: new energy, direction, time, counter
  const double s2 = v1[0] * v1[0] + v1[1] * v1[1] + v1[2] * v1[2];
  const double e1 = std::max(s2 * INV_C2SQ, EPS_FLOOR);
  double k1[3] = {el.kx, el.ky, el.kz};
  if (s2 > 0.0) { const double nrm = std::sqrt(s2); k1[0] = v1[0] / nrm; k1[1] = v1[1] / nrm; k1[2] = v1[2] / nrm; }
  const double t1 = el.t + dt;
  if (tl) {
    tl->n_steps++;
    tl->sdx += r1[0] - r0[0]; tl->sdy += r1[1] - r0[1]; tl->sdz += r1[2] - r0[2]; tl->sdt += dt;
  }
  el.x = r1[0]; el.y = r1[1]; el.z = r1[2]; el.t = t1; el.e = e1; el.kx = k1[0]; el.ky = k1[1]; el.kz = k1[2];
  el.n = n_s + 1;
  // S5: terminate at r' — bounds, then material, then time limit (R13: no back-projection)
  double E1[3], m1;
  int s1 = field_at(f, r1[0], r1[1], r1[2], E1, m1);
  if (s1 < 0) { el.status = -s1; return; }
  if (m1 < 0.5) { el.status = AVMO_MATERIAL; return; }
  if (t1 > t_max) { el.status = AVMO_TIME_LIMIT; return; }
  if (el.n >= N_STEP_LIMIT) { el.status = AVMO_STEP_LIMIT; return; }
  // S6: energy bin (R5: piecewise constant, clamp and count)
  const double sb = e1 * g.inv_de;
  int b;
  if (sb >= (double)g.nb) { b = g.nb - 1; if (tl) tl->n_overflow++; } else b = (int)sb;
  so.bin = b;
  const double* row = g.cum + (size_t)b * g.L;
  // S7: null or real (R7: one uniform decides both).  N6: a flight that was cut is a null collision; the band's rate must
  // bound the total rate of the bin reached (counted when it does not: never, by construction)
  if (cut) { so.event = -1; if (tl) tl->n_null++; return; }
  if (tl && row[g.L - 1] > nu_hat) tl->n_viol++;
  const double xr = u2 * nu_hat;
  if (xr >= row[g.L - 1]) { so.event = -1; if (tl) tl->n_null++; return; }
  // S8: level = smallest index with cum[b][l] > x
  int l = 0;
  while (row[l] <= xr) ++l;
  so.event = l;
  if (tl) { tl->n_real++; tl->level[l]++; }
  // S9a: attachment
  if (g.type[l] == AVMO_ATTACHMENT) { el.status = AVMO_ATTACHED; return; }
  // S9b: deflection angles
  double u3, u4;
  uniform_pair(seed, el.id, n_s, 1, u3, u4);
  double ct = 1.0 - 2.0 * u3;
  double st = 2.0 * std::sqrt(u3 * (1.0 - u3));
  if (g.xi) {
    // X1: forward-peaked deflection, cos(theta) = (c0 + xi) / (1 + xi c0) with c0 = 1 - 2 u3 uniform in (-1, 1) and xi the
    // table entry of this bin and level; sin(theta) in the cancellation-free form sqrt((1 - ct)(1 + ct)) =
    // 2 sqrt(u3 (1 - u3)) sqrt(1 - xi^2) / (1 + xi c0)
    const double xi = g.xi[(size_t)b * g.L + l];
    const double den = 1.0 + xi * ct;
    st = st * std::sqrt(1.0 - xi * xi) / den;
    ct = (ct + xi) / den;
  }
  const double phi = TWO_PI * u4;
  const double sphi = std::sin(phi), cphi = std::cos(phi);
  // S9c: energy after the collision
  double e2;
  bool thermal = false;
  double V[3] = {0.0, 0.0, 0.0};
  if (g.type[l] == AVMO_ELASTIC && g.kT > 0.0 && g.recoil[l] > 0.0) {
    // X3: the gas atom moves.  Its velocity components are normal with variance kT / M, M / m = 2 / r (R9's order):
    // sigma = c2 sqrt(kT r / 4); Box-Muller from blocks 2 and 3.  The cold-gas collision (S9b-S9d) is applied to the
    // electron's velocity RELATIVE to the atom, w = v' - V, and the atom's velocity is added back.
    double u5, u6, u7, u8;
    uniform_pair(seed, el.id, n_s, 2, u5, u6);
    uniform_pair(seed, el.id, n_s, 3, u7, u8);
    const double sigma = C2 * std::sqrt(g.kT * g.recoil[l] * 0.25);
    const double ra = std::sqrt(-2.0 * std::log(u5)), rb = std::sqrt(-2.0 * std::log(u7));
    V[0] = sigma * ra * std::cos(TWO_PI * u6);
    V[1] = sigma * ra * std::sin(TWO_PI * u6);
    V[2] = sigma * rb * std::cos(TWO_PI * u8);
    const double w[3] = {v1[0] - V[0], v1[1] - V[1], v1[2] - V[2]};
    const double w2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2];
    const double ew = std::max(w2 * INV_C2SQ, EPS_FLOOR);
    if (w2 > 0.0) { const double nrm = std::sqrt(w2); k1[0] = w[0] / nrm; k1[1] = w[1] / nrm; k1[2] = w[2] / nrm; }
    e2 = ew * (1.0 - g.recoil[l] * (1.0 - ct));                    // relative-frame energy after the collision
    thermal = true;
  } else if (g.type[l] == AVMO_ELASTIC) {
    e2 = e1 * (1.0 - g.recoil[l] * (1.0 - ct));                    // R9
    if (tl) tl->sloss += e1 - e2;
  } else if (g.type[l] == AVMO_EXCITATION) {
    e2 = std::max(e1 - g.loss[l], EPS_FLOOR);                      // R11
    if (tl) tl->sloss += e1 - e2;
    if (g.pen_p && g.pen_p[l] > 0.0) {
      // X2: Penning transfer — with probability p_l the excited atom ionises the admixture: one more electron at r', t'
      // with energy u8 x (available energy), isotropic direction from (u6, u7), id hashed like an ionisation's child
      double u5, u6, u7, u8;
      uniform_pair(seed, el.id, n_s, 2, u5, u6);
      uniform_pair(seed, el.id, n_s, 3, u7, u8);
      if (u5 < g.pen_p[l]) {
        Electron& c = so.c;
        c.x = r1[0]; c.y = r1[1]; c.z = r1[2]; c.t = t1;
        c.e = std::max(u8 * g.pen_e[l], EPS_FLOOR);
        const double sc = 2.0 * std::sqrt(u6 * (1.0 - u6));
        const double pc = TWO_PI * u7;
        c.kx = sc * std::cos(pc); c.ky = sc * std::sin(pc); c.kz = 1.0 - 2.0 * u6;
        uint32_t wd[4];
        philox_block(seed, el.id, n_s, BLOCK_CHILD_ID, wd);
        c.id = (uint64_t)wd[0] + ((uint64_t)wd[1] << 32);
        c.n = 0; c.aval = el.aval; c.status = AVMO_ACTIVE; c.primary = false;
        c.birth[0] = c.x; c.birth[1] = c.y; c.birth[2] = c.z; c.birth[3] = c.t; c.birth[4] = c.e;
        so.child = true;
        if (tl) tl->n_penning++;
      }
    }
  } else {                                                         // ionisation, R10 (Opal-Peterson-Beaty)
    double u5, u6, u7, u8;
    uniform_pair(seed, el.id, n_s, 2, u5, u6);
    uniform_pair(seed, el.id, n_s, 3, u7, u8);
    const double ea = std::max(e1 - g.loss[l], 0.0);
    const double w = g.w[l];
    const double es = w * std::tan(u5 * std::atan(ea / (2.0 * w)));
    e2 = std::max(ea - es, EPS_FLOOR);
    Electron& c = so.c;
    c.x = r1[0]; c.y = r1[1]; c.z = r1[2]; c.t = t1;
    c.e = std::max(es, EPS_FLOOR);
    const double sc = 2.0 * std::sqrt(u6 * (1.0 - u6));
    const double pc = TWO_PI * u7;
    c.kx = sc * std::cos(pc); c.ky = sc * std::sin(pc); c.kz = 1.0 - 2.0 * u6;
    uint32_t wd[4];
    philox_block(seed, el.id, n_s, BLOCK_CHILD_ID, wd);             // R16: schedule-independent child id
    c.id = (uint64_t)wd[0] + ((uint64_t)wd[1] << 32);
    c.n = 0; c.aval = el.aval; c.status = AVMO_ACTIVE; c.primary = false;
    c.birth[0] = c.x; c.birth[1] = c.y; c.birth[2] = c.z; c.birth[3] = c.t; c.birth[4] = c.e;
    so.child = true;
    if (tl) tl->sloss += e1 - e2 - c.e;
  }
  el.e = e2;
  // S9d: new direction — branch-free orthonormal basis about k' (Duff et al. 2017), then renormalise
  const double sg = std::copysign(1.0, k1[2]);
  const double A = -1.0 / (sg + k1[2]);
  const double Bq = k1[0] * k1[1] * A;
  const double b1[3] = {1.0 + sg * k1[0] * k1[0] * A, sg * Bq, -sg * k1[0]};
  const double b2[3] = {Bq, sg + k1[1] * k1[1] * A, -k1[1]};
  double k2[3];
  for (int i = 0; i < 3; ++i) k2[i] = ct * k1[i] + st * (cphi * b1[i] + sphi * b2[i]);
  const double nk = std::sqrt(k2[0] * k2[0] + k2[1] * k2[1] + k2[2] * k2[2]);
  el.kx = k2[0] / nk; el.ky = k2[1] / nk; el.kz = k2[2] / nk;
  if (thermal) {
    // X3, back to the laboratory frame: v'' = c2 sqrt(e2) k'' + V; energy and direction from v''
    const double sw = C2 * std::sqrt(e2);
    const double v2[3] = {sw * el.kx + V[0], sw * el.ky + V[1], sw * el.kz + V[2]};
    const double s22 = v2[0] * v2[0] + v2[1] * v2[1] + v2[2] * v2[2];
    el.e = std::max(s22 * INV_C2SQ, EPS_FLOOR);
    if (s22 > 0.0) { const double nrm = std::sqrt(s22); el.kx = v2[0] / nrm; el.ky = v2[1] / nrm; el.kz = v2[2] / nrm; }
    if (tl) tl->sloss += e1 - el.e;
  }
}

struct Record { Electron el; };

// The avalanche driver: transport until status != 0, push newly created electrons, repeat.
// Serial: one electron at a time from a stack.  Order is irrelevant because draws are keyed by (id, n).
void run_range(const Gas& g, const avmo_field_desc* f, const double* prim, int64_t p0, int64_t p1, uint64_t seed,
               uint64_t id_offset, double t_max, bool banded, std::vector<Electron>& done, Tally& tl,
               const avmo_signal* sg = nullptr, double* sig_acc = nullptr) {
  std::vector<Electron> stack;
  StepOut so;
  for (int64_t p = p0; p < p1; ++p) {
    const double* q = prim + p * 8;
    Electron el;
    el.x = q[0]; el.y = q[1]; el.z = q[2]; el.t = q[3]; el.e = std::max(q[4], EPS_FLOOR);
    double nk = std::sqrt(q[5] * q[5] + q[6] * q[6] + q[7] * q[7]);
    if (!(nk > 0)) { el.kx = 0; el.ky = 0; el.kz = 1; } else { el.kx = q[5] / nk; el.ky = q[6] / nk; el.kz = q[7] / nk; }
    el.id = id_offset + (uint64_t)p; el.n = 0; el.aval = (uint32_t)p; el.status = AVMO_ACTIVE; el.primary = true;
    el.birth[0] = el.x; el.birth[1] = el.y; el.birth[2] = el.z; el.birth[3] = el.t; el.birth[4] = el.e;
    // a-1: reject out-of-domain primaries (status set, endpoint = birth point)
    double E[3], m;
    int si = field_at(f, el.x, el.y, el.z, E, m);
    if (si < 0) el.status = -si;
    else if (m < 0.5) el.status = AVMO_MATERIAL;
    else if (el.t > t_max) el.status = AVMO_TIME_LIMIT;
    stack.push_back(el);
    while (!stack.empty()) {
      Electron cur = stack.back();
      stack.pop_back();
      while (cur.status == AVMO_ACTIVE) {
        step(g, f, seed, t_max, banded, cur, so, &tl, sg, sig_acc);
        if (so.child) stack.push_back(so.c);
      }
      done.push_back(cur);
    }
  }
}

}  // namespace

extern "C" {

const char* avmo_last_error(void) { return g_err.c_str(); }

int32_t avmo_majorant(const avmo_gas_desc* gd, int32_t* shape3, double* a2, double* nu, double* dtmax) {
  Gas g;
  if (!load_gas(gd, g) || !shape3) return AVMO_ERR_INVALID_ARG;
  shape3[0] = g.M.K; shape3[1] = g.M.J; shape3[2] = g.M.shift;
  if (a2) std::copy(g.M.a2.begin(), g.M.a2.end(), a2);
  if (nu) std::copy(g.M.nu.begin(), g.M.nu.end(), nu);
  if (dtmax) std::copy(g.M.dtmax.begin(), g.M.dtmax.end(), dtmax);
  return AVMO_OK;
}

void avmo_philox(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, uint32_t out[4]) { philox_block(seed, id, n, block, out); }

void avmo_uniform_pair(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, double out[2]) {
  uniform_pair(seed, id, n, block, out[0], out[1]);
}

int32_t avmo_field_eval(const avmo_field_desc* f, int64_t n, const double* r, double* E, double* mask, int32_t* slab) {
  if (!check_field(f) || n < 0 || !r || !E || !mask || !slab) return AVMO_ERR_INVALID_ARG;
  const PreparedField pf(f);
  f = &pf;
  for (int64_t i = 0; i < n; ++i) {
    double e[3] = {0, 0, 0}, m = 0;
    int si = field_at(f, r[i], r[n + i], r[2 * n + i], e, m);
    E[i] = e[0]; E[n + i] = e[1]; E[2 * n + i] = e[2]; mask[i] = m; slab[i] = si < 0 ? -1 : si;
  }
  return AVMO_OK;
}

int32_t avmo_step_batch(const avmo_gas_desc* gd, const avmo_field_desc* f, uint64_t seed, double t_max, int64_t n,
                        const double* in, const uint64_t* id, const uint32_t* n_idx, double* out, int32_t* event,
                        int32_t* status, int32_t* bin, double* child, uint64_t* child_id, uint32_t flags) {
  Gas g;
  if (!load_gas(gd, g) || !check_field(f)) return AVMO_ERR_INVALID_ARG;
  if (n < 0 || !in || !id || !n_idx || !out || !event || !status || !bin || !child || !child_id) { g_err = "step_batch: null"; return AVMO_ERR_INVALID_ARG; }
  const PreparedField pf(f);
  f = &pf;
  StepOut so;
  for (int64_t i = 0; i < n; ++i) {
    Electron el;
    el.x = in[i]; el.y = in[n + i]; el.z = in[2 * n + i]; el.t = in[3 * n + i]; el.e = in[4 * n + i];
    el.kx = in[5 * n + i]; el.ky = in[6 * n + i]; el.kz = in[7 * n + i];
    el.id = id[i]; el.n = n_idx[i]; el.aval = 0; el.status = AVMO_ACTIVE;
    step(g, f, seed, t_max, (flags & AVMO_BANDED) != 0, el, so, nullptr);
    out[i] = el.x; out[n + i] = el.y; out[2 * n + i] = el.z; out[3 * n + i] = el.t; out[4 * n + i] = el.e;
    out[5 * n + i] = el.kx; out[6 * n + i] = el.ky; out[7 * n + i] = el.kz;
    event[i] = so.event; status[i] = el.status; bin[i] = so.bin;
    for (int c = 0; c < 8; ++c) child[c * n + i] = 0.0;
    child_id[i] = 0;
    if (so.child) {
      const Electron& c = so.c;
      child[i] = c.x; child[n + i] = c.y; child[2 * n + i] = c.z; child[3 * n + i] = c.t; child[4 * n + i] = c.e;
      child[5 * n + i] = c.kx; child[6 * n + i] = c.ky; child[7 * n + i] = c.kz;
      child_id[i] = c.id;
    }
  }
  return AVMO_OK;
}

int32_t avmo_ion_drift(const avmo_field_desc* f, const avmo_signal* sg, const avmo_ion_opts* io, int64_t n, int64_t n_prim,
                       int64_t ldb, const double* birth, int64_t lde, const double* end, const int32_t* status,
                       double* ion_end, int32_t* ion_status, uint32_t* ion_steps) {
  if (!check_field(f) || !io || n < 0 || !birth || !end || !status || !ion_end || !ion_status || !ion_steps) { g_err = "ion_drift: null"; return AVMO_ERR_INVALID_ARG; }
  if (!(io->step_cm > 0) || !(io->mobility_pos > 0) || !(io->mobility_neg > 0) || io->max_steps < 1) { g_err = "ion_drift: options"; return AVMO_ERR_INVALID_ARG; }
  if (sg && (!sg->weighting || !check_field(sg->weighting) || !(sg->dt_bin > 0) || sg->n_bins < 1 || !sg->signal)) { g_err = "ion_drift: signal description"; return AVMO_ERR_INVALID_ARG; }
  const PreparedField pf(f);
  f = &pf;
  std::unique_ptr<PreparedField> pw;
  avmo_signal sg_local;
  if (sg) { pw = std::make_unique<PreparedField>(sg->weighting); sg_local = *sg; sg_local.weighting = pw.get(); sg = &sg_local; }
  const int64_t N = 2 * n;
  for (int64_t i = 0; i < N; ++i) {
    const int64_t s = i < n ? i : i - n;
    const bool pos = i < n;
    ion_status[i] = -1; ion_steps[i] = 0;
    for (int c = 0; c < 4; ++c) ion_end[c * N + i] = 0.0;
    if (pos ? s < n_prim : status[s] != AVMO_ATTACHED) continue;           // W3: which ions exist
    double r[3], t;
    if (pos) { r[0] = birth[s]; r[1] = birth[ldb + s]; r[2] = birth[2 * ldb + s]; t = birth[3 * ldb + s]; }
    else { r[0] = end[s]; r[1] = end[lde + s]; r[2] = end[2 * lde + s]; t = end[3 * lde + s]; }
    const double q = pos ? 1.0 : -1.0, mu = pos ? io->mobility_pos : io->mobility_neg;
    int st = AVMO_ACTIVE;
    uint32_t ns = 0;
    double E[3], m;
    int si = field_at(f, r[0], r[1], r[2], E, m);
    if (si < 0) st = -si; else if (m < 0.5) st = AVMO_MATERIAL;
    while (st == AVMO_ACTIVE) {                                              // W4: explicit midpoint, fixed step length
      if (ns >= (uint32_t)io->max_steps) { st = AVMO_STEP_LIMIT; break; }
      const double k1[3] = {q * mu * E[0], q * mu * E[1], q * mu * E[2]};
      const double n1 = std::sqrt(k1[0] * k1[0] + k1[1] * k1[1] + k1[2] * k1[2]);
      if (!(n1 > 0.0)) { st = AVMO_STEP_LIMIT; break; }
      const double hh = 0.5 * io->step_cm / n1;
      const double rm[3] = {r[0] + hh * k1[0], r[1] + hh * k1[1], r[2] + hh * k1[2]};
      double Em[3], mm;
      if (field_at(f, rm[0], rm[1], rm[2], Em, mm) < 0) { Em[0] = E[0]; Em[1] = E[1]; Em[2] = E[2]; }   // midpoint outside: Euler step
      const double k2[3] = {q * mu * Em[0], q * mu * Em[1], q * mu * Em[2]};
      const double n2 = std::sqrt(k2[0] * k2[0] + k2[1] * k2[1] + k2[2] * k2[2]);
      if (!(n2 > 0.0)) { st = AVMO_STEP_LIMIT; break; }
      const double h2 = io->step_cm / n2;
      const double r1[3] = {r[0] + h2 * k2[0], r[1] + h2 * k2[1], r[2] + h2 * k2[2]};
      if (sg) induce(sg, sg->signal, q, rm, r, r1, t);
      r[0] = r1[0]; r[1] = r1[1]; r[2] = r1[2];
      t = t + h2;
      ++ns;
      si = field_at(f, r[0], r[1], r[2], E, m);
      if (si < 0) st = -si;
      else if (m < 0.5) st = AVMO_MATERIAL;
      else if (t > io->t_max) st = AVMO_TIME_LIMIT;
    }
    ion_end[i] = r[0]; ion_end[N + i] = r[1]; ion_end[2 * N + i] = r[2]; ion_end[3 * N + i] = t;
    ion_status[i] = st; ion_steps[i] = ns;
  }
  return AVMO_OK;
}

int32_t avmo_run(const avmo_gas_desc* gd, const avmo_field_desc* f, const double* prim, int64_t np,
                 const avmo_run_opts* opts, avmo_outputs* o, int64_t* n_out) {
  Gas g;
  if (!load_gas(gd, g) || !check_field(f)) return AVMO_ERR_INVALID_ARG;
  if (np < 0 || (np > 0 && !prim) || !opts || !o || !n_out || o->capacity < 0) { g_err = "run: null/negative"; return AVMO_ERR_INVALID_ARG; }
  if (np > 0xFFFFFFFFll) { g_err = "run: too many primaries"; return AVMO_ERR_INVALID_ARG; }
  const bool banded = (opts->flags & AVMO_BANDED) != 0;
  int nt = std::max(1, opts->n_threads);
  nt = (int)std::min<int64_t>(nt, std::max<int64_t>(np, 1));
  std::vector<std::vector<Electron>> done(nt);
  std::vector<Tally> tl(nt);
  for (auto& t : tl) t.level.assign(g.L, 0);
  const avmo_signal* sg = opts->signal;
  if (sg && (!sg->weighting || !check_field(sg->weighting) || !(sg->dt_bin > 0) || sg->n_bins < 1 || !sg->signal)) { g_err = "run: signal description"; return AVMO_ERR_INVALID_ARG; }
  const PreparedField pf(f);
  f = &pf;
  std::unique_ptr<PreparedField> pw;
  avmo_signal sg_local;
  if (sg) { pw = std::make_unique<PreparedField>(sg->weighting); sg_local = *sg; sg_local.weighting = pw.get(); sg = &sg_local; }
  std::vector<std::vector<double>> sacc(nt);
  if (sg) for (auto& a : sacc) a.assign(sg->n_bins, 0.0);
  if (nt == 1) {
    run_range(g, f, prim, 0, np, opts->seed, opts->id_offset, opts->t_max, banded, done[0], tl[0], sg, sg ? sacc[0].data() : nullptr);
  } else {                       // timed multi-core baseline only: disjoint primary ranges, identical results
    std::vector<std::thread> th;
    for (int t = 0; t < nt; ++t) {
      int64_t p0 = np * t / nt, p1 = np * (t + 1) / nt;
      th.emplace_back([&, t, p0, p1] { run_range(g, f, prim, p0, p1, opts->seed, opts->id_offset, opts->t_max, banded, done[t], tl[t], sg, sg ? sacc[t].data() : nullptr); });
    }
    for (auto& x : th) x.join();
  }
  if (sg) for (auto& a : sacc) for (int i = 0; i < sg->n_bins; ++i) sg->signal[i] += a[i];
  // outputs
  int64_t total = 0;
  for (auto& d : done) total += (int64_t)d.size();
  const int64_t cap = o->capacity;
  if (o->per_avalanche) std::memset(o->per_avalanche, 0, sizeof(uint64_t) * 3 * (size_t)np);
  // entries in creation order as far as it is defined: the primaries first, in primary order (threads own ascending
  // ranges), then the secondaries (order unspecified; compare after sorting by id, R17)
  int64_t w = 0;
  for (int pass = 0; pass < 2; ++pass)
  for (auto& d : done)
    for (auto& el : d) {
      if (el.primary != (pass == 0)) continue;
      if (o->per_avalanche) {                 // a-12 / C11: ions = ionisations = endpoints - 1 per avalanche
        o->per_avalanche[3 * (size_t)el.aval + 0]++;
        if (el.status == AVMO_ATTACHED) o->per_avalanche[3 * (size_t)el.aval + 2]++;
      }
      if (w >= cap) { ++w; continue; }
      if (o->id) o->id[w] = el.id;
      if (o->avalanche) o->avalanche[w] = el.aval;
      if (o->status) o->status[w] = el.status;
      if (o->n_steps) o->n_steps[w] = el.n;
      if (o->birth) for (int c = 0; c < 5; ++c) o->birth[c * cap + w] = el.birth[c];
      if (o->end) {
        const double e8[8] = {el.x, el.y, el.z, el.t, el.e, el.kx, el.ky, el.kz};
        for (int c = 0; c < 8; ++c) o->end[c * cap + w] = e8[c];
      }
      ++w;
    }
  if (o->per_avalanche)
    for (int64_t p = 0; p < np; ++p) o->per_avalanche[3 * p + 1] = o->per_avalanche[3 * p] > 0 ? o->per_avalanche[3 * p] - 1 : 0;
  if (o->tallies_u64) {
    for (int l = 0; l < g.L + 6; ++l) o->tallies_u64[l] = 0;
    for (auto& t : tl) {
      for (int l = 0; l < g.L; ++l) o->tallies_u64[l] += t.level[l];
      o->tallies_u64[g.L] += t.n_null; o->tallies_u64[g.L + 1] += t.n_real;
      o->tallies_u64[g.L + 2] += t.n_overflow; o->tallies_u64[g.L + 3] += t.n_steps; o->tallies_u64[g.L + 4] += t.n_penning;
      o->tallies_u64[g.L + 5] += t.n_viol;
    }
  }
  if (o->tallies_f64) {
    for (int c = 0; c < 5; ++c) o->tallies_f64[c] = 0;
    for (auto& t : tl) {
      o->tallies_f64[0] += t.sdx; o->tallies_f64[1] += t.sdy; o->tallies_f64[2] += t.sdz;
      o->tallies_f64[3] += t.sdt; o->tallies_f64[4] += t.sloss;
    }
  }
  *n_out = std::min(total, cap);
  if (total > cap) { g_err = "run: capacity exceeded"; return AVMO_ERR_CAPACITY; }
  return AVMO_OK;
}

}  // extern "C"
