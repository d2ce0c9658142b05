/* avmo — the ORACLE: plain, serial, slow, obviously-correct CPU implementation of microscopic electron
 * avalanche transport (null-collision Monte Carlo).  TEST INFRASTRUCTURE ONLY: used by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.  It shares no code with the
 * CUDA path (paper_2509_15377_b200/csrc/) and the product never routes through it.
 *
 * What it follows.  The paper (arxiv 2509.15377, /root/reference/PAPER.md) describes the algorithm only in
 * outline: "electron transport" for every active electron, then "stack processing", until every electron
 * has a non-zero status (Fig. 2 at PAPER.md:89); it names its method's sources as the
 * semi-classical null-collision Monte Carlo technique (ref [8]) over per-process cross
 * sections (ref [9]).  Every numeric choice the paper leaves open is fixed by the readings
 * R1-R20 and steps S0-S9 of SURVEY.md §8(c), restated in DESIGN.md §3; the functions below cite them.
 *
 * Units: cm, ns, eV, V/cm, tesla.  All arithmetic fp64; grid nodes are fp32 storage, fp64 arithmetic.
 * All pointers are HOST pointers.  Parity status of each function: see DESIGN.md §5 (pins C1-C17 of the base model; the
 * NEXT rows' pins: tests/test_oracle_pins_banded.py, _next2.py, _next3.py, _next4.py — every function has a pin);
 * absolute values of the synthetic-gas results (gain, alpha, W of configs 1-5) are "parity unpinned"
 * (no reference values exist anywhere) — they are pinned GPU-vs-oracle only.
 */
#ifndef AVMO_H
#define AVMO_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { AVMO_OK = 0, AVMO_ERR_INVALID_ARG = -1, AVMO_ERR_CAPACITY = -2 };
enum { AVMO_ELASTIC = 0, AVMO_EXCITATION = 1, AVMO_IONISATION = 2, AVMO_ATTACHMENT = 3 };
enum { AVMO_ACTIVE = 0, AVMO_LEFT_ZLO = 1, AVMO_LEFT_ZHI = 2, AVMO_LEFT_XY = 3, AVMO_MATERIAL = 4,
       AVMO_ATTACHED = 5, AVMO_TIME_LIMIT = 6, AVMO_STEP_LIMIT = 7 };

typedef struct {
  int32_t n_bins;  double e_max_eV;
  int32_t n_levels;
  const double*  cum_rate;        /* [n_bins][n_levels] ns^-1, non-decreasing along levels */
  const uint8_t* level_type;
  const double*  level_loss_eV;
  const double*  level_recoil;
  const double*  level_ob_w_eV;
  double nu_hat;                  /* <= 0: max_b cum_rate[b][L-1] */
  /* NEXT-3 (DESIGN.md §3.6 readings X1-X3); every one optional (NULL / 0 = the base model R8, R9): */
  const double*  scat_xi;            /* X1 [n_bins][n_levels]: forward-scattering parameter xi in (-1, 1) of S9b, 0 = isotropic */
  const double*  level_penning_prob; /* X2 [n_levels]: probability that an excitation of the level ionises the admixture */
  const double*  level_penning_eV;   /* X2 [n_levels]: energy available to that electron (excitation energy - ionisation potential) */
  double kT_eV;                      /* X3: gas temperature (0.02526 eV at 293.15 K); 0 = cold gas */
} avmo_gas_desc;

typedef struct {
  double z_lo, z_hi;  int32_t kind;           /* 0 uniform, 1 grid */
  double E[3];
  const float* nodes;                          /* grid: [nz][ny][nx][4] = Ex,Ey,Ez,mask */
  int32_t nx, ny, nz;  double origin[3], spacing[3];
  int32_t bc_x, bc_y;                          /* 0 none, 1 periodic, 2 mirror */
  double period_x, period_y;
  /* kind 2 (NEXT-2; DESIGN.md §3.8 readings F1-F4): an unstructured mesh of 10-node (quadratic)
   * tetrahedra with straight edges, as ANSYS SOLID123 exports them.  Coordinates are relative to `origin`
   * (x, y after the fold of bc_x / bc_y, as for a grid).  tet_nodes[e] = 4 vertices then the mid-edge nodes of edges
   * (0,1) (0,2) (0,3) (1,2) (1,3) (2,3); node_V = potential [V] at every node; tet_gas[e] = 1 gas, 0 solid.  Inside an
   * element V = sum_i V_i N_i(lambda), N_vertex = l(2l - 1), N_edge = 4 l_a l_b, E = -grad V; the mask is the element's flag;
   * a point of the slab inside no element is solid (an unmeshed electrode). */
  int64_t n_mesh_nodes, n_tets;
  const double* node_xyz;                      /* [n_mesh_nodes][3] */
  const double* node_V;                        /* [n_mesh_nodes] */
  const int32_t* tet_nodes;                    /* [n_tets][10] */
  const uint8_t* tet_gas;                      /* [n_tets] */
} avmo_slab;

typedef struct { const avmo_slab* slabs; int32_t n_slabs; double B[3]; double xy_lo[2], xy_hi[2]; } avmo_field_desc;

/* flags.  AVMO_BANDED: the null-collision rate of a flight is the one of the
 * electron's energy band and of the flight's acceleration class instead of the global maximum; flights longer than the
 * band's validity time are cut and count as null collisions.  Same physics, fewer null steps, other random streams. */
enum { AVMO_BANDED = 1u };
/* NEXT-4 (DESIGN.md §3.7 readings W1-W4): induced-signal accumulation (Shockley-Ramo).  weighting = the
 * weighting field E_w [1/cm] of the read-out electrode as a field description (mask and B ignored; outside it E_w = 0).
 * Every flight r -> r' that starts at time t adds q E_w(r) . (r' - r), q = -1, to signal[floor((t - t0) / dt_bin)] (flights
 * starting outside the bins are dropped).  signal: [n_bins] induced charge per bin in units of e, ADDED to. */
typedef struct { const avmo_field_desc* weighting; double t0, dt_bin; int32_t n_bins; double* signal; } avmo_signal;
/* id_offset: primary p gets electron id id_offset + p (shards of one job use disjoint id ranges); avalanche stays p. */
typedef struct { uint64_t seed; double t_max; int32_t n_threads; uint64_t id_offset; uint32_t flags;
                 const avmo_signal* signal; /* NULL: none */ } avmo_run_opts;

/* Ion drift (W3, W4): every electron s >= n_primaries left a positive ion at its birth point, every attached electron
 * (status 5) a negative ion at its endpoint.  Ion i = s (positive) or n + s (negative) of 2 n entries; status -1 = no such
 * ion.  An ion of charge q moves with v = q mu E(r) (mu: mobility [cm^2 / (V ns)], constant), integrated by the explicit
 * midpoint rule in steps of fixed LENGTH step_cm: k1 = v(r), r_m = r + (step/2) k1/|k1|, k2 = v(r_m), r' = r + step k2/|k2|,
 * dt = step / |k2|; it stops at the first sampled point outside the domain (status 1-3), inside material (4), after t_max
 * (6), after max_steps or where the field vanishes (7).  With a signal, each step adds q E_w(r_m) . (r' - r) to the bin of
 * the step's start time.  ion_end: [4][2n] x, y, z, t. */
typedef struct { double mobility_pos, mobility_neg, step_cm, t_max; int32_t max_steps; } avmo_ion_opts;
int32_t avmo_ion_drift(const avmo_field_desc* field, const avmo_signal* signal, const avmo_ion_opts* opts, int64_t n,
                       int64_t n_primaries, int64_t ld_birth, const double* birth /*[5][ld]*/, int64_t ld_end,
                       const double* end /*[8][ld]*/, const int32_t* status, double* ion_end, int32_t* ion_status,
                       uint32_t* ion_steps);

typedef struct {
  int64_t capacity;
  uint64_t* id; uint32_t* avalanche; int32_t* status; uint32_t* n_steps;
  double* birth;            /* [5][capacity]: x0,y0,z0,t0,e0 */
  double* end;              /* [8][capacity]: x1,y1,z1,t1,e1,kx,ky,kz */
  uint64_t* per_avalanche;  /* [Np][3]: endpoints, ions, negative ions */
  uint64_t* tallies_u64;    /* [n_levels+6]: per level, null, real, overflow, steps, Penning transfers, banded-rate violations (always 0) */
  double*   tallies_f64;    /* [5]: sum dx,dy,dz over all flights, sum dt, sum energy loss */
} avmo_outputs;

/* Philox4x32-10 block for (seed, electron id, collision index n, block) -> 4 words / 2 uniforms. */
void avmo_philox(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, uint32_t out[4]);
void avmo_uniform_pair(uint64_t seed, uint64_t id, uint32_t n, uint32_t block, double out[2]);

/* Field at n points r[3][n] -> E[3][n], mask[n], slab[n] (-1 outside the domain / bounds). */
int32_t avmo_field_eval(const avmo_field_desc*, int64_t n, const double* r, double* E, double* mask, int32_t* slab);

/* One step S0-S9 each from given states (state [8][n] = x,y,z,t,e,kx,ky,kz).  Outputs: state_out [8][n];
 * event[n]: -1 null collision, l>=0 selected level, -2 terminated before the collision decision;
 * status[n]; bin[n] (-1 if not reached); child [8][n] + child_id[n] valid where level type is ionisation. */
int32_t avmo_step_batch(const avmo_gas_desc*, const avmo_field_desc*, uint64_t seed, double t_max, int64_t n,
                        const double* state_in, const uint64_t* id, const uint32_t* n_idx,
                        double* state_out, int32_t* event, int32_t* status, int32_t* bin,
                        double* child_out, uint64_t* child_id, uint32_t flags);

/* The table of banded rates built for this gas (pins): shape3 = (K bands, J classes, shift); a2 [J] squared class edges;
 * nu, dtmax [K][J+1].  Any output pointer may be NULL. */
int32_t avmo_majorant(const avmo_gas_desc*, int32_t* shape3, double* a2, double* nu, double* dtmax);

/* Whole avalanches: stack driver.  primaries: [Np][8] AoS.  Returns AVMO_ERR_CAPACITY when more than
 * `capacity` electrons are created (outputs then hold the first `capacity` finished ones). */
int32_t avmo_run(const avmo_gas_desc*, const avmo_field_desc*, const double* primaries, int64_t n_primaries,
                 const avmo_run_opts*, avmo_outputs*, int64_t* n_endpoints_out);

const char* avmo_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
