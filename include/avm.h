/* avm.h — C ABI of libavm: microscopic (collision-by-collision) electron avalanche transport on one B200.
 *
 * What the library computes.  The hot path of the paper "Accelerating Garfield++ with CUDA"
 * (arxiv 2509.15377, PAPER.md): for every active electron an "electron transport" stage, then "stack
 * processing" (finished electrons removed, newly created ones added), repeated until every electron has a
 * non-zero status code (Fig. 2 at PAPER.md:89).  The transport stage is the semi-classical
 * null-collision Monte Carlo technique the paper names as its method's source (refs [8], [9] at
 * PAPER.md:189-190).  The paper prints no equations; every numeric choice is fixed by readings R1-R20 and
 * steps S0-S9 of SURVEY.md §8(c), restated in DESIGN.md §3.
 *
 * Conventions.
 *  - Units: cm, ns, eV, V/cm, tesla.  All arithmetic fp64; grid-map nodes are fp32 storage, fp64 arithmetic.
 *  - Every function returns int32_t: AVM_OK or a negative AVM_ERR_*; avm_last_error() gives a thread-local
 *    message.  No exception crosses the boundary.
 *  - The library NEVER allocates device memory and has no CPU fallback: the caller provides every device
 *    buffer and the CUDA stream (PyTorch in this repo: torch.empty(..., device="cuda"), stream handle).
 *  - "host" / "device" is stated for every pointer.  Host arrays are borrowed for the duration of the call;
 *    device buffers given at creation are borrowed until the matching destroy.
 *  - Work is enqueued on the context's stream.  avm_run and avm_fetch synchronise that stream before they
 *    return (a count is returned to the host); avm_step_batch and avm_field_eval do not.
 *  - Random numbers: counter-based Philox4x32-10, counter = (n, block, id_lo, id_hi), key = (seed_lo,
 *    seed_hi); n = the electron's collision index, id = its 64-bit id.  This replaces the paper's
 *    pre-generated numbers selected by electron ID: results do not depend on scheduling.
 */
#ifndef AVM_H
#define AVM_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { AVM_OK = 0, AVM_ERR_INVALID_ARG = -1, AVM_ERR_CAPACITY = -2, AVM_ERR_CUDA = -3, AVM_ERR_STATE = -4 };
/* collision level types */
enum { AVM_ELASTIC = 0, AVM_EXCITATION = 1, AVM_IONISATION = 2, AVM_ATTACHMENT = 3 };
/* electron status codes: "non-zero status code" = finished */
enum { AVM_ACTIVE = 0, AVM_LEFT_ZLO = 1, AVM_LEFT_ZHI = 2, AVM_LEFT_XY = 3, AVM_MATERIAL = 4,
       AVM_ATTACHED = 5, AVM_TIME_LIMIT = 6, AVM_STEP_LIMIT = 7 };
enum { AVM_MAX_LEVELS = 64, AVM_MAX_SLABS = 8 };

typedef struct avm_ctx avm_ctx;
typedef struct avm_gas avm_gas;
typedef struct avm_field avm_field;

/* Thread-local message of the last failing call on this thread ("" if none). */
const char* avm_last_error(void);

/* ---- context: "run on a chosen GPU" (SetRunModeOptions(mode, device)) ----------------
 * device: CUDA ordinal.  cuda_stream: a cudaStream_t (NULL = the legacy default stream).  The context
 * records device properties (SM count) used to size the persistent grid.  Fails with AVM_ERR_CUDA when the
 * device is missing or is not compute capability 10.x. */
int32_t avm_ctx_create(int32_t device, void* cuda_stream, avm_ctx** out);
int32_t avm_ctx_destroy(avm_ctx*);
/* Number of SMs of the context's device (grid sizing; reported by the bench). */
int32_t avm_ctx_sm_count(const avm_ctx*);

/* ---- gas: cumulative collision-rate tables ("GPU versions" of the Medium data; S6-S9) -------
 * All pointers HOST.  cum_rate[b][l] = sum of the rates [ns^-1] of levels 0..l in energy bin b; bins are
 * uniform on [0, e_max), bin = floor(e * n_bins / e_max), energies >= e_max use the last bin and are
 * counted (R5).  Rates are piecewise constant per bin.  nu_hat is the null-collision rate (R4); it must be
 * >= every cum_rate[b][n_levels-1]; <= 0 selects that maximum. */
typedef struct {
  int32_t n_bins;
  double e_max_eV;
  int32_t n_levels;               /* 1..AVM_MAX_LEVELS */
  const double* cum_rate;         /* host [n_bins][n_levels], non-decreasing along levels */
  const uint8_t* level_type;      /* host [n_levels], AVM_ELASTIC.. */
  const double* level_loss_eV;    /* host [n_levels]: threshold = energy loss (excitation, ionisation) */
  const double* level_recoil;     /* host [n_levels]: r = 2mM/(m+M)^2 (elastic) */
  const double* level_ob_w_eV;    /* host [n_levels]: Opal-Beaty w (ionisation) */
  double nu_hat;
  /* NEXT-3 (DESIGN.md §3.6 readings X1-X3; PAPER.md:121 for Penning transfer, the feature the paper had to
   * switch off).  All optional: NULL / 0 = the base model (isotropic deflection R9, no transfer, cold gas R8). */
  const double* scat_xi;            /* host [n_bins][n_levels]: forward-scattering parameter xi in (-1, 1) of the bin and
                                     * level: cos(theta) = (c0 + xi) / (1 + xi c0), c0 = 1 - 2 u3 (0 = isotropic) */
  const double* level_penning_prob; /* host [n_levels]: probability that an excitation of the level ionises the admixture */
  const double* level_penning_eV;   /* host [n_levels]: energy available to that electron (its energy is uniform in it) */
  double kT_eV;                     /* gas temperature for elastic collisions (0.02526 eV at 293.15 K); 0 = cold gas */
} avm_gas_desc;
/* Bytes of device memory avm_gas_create needs for this table (0 on an invalid description). */
size_t avm_gas_bytes(const avm_gas_desc*);
/* Validates the table, lays it out in dev_buf (DEVICE, >= avm_gas_bytes, 256-byte aligned; borrowed until
 * avm_gas_destroy) and uploads it on the context's stream.  Layout: DESIGN.md §4. */
int32_t avm_gas_create(avm_ctx*, const avm_gas_desc*, void* dev_buf, size_t dev_bytes, avm_gas** out);
int32_t avm_gas_destroy(avm_gas*);
/* The resolved null-collision rate [ns^-1]. */
double avm_gas_nu_hat(const avm_gas*);
/* The table of energy-banded null-collision rates avm_gas_create built for this gas (AVM_RUN_BANDED; DESIGN.md §3.5,
 * readings N1-N4, "revisiting the algorithms").  shape3 (HOST) = (K energy bands, J
 * acceleration classes, shift: a band is 2^shift energy bins); a2: HOST [J] squared upper edges of the classes
 * [(cm/ns^2)^2]; nu, dtmax: HOST [K][J + 1] rate [ns^-1] and validity time [ns] (+inf = no cut) per band and class, column
 * J = accelerations above every class.  a2, nu, dtmax may be NULL.  Lets the tests compare the table with the oracle's. */
int32_t avm_gas_bands(const avm_gas*, int32_t* shape3, double* a2, double* nu, double* dtmax);

/* ---- field: uniform, uniform + B, or regular-grid map(s) (S0, R14, R15) ---------------------------------
 * A stack of z-slabs, ascending and contiguous (slab[i].z_hi == slab[i+1].z_lo).  kind 2: see below.  kind 0: uniform field
 * vector E (the force on an electron is -E).  kind 1: regular grid of float4 nodes (Ex, Ey, Ez, gas-mask)
 * laid out [nz][ny][nx][4], trilinear interpolation (x, then y, then z); mask < 0.5 = solid material, the
 * electron is absorbed (R14).  bc 0: leaving the grid in x/y ends the electron (status 3); 1: periodic with
 * the given period; 2: mirror-periodic — fold into [0, period], the field component normal to the mirror
 * changes sign (R15).  The map is fp32 storage; all arithmetic on it is fp64.  B is one constant vector for the whole run (exact helical flight when non-zero).
 * xy_lo/xy_hi: absorbing bounds in x and y (+-inf allowed). */
typedef struct {
  double z_lo, z_hi;
  int32_t kind;
  double E[3];
  const float* nodes_dev;         /* DEVICE [nz][ny][nx][4], 16-byte aligned, borrowed until avm_field_destroy */
  int32_t nx, ny, nz;
  double origin[3], spacing[3];
  int32_t bc_x, bc_y;
  double period_x, period_y;
  double* nodes_f64_dev;          /* DEVICE scratch or NULL: [nz][ny][nx][4] doubles, 16-byte aligned, borrowed until
                                   * avm_field_destroy.  When given, avm_field_create widens the fp32 map into it once
                                   * (same values) and lookups read it: no float-to-double conversion per step, twice
                                   * the bytes.  Results are identical either way. */
  /* kind 2 (NEXT-2: SURVEY.md §8(f), DESIGN.md §3.8 readings F1-F4; PAPER.md:121 — the paper's maps are ANSYS meshes of
   * 10-node tetrahedra, found through an octree): an unstructured mesh of quadratic tetrahedra with straight
   * edges.  Coordinates are relative to `origin`, x and y after the fold of bc_x / bc_y (as for a grid; bc none: no fold).
   * tet_nodes[e] = 4 vertices, then the mid-edge nodes of edges (0,1) (0,2) (0,3) (1,2) (1,3) (2,3); node_V = potential
   * [V] at every node.  Inside an element V = sum_i V_i N_i(lambda) (N_vertex = l (2l - 1), N_edge = 4 l_a l_b), E = -grad V,
   * the mask is tet_gas[e] (1 gas, 0 solid); the element of a point is the lowest-numbered one whose barycentric
   * coordinates are all >= -1e-10; a point of the slab inside no element is solid (an unmeshed electrode).  The four host
   * arrays are read by avm_field_create only; mesh_dev (DEVICE, >= avm_tetmesh_bytes(slab), 256-byte aligned) receives the
   * per-element records and the bucket-grid index and is borrowed until avm_field_destroy. */
  int64_t n_mesh_nodes, n_tets;
  const double* node_xyz;         /* HOST [n_mesh_nodes][3] */
  const double* node_V;           /* HOST [n_mesh_nodes] */
  const int32_t* tet_nodes;       /* HOST [n_tets][10] */
  const uint8_t* tet_gas;         /* HOST [n_tets] */
  void* mesh_dev;
  size_t mesh_dev_bytes;
} avm_slab;
/* Bytes of device memory avm_field_create needs for the mesh of a kind-2 slab (0 for other kinds or an invalid mesh). */
size_t avm_tetmesh_bytes(const avm_slab*);
typedef struct {
  const avm_slab* slabs;          /* host [n_slabs], 1..AVM_MAX_SLABS */
  int32_t n_slabs;
  double B[3];
  double xy_lo[2], xy_hi[2];
} avm_field_desc;
int32_t avm_field_create(avm_ctx*, const avm_field_desc*, avm_field** out);
int32_t avm_field_destroy(avm_field*);
/* Field and gas-mask at n points.  r: DEVICE [3][n]; E: DEVICE [3][n]; mask: DEVICE [n]; slab: DEVICE [n]
 * (-1 = outside the domain).  Asynchronous on the context's stream. */
int32_t avm_field_eval(avm_ctx*, const avm_field*, int64_t n, const double* r, double* E, double* mask,
                       int32_t* slab);

/* ---- run: whole avalanches --------------------------------------------------------------
 * Primaries: [n_primaries][8] = x, y, z, t, energy, kx, ky, kz (AoS).  HOST by default (the H2D copy is part
 * of the call, as in the paper's timing convention); DEVICE with AVM_RUN_PRIMARIES_ON_DEVICE.
 * Primary p gets id = p + id_offset and avalanche index p; secondaries get id = Philox(n_s, 0xFFFFFFFF, parent
 * id) (R16) and inherit the avalanche index.  A primary outside the domain / inside material is finished at
 * its birth point with the corresponding status. */
enum {
  AVM_RUN_PRIMARIES_ON_DEVICE = 1u,
  /* bit 2u is unused (it was AVM_RUN_NO_TALLIES, a flag without effect: tallies are three per-thread counters) */
  /* Launch shape of the transport kernel.  Default: chosen from n_primaries (wide when the primaries alone outnumber
   * the lanes of the latency shape).  Results do not depend on the shape. */
  AVM_RUN_SHAPE_WIDE = 4u,        /* 768 threads per SM: most lanes, for runs that keep them busy */
  AVM_RUN_SHAPE_LATENCY = 8u,     /* 512 threads per SM with time-parallel batches: fewest cycles per step */
  /* Energy-banded null-collision rate (DESIGN.md §3.5 readings N1-N6): the rate of a flight is the
   * one of the electron's energy band and of the acceleration class of the field at its position (avm_gas_bands) instead
   * of the global nu_hat; a flight longer than the band's validity time is cut there and ends in a null collision.  The
   * same collision physics (thinning with a piecewise-constant majorant is exact) in 1.6-5x fewer steps; the random streams
   * are consumed differently, so a banded run is compared with a banded oracle run.  NOT identical at absorbing planes:
   * an electron is tested for having left the domain only where a flight ends, and banded flights are longer, so fewer
   * electrons are lost at a plane they start on or linger near (config 1, primaries on the cathode plane: mean gain +1.1 %,
   * share ending at the cathode -2.1 points against the global rate, N7).  Use the global rate when such
   * losses matter.  Runs take serial batches and full-warp
   * iterations only (no time-parallel batches: a flight's rate depends on the energy the previous flight ended with). */
  AVM_RUN_BANDED = 16u
};
/* NEXT-4 ("induced-signal accumulation (weighting-field dot velocity per flight) and ion drift";
 * what the endpoints feed; DESIGN.md §3.7 readings W1-W4).  weighting: the weighting field E_w [1/cm] of the
 * read-out electrode as an avm_field (uniform slabs or grid maps only — a field with a tetrahedral slab is refused with
 * AVM_ERR_INVALID_ARG; mask and B ignored; E_w = 0 outside it).  Every step
 * r -> r' of a charge q [e] that starts at time t adds q E_w . (r' - r) to signal_dev[floor((t - t0) / dt_bin)]; steps that
 * start outside the bins are dropped.  Electron flights: q = -1, E_w at r.  signal_dev: DEVICE [n_bins] doubles, ADDED to
 * (the caller zeroes it); induced charge per bin, current = charge / dt_bin. */
typedef struct {
  const avm_field* weighting;
  double t0, dt_bin;
  int32_t n_bins;
  double* signal_dev;
} avm_signal;

typedef struct {
  uint64_t seed;
  double t_max;                   /* ns; electrons with t > t_max stop with status 6 (+inf: none) */
  uint32_t flags;
  uint32_t max_iters_per_launch;  /* guard: working iterations per warp and launch (0 = default 2^22); the warp that
                                   * reaches it stops the launch, live electrons are parked, the host relaunches */
  uint64_t id_offset;             /* id of primary 0 (replicas / shards of one job use disjoint ranges) */
  int32_t max_ctas;               /* 0 = one CTA per SM; else at most this many CTAs (results do not depend on it) */
  const avm_signal* signal;       /* HOST struct or NULL: accumulate the electrons' induced signal during the run */
} avm_run_opts;

/* Caller-provided DEVICE buffers; `capacity` = maximum number of electrons ever created (primaries +
 * secondaries).  Slot s holds electron s for the whole run: while the electron is active its `end` column
 * is its live state, afterwards its endpoint.  Slots are in creation order (primaries first); the order of
 * secondaries is unspecified (compare after sorting by id, R17).  id, avalanche, status, n_steps and end are
 * required; per_avalanche and tallies_* may be NULL; birth may be NULL only when tallies_f64 is NULL too
 * (the flight sums are taken as sum over electrons of endpoint - birth point). */
typedef struct {
  int64_t capacity;
  void* workspace;                /* DEVICE, >= avm_run_workspace_bytes(capacity), 256-byte aligned */
  size_t workspace_bytes;
  uint64_t* id;                   /* [capacity] */
  uint32_t* avalanche;            /* [capacity] */
  int32_t* status;                /* [capacity] */
  uint32_t* n_steps;              /* [capacity] collision index n reached (real + null steps taken) */
  double* birth;                  /* [5][capacity]: x0, y0, z0, t0, e0; may be NULL */
  double* end;                    /* [8][capacity]: x1, y1, z1, t1, e1, kx, ky, kz */
  uint64_t* per_avalanche;        /* [n_primaries][3]: endpoints, ions (= endpoints - 1), negative ions; may be NULL */
  uint64_t* tallies_u64;          /* [n_levels + 5]: per level, null, real, energy overflow, steps, Penning transfers; may be NULL */
  double* tallies_f64;            /* [5]: sum dx, dy, dz over all flights, sum dt, sum energy loss; may be NULL */
} avm_outputs;
size_t avm_run_workspace_bytes(const avm_ctx*, int64_t capacity);
/* Runs all avalanches to completion.  *n_endpoints_out = electrons created = endpoints written (<= capacity).
 * AVM_ERR_CAPACITY: more than `capacity` electrons would exist; the run still terminates, outputs hold the
 * electrons that fit (children that did not fit are dropped and counted in the message).
 * A signal or a gas with NEXT-3 extensions needs the kernel variant that keeps the threshold table in shared memory: gases of
 * more than ~24000 energy bins are refused for those runs (AVM_ERR_INVALID_ARG, before anything is queued). */
int32_t avm_run(avm_ctx*, const avm_gas*, const avm_field*, const double* primaries, int64_t n_primaries,
                const avm_run_opts*, const avm_outputs*, int64_t* n_endpoints_out);
/* avm_run for callers that have no device workspace to give.
 *
 * Who this is for.  avm_run needs a `workspace`: scratch in device memory that the persistent transport kernel uses for
 * its run-control block (live / created electron counters, the ticket queue head, per-CTA stop flags, the tally
 * accumulators) and that stages the primaries' host-to-device copy.  Normally the caller allocates it next to the output
 * arrays.  Some callers cannot: a plug-in that is handed its output buffers by a host framework and is forbidden to call
 * the CUDA allocator itself; a service whose memory pool is sized and frozen at start-up; code that runs where
 * cudaMalloc would synchronise the device or is simply not permitted.  For them the library carries ONE fixed scratch
 * block of its own: a file-scope `static __device__` array in the library image, avm_run_static_bytes() bytes (4 MiB +
 * 36 KiB), which every GPU that loads the library holds from module load until the process exits, used or not.
 *
 * What it does.  Exactly avm_run — same kernels, same arguments, same results, same return codes — except that
 * outputs->workspace and outputs->workspace_bytes are IGNORED (pass NULL / 0) and the built-in block is used instead.
 * All input and output arrays are still the caller's.  The call itself allocates nothing: no cudaMalloc, cudaFree, or
 * library routine that allocates device memory is reached from it.
 *
 * Limit.  outputs->capacity <= AVM_RUN_STATIC_MAX_CAPACITY (65536 electrons, primaries + secondaries: the staging part of
 * the block is sized for that many primaries).  A larger capacity fails at once with AVM_ERR_INVALID_ARG and a message
 * that names the limit; nothing is queued.  Use avm_run with your own workspace for bigger runs.
 *
 * First call on a device.  The array's device address is looked up (cudaGetSymbolAddress, with the context's device
 * current) the first time the entry point is called for that device, and remembered.  Make that first call outside any
 * CUDA stream capture.
 *
 * Sharing.  There is one block per GPU and every avm_run_static call on that GPU uses it, whatever the context or the
 * stream.  It still holds the previous call's contents when the next one starts; the call re-zeroes the run-control part
 * on its stream before any kernel reads it, and the staging part is overwritten before it is read, so nothing of an
 * earlier run leaks into a later one.  Because avm_run synchronises its stream before it returns, calls made one after
 * the other from one host thread never overlap.  Calls issued from different host threads of one process to the same
 * GPU at the same time DO overlap on the device and race on the block: serialise them yourself.  (Separate processes
 * each load their own copy of the library image, so they do not share a block.) */
enum { AVM_RUN_STATIC_MAX_CAPACITY = 65536 };
size_t avm_run_static_bytes(void);
int32_t avm_run_static(avm_ctx*, const avm_gas*, const avm_field*, const double* primaries, int64_t n_primaries,
                       const avm_run_opts*, const avm_outputs*, int64_t* n_endpoints_out);
/* Launch statistics of the last avm_run on this context: kernels launched, persistent-kernel launches. */
int32_t avm_run_stats(const avm_ctx*, int64_t* n_kernel_launches, int64_t* n_transport_launches);
/* Device time [ms] of the transport-kernel launches of the last avm_run on this context, summed (CUDA events
 * recorded on the context's stream around each launch).  *ms_out is HOST.  bench.py's roofline uses it. */
int32_t avm_run_transport_ms(const avm_ctx*, float* ms_out);

/* Ion drift after a run (W3, W4).  Every electron s >= n_primaries left a positive ion at its birth point, every attached
 * electron (status 5) a negative ion at its endpoint.  Ion i = s (positive) or n + s (negative) of 2 n entries; status -1 =
 * no such ion.  An ion of charge q moves with v = q mu E(r), mu the mobility [cm^2 / (V ns)], integrated by the explicit
 * midpoint rule in steps of fixed LENGTH step_cm (k1 = v(r), r_m = r + (step/2) k1/|k1|, k2 = v(r_m), r' = r + step k2/|k2|,
 * dt = step / |k2|); it stops at the first sampled point outside the domain (status 1-3), inside material (4), after t_max
 * (6), after max_steps or where the field vanishes (7).  With a signal, each step adds q E_w(r_m) . (r' - r) to the bin of the
 * step's start time.  run: the avm_outputs of the finished avm_run (birth, end, status DEVICE arrays are read; n = its
 * endpoint count).  ion_end: DEVICE [4][2n] x, y, z, t; ion_status: DEVICE [2n]; ion_steps: DEVICE [2n].  Asynchronous on
 * the context's stream.  n_primaries <= n <= run->capacity is required; slots whose status is <= 0 (no finished electron:
 * n was larger than the run's endpoint count) yield no ion (status -1). */
typedef struct { double mobility_pos, mobility_neg, step_cm, t_max; int32_t max_steps; } avm_ion_opts;
int32_t avm_ion_drift(avm_ctx*, const avm_field* field, const avm_signal* signal, const avm_ion_opts*, const avm_outputs* run,
                      int64_t n, int64_t n_primaries, double* ion_end, int32_t* ion_status, uint32_t* ion_steps);

/* Device -> host copy of the first n entries of every non-NULL array of `host` from the same-named array of
 * `dev` ("retrieve the electron endpoints").  `host` is an avm_outputs whose pointers are HOST
 * arrays with leading dimension host->capacity (workspace ignored); per_avalanche needs n_primaries,
 * tallies_u64 needs n_levels (0 skips them).  Synchronises the stream. */
int32_t avm_fetch(avm_ctx*, const avm_outputs* dev, int64_t n, int64_t n_primaries, int32_t n_levels,
                  const avm_outputs* host);

/* ---- parity hook: ONE step S0-S9 from each of n given states (no loop, no append) -----------------------
 * All arrays DEVICE, length n ([8][n] for states = x,y,z,t,e,kx,ky,kz).  event: -1 null collision, l >= 0
 * selected level, -2 terminated before the collision decision.  status: as above.  bin: energy bin used
 * (-1 if not reached).  child/child_id: valid where the level is an ionisation, else zero. */
int32_t avm_step_batch(avm_ctx*, const avm_gas*, const avm_field*, uint64_t seed, double t_max, int64_t n,
                       const double* state_in, const uint64_t* id, const uint32_t* n_idx, double* state_out,
                       int32_t* event, int32_t* status, int32_t* bin, double* child_out, uint64_t* child_id);

/* The same hook through the step FORMS the persistent kernel runs (the device functions of
 * csrc/avm_forms.cuh, shared by the kernel and this hook) — north_star "per-collision steps ... relative 1e-12" on the
 * instruction sequences that earn the bench number (PAPER.md:65-69 for what a step is).
 *  form 0: the general sequence (= avm_step_batch).  Arrays of length n.
 *  form 1: the full-warp form: 16-bit threshold filter + exact record inside a band, the next flight's draws hoisted
 *          behind the record load, deflection drawn in the collision phase.  Arrays of length n.
 *  form 2: one time-parallel batch per warp (one uniform slab only): k electrons per warp (1..16, n a multiple of k) on
 *          scattered lanes, gl = 32 / 2^ceil(log2 k) consecutive steps of each, evaluated as composed flights.
 *  form 3: one serial batch per warp (any field): cooperative draws through shared memory, then every owner lane takes
 *          its electron's gl steps one after the other in straight-line code.  Same k, gl and layout as form 2.
 *          For forms 2 and 3 the output arrays have n * gl entries ([8][n * gl] for states): entry i * gl + s = the result of step s of electron i,
 *          in the sense of avm_step_batch (state after the step, event, status, bin, child).  Entries of steps the
 *          electron does not reach (it finished earlier in the batch) are left untouched: pre-fill event with -3.
 * k is ignored for forms 0 and 1.  flags: 0 or AVM_RUN_BANDED (forms 1 and 3 only: the forms a banded run takes). */
int32_t avm_step_batch_form(avm_ctx*, const avm_gas*, const avm_field*, uint64_t seed, double t_max, int32_t form,
                            int32_t k, int64_t n, const double* state_in, const uint64_t* id, const uint32_t* n_idx,
                            double* state_out, int32_t* event, int32_t* status, int32_t* bin, double* child_out,
                            uint64_t* child_id, uint32_t flags);

/* Philox block (seed, id, n, block) -> words[4] and two uniforms, for n_items items.  All arrays DEVICE.
 * Pin C1: lets the tests compare the device generator bit for bit. */
int32_t avm_philox_batch(avm_ctx*, uint64_t seed, int64_t n_items, const uint64_t* id, const uint32_t* n_idx,
                         const uint32_t* block, uint32_t* words_out /*[n_items][4]*/, double* u_out /*[n_items][2]*/);

/* FP64 issue-rate probe: runs a chain of dependent-free DFMA streams (n_threads threads, iters iterations of
 * 8 independent FMAs each) and writes the elapsed milliseconds; used by bench.py to measure the ALU roofline
 * denominator on the box it runs on.  sink: DEVICE [n_blocks * n_threads_per_block] doubles. */
int32_t avm_fp64_probe(avm_ctx*, int32_t n_blocks, int32_t n_threads_per_block, int64_t iters, double* sink,
                       float* ms_out /*host*/);

/* Random-gather probe: every thread issues `iters` independent 32-byte (one-sector) loads at random sector indices of
 * the working set buf[0, bytes), bypassing L1.  With the working set inside L2 it measures the L2-resident random-sector
 * rate, far beyond L2 the HBM one: the denominators of the field-gather roofline of the map configs (SURVEY.md §7 stage
 * 0, §8(d): steps/s x 128 B / measured gather bandwidth; PAPER.md:83 for the field data that is gathered).  buf: DEVICE,
 * 32-byte aligned, contents irrelevant; sink: DEVICE [n_blocks * n_threads_per_block] u64; n_threads_per_block <= 256.
 * Bytes moved = n_blocks * n_threads_per_block * iters * 32. */
int32_t avm_gather_probe(avm_ctx*, const void* buf, size_t bytes, int32_t n_blocks, int32_t n_threads_per_block,
                         int64_t iters, uint64_t* sink, float* ms_out /*host*/);
/* Shared-memory random-load probe: `iters` random 8-byte loads per thread from a table of table_bytes in dynamic shared
 * memory (the access pattern of the threshold table, one record per step).  sink as above;
 * n_threads_per_block <= 512.  Loads = n_blocks * n_threads_per_block * iters. */
int32_t avm_smem_probe(avm_ctx*, int32_t table_bytes, int32_t n_blocks, int32_t n_threads_per_block, int64_t iters,
                       uint64_t* sink, float* ms_out /*host*/);

#ifdef __cplusplus
}
#endif
#endif
