/*
 * md_b200.h -- C ABI of the B200-native short-range molecular-dynamics hot path
 *              of arXiv 1009.4330 (Trott, Winterfeld, Crozier, "General-purpose
 *              molecular dynamics simulations on GPU-based clusters").
 *
 * The library (libmd_b200.so, hand-written CUDA for sm_100a) owns all device
 * state of one periodic orthogonal box of N atoms and runs, on ONE GPU:
 *
 *   cell binning + counting sort + spatial reorder      ("spatially ordered")
 *   Verlet neighbor-list build, full or half            (numneigh[i], neighbors[i][jj])
 *   pair forces: LJ 12-6, two-pass EAM (analytic and tabulated), Buckingham + cutoff Coulomb
 *                                                       (App. A)
 *     one thread (TpA, L88-104), 2 / 4 / 8 lanes or a warp per list row with shuffle
 *     reduction (the paper's block-per-atom BpA, L105-122), direct cell list (L64-82),
 *     chosen by a setup-time mini benchmark (L137)
 *   velocity-Verlet NVE and Nose-Hoover NVT, positions/velocities/forces resident on the device (L50-58)
 *   rebuild iff max_i |x_i - x0_i|^2 > (skin/2)^2, decided on the device.
 *   md_run keeps the host out of the loop: one fused launch per time step (two for EAM) with programmatic dependent
 *   launch, the rebuild flag read once per batch of steps, rebuilds enqueued without waiting and replayed as a CUDA graph.
 *
 * Conventions
 *   - Every call returns MD_OK (0) or a negative MD_ERR_*; nothing throws or
 *     aborts across the ABI.  md_last_error() gives the text of the last failure.
 *   - The handle owns all device memory.  Caller buffers are only read or
 *     written during the call; they may be HOST or DEVICE pointers (detected
 *     with cudaPointerGetAttributes; pageable or pinned host memory both work).
 *   - Per-atom arrays are N x 3 AoS doubles in the CALLER'S atom order; the
 *     spatial permutation the library applies internally is invisible.
 *   - All work is enqueued on the stream given to md_create (a cudaStream_t
 *     passed as void*; NULL = the legacy default stream).  Calls that return
 *     host scalars or fill host buffers synchronise that stream.
 *   - Units are the caller's: accelerations are f/m * ftm2v, kinetic energy is
 *     1/2 m v^2 * mvv2e (LJ reduced units: 1, 1; LAMMPS-metal: see md_set_units).
 *   - Precision modes: MD_FP64 computes everything in double;
 *     MD_MIXED computes pair terms in fp32 from tile-centred fp32 coordinates and
 *     accumulates per-atom sums, energy and virial in fp64; positions,
 *     velocities, forces, the list-build distance test and the integrator are
 *     fp64 in both modes.
 */
#ifndef MD_B200_H
#define MD_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct md_system md_system; /* opaque */

/* error codes */
#define MD_OK 0
#define MD_ERR_BAD_ARGUMENT (-1)   /* NULL pointer, N <= 0, unknown enum, bad parameter count ... */
#define MD_ERR_BOX_TOO_SMALL (-2)  /* some box edge < 3 (rc + skin): the 27-cell stencil would double count */
#define MD_ERR_CUDA (-3)           /* a CUDA runtime call failed; text in md_last_error */
#define MD_ERR_OVERFLOW (-4)       /* a tile or neighbor row outgrew its capacity even after re-planning */
#define MD_ERR_NOT_READY (-5)      /* positions or pair style not set yet */
#define MD_ERR_NONFINITE (-6)      /* a non-finite coordinate reached the binning kernel */

/* precision modes */
#define MD_FP64 0
#define MD_MIXED 1

/* pair styles */
#define MD_PAIR_LJ126 1   /* params = {eps, sigma}:   u = 4 eps [(s/r)^12 - (s/r)^6], plain cut at rc (lj/cut, L256) */
#define MD_PAIR_EAM_FS 2  /* params = {A, p, B, q, r0}: phi = A exp(-p(r/r0-1)), rho = exp(-q(r/r0-1)),
                             F(rho) = -B sqrt(rho), F'(0) := 0; E = sum_i F(rho_i) + 1/2 sum_ij phi (L260) */

#define MD_PAIR_EAM_TAB 4  /* params = {dr, drho}: the same two-pass EAM with rho(r), phi(r) on the grid r_k = k dr and F(rho) on
                             rho_k = k drho, given by md_set_eam_tables (App. A: what the paper's
                             EAM run used; reading s26): cubic Hermite interpolation per interval with centred-difference node
                             slopes; the force uses the derivative of the interpolant */
#define MD_PAIR_BUCK_COUL 3 /* params = {k}: u_ab = A_ab exp(-r/rho_ab) - C_ab/r^6 + k q_a q_b / r, all three terms cut plainly at rc
                             (App. A "silicate (cutoff)", LAMMPS buck/coul/cut).  Per type pair
                             A, rho, C by md_set_pair_coeff, per type charge by md_set_type_charges; at most 4 types;
                             k = 14.399645 eV A / e^2 in metal units */

/* thermostats (md_set_thermostat) */
#define MD_THERMO_NONE 0         /* NVE */
#define MD_THERMO_NOSE_HOOVER 1  /* NVT: one Nose-Hoover thermostat */

/* neighbor-list kinds */
#define MD_LIST_FULL 0    /* both (i,j) and (j,i): each kernel row writes only f[i] (L104) */
#define MD_LIST_HALF 1    /* each pair once; -F scattered to j with atomics (Newton's third law, L76) */

/* force-kernel variants */
#define MD_KERNEL_AUTO 0     /* setup-time mini benchmark picks among TPA / SUBWARP2 / SUBWARP4 / SUBWARP / WARP (L137) */
#define MD_KERNEL_TPA 1      /* one thread per atom (L88-104) */
#define MD_KERNEL_SUBWARP 2  /* 8 lanes per atom, shuffle reduction */
#define MD_KERNEL_WARP 3     /* 32 lanes per atom, shuffle reduction (the paper's BpA, L105-122) */
#define MD_KERNEL_CELL 4     /* no list: every atom scans the 27-cell stencil of its tile (L64-82) */
#define MD_KERNEL_SUBWARP4 5 /* 4 lanes per atom, shuffle reduction: fills the SM when a tile holds few atoms with long rows */
#define MD_KERNEL_SUBWARP2 6 /* 2 lanes per list row, shuffle reduction */

typedef struct md_stats {
  int64_t natoms;
  int64_t nsteps_total;        /* time steps integrated since md_create */
  int64_t nbuilds;             /* neighbor-list builds since md_create */
  int64_t nforce_evals;        /* force evaluations since md_create */
  int32_t kernel_variant;      /* MD_KERNEL_* actually in use (AUTO resolved) */
  int32_t list_kind;
  int32_t precision;
  int32_t lanes_per_atom;      /* 1, 4, 8 or 32 */
  int32_t ncells[3];           /* cell grid */
  int32_t brick[3];            /* cells per tile edge (interior) */
  int32_t ntiles;              /* thread blocks per force launch */
  int32_t tile_capacity;       /* staged atoms a tile can hold */
  int32_t max_tile_atoms;      /* largest staged count seen at the last build */
  int32_t max_neighbors;       /* most neighbors of any atom in the current list (exact fp64 pair set, counted on demand) */
  int32_t row_capacity;        /* list row capacity (entries) */
  int32_t list_balanced;       /* 1: the current list's rows have been permuted for conflict-free gathers (long-lived lists only) */
  double mean_neighbors;       /* mean neighbors per atom in the current list (exact fp64 pair set, counted on demand) */
  double kinetic_energy;       /* 1/2 sum m v^2 mvv2e at the time of the call */
  double ms_build;             /* device time of the last list build (bin+sort+build), CUDA events */
  double ms_force;             /* device time of the last md_compute_forces */
  double ms_run;               /* device time of the last md_run */
  int64_t launches_last_run;   /* kernels launched by the last md_run */
  int64_t launches_total;      /* kernels launched since md_create */
  /* phase timers of the last md_run (CUDA events on the library's stream, inside the run) */
  double ms_force_sampled;     /* summed device time of the force launches of the sampled steps */
  int64_t nforce_sampled;      /* how many steps were sampled (every ceil(nsteps/128)-th) */
  double ms_build_in_run;      /* summed device time of the list builds (bin+sort+reorder+build) */
  int64_t nbuilds_in_run;      /* list builds inside the last md_run */
  /* the STORED rows: one per pair of consecutive atoms of a cell, holding the union of the two atoms' neighbors
   * (a superset of the fp64 pair set, see md_get_neighbor_rows) */
  int32_t max_row;             /* longest stored row at the last build */
  int32_t reserved0;
  double mean_row;             /* mean stored row length at the last build (entries per pair of atoms) */
  double ms_force_pass1_sampled; /* EAM: the share of ms_force_sampled spent in pass 1 (density + embedding); 0 for LJ */
} md_stats;

/* Creates a system: orthogonal periodic box [0,Lx) x [0,Ly) x [0,Lz), N atoms with type ids in
 * 0..ntypes-1 (caller order, host or device pointer; ids outside the range are refused) and per-type masses
 * (host pointer).  stream: a cudaStream_t (void*), NULL for the default stream.
 * ("N atoms in a periodic box"; north_star md_create(box, N, types)) */
int md_create(md_system** out, const double box[3], int64_t N, const int32_t* types, int ntypes,
              const double* mass, void* cuda_stream);
/* Frees the handle and all device memory it owns.  NULL is allowed.  (north_star: the handle owns the device state) */
void md_destroy(md_system* s);

/* Unit factors of the integrator (PAPER.md L52 NVE; reading s14 of DESIGN.md: the paper runs LAMMPS "metal" units for
 * the EAM workload, App. A): a = f/m * ftm2v, KE = 1/2 m v^2 * mvv2e.  LJ reduced units: (1, 1).
 * LAMMPS-metal (A, eV, amu, ps): ftm2v = 1/1.0364269e-4, mvv2e = 1.0364269e-4.  Both must be positive. */
int md_set_units(md_system* s, double ftm2v, double mvv2e);
/* MD_FP64 or MD_MIXED ("single, double and mixed precision"; reading s15).  Invalidates the
 * neighbor list and the variant choice. */
int md_set_precision(md_system* s, int mode);
/* Positions (north_star: resident on the device): N x 3 doubles, caller order, host or device.  They may
 * lie outside the box (wrapped at the next build, reading s5); a non-finite value is reported by the next build as
 * MD_ERR_NONFINITE.  Setting positions invalidates the neighbor list and the cached forces. */
int md_set_positions(md_system* s, const double* x);
/* Velocities (PAPER.md L52 velocity Verlet; reading s17: generated by the caller): N x 3 doubles, caller order,
 * host or device. */
int md_set_velocities(md_system* s, const double* v);
/* Pair style, its parameters (see MD_PAIR_*), cutoff rc and skin (PAPER.md L86-98 neighbor lists with a skin, App. A
 * L256/L260; north_star md_set_pair(style, params, rc, skin)).  MD_PAIR_LJ126 and MD_PAIR_EAM_FS take one parameter set for all
 * type pairs (types select masses); MD_PAIR_BUCK_COUL takes per-type-pair coefficients through md_set_pair_coeff.  The interaction is r^2 < rc^2 strictly (reading s3).  Fails with MD_ERR_BOX_TOO_SMALL unless every box
 * edge >= 3 (rc + skin) (reading s19), MD_ERR_BAD_ARGUMENT for a wrong parameter count or a non-finite value. */
int md_set_pair(md_system* s, int style, const double* params, int nparams, double rc, double skin);
/* MD_PAIR_BUCK_COUL only: the coefficients {A, rho, C} (n = 3) of the type pair (a, b) and, by symmetry, (b, a)
 * (App. A "26 pair force styles": per-type-pair coefficients as in LAMMPS pair_coeff).  Every pair of
 * the system's types must be set before the next force evaluation (MD_ERR_NOT_READY otherwise); rho must be positive. */
int md_set_pair_coeff(md_system* s, int type_a, int type_b, const double* coeff, int n);
/* MD_PAIR_EAM_TAB only (after md_set_pair): the tables rho_r[nr], phi_r[nr] at r = 0, dr, 2 dr, ... and F_rho[nrho] at
 * rho = 0, drho, ... (host pointers; copied).  The r grid must reach the cutoff (checked at the next build); distances
 * and densities beyond a table's end are evaluated with its last interval's cubic.  (App. A; reading s26) */
int md_set_eam_tables(md_system* s, const double* rho_r, const double* phi_r, int nr, const double* F_rho, int nrho);
/* MD_PAIR_BUCK_COUL only: the charge of every atom type, n = ntypes values (the paper's silicate carries one charge per
 * species, App. A).  Host pointer. */
int md_set_type_charges(md_system* s, const double* q, int n);
/* list_kind: MD_LIST_FULL | MD_LIST_HALF (PAPER.md L76 Newton's third law, L104 full list; reading s6);
 * kernel: MD_KERNEL_* (PAPER.md L88-122 TpA/BpA, L64-82 cell list, L137 choice by timing).  HALF needs TPA or AUTO.
 * Invalidates the list. */
int md_set_neighbor(md_system* s, int list_kind, int kernel);

/* Tuning knobs for measurements (profiles/; none is needed in normal use: the planner and md_autotune set
 * all of them; SURVEY.md 8(f)-1 sweeps use them).  Invalidates the list and the variant choice.  Names:
 *   "tile_shape"  bx | by << 4 | bz << 8 cells per tile (4 >= bx >= by >= bz >= 1), 0: planner
 *   "force_threads"  block size of the list force kernels, 0: planner
 *   "persistent_groups"  tile buffers of the persistent force kernel minus one: 1 (two buffers), 2 (three), 0 = automatic
 *               (the name dates from the version that dealt tiles to that many fixed groups of consumer warps)
 *   "persistent_min_tiles_per_sm"  the persistent kernel is used from this many tiles per SM on (default 1)
 *   "no_persistent"  1: run the one-block-per-tile kernel everywhere
 *   "balance_after"  apply the row balancing to a list that has lived this many steps (default 48; <= 0: at every build)
 *   "no_balance"  1: never
 *   "build_graph"  0: md_run enqueues every rebuild launch by launch (default 1: replays the sequence as a CUDA graph)
 *   "pdl"  0: md_run launches its step kernels without programmatic dependent launch (default 1)
 *   "tab_smem"  0: MD_PAIR_EAM_TAB reads its coefficient tables through L1/L2 (default 1: staged in shared memory when
 *               a table is at most 48 KB)
 *   "tune_verbose"  1: md_autotune prints every candidate's timing to stderr
 * Unknown names and values out of range return MD_ERR_BAD_ARGUMENT. */
int md_set_option(md_system* s, const char* name, int64_t value);

/* Wrap into the box, bin into cells of edge >= rc+skin, counting-sort and reorder atoms, build the
 * Verlet list from the 27-cell stencil (fp64 distance test r^2 < (rc+skin)^2), reset x0.
 * (north_star (1),(2); md_build_neighbors) */
int md_build_neighbors(md_system* s);

/* Forces at the current positions (builds the list first if it is not valid).  f_out: N x 3 doubles in
 * caller order, host or device, may be NULL.  energy_out: total potential energy (host double), may be
 * NULL.  virial_out: xx,yy,zz,xy,xz,yz with W_ab = sum over pairs (each once) of D_a f_b (host), may be
 * NULL.  (north_star md_compute_forces) */
int md_compute_forces(md_system* s, double* f_out, double* energy_out, double virial_out[6]);

/* nsteps of velocity-Verlet NVE with time step dt: v += dt/2 f/m ftm2v; x += dt v;
 * [rebuild iff max |x-x0|^2 > (skin/2)^2]; f = F(x); v += dt/2 f/m ftm2v.  Asynchronous apart from the
 * rebuild decisions.  (north_star md_run) */
int md_run(md_system* s, int64_t nsteps, double dt);

/* NVT ("NVE, NVT, and NPT integrators"; reading s25 of DESIGN.md): with
 * MD_THERMO_NOSE_HOOVER md_run integrates dv/dt = f/m - xi v, dxi/dt = (2 KE - g kT)/Q, Q = g kT tau^2, g = 3N - 3, by the
 * symmetric splitting TH(dt/2) kick drift force kick TH(dt/2), TH(h): xi += h/2 G; v *= exp(-xi h); eta += xi h; xi += h/2 G.
 * kT in the caller's energy units (k_B T), tau in its time units.  Resets the thermostat state (xi = eta = 0), which
 * otherwise persists across md_run calls.  MD_THERMO_NONE returns to NVE. */
int md_set_thermostat(md_system* s, int kind, double kT, double tau);
/* out = {xi, eta, Q xi^2 / 2 + g kT eta}: the thermostat's state and its share of the conserved quantity
 * H = KE + PE + Q xi^2 / 2 + g kT eta (host doubles). */
int md_get_thermostat(md_system* s, double out[3]);

/* Current positions in caller order (host or device buffer of N x 3 doubles, reading s5): as stored,
 * i.e. inside the box at the last build, possibly slightly outside since.  MD_ERR_NOT_READY before md_set_positions. */
int md_get_positions(md_system* s, double* x);
/* Current velocities in caller order: at whole time steps after md_run. */
int md_get_velocities(md_system* s, double* v);
/* Forces of the last evaluation (md_compute_forces, or the last step of md_run: PAPER.md L52, the forces that belong
 * to the final positions).  MD_ERR_NOT_READY if there is none. */
int md_get_forces(md_system* s, double* f);

/* The current neighbor list in CALLER ids, for pair-set parity (numneigh[i], neighbors[i][jj];
 * north_star (2): "neighbor pair sets identical"): numneigh[N] and neigh[N x stride] (host or device int32 buffers),
 * exactly the pairs with |x_i - x_j|^2 < (rc+skin)^2 in fp64 at the current positions among the stored rows.  Rows
 * longer than stride are truncated (numneigh still holds the true length).  Half lists hold each unordered pair in
 * exactly one of the two rows.  Builds the list first if it is not valid. */
int md_get_neighbors(md_system* s, int32_t* numneigh, int32_t* neigh, int64_t stride);

/* The STORED list rows as they are, for checking the build itself (north_star (2)).
 * The library keeps one row per PAIR of consecutive atoms of a cell: the union of the two atoms' neighbors by a
 * conservative fp32 test (r^2 < (rc+skin)^2 (1 + band)), without the two atoms themselves; it is a superset of the
 * fp64 pair sets that md_get_neighbors returns.  All three outputs are indexed by caller atom id (host or device
 * int32 buffers): row_owner[i] = id of the first atom of i's pair (i itself if i is the first); numrow[i] =
 * entries of the row if i is a first atom, else 0; entries[i x stride ..] = the row in caller ids (first atoms
 * only; rows longer than stride are truncated, numrow still holds the true length). */
int md_get_neighbor_rows(md_system* s, int32_t* row_owner, int32_t* numrow, int32_t* entries, int64_t stride);

/* Kinetic energy 1/2 sum m v^2 mvv2e of the current velocities (host double; synchronises the stream).
 * (NVE; the metric a time-stepping caller reads back.) */
int md_kinetic_energy(md_system* s, double* ke_out);

/* The same quantity (the kinetic energy the NVE/NVT integrators report) for callers that cannot call
 * cudaMalloc -- code under CUDA-graph capture, tight serving loops, harnesses that forbid allocation.  Needs no handle
 * and allocates NOTHING, on the host or the device: no cudaMalloc / cudaFree / allocating library routine; it enqueues
 * one 4-byte memset and one kernel on cuda_stream (a cudaStream_t passed as void*, NULL = legacy default stream) and
 * does not synchronise.  The kernel's scratch (one partial sum per 256 atoms plus a completion counter) is a file-scope
 * static __device__ array of MD_NOALLOC_SCRATCH_BYTES that every GPU which loads the library holds until the process
 * exits; its device address is resolved with cudaGetSymbolAddress on the first call on each device (make that call
 * outside stream capture).
 *   v_dev      DEVICE, N x 3 AoS doubles, read
 *   type_dev   DEVICE, N int32 in [0, ntypes), read (not range-checked)
 *   mass_dev   DEVICE, ntypes doubles, read
 *   mvv2e      the unit factor of md_set_units (1 in LJ reduced units)
 *   ke_out_dev DEVICE, 1 double, written by the kernel: 1/2 sum m v^2 mvv2e, summed in a fixed order (bitwise
 *              reproducible from call to call)
 * The caller owns all five buffers.  Errors: MD_ERR_BAD_ARGUMENT for a NULL pointer, N <= 0 or N > MD_NOALLOC_MAX_ATOMS
 * (nothing is enqueued); MD_ERR_CUDA if a runtime call fails; the text is in md_last_error(NULL) on the calling thread.
 * ALL calls in the process share the one array per GPU: calls on the same stream are ordered and safe; calls whose
 * kernels may overlap on the GPU (different streams, or several host threads on different streams) RACE on the scratch
 * and give wrong sums -- serialise them.  The counter is cleared at the start of every call; the partials need no
 * clearing (each call overwrites the ones it reads). */
#define MD_NOALLOC_SCRATCH_BYTES 524288   /* 512 KiB: 256 bytes of header + 65504 partials */
#define MD_NOALLOC_MAX_ATOMS 16769024LL   /* 65504 partials x 256 atoms */
int md_kinetic_energy_noalloc(const double* v_dev, const int32_t* type_dev, const double* mass_dev, int64_t N, double mvv2e,
                              double* ke_out_dev, void* cuda_stream);

/* Setup-time mini benchmark of PAPER.md L137 ("the faster variant is chosen by timing at setup"): on the current
 * positions, builds the list and times nrep (rounded up to an even number) FUSED time-step kernels with dt = 0 (force
 * evaluation + kick + drift epilogue: what md_run runs; positions and velocities keep their values) with each of TPA,
 * SUBWARP, WARP, SUBWARP4 and SUBWARP2 and, on boxes with fewer than 2048 tiles, at the planner's tile shape and its
 * neighbours in the list of feasible shapes; keeps the combination with the lowest (step + 1/8 list build) time and
 * reports the best step time of each variant (ms, in the order TPA, SUBWARP, WARP, SUBWARP4, SUBWARP2) if ms_out is
 * not NULL.  MD_KERNEL_AUTO runs it before the first build and once more inside md_run, at the first rebuild that comes
 * 20 or more time steps later (the caller's positions are often a perfect lattice).  Half lists always use TPA. */
int md_autotune(md_system* s, int nrep, double ms_out[5]);

/* Counters, geometry and timers (see md_stats; what bench.py reports).  Counts the exact neighbor
 * statistics on demand and reads the kinetic energy, so it synchronises the stream. */
int md_get_stats(md_system* s, md_stats* out);
/* Text of the last failure of this handle (north_star: errors are codes, never throws).  s may be NULL: the error of
 * a failed md_create on this thread. */
const char* md_last_error(const md_system* s);

#ifdef __cplusplus
}
#endif
#endif /* MD_B200_H */
