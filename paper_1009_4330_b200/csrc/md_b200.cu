// md_b200.cu -- host side of the C ABI declared in include/md_b200.h.
// Every step of the hot path runs in the kernels of md_kernels.cuh; this file owns device memory,
// plans tile geometry, launches, and marshals caller buffers.  There is no CPU fallback: any CUDA
// failure is reported as MD_ERR_CUDA.
#include "../../include/md_b200.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <type_traits>
#include <string>
#include <vector>

#include "md_kernels.cuh"

using namespace mdk;

namespace {

thread_local std::string g_create_error;

struct md_system_impl {
  int64_t N = 0;
  size_t ld = 0;   // leading dimension of SoA arrays (N rounded up to 32)
  cudaStream_t stream = nullptr;
  double box[3] = {0, 0, 0};
  int ntypes = 0;
  double ftm2v = 1.0, mvv2e = 1.0;
  int precision = MD_FP64;
  int style = 0;
  double params[5] = {0, 0, 0, 0, 0};
  // MD_PAIR_BUCK_COUL: per type pair A, rho, C (md_set_pair_coeff) and per type charge (md_set_type_charges)
  double pair_coef[MAX_PAIR_TYPES][MAX_PAIR_TYPES][3] = {};
  bool pair_coef_set[MAX_PAIR_TYPES][MAX_PAIR_TYPES] = {};
  double qtype[MAX_PAIR_TYPES] = {0, 0, 0, 0};
  // MD_PAIR_EAM_TAB: per-interval cubic coefficients of rho(r), phi(r) (float4 and double4 copies) and F(rho) (double4)
  int eam_nr = 0, eam_nrho = 0;
  float4* tab_rho_f = nullptr; float4* tab_phi_f = nullptr;
  double4* tab_rho_dd = nullptr; double4* tab_phi_dd = nullptr; double4* tab_F_dd = nullptr;
  double rc = 0, skin = 0;
  int list_kind = MD_LIST_FULL;
  int kernel_req = MD_KERNEL_TPA;
  int kernel_eff = MD_KERNEL_TPA;
  bool autotuned = false;
  int tune_stage = 0;            // 1: variant chosen on the caller's positions at setup; 2: confirmed on evolved positions (md_run)
  int64_t tune_step = 0;         // nsteps_total at the setup-time choice
  bool have_x = false, pair_set = false, planned = false, list_valid = false, forces_valid = false;
  bool list_built_for_export = false;

  // device arrays (sorted order, SoA with leading dimension ld)
  double* x[2] = {nullptr, nullptr};
  double* v[2] = {nullptr, nullptr};
  int* id[2] = {nullptr, nullptr};
  int* type[2] = {nullptr, nullptr};
  int cur = 0;    // buffer of v, id, type (flips at every build)
  int xcur = 0;   // buffer of x (flips at every build and at every fused kick+drift step)
  int force_threads = 256, batch = 8;
  int build_attempts = 0;   // builds in a row that md_run found too small for their capacities
  // the build's launch sequence as CUDA graphs, one per (cur, xcur) buffer state; captured on capture_stream (the
  // caller's stream may be the legacy default stream, which cannot be captured) and launched on the caller's stream
  struct BuildGraph { cudaGraphExec_t exec = nullptr; uint64_t key = 0; int64_t nlaunch = 0; };
  BuildGraph build_graph[4];
  cudaStream_t capture_stream = nullptr;
  uint64_t plan_epoch = 0;    // bumped by every plan(): graphs captured for an older geometry are stale
  bool opt_build_graph = true;   // md_set_option("build_graph")
  bool opt_pdl = true;           // md_set_option("pdl"): programmatic dependent launch of the step kernels
  bool opt_tab_smem = true;      // md_set_option("tab_smem"): tabulated EAM stages its coefficient tables in shared memory
  int num_sms = 148;
  bool force_timing_pending = false;
  bool list_balanced = false;
  int64_t steps_since_build = 0;
  int balance_after = 0;     // BALANCE_AFTER, or MD_B200_BALANCE_AFTER (tuning experiments)
  bool no_balance = false;   // MD_B200_NO_BALANCE=1: skip the row-balancing pass (for A/B measurements)
  int p_min_tiles_per_sm = 1;   // k_tile_force_p is used from this many tiles per SM on (MD_B200_PMIN; measured: cfg 4 -4 % at 2-3 tiles per SM)
  int p_groups = 0;             // tile buffers of the persistent force kernel minus one; 0: two (three buffers) if they fit, else one
  bool no_persistent = false;   // MD_B200_NO_PERSISTENT=1: run k_tile_force where k_tile_force_p would be used (A/B measurements)
  int brick_forced = 0;   // tile shape chosen by the autotuner, bx | by << 4 | bz << 8 (0: the planner's own pick)
  int opt_tile_shape = 0;     // md_set_option("tile_shape"): bx | by << 4 | bz << 8, 0: planner
  int opt_force_threads = 0;  // md_set_option("force_threads"): block size of the list force kernels, 0: planner
  bool tune_verbose = false;  // md_set_option("tune_verbose")
  int shape_index = 0, shape_count = 0, build_threads = 256;
  int shape_codes[64] = {};   // the feasible tile shapes of the last plan(), largest first (bx | by << 4 | bz << 8)
  double *f = nullptr, *x0 = nullptr, *rho = nullptr, *fp = nullptr;
  void* xr[2] = {nullptr, nullptr};   // packed cell-relative positions (Vec4<T>, 32 B per atom reserved), buffer index = xcur
  int* tab = nullptr;                 // per-tile tables of the last build
  size_t tab_alloc = 0;
  int *cell_of = nullptr, *rank = nullptr, *perm = nullptr, *mkey = nullptr, *numneigh = nullptr;
  int* nstat_d = nullptr;            // 4 ints: exact neighbor statistics of k_export_list (max; sum as 64 bits at [2])
  int* export_buf = nullptr;         // staging for md_get_neighbors / md_get_neighbor_rows into host buffers
  size_t export_alloc = 0;
  bool counts_valid = false;         // max_nb_exact / mean_nb_exact belong to the current list
  int max_nb_exact = 0;
  double mean_nb_exact = 0;
  size_t numneigh_alloc = 0;
  int *cell_count = nullptr, *cell_start = nullptr;
  size_t cell_alloc = 0;
  uint4* list = nullptr;
  size_t list_words = 0;
  double* mass_d = nullptr;
  double* dtf_d = nullptr;       // [ntypes]: dt/2 ftm2v / mass of the current md_run
  // NVT (md_set_thermostat): one Nose-Hoover thermostat; state xi, eta persists across md_run calls
  int thermostat = MD_THERMO_NONE;
  double thermo_kT = 0, thermo_tau = 0, thermo_xi = 0, thermo_eta = 0;
  double* thermo_d = nullptr;    // 8 doubles: xi, eta, KE, scale, g kT, Q
  double* ke_partial_d = nullptr;   // one kinetic-energy partial per block of k_final_integrate_ke
  std::vector<double> mass_h;
  double* ev_partials = nullptr;
  size_t ev_tiles_alloc = 0;
  double* scalars_d = nullptr;   // 16 doubles: [0..7] energy/virial, [8] kinetic
  double* io_d = nullptr;        // 3N doubles, staging for host pointers
  int* io_i = nullptr;           // N ints staging
  int* types_caller = nullptr;   // types in caller order (device)
  Flags* flags_d = nullptr;
  Flags* flags_h = nullptr;      // pinned
  double* scalars_h = nullptr;   // pinned, 16 doubles

  Geom g{};
  PairParams P{};
  double cap_scale_tile = 1.0, cap_scale_int = 1.0, cap_scale_row = 1.0;

  // stats
  int64_t nsteps_total = 0, nbuilds = 0, nforce = 0, launches = 0, launches_last_run = 0;
  int max_tile_atoms = 0, max_row = 0;   // max_row / mean_row: the stored PAIR rows (union of the two atoms' neighbors)
  double mean_row = 0;
  double ms_build = 0, ms_force = 0, ms_run = 0;
  cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev2 = nullptr, ev3 = nullptr, ev4 = nullptr, ev5 = nullptr;   // run, build, autotune
  static constexpr int NSAMPLE = 128;          // sampled force timings per md_run
  cudaEvent_t pev[2 * NSAMPLE] = {};
  cudaEvent_t pev_mid[NSAMPLE] = {};           // EAM: between the two passes of a sampled force evaluation
  cudaEvent_t mid_event = nullptr;             // recorded by the next EAM force evaluation after its first pass (md_run sets it)
  double ms_pass1_sampled = 0;
  double ms_force_sampled = 0, ms_build_in_run = 0;
  int64_t nforce_sampled = 0, nbuilds_in_run = 0, nforce_sampled_acc = 0;

  std::string err;
};

}  // namespace

struct md_system : md_system_impl {};

namespace {

int fail(md_system* s, int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (s) s->err = buf; else g_create_error = buf;
  return code;
}

#define CK(call)                                                                                         \
  do {                                                                                                   \
    cudaError_t e_ = (call);                                                                             \
    if (e_ != cudaSuccess) return fail(s, MD_ERR_CUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

// Kernels that need more than the default 48 KB of dynamic shared memory are opted in ONCE per process to the
// device's maximum: the attribute belongs to the kernel (per context), not to a handle, so it must never be
// lowered by another handle with a smaller tile geometry.
std::mutex g_attr_mutex;
std::map<const void*, int> g_attr_set;
template <class Kern>
cudaError_t opt_in_smem(Kern kern) {
  const void* key = reinterpret_cast<const void*>(kern);
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(g_attr_mutex);
  auto it = g_attr_set.find(key);
  if (it != g_attr_set.end() && (it->second >> dev & 1)) return cudaSuccess;
  int optin = 0;
  e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (e != cudaSuccess) return e;
  cudaFuncAttributes fa;
  e = cudaFuncGetAttributes(&fa, kern);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
  if (e != cudaSuccess) return e;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
  if (e != cudaSuccess) return e;
  g_attr_set[key] |= 1 << (dev & 31);
  return cudaSuccess;
}

template <class Kern, class... Args>
cudaError_t launch(md_system* s, Kern kern, unsigned grid, unsigned block, size_t smem, Args... args) {
  if (grid == 0) return cudaSuccess;
  if (smem > 40 * 1024) {   // static shared memory (reduction scratch) counts against the 48 KB default too
    cudaError_t e = opt_in_smem(kern);
    if (e != cudaSuccess) return e;
  }
  kern<<<grid, block, smem, s->stream>>>(args...);
  s->launches++;
  return cudaGetLastError();
}

// A step kernel of md_run's batches: programmatic dependent launch, so that the launch itself (grid set-up, block
// scheduling) overlaps the tail of the previous step kernel; the kernels call pdl_wait_then_release() before they read
// anything (md_kernels.cuh).
template <class Kern, class... Args>
cudaError_t launch_pdl(md_system* s, bool pdl, Kern kern, unsigned grid, unsigned block, size_t smem, Args... args) {
  if (!pdl) return launch(s, kern, grid, block, smem, args...);
  if (grid == 0) return cudaSuccess;
  if (smem > 40 * 1024) {
    cudaError_t e = opt_in_smem(kern);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = s->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  s->launches++;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}

inline unsigned blocks_for(int64_t n, int block) { return (unsigned)((n + block - 1) / block); }

bool is_device_ptr(const void* p) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, p);
  if (e != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

template <class T>
cudaError_t dalloc(T** p, size_t n) { return cudaMalloc((void**)p, std::max<size_t>(n, 1) * sizeof(T)); }

int lanes_for(int kernel) {
  return kernel == MD_KERNEL_SUBWARP ? 8 : (kernel == MD_KERNEL_WARP ? 32 : (kernel == MD_KERNEL_SUBWARP4 ? 4 : (kernel == MD_KERNEL_SUBWARP2 ? 2 : 1)));
}

// ---- planning: cell grid, tile width, capacities -----------------------------------------------------
size_t elem_size(const md_system* s) { return s->precision == MD_FP64 ? sizeof(double) : sizeof(float); }
int capA_of(const Geom& g) { return (g.tile_cap + 8) & ~3; }
size_t force_smem(const md_system* s, const Geom& g, bool half) {
  return sizeof(TileTables) + 4 * (size_t)(capA_of(g) + tile_tab_cells(g)) * elem_size(s) + (size_t)g.interior_cap * 2 +
         (size_t)((tile_tab_quads(g) + 7) & ~7) * 2 + (half ? (size_t)capA_of(g) * 4 : 0) + 16;
}
size_t cell_smem(const md_system* s, const Geom& g) { return sizeof(TileTables) + 4 * (size_t)capA_of(g) * elem_size(s) + 16; }
size_t build_smem(const Geom& g, int threads) {
  return sizeof(TileTables) + (size_t)tile_tab_cells(g) * 16 + (size_t)build_rowcell_len(g) * 2 + 3 * (size_t)capA_of(g) * sizeof(float) +
         (size_t)threads * RING_STRIDE + 16;
}
// threads per block of the list build: 256 when three such blocks fit an SM's shared memory, else 384 (two blocks):
// 24 warps per SM either way
int build_threads(const Geom& g) {
  const size_t sm_total = 227 * 1024, reserve = 1024 + 512;
  if (3 * (build_smem(g, BUILD_THREADS) + reserve) <= sm_total) return BUILD_THREADS;
  if (2 * (build_smem(g, BUILD_MAX_THREADS) + reserve) <= sm_total) return BUILD_MAX_THREADS;
  if (2 * (build_smem(g, BUILD_THREADS) + reserve) <= sm_total) return BUILD_THREADS;
  return BUILD_MAX_THREADS;   // one block per SM: as many warps as the kernel is compiled for
}
size_t export_smem(const Geom& g) { return sizeof(TileTables) + (size_t)capA_of(g) * (2 * sizeof(int) + 2) + 16; }

// The persistent, warp-specialised force kernel (k_tile_force_p) serves the mixed-precision full-list variants; it
// needs three tile buffers in shared memory.  Everything else (fp64, energy/virial, half list) runs k_tile_force.
constexpr size_t SMEM_OPTIN_BUDGET = 227 * 1024 - 1024;
bool persistent_eligible(const md_system* s) {
  return s->precision == MD_MIXED && s->list_kind == MD_LIST_FULL && s->kernel_eff != MD_KERNEL_CELL && !s->no_persistent;
}
// Tabulated EAM: the two coefficient tables (rho, phi: 16 bytes per interval) are staged in shared memory behind the
// tile buffers when they are small enough to leave room for two buffers; bytes of ONE table, 0: read through L1/L2.
size_t p_table_bytes(const md_system* s) {
  if (s->style != MD_PAIR_EAM_TAB || s->precision != MD_MIXED || !s->opt_tab_smem || s->eam_nr < 2) return 0;
  const size_t one = (size_t)(s->eam_nr - 1) * 16;
  return one <= 48 * 1024 ? one : 0;
}
// Tile buffers per block minus one (historically: consumer groups): two, i.e. three buffers, when they fit the
// SM's shared memory; else one, i.e. two buffers (rc = 5 sigma: a 3x1x1 tile stages 108 KB); 0: does not fit.
int p_groups(const md_system* s, const Geom& g) {
  const size_t extra = 2 * p_table_bytes(s);
  if (s->p_groups > 0) return force_p_smem(g, s->p_groups + 1) + extra <= SMEM_OPTIN_BUDGET ? s->p_groups : 0;
  if (force_p_smem(g, 3) + extra <= SMEM_OPTIN_BUDGET) return 2;
  return force_p_smem(g, 2) + extra <= SMEM_OPTIN_BUDGET ? 1 : 0;
}
int p_nbuf(const md_system* s, const Geom& g) { return p_groups(s, g) + 1; }             // tile buffers: one per group + one being loaded
int p_max_group_threads(const md_system* s, const Geom& g) {   // whole warpgroups (register split)
  return ((FORCE_P_MAX_THREADS - 32 * FORCE_P_NPROD) / std::max(1, p_groups(s, g))) / 128 * 128;
}
// ... and enough tiles per SM for the producer to run ahead
bool use_persistent(const md_system* s, const Geom& g) {
  return persistent_eligible(s) && g.ntiles >= s->p_min_tiles_per_sm * s->num_sms && p_groups(s, g) > 0;
}

void fill_geom_for_b(const md_system* s, const int shape[3], Geom& g) {
  double rl = s->rc + s->skin;
  g.ncell = 1;
  for (int d = 0; d < 3; ++d) {
    g.L[d] = s->box[d];
    g.nc[d] = (int)std::floor(s->box[d] / rl);
    g.edge[d] = s->box[d] / g.nc[d];
    g.inv_edge[d] = g.nc[d] / s->box[d];
    {   // anchor spacing: edge rounded to `bits` significant bits, so that k * h/2 is exact in fp32 for |k| <= 2 nc
      int lg = 1;
      while ((1 << lg) < 2 * g.nc[d] + 4) ++lg;
      const int bits = std::max(4, 23 - lg);
      int e;
      const double m = std::frexp(g.edge[d], &e);                 // edge = m 2^e, m in [0.5, 1)
      g.h[d] = std::ldexp(std::nearbyint(std::ldexp(m, bits)), e - bits);
    }
    g.b[d] = std::min(shape[d], g.nc[d]);
    g.nb[d] = (g.nc[d] + g.b[d] - 1) / g.b[d];
    g.ncell *= g.nc[d];
  }
  g.ntiles = g.nb[0] * g.nb[1] * g.nb[2];
  double per_cell = (double)s->N / g.ncell + 1.5;   // cells are padded to multiples of 4 slots
  double staged = per_cell * (g.b[0] + 2) * (g.b[1] + 2) * (g.b[2] + 2);
  double interior = (per_cell - 1.0) * g.b[0] * g.b[1] * g.b[2];   // list rows: cells padded to multiples of 2
  // slack over the mean: five standard deviations of a Poisson count (a liquid fluctuates less), i.e. 7 % for the
  // ~5000 staged atoms of an rc = 5 sigma tile and 9 % at cfg 5, where a flat 20 % would cost a resident block;
  // an overflow is detected by the kernels and re-planned with a larger factor
  g.tile_cap = (int)(staged * (1.0 + 5.0 / std::sqrt(std::max(staged, 1.0))) * s->cap_scale_tile + 64);
  g.tile_cap = (g.tile_cap + 7) & ~7;
  g.interior_cap = (int)(interior * 1.25 * s->cap_scale_int + 32);
  g.interior_cap = (g.interior_cap + 31) & ~31;
  g.K = lanes_for(s->kernel_eff);
  g.half = s->list_kind == MD_LIST_HALF ? 1 : 0;
  g.code_shift = s->precision == MD_FP64 ? 4 : 3;
  double vol = s->box[0] * s->box[1] * s->box[2];
  // (a half list keeps or drops another cell whole, so its rows range from empty to nearly the full neighborhood:
  // the row capacity is that of the full list)
  double mean_nb = 4.0 / 3.0 * M_PI * rl * rl * rl * s->N / vol;
  int unit = 8 * g.K;
  // a stored row is the union of the neighbors of two atoms ~1.4 sigma apart: ~1.4 x the single-atom mean (measured
  // 1.38 in the LJ liquid), times the same 1.5 x slack over the mean as before
  g.row_cap = (int)(mean_nb * 1.4 * 1.5 * s->cap_scale_row + 24);
  g.row_cap = ((g.row_cap + unit - 1) / unit) * unit;
  g.chunk_cap = g.row_cap / unit;
}

// Candidate tile shapes (cells per tile edge, bx >= by >= bz, (bx+2)(by+2)(bz+2) <= MAX_TILE_CELLS), largest first.
struct TileShape { int b[3]; };
int tile_shapes(TileShape* out) {
  int n = 0;
  for (int cells = 64; cells >= 1; --cells)
    for (int bx = 4; bx >= 1; --bx)
      for (int by = bx; by >= 1; --by)
        for (int bz = by; bz >= 1; --bz)
          if (bx * by * bz == cells && (bx + 2) * (by + 2) * (bz + 2) <= MAX_TILE_CELLS) out[n++] = TileShape{{bx, by, bz}};
  return n;
}

int plan(md_system* s) {
  double rl = s->rc + s->skin;
  for (int d = 0; d < 3; ++d)
    if (s->box[d] < 3.0 * rl) return fail(s, MD_ERR_BOX_TOO_SMALL, "box edge %d = %g < 3 (rc+skin) = %g", d, s->box[d], 3.0 * rl);
  double vol = s->box[0] * s->box[1] * s->box[2];
  double lscale = std::cbrt(vol / (double)s->N);   // ~ nearest-neighbor distance
  Geom g{};
  const size_t smem_hard = 200 * 1024;
  // three force blocks per SM: their phases (staging, list loop, epilogue) overlap better than those of two bigger ones
  const size_t smem_three = (227 * 1024) / 3 - 1536 - 3200;
  const int code_shift = s->precision == MD_FP64 ? 4 : 3;
  TileShape shapes[64];
  const int nshapes = tile_shapes(shapes);
  // feasible[]: shapes within the hard limits, largest first; `pick`: the first one that also meets the preferences
  // of pass 0 (all), pass 1 (all but the tile count) or pass 2 (none)
  int feasible[64], nfeas = 0, pick = -1;
  int forced_shape[3] = {0, 0, 0};
  if (s->opt_tile_shape) { forced_shape[0] = s->opt_tile_shape & 15; forced_shape[1] = (s->opt_tile_shape >> 4) & 15; forced_shape[2] = (s->opt_tile_shape >> 8) & 15; }
  for (int i = 0; i < nshapes; ++i) {
    fill_geom_for_b(s, shapes[i].b, g);
    if (g.b[0] != shapes[i].b[0] || g.b[1] != shapes[i].b[1] || g.b[2] != shapes[i].b[2]) continue;   // wider than the box
    if (g.tile_cap > (65535 >> code_shift)) continue;       // 16-bit slot codes
    size_t sm = std::max(std::max(force_smem(s, g, g.half), build_smem(g, build_threads(g))), cell_smem(s, g));
    if (sm > smem_hard) continue;
    if (forced_shape[0] && (forced_shape[0] != g.b[0] || forced_shape[1] != g.b[1] || forced_shape[2] != g.b[2])) continue;
    feasible[nfeas++] = i;
  }
  if (!nfeas) return fail(s, MD_ERR_OVERFLOW, "no tile shape fits shared memory or the 16-bit slot codes (too many atoms per cell of edge rc+skin)");
  // Preferences, dropped one level at a time until a shape qualifies (largest shape first within a level):
  //   level 0: shared memory for three resident blocks (or the persistent kernel's two groups + three tile buffers), fp32 tile extent,
  //            enough tiles for two per SM, one round of rows, halo not more than 18 staged cells per interior cell
  //   level 1: the same without the tile count
  //   level 2: shared memory for two resident blocks (or the persistent kernel with one group + two buffers)
  //   level 3: anything feasible
  const size_t smem_two = (227 * 1024) / 2 - 1536 - 3200;
  for (int pass = 0; pass < 4 && pick < 0; ++pass) {
    for (int f = 0; f < nfeas && pick < 0; ++f) {
      fill_geom_for_b(s, shapes[feasible[f]].b, g);
      if (pass < 3) {
        const bool pers = use_persistent(s, g);
        if (pass < 2 ? !(pers && p_groups(s, g) == 2) && force_smem(s, g, g.half) > smem_three : !pers && force_smem(s, g, g.half) > smem_two) continue;
        double half_extent = 0;
        for (int d = 0; d < 3; ++d) half_extent = std::max(half_extent, 0.5 * (g.b[d] + 2) * g.edge[d]);
        // fp32 tile coordinates: |value| <= 13.5 nearest-neighbor distances keeps the ulp at 1e-6 of one (cfg 3's 3x1x1
        // tiles, 13.2, meet the 1e-5 force tolerance at full size: tests/test_gpu_fullsize.py)
        if (s->precision == MD_MIXED && half_extent > 13.5 * lscale && g.b[0] > 1) continue;
        if (pass == 0 && g.ntiles < 2 * 148) continue;
        if ((g.b[0] + 2) * (g.b[1] + 2) * (g.b[2] + 2) > 18 * g.b[0] * g.b[1] * g.b[2] && g.nc[0] * g.nc[1] * g.nc[2] > 27) continue;
        // thread-per-row: the tile's pair rows (+ 5 % for the fullest tiles) should fit ONE round of a block small
        // enough for three resident blocks (384 threads of <= 56 registers); a second, nearly empty round costs
        // more than the smaller tile does
        if (g.K == 1 && 0.5 * ((double)s->N / g.ncell + 0.5) * g.b[0] * g.b[1] * g.b[2] * 1.05 > (pers ? (double)p_max_group_threads(s, g) : 384.0)) continue;
      }
      pick = f;
    }
  }
  // the autotuner may name a shape itself; if that shape is not feasible (any more: the capacities may have grown
  // after an overflow), the planner's own pick stands
  if (s->brick_forced) {
    int found = -1;
    for (int f = 0; f < nfeas; ++f) {
      const int* b = shapes[feasible[f]].b;
      if ((b[0] | b[1] << 4 | b[2] << 8) == s->brick_forced) found = f;
    }
    if (found >= 0) pick = found; else s->brick_forced = 0;
  }
  s->shape_index = pick; s->shape_count = nfeas;
  for (int f = 0; f < nfeas; ++f) s->shape_codes[f] = shapes[feasible[f]].b[0] | shapes[feasible[f]].b[1] << 4 | shapes[feasible[f]].b[2] << 8;
  fill_geom_for_b(s, shapes[feasible[pick]].b, g);
  s->g = g;
  // block size of the list force kernels: the tile's pair rows should fill whole rounds of the block
  {
    double rows = 0.5 * ((double)s->N / g.ncell + 0.5) * g.b[0] * g.b[1] * g.b[2] * 1.05;
    double lanes = rows * g.K;
    int tmax = s->precision == MD_FP64 ? FORCE_MAX_THREADS_WIDE : FORCE_MAX_THREADS;
    if (use_persistent(s, g)) tmax = p_max_group_threads(s, g);                     // threads of ONE consumer group
    else if (force_smem(s, g, g.half) <= smem_three) tmax = std::min(tmax, 384);   // three resident blocks of <= 56 registers
    int rounds = (int)std::ceil(lanes / tmax);
    int t = (int)std::ceil(lanes / std::max(rounds, 1));
    t = ((t + 31) / 32) * 32;
    s->force_threads = std::min(std::max(t, 32), tmax);
    if (s->opt_force_threads) s->force_threads = std::min(std::max(s->opt_force_threads / 32 * 32, 32), tmax);
  }
  // pair constants
  PairParams& P = s->P;
  P = PairParams{};
  P.rc2 = s->rc * s->rc;
  if (s->style == MD_PAIR_LJ126) {
    double eps = s->params[0], sg = s->params[1];
    double s6 = std::pow(sg, 6), s12 = s6 * s6;
    P.lj1 = 48.0 * eps * s12; P.lj2 = 24.0 * eps * s6; P.lj3 = 4.0 * eps * s12; P.lj4 = 4.0 * eps * s6;
  } else if (s->style == MD_PAIR_EAM_TAB) {
    if (!s->tab_F_dd) return fail(s, MD_ERR_NOT_READY, "md_set_eam_tables has not been called");
    const double rmax = (s->eam_nr - 1) * s->params[0];
    if (rmax < s->rc) return fail(s, MD_ERR_BAD_ARGUMENT, "the EAM tables end at r = %g, before the cutoff %g", rmax, s->rc);
    P.tab_rho = s->precision == MD_FP64 ? (const void*)s->tab_rho_dd : (const void*)s->tab_rho_f;
    P.tab_phi = s->precision == MD_FP64 ? (const void*)s->tab_phi_dd : (const void*)s->tab_phi_f;
    P.tab_F = s->tab_F_dd;
    P.tab_nr = s->eam_nr; P.tab_nrho = s->eam_nrho;
    P.inv_dr = 1.0 / s->params[0]; P.inv_drho = 1.0 / s->params[1];
  } else if (s->style == MD_PAIR_BUCK_COUL) {
    if (s->ntypes > MAX_PAIR_TYPES) return fail(s, MD_ERR_BAD_ARGUMENT, "MD_PAIR_BUCK_COUL supports at most %d atom types", MAX_PAIR_TYPES);
    for (int a = 0; a < s->ntypes; ++a)
      for (int b = 0; b < s->ntypes; ++b) {
        if (!s->pair_coef_set[a][b]) return fail(s, MD_ERR_NOT_READY, "md_set_pair_coeff has not been called for the type pair (%d, %d)", a, b);
        double* e = P.bc[MAX_PAIR_TYPES * a + b];
        e[0] = s->pair_coef[a][b][0]; e[1] = 1.0 / s->pair_coef[a][b][1]; e[2] = s->pair_coef[a][b][2];
        e[3] = s->params[0] * s->qtype[a] * s->qtype[b];
      }
  } else {
    P.A = s->params[0]; P.p = s->params[1]; P.B = s->params[2]; P.q = s->params[3];
    P.inv_r0 = 1.0 / s->params[4]; P.p_r0 = P.p * P.inv_r0; P.q_r0 = P.q * P.inv_r0;
  }
  P.fill_float_copies();
  // (re)allocate what depends on the geometry
  if ((size_t)g.ncell + 1 > s->cell_alloc) {
    cudaFree(s->cell_count); cudaFree(s->cell_start);
    s->cell_alloc = (size_t)g.ncell + 1;
    CK(dalloc(&s->cell_count, s->cell_alloc + s->cell_alloc / SCAN_BLOCK + 2));   // + the scan's block sums
    CK(dalloc(&s->cell_start, s->cell_alloc));
  }
  size_t words = (size_t)g.ntiles * g.chunk_cap * prow_cap(g) * g.K;
  if (words > s->list_words) {
    cudaFree(s->list);
    s->list = nullptr; s->list_words = 0;
    CK(dalloc(&s->list, words));
    s->list_words = words;
  }
  size_t rows = (size_t)g.ntiles * prow_cap(g);
  if (rows > s->numneigh_alloc) {
    cudaFree(s->numneigh);
    s->numneigh = nullptr; s->numneigh_alloc = 0;
    CK(dalloc(&s->numneigh, rows));
    s->numneigh_alloc = rows;
  }
  size_t tab_ints = (size_t)g.ntiles * tile_tab_stride(g);
  if (tab_ints > s->tab_alloc) {
    cudaFree(s->tab);
    s->tab = nullptr; s->tab_alloc = 0;
    CK(dalloc(&s->tab, tab_ints));
    s->tab_alloc = tab_ints;
  }
  if ((size_t)g.ntiles > s->ev_tiles_alloc) {
    cudaFree(s->ev_partials);
    s->ev_tiles_alloc = g.ntiles;
    CK(dalloc(&s->ev_partials, (size_t)g.ntiles * 8));
  }
  s->planned = true;
  s->plan_epoch++;
  s->list_valid = false;
  return MD_OK;
}

// ---- build ------------------------------------------------------------------------------------------
int build_list_only(md_system* s) {
  const Geom& g = s->g;
  double rl = s->rc + s->skin;
  BuildArgs B{};
  B.g = g; B.tab = s->tab;
  B.xr = s->xr[s->xcur]; B.xr_double = s->precision == MD_FP64 ? 1 : 0;
  // guard band of the fp32 distance test: tile-centred coordinates up to E are
  // rounded to fp32, so r^2 carries a relative error of about (7 E / rl + 3) 2^-24; four times that is used.
  // The stored rows are a superset of the fp64 pair set: everything with fp32 r^2 < rl^2 (1 + band).
  double E = 0;
  for (int d = 0; d < 3; ++d) E = std::max(E, 0.5 * (g.b[d] + 2) * g.edge[d] + s->skin);
  double band = 4.0 * (7.0 * E / rl + 3.0) * std::ldexp(1.0, -24);
  B.rl2_hi = std::nextafterf((float)(rl * rl * (1.0 + band)), INFINITY);
  B.list = s->list; B.numneigh = s->numneigh; B.flags = s->flags_d;
  const bool s4 = g.code_shift == 4;
  const int bt = build_threads(g);
  const size_t sm = build_smem(g, bt);
  if (g.half) {
    if (s4) CK(launch(s, k_build_list<true, 0, 4>, g.ntiles, bt, sm, B));
    else CK(launch(s, k_build_list<true, 0, 3>, g.ntiles, bt, sm, B));
  } else if (g.K == 1) {
    if (s4) CK(launch(s, k_build_list<false, 0, 4>, g.ntiles, bt, sm, B));
    else CK(launch(s, k_build_list<false, 0, 3>, g.ntiles, bt, sm, B));
  } else if (g.K == 2) {
    if (s4) CK(launch(s, k_build_list<false, 1, 4>, g.ntiles, bt, sm, B));
    else CK(launch(s, k_build_list<false, 1, 3>, g.ntiles, bt, sm, B));
  } else if (g.K == 4) {
    if (s4) CK(launch(s, k_build_list<false, 2, 4>, g.ntiles, bt, sm, B));
    else CK(launch(s, k_build_list<false, 2, 3>, g.ntiles, bt, sm, B));
  } else if (g.K == 8) {
    if (s4) CK(launch(s, k_build_list<false, 3, 4>, g.ntiles, bt, sm, B));
    else CK(launch(s, k_build_list<false, 3, 3>, g.ntiles, bt, sm, B));
  } else {
    if (s4) CK(launch(s, k_build_list<false, 5, 4>, g.ntiles, bt, sm, B));
    else CK(launch(s, k_build_list<false, 5, 3>, g.ntiles, bt, sm, B));
  }
  return MD_OK;
}

// Row balancing (md_kernels.cuh): permutes every list row in place for conflict-free shared-memory gathers.  It
// costs about as much as a few force evaluations and makes one 4-20 % faster, so it pays only for a list that
// lives long: md_run applies it once a list has survived BALANCE_AFTER steps (a cold solid such as cfg 4 keeps
// its list for hundreds of steps; a hot liquid rebuilds every ~6 and never gets there).
constexpr int BALANCE_AFTER = 48;
int balance_rows(md_system* s) {
  const Geom& g = s->g;
  if (s->no_balance || s->list_balanced || !s->list_valid || !s->list_built_for_export) return MD_OK;
  BalanceArgs R{};
  R.g = g; R.tab = s->tab; R.list = s->list; R.numneigh = s->numneigh;
  R.row_bytes = g.row_cap * 2 + 16;
  if ((R.row_bytes / 16) % 2 == 0) R.row_bytes += 16;
  int threads = (int)std::min<size_t>(256, (160 * 1024) / (size_t)R.row_bytes) / 32 * 32;
  if (threads >= 32) {
    const size_t bsm = (size_t)threads * R.row_bytes;
    if (g.K == 1) CK(launch(s, k_balance_rows<0>, g.ntiles, threads, bsm, R));
    else if (g.K == 2) CK(launch(s, k_balance_rows<1>, g.ntiles, threads, bsm, R));
    else if (g.K == 4) CK(launch(s, k_balance_rows<2>, g.ntiles, threads, bsm, R));
    else if (g.K == 8) CK(launch(s, k_balance_rows<3>, g.ntiles, threads, bsm, R));
    else CK(launch(s, k_balance_rows<5>, g.ntiles, threads, bsm, R));
  }
  s->list_balanced = true;
  return MD_OK;
}

// One build, enqueued on the stream without waiting for it: bin, scan, rank sort, reorder (which flips the buffers), tile
// tables and the list.  What the kernels found (capacities needed, non-finite coordinates, row statistics) is in
// flags_d afterwards; build_finish() judges a host copy of it.
int build_launches(md_system* s, bool do_list) {
  const Geom& g = s->g;
  const int N = (int)s->N;
  CK(cudaMemsetAsync(s->flags_d, 0, sizeof(Flags), s->stream));
  CK(cudaMemsetAsync(s->cell_count, 0, (size_t)(g.ncell + 1) * sizeof(int), s->stream));
  int c = s->cur, o = 1 - c, xc = s->xcur, xo = 1 - xc;
  CK(launch(s, k_bin, blocks_for(N, 256), 256, 0, g, N, s->x[xc], s->x[xc] + s->ld, s->x[xc] + 2 * s->ld, s->cell_of, s->rank,
            s->cell_count, s->flags_d));
  {
    // block sums live in the tail of cell_count's allocation (cell_alloc has SCAN slack, see plan())
    const unsigned nblk = blocks_for(g.ncell, SCAN_BLOCK);
    int* bsum = s->cell_count + (g.ncell + 1);
    CK(launch(s, k_scan_block_sums, nblk, 1024, 0, g.ncell, (const int*)s->cell_count, bsum));
    CK(launch(s, k_scan_cells, nblk, 1024, 0, g.ncell, (const int*)s->cell_count, (const int*)bsum, s->cell_start));
  }
  CK(launch(s, k_fill_perm, blocks_for(N, 256), 256, 0, N, (const int*)s->cell_of, (const int*)s->rank, (const int*)s->cell_start,
            s->perm, s->mkey));
  CK(launch(s, k_sort_cells, std::min<unsigned>(blocks_for(g.ncell, 8), 148u * 8u), 256, 0, g.ncell, (const int*)s->cell_start,
            s->perm, s->mkey));   // a warp per cell, grid-stride
  if (s->precision == MD_FP64)
    CK(launch(s, k_permute<double>, blocks_for(N, 256), 256, 0, g, N, (const int*)s->perm, (const double*)s->x[xc], (const double*)s->v[c],
              (const int*)s->id[c], (const int*)s->type[c], s->x[xo], s->v[o], s->id[o], s->type[o], s->x0, (double4*)s->xr[xo], s->ld));
  else
    CK(launch(s, k_permute<float>, blocks_for(N, 256), 256, 0, g, N, (const int*)s->perm, (const double*)s->x[xc], (const double*)s->v[c],
              (const int*)s->id[c], (const int*)s->type[c], s->x[xo], s->v[o], s->id[o], s->type[o], s->x0, (float4*)s->xr[xo], s->ld));
  CK(launch(s, k_tile_tables, g.ntiles, 128, 0, g, (const int*)s->cell_start, s->tab, s->flags_d));
  s->cur = o; s->xcur = xo;   // host state only: the list is built from the reordered buffers
  s->forces_valid = false;
  if (do_list) { int rc = build_list_only(s); if (rc) return rc; }
  return MD_OK;
}

// use_graph: replay the sequence as a CUDA graph (md_run's rebuilds: the same dozen launches every few steps, which at
// small N cost more to launch than to run); the graph of a buffer state is captured the first time that state builds.
int build_enqueue(md_system* s, bool need_list, bool* did_list, bool use_graph = false) {
  if (!s->planned) { int rc = plan(s); if (rc) return rc; }
  const bool do_list = need_list || s->kernel_eff != MD_KERNEL_CELL;
  *did_list = do_list;
  CK(cudaEventRecord(s->ev2, s->stream));
  if (use_graph && s->opt_build_graph && s->capture_stream) {
    md_system_impl::BuildGraph& G = s->build_graph[s->cur * 2 + s->xcur];
    const uint64_t key = (s->plan_epoch << 8) | (uint64_t)(s->precision << 4) | (uint64_t)(s->kernel_eff << 1) | (do_list ? 1u : 0u);
    if (!G.exec || G.key != key) {
      if (G.exec) { cudaGraphExecDestroy(G.exec); G.exec = nullptr; }
      const int cur0 = s->cur, xcur0 = s->xcur;
      const int64_t l0 = s->launches;
      cudaStream_t user = s->stream;
      cudaGraph_t graph = nullptr;
      CK(cudaStreamBeginCapture(s->capture_stream, cudaStreamCaptureModeRelaxed));
      s->stream = s->capture_stream;
      const int rc = build_launches(s, do_list);
      s->stream = user;
      const cudaError_t e = cudaStreamEndCapture(s->capture_stream, &graph);
      G.nlaunch = s->launches - l0;
      s->launches = l0; s->cur = cur0; s->xcur = xcur0;   // nothing has run yet
      if (rc || e != cudaSuccess) {
        if (graph) cudaGraphDestroy(graph);
        if (rc) return rc;
        return fail(s, MD_ERR_CUDA, "capturing the build sequence failed: %s", cudaGetErrorString(e));
      }
      const cudaError_t ei = cudaGraphInstantiate(&G.exec, graph, 0);
      cudaGraphDestroy(graph);
      if (ei != cudaSuccess) { G.exec = nullptr; return fail(s, MD_ERR_CUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(ei)); }
      G.key = key;
    }
    CK(cudaGraphLaunch(G.exec, s->stream));
    s->launches += G.nlaunch;
    s->cur ^= 1; s->xcur ^= 1;
    s->forces_valid = false;
  } else {
    int rc = build_launches(s, do_list);
    if (rc) return rc;
  }
  CK(cudaEventRecord(s->ev3, s->stream));
  return MD_OK;
}

// Judges a finished build from the host copy F of its flags (the stream has been synchronised since ev3).
// *again: a capacity was too small; the cap scales are raised and the geometry has to be planned anew.
int build_finish(md_system* s, const Flags& F, bool did_list, bool* again) {
  const Geom& g = s->g;
  float ms = 0;
  cudaEventElapsedTime(&ms, s->ev2, s->ev3);
  s->ms_build = ms;
  s->nbuilds++;
  *again = false;
  if (F.nonfinite) return fail(s, MD_ERR_NONFINITE, "a non-finite coordinate reached the binning kernel");
  if (F.need_tile_cap > g.tile_cap) { s->cap_scale_tile *= 1.1 * (double)F.need_tile_cap / g.tile_cap; *again = true; }
  if (F.need_interior_cap > g.interior_cap) { s->cap_scale_int *= 1.1 * (double)F.need_interior_cap / g.interior_cap; *again = true; }
  if (F.need_row_cap > g.row_cap) { s->cap_scale_row *= 1.1 * (double)F.need_row_cap / g.row_cap; *again = true; }
  if (*again) { s->planned = false; return MD_OK; }
  s->max_tile_atoms = F.max_tile_atoms;
  s->max_row = F.max_row;
  s->mean_row = (double)F.sum_rows / (0.5 * (double)s->N);   // entries per stored pair row
  s->list_valid = true;
  s->list_built_for_export = did_list;
  s->list_balanced = false;
  s->steps_since_build = 0;
  s->build_attempts = 0;
  return MD_OK;
}

int build(md_system* s, bool need_list) {
  if (!s->have_x || !s->pair_set) return fail(s, MD_ERR_NOT_READY, "positions and pair style must be set before building");
  // nothing of the previous list survives a build, successful or not
  s->list_valid = false; s->forces_valid = false; s->list_built_for_export = false; s->counts_valid = false;
  for (int attempt = 0; attempt < 6; ++attempt) {
    bool did_list = false, again = false;
    int rc = build_enqueue(s, need_list, &did_list);
    if (rc) return rc;
    CK(cudaMemcpyAsync(s->flags_h, s->flags_d, sizeof(Flags), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    rc = build_finish(s, *s->flags_h, did_list, &again);
    if (rc) return rc;
    if (again) continue;
    if (s->balance_after <= 0 && did_list) { int rcb = balance_rows(s); if (rcb) return rcb; }   // tuning experiments only
    return MD_OK;
  }
  return fail(s, MD_ERR_OVERFLOW, "tile or neighbor-row capacity still exceeded after re-planning");
}

// ---- force dispatch ------------------------------------------------------------------------------------
// how a force evaluation is embedded in time stepping (ForceArgs.epi / in_run / parity)
struct StepMode {
  int epi = EPI_FORCES;
  int in_run = 0;
  int parity = 0;
  double dt = 0, hdtf = 0, trigger = 0;
  int xbuf = -1;                  // x / xr buffer read (default: the current one); EPI_KICK_DRIFT writes the other one
};

template <typename T, template <typename, bool> class BodyT, int MODE, bool EV>
int launch_force_variant(md_system* s, const ForceArgs& A) {
  using Body = BodyT<T, EV>;
  const Geom& g = s->g;
  const bool half = g.half != 0;
  // the energy/virial and fp64 instantiations are compiled for more registers, hence smaller blocks
  const int threads = (EV || sizeof(T) == 8) ? std::min(s->force_threads, FORCE_MAX_THREADS_WIDE) : s->force_threads;
  const bool pdl = A.in_run != 0 && s->opt_pdl;   // the fused step launches of md_run's batches
  if (s->kernel_eff == MD_KERNEL_CELL) {
    CK(launch(s, k_cell_force<T, Body, MODE, EV>, g.ntiles, BUILD_THREADS, cell_smem(s, g), A));
  } else if (half) {
    // each pair once: the term of the row's atoms in registers, the term of j scattered with fp64 atomics
    if (MODE == 0) CK(cudaMemsetAsync(A.f, 0, 3 * s->ld * sizeof(double), s->stream));
    else CK(cudaMemsetAsync(A.rho, 0, s->ld * sizeof(double), s->stream));
    CK(launch(s, k_tile_force<T, Body, 1, MODE, EV, true>, g.ntiles, threads, force_smem(s, g, true), A));
  } else {
    if constexpr (std::is_same<T, float>::value && !EV) {
      if (use_persistent(s, g)) {
        // persistent, warp-specialised path: one block per SM, ng * gth consumer threads (tasks dealt to warps) + the producer warps
        const int ng = p_groups(s, g), nb = p_nbuf(s, g);
        // all the consumer warps the register budget allows: the kernel deals 32-lane tasks to whichever warp is free,
        // so the tile's row count no longer has to match a group's size
        const int gth = p_max_group_threads(s, g);   // whole warpgroups
        const unsigned grid = (unsigned)std::min(g.ntiles, s->num_sms);
        const unsigned block = (unsigned)(ng * gth + 32 * FORCE_P_NPROD);
        const size_t sm = force_p_smem(g, nb) + 2 * p_table_bytes(s);
        if (g.K == 1) CK(launch_pdl(s, pdl, k_tile_force_p<Body, 1, MODE>, grid, block, sm, A, gth, ng, nb));
        else if (g.K == 2) CK(launch_pdl(s, pdl, k_tile_force_p<Body, 2, MODE>, grid, block, sm, A, gth, ng, nb));
        else if (g.K == 4) CK(launch_pdl(s, pdl, k_tile_force_p<Body, 4, MODE>, grid, block, sm, A, gth, ng, nb));
        else if (g.K == 8) CK(launch_pdl(s, pdl, k_tile_force_p<Body, 8, MODE>, grid, block, sm, A, gth, ng, nb));
        else CK(launch_pdl(s, pdl, k_tile_force_p<Body, 32, MODE>, grid, block, sm, A, gth, ng, nb));
        return MD_OK;
      }
    }
    const unsigned nt = (unsigned)g.ntiles, th = (unsigned)threads;
    if (g.K == 1) CK(launch_pdl(s, pdl, k_tile_force<T, Body, 1, MODE, EV, false>, nt, th, force_smem(s, g, false), A));
    else if (g.K == 2) CK(launch_pdl(s, pdl, k_tile_force<T, Body, 2, MODE, EV, false>, nt, th, force_smem(s, g, false), A));
    else if (g.K == 4) CK(launch_pdl(s, pdl, k_tile_force<T, Body, 4, MODE, EV, false>, nt, th, force_smem(s, g, false), A));
    else if (g.K == 8) CK(launch_pdl(s, pdl, k_tile_force<T, Body, 8, MODE, EV, false>, nt, th, force_smem(s, g, false), A));
    else CK(launch_pdl(s, pdl, k_tile_force<T, Body, 32, MODE, EV, false>, nt, th, force_smem(s, g, false), A));
  }
  return MD_OK;
}

template <typename T, bool EV>
int launch_force_T(md_system* s, const StepMode& M) {
  const Geom& g = s->g;
  ForceArgs A{};
  const int xb = M.xbuf >= 0 ? M.xbuf : s->xcur;
  A.g = g; A.P = s->P; A.cell_start = s->cell_start; A.tab = s->tab; A.x = s->x[xb]; A.xr = s->xr[xb]; A.ld = s->ld; A.list = s->list;
  A.numneigh = s->numneigh; A.fp_in = nullptr; A.f = s->f; A.rho = s->rho; A.fp_out = s->fp; A.ev_partials = s->ev_partials;
  A.epi = M.epi; A.in_run = M.in_run; A.parity = M.parity;
  A.v = s->v[s->cur]; A.x_new = s->x[xb ^ 1]; A.xr_new = s->xr[xb ^ 1]; A.x0 = s->x0; A.type = s->type[s->cur]; A.mass = s->mass_d;
  A.dtf_type = s->dtf_d;
  A.tab_smem_bytes = (int)p_table_bytes(s);
  A.dt = M.dt; A.half_dt_ftm2v = M.hdtf; A.trigger = M.trigger; A.flags = s->flags_d;
  if (s->style == MD_PAIR_LJ126) {
    int rc = launch_force_variant<T, LJBody, 0, EV>(s, A);
    if (rc) return rc;
    if (EV) CK(launch(s, k_reduce_ev, 1, 256, 0, g.ntiles, (const double*)s->ev_partials, s->scalars_d, 0));
  } else if (s->style == MD_PAIR_BUCK_COUL) {
    int rc = launch_force_variant<T, BuckCoulBody, 0, EV>(s, A);
    if (rc) return rc;
    if (EV) CK(launch(s, k_reduce_ev, 1, 256, 0, g.ntiles, (const double*)s->ev_partials, s->scalars_d, 0));
  } else {
    const bool tab = s->style == MD_PAIR_EAM_TAB;
    int rc = tab ? launch_force_variant<T, EamTabDensityBody, 1, EV>(s, A)
                 : launch_force_variant<T, EamDensityBody, 1, EV>(s, A);   // pass 1: rho, F'(rho), sum F(rho)
    if (rc) return rc;
    if (EV) CK(launch(s, k_reduce_ev, 1, 256, 0, g.ntiles, (const double*)s->ev_partials, s->scalars_d, 0));
    if (g.half && s->kernel_eff != MD_KERNEL_CELL)   // half list: rho was scattered with atomics, so F'(rho) needs its own pass
      CK(launch(s, k_eam_embed<T>, blocks_for(s->N, 256), 256, 0, (int)s->N, s->P, (const double*)s->rho, s->fp, (T*)s->xr[xb],
                EV ? s->scalars_d : (double*)nullptr));
    if (s->mid_event) CK(cudaEventRecord(s->mid_event, s->stream));
    A.fp_in = s->fp;
    rc = tab ? launch_force_variant<T, EamTabForceBody, 0, EV>(s, A) : launch_force_variant<T, EamForceBody, 0, EV>(s, A);   // pass 2: forces
    if (rc) return rc;
    if (EV) CK(launch(s, k_reduce_ev, 1, 256, 0, g.ntiles, (const double*)s->ev_partials, s->scalars_d, 1));
  }
  s->nforce++;
  return MD_OK;
}

int compute_forces_device(md_system* s, bool ev, const StepMode& M = StepMode()) {
  int rc;
  if (s->precision == MD_FP64) rc = ev ? launch_force_T<double, true>(s, M) : launch_force_T<double, false>(s, M);
  else rc = ev ? launch_force_T<float, true>(s, M) : launch_force_T<float, false>(s, M);
  if (rc == MD_OK && M.epi == EPI_FORCES) s->forces_valid = true;
  return rc;
}

int autotune(md_system* s, int nrep, double* ms_out);

int initial_integrate(md_system* s, double dt, double hdtf, bool in_run = false, const double* vscale = nullptr) {
  const Flags* rf = in_run ? s->flags_d : nullptr;
  const int N = (int)s->N;
  if (s->precision == MD_FP64)
    CK(launch(s, k_initial_integrate<double>, blocks_for(N, 256), 256, 0, s->g, N, s->ld, s->x[s->xcur], s->v[s->cur], (const double*)s->f,
              (const double*)s->x0, (const int*)s->type[s->cur], (const double*)s->mass_d, (double4*)s->xr[s->xcur], dt, hdtf,
              &s->flags_d->max_disp2_bits[0], rf, vscale));
  else
    CK(launch(s, k_initial_integrate<float>, blocks_for(N, 256), 256, 0, s->g, N, s->ld, s->x[s->xcur], s->v[s->cur], (const double*)s->f,
              (const double*)s->x0, (const int*)s->type[s->cur], (const double*)s->mass_d, (float4*)s->xr[s->xcur], dt, hdtf,
              &s->flags_d->max_disp2_bits[0], rf, vscale));
  return MD_OK;
}

int ensure_list(md_system* s) {
  if (!s->have_x || !s->pair_set) return fail(s, MD_ERR_NOT_READY, "positions and pair style must be set first");
  if (s->kernel_req == MD_KERNEL_AUTO && !s->autotuned) {
    int rc = autotune(s, 5, nullptr);
    if (rc) return rc;
  }
  if (!s->list_valid) return build(s, false);
  return MD_OK;
}

int autotune(md_system* s, int nrep, double* ms_out) {
  if (!s->have_x || !s->pair_set) return fail(s, MD_ERR_NOT_READY, "positions and pair style must be set first");
  if (s->list_kind == MD_LIST_HALF) { s->kernel_eff = MD_KERNEL_TPA; s->autotuned = true; s->planned = false; return MD_OK; }
  if (nrep < 1) nrep = 1;
  // The setup-time mini benchmark of PAPER.md L137, over lanes per row (1, 2, 4, 8, 32) and, because the best tile
  // shape depends on how many tiles the box yields, over the planner's shape and its neighbours in the list of feasible
  // shapes.  What is timed is what md_run runs: the FUSED step kernel (force evaluation + kick + drift epilogue), with
  // dt = 0 so that positions and velocities keep their values while the kernel does all of its work (a plain force
  // evaluation misjudges the variants with few lanes per row, whose epilogue is the more expensive one).  Score of a
  // candidate: one step plus an eighth of a list build (a typical rebuild interval).
  const int cand[5] = {MD_KERNEL_TPA, MD_KERNEL_SUBWARP, MD_KERNEL_WARP, MD_KERNEL_SUBWARP4, MD_KERNEL_SUBWARP2};
  s->brick_forced = 0;
  s->kernel_eff = MD_KERNEL_TPA;
  s->cap_scale_tile = s->cap_scale_int = s->cap_scale_row = 1.0;   // the candidate list below must be the one the loop plans with
  s->planned = false;
  int rc = plan(s);
  if (rc) return rc;
  double best_score = 1e300;
  int best = MD_KERNEL_TPA, best_b = 0;
  if (ms_out) for (int k = 0; k < 5; ++k) ms_out[k] = 1e300;
  // with thousands of tiles the planner's pick is right and the SMs are full either way; the tile shape matters when
  // the box yields few tiles: then its neighbours in the candidate list (two larger, two smaller) are timed too
  const bool sweep = s->g.ntiles < 2048;
  const int i0 = s->shape_index, nfeas = s->shape_count;
  nrep = (nrep + 1) & ~1;                                   // an even number of buffer flips
  CK(cudaMemsetAsync(s->dtf_d, 0, (size_t)s->ntypes * sizeof(double), s->stream));   // kick factors of a dt = 0 step
  int codes[64];
  for (int f = 0; f < nfeas; ++f) codes[f] = s->shape_codes[f];
  for (int idx = sweep ? std::max(0, i0 - 2) : i0; idx <= (sweep ? std::min(nfeas - 1, i0 + 2) : i0); ++idx) {
    for (int kk = 0; kk < 5; ++kk) {
      static const int by_lanes[5] = {0, 4, 3, 1, 2};   // cand[] in the order 1, 2, 4, 8, 32 lanes per row
      const int k = by_lanes[kk];
      s->kernel_eff = cand[k];
      s->brick_forced = codes[idx];
      s->cap_scale_tile = s->cap_scale_int = s->cap_scale_row = 1.0;   // an overflow of one shape must not inflate the next
      s->planned = false;
      rc = build(s, true);
      if (rc && s->tune_verbose)
        fprintf(stderr, "autotune: K=%d shape %d (%dx%dx%d): build failed (%d) %s\n", lanes_for(cand[k]), idx, s->g.b[0], s->g.b[1], s->g.b[2], rc, s->err.c_str());
      if (rc == MD_ERR_OVERFLOW && idx != i0) continue;   // this shape does not fit with this many lanes per row
      if (rc) return rc;
      if ((s->g.b[0] | s->g.b[1] << 4 | s->g.b[2] << 8) != codes[idx]) continue;   // the build had to fall back to another shape
      const double ms_build = s->ms_build;
      auto step = [&](int r) {
        StepMode M;
        M.epi = EPI_KICK_DRIFT; M.in_run = 0; M.parity = r & 1; M.dt = 0.0; M.hdtf = 0.0; M.trigger = 1e300;
        M.xbuf = s->xcur ^ (r & 1);
        return compute_forces_device(s, false, M);
      };
      for (int r = 0; r < 2; ++r) { rc = step(r); if (rc) return rc; }   // warm-up
      float ms = 0;
      int reps = nrep;
      for (int pass = 0; pass < 2; ++pass) {
        CK(cudaEventRecord(s->ev4, s->stream));
        for (int r = 0; r < reps; ++r) { rc = step(r); if (rc) return rc; }
        CK(cudaEventRecord(s->ev5, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        cudaEventElapsedTime(&ms, s->ev4, s->ev5);
        if (ms >= 1.0f) break;   // short steps (small boxes) are timed over four times as many launches: the candidates
        if (pass == 0) reps *= 4;   // differ by a few percent there, which a handful of 20-100 us launches does not resolve
      }
      const double per = ms / reps, score = per + ms_build / 8.0;
      if (s->tune_verbose)
        fprintf(stderr, "autotune: K=%d shape %d of %d (%dx%dx%d) tiles %d threads %d step %.4f ms build %.4f ms score %.4f\n", lanes_for(cand[k]), idx,
                nfeas, s->g.b[0], s->g.b[1], s->g.b[2], s->g.ntiles, s->force_threads, per, ms_build, score);
      if (ms_out && per < ms_out[k]) ms_out[k] = per;
      // more lanes per row must win by 2 % (timing noise)
      if (score < (best_score < 1e299 && lanes_for(cand[k]) > lanes_for(best) ? 0.98 * best_score : best_score)) {
        best_score = score; best = cand[k]; best_b = s->brick_forced;
      }
    }
  }
  s->kernel_eff = best;
  s->brick_forced = best_b;
  s->cap_scale_tile = s->cap_scale_int = s->cap_scale_row = 1.0;
  s->autotuned = true;
  s->tune_stage = s->tune_stage == 0 ? 1 : 2;
  s->tune_step = s->nsteps_total;
  s->planned = false;
  s->list_valid = false;
  return MD_OK;
}

// ---- caller-order I/O -----------------------------------------------------------------------------------
int set_vec3(md_system* s, const double* in, double* dst) {
  const double* src = in;
  if (!is_device_ptr(in)) {
    CK(cudaMemcpyAsync(s->io_d, in, 3 * (size_t)s->N * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    src = s->io_d;
  }
  CK(launch(s, k_scatter_in, blocks_for(s->N, 256), 256, 0, (int)s->N, (const int*)s->id[s->cur], src, dst, s->ld));
  if (src == s->io_d) CK(cudaStreamSynchronize(s->stream));   // the caller may reuse its buffer
  return MD_OK;
}
int get_vec3(md_system* s, const double* srcv, double* out) {
  bool dev = is_device_ptr(out);
  double* dst = dev ? out : s->io_d;
  CK(launch(s, k_gather_out, blocks_for(s->N, 256), 256, 0, (int)s->N, (const int*)s->id[s->cur], srcv, dst, s->ld));
  if (!dev) {
    CK(cudaMemcpyAsync(out, s->io_d, 3 * (size_t)s->N * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
  }
  return MD_OK;
}

}  // namespace

// =====================================================================================================
// C ABI
// =====================================================================================================
extern "C" {

const char* md_last_error(const md_system* s) { return s ? s->err.c_str() : g_create_error.c_str(); }

int md_create(md_system** out, const double box[3], int64_t N, const int32_t* types, int ntypes, const double* mass,
              void* cuda_stream) {
  md_system* s = nullptr;
  if (!out || !box || !types || !mass || N <= 0 || ntypes <= 0 || N > 2000000000LL)
    return fail(nullptr, MD_ERR_BAD_ARGUMENT, "md_create: bad argument");
  for (int d = 0; d < 3; ++d)
    if (!(box[d] > 0.0) || !std::isfinite(box[d])) return fail(nullptr, MD_ERR_BAD_ARGUMENT, "md_create: box edge must be positive");
  for (int t = 0; t < ntypes; ++t)
    if (!(mass[t] > 0.0)) return fail(nullptr, MD_ERR_BAD_ARGUMENT, "md_create: masses must be positive");
  s = new md_system();
  s->balance_after = BALANCE_AFTER;
  auto bail = [&](int code) { std::string e = s->err; md_destroy(s); g_create_error = e; return code; };
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) s->num_sms = sms;
  }
  s->N = N;
  s->ld = ((size_t)N + 31) & ~(size_t)31;
  s->stream = (cudaStream_t)cuda_stream;
  s->ntypes = ntypes;
  for (int d = 0; d < 3; ++d) s->box[d] = box[d];
#define CKC(call)                                                                                     \
  do {                                                                                                \
    cudaError_t e_ = (call);                                                                          \
    if (e_ != cudaSuccess) { fail(s, MD_ERR_CUDA, "%s failed: %s", #call, cudaGetErrorString(e_)); return bail(MD_ERR_CUDA); } \
  } while (0)
  for (int k = 0; k < 2; ++k) {
    CKC(dalloc(&s->x[k], 3 * s->ld)); CKC(dalloc(&s->v[k], 3 * s->ld));
    CKC(dalloc(&s->id[k], s->ld)); CKC(dalloc(&s->type[k], s->ld));
    CKC(cudaMalloc(&s->xr[k], (s->ld + 8) * 32));
    CKC(cudaMemsetAsync(s->x[k], 0, 3 * s->ld * sizeof(double), s->stream));
    CKC(cudaMemsetAsync(s->v[k], 0, 3 * s->ld * sizeof(double), s->stream));
  }
  CKC(dalloc(&s->f, 3 * s->ld)); CKC(dalloc(&s->x0, 3 * s->ld)); CKC(dalloc(&s->rho, s->ld)); CKC(dalloc(&s->fp, s->ld));
  CKC(cudaMemsetAsync(s->f, 0, 3 * s->ld * sizeof(double), s->stream));
  CKC(dalloc(&s->cell_of, s->ld)); CKC(dalloc(&s->rank, s->ld)); CKC(dalloc(&s->perm, s->ld)); CKC(dalloc(&s->mkey, s->ld));
  CKC(dalloc(&s->nstat_d, (size_t)4));
  CKC(dalloc(&s->mass_d, (size_t)ntypes)); CKC(dalloc(&s->dtf_d, (size_t)ntypes));
  CKC(dalloc(&s->thermo_d, (size_t)8)); CKC(dalloc(&s->ke_partial_d, (size_t)blocks_for(N, 256)));
  s->mass_h.assign(mass, mass + ntypes); CKC(dalloc(&s->scalars_d, 16)); CKC(dalloc(&s->io_d, 3 * s->ld));
  CKC(dalloc(&s->io_i, s->ld)); CKC(dalloc(&s->types_caller, s->ld)); CKC(dalloc(&s->flags_d, 1));
  CKC(cudaMallocHost((void**)&s->flags_h, sizeof(Flags))); CKC(cudaMallocHost((void**)&s->scalars_h, 16 * sizeof(double)));
  CKC(cudaEventCreate(&s->ev0)); CKC(cudaEventCreate(&s->ev1)); CKC(cudaEventCreate(&s->ev2)); CKC(cudaEventCreate(&s->ev3)); CKC(cudaEventCreate(&s->ev4)); CKC(cudaEventCreate(&s->ev5));
  CKC(cudaStreamCreateWithFlags(&s->capture_stream, cudaStreamNonBlocking));
  for (int k = 0; k < 2 * md_system_impl::NSAMPLE; ++k) CKC(cudaEventCreate(&s->pev[k]));
  for (int k = 0; k < md_system_impl::NSAMPLE; ++k) CKC(cudaEventCreate(&s->pev_mid[k]));
  CKC(cudaMemcpyAsync(s->mass_d, mass, ntypes * sizeof(double), cudaMemcpyHostToDevice, s->stream));
  CKC(cudaMemcpyAsync(s->types_caller, types, (size_t)N * sizeof(int), is_device_ptr(types) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                      s->stream));
  CKC(cudaMemsetAsync(s->flags_d, 0, sizeof(Flags), s->stream));
  CKC(launch(s, k_iota, blocks_for(N, 256), 256, 0, (int)N, s->id[0]));
  CKC(cudaMemcpyAsync(s->type[0], s->types_caller, (size_t)N * sizeof(int), cudaMemcpyDeviceToDevice, s->stream));
  {   // type ids index the mass table on the device: refuse anything outside 0..ntypes-1
    CKC(cudaMemsetAsync(s->nstat_d, 0, 4 * sizeof(int), s->stream));
    CKC(launch(s, k_check_types, blocks_for(N, 256), 256, 0, (int)N, (const int*)s->types_caller, ntypes, s->nstat_d));
    CKC(cudaMemcpyAsync(s->flags_h, s->nstat_d, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  }
  CKC(cudaStreamSynchronize(s->stream));
  if (*reinterpret_cast<const int*>(s->flags_h) != 0) {
    fail(s, MD_ERR_BAD_ARGUMENT, "md_create: type ids must lie in 0..ntypes-1");
    return bail(MD_ERR_BAD_ARGUMENT);
  }
#undef CKC
  *out = s;
  return MD_OK;
}

void md_destroy(md_system* s) {
  if (!s) return;
  for (int k = 0; k < 2; ++k) { cudaFree(s->x[k]); cudaFree(s->v[k]); cudaFree(s->id[k]); cudaFree(s->type[k]); cudaFree(s->xr[k]); }
  cudaFree(s->tab);
  cudaFree(s->f); cudaFree(s->x0); cudaFree(s->rho); cudaFree(s->fp); cudaFree(s->cell_of); cudaFree(s->rank); cudaFree(s->perm); cudaFree(s->mkey);
  cudaFree(s->nstat_d); cudaFree(s->export_buf);
  cudaFree(s->numneigh); cudaFree(s->cell_count); cudaFree(s->cell_start); cudaFree(s->list); cudaFree(s->mass_d); cudaFree(s->dtf_d); cudaFree(s->thermo_d); cudaFree(s->ke_partial_d);
  cudaFree(s->tab_rho_f); cudaFree(s->tab_phi_f); cudaFree(s->tab_rho_dd); cudaFree(s->tab_phi_dd); cudaFree(s->tab_F_dd);
  cudaFree(s->ev_partials); cudaFree(s->scalars_d); cudaFree(s->io_d); cudaFree(s->io_i); cudaFree(s->types_caller); cudaFree(s->flags_d);
  if (s->flags_h) cudaFreeHost(s->flags_h);
  if (s->scalars_h) cudaFreeHost(s->scalars_h);
  for (auto& G : s->build_graph) if (G.exec) cudaGraphExecDestroy(G.exec);
  if (s->capture_stream) cudaStreamDestroy(s->capture_stream);
  if (s->ev0) cudaEventDestroy(s->ev0);
  if (s->ev1) cudaEventDestroy(s->ev1);
  if (s->ev2) cudaEventDestroy(s->ev2);
  if (s->ev3) cudaEventDestroy(s->ev3);
  if (s->ev4) cudaEventDestroy(s->ev4);
  if (s->ev5) cudaEventDestroy(s->ev5);
  for (cudaEvent_t e : s->pev) if (e) cudaEventDestroy(e);
  for (cudaEvent_t e : s->pev_mid) if (e) cudaEventDestroy(e);
  delete s;
}

int md_set_units(md_system* s, double ftm2v, double mvv2e) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  if (!(ftm2v > 0.0) || !(mvv2e > 0.0)) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_units: factors must be positive");
  s->ftm2v = ftm2v; s->mvv2e = mvv2e;
  return MD_OK;
}

int md_set_option(md_system* s, const char* name, int64_t value) {
  if (!s || !name) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_option: NULL") : MD_ERR_BAD_ARGUMENT;
  const std::string n(name);
  if (n == "tile_shape") {
    const int bx = (int)(value & 15), by = (int)((value >> 4) & 15), bz = (int)((value >> 8) & 15);
    if (value != 0 && (value < 0 || value > 0xfff || bx < 1 || bx > 4 || by < 1 || by > bx || bz < 1 || bz > by))
      return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_option: tile_shape wants bx | by << 4 | bz << 8 with 4 >= bx >= by >= bz >= 1, or 0");
    s->opt_tile_shape = (int)value;
  } else if (n == "force_threads") {
    if (value < 0 || value > 1024) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_option: force_threads wants 0..1024");
    s->opt_force_threads = (int)value;
  } else if (n == "balance_after") {
    s->balance_after = (int)std::max<int64_t>(-1, std::min<int64_t>(value, 1 << 30));
  } else if (n == "no_balance") {
    s->no_balance = value != 0;
  } else if (n == "no_persistent") {
    s->no_persistent = value != 0;
  } else if (n == "persistent_groups") {
    if (value < 0 || value > 2) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_option: persistent_groups wants 0 (automatic), 1 or 2");
    s->p_groups = (int)value;
  } else if (n == "persistent_min_tiles_per_sm") {
    if (value < 0) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_option: persistent_min_tiles_per_sm wants >= 0");
    s->p_min_tiles_per_sm = (int)std::min<int64_t>(value, 1 << 20);
  } else if (n == "build_graph") {
    s->opt_build_graph = value != 0;
  } else if (n == "pdl") {
    s->opt_pdl = value != 0;
  } else if (n == "tab_smem") {
    s->opt_tab_smem = value != 0;
  } else if (n == "tune_verbose") {
    s->tune_verbose = value != 0;
  } else {
    return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_option: unknown option '%s'", name);
  }
  s->planned = false; s->list_valid = false; s->forces_valid = false; s->autotuned = false; s->tune_stage = 0; s->brick_forced = 0;
  return MD_OK;
}

int md_set_precision(md_system* s, int mode) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  if (mode != MD_FP64 && mode != MD_MIXED) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_precision: unknown mode %d", mode);
  if (mode != s->precision) { s->precision = mode; s->planned = false; s->list_valid = false; s->forces_valid = false; s->autotuned = false; s->tune_stage = 0; s->brick_forced = 0; }
  return MD_OK;
}

int md_set_positions(md_system* s, const double* x) {
  if (!s || !x) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_positions: NULL") : MD_ERR_BAD_ARGUMENT;
  int rc = set_vec3(s, x, s->x[s->xcur]);
  if (rc) return rc;
  s->have_x = true; s->list_valid = false; s->forces_valid = false;
  return MD_OK;
}

int md_set_velocities(md_system* s, const double* v) {
  if (!s || !v) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_velocities: NULL") : MD_ERR_BAD_ARGUMENT;
  return set_vec3(s, v, s->v[s->cur]);
}

int md_set_pair(md_system* s, int style, const double* params, int nparams, double rc, double skin) {
  if (!s || !params) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: NULL") : MD_ERR_BAD_ARGUMENT;
  int need = style == MD_PAIR_LJ126 ? 2 : (style == MD_PAIR_EAM_FS ? 5 : (style == MD_PAIR_BUCK_COUL ? 1 : (style == MD_PAIR_EAM_TAB ? 2 : -1)));
  if (need < 0) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: unknown style %d", style);
  if (nparams != need) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: style %d takes %d parameters, got %d", style, need, nparams);
  if (!(rc > 0.0) || !(skin >= 0.0) || !std::isfinite(rc) || !std::isfinite(skin)) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: bad rc/skin");
  for (int k = 0; k < need; ++k)
    if (!std::isfinite(params[k])) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: non-finite parameter");
  if (style == MD_PAIR_EAM_FS && !(params[4] > 0.0)) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: r0 must be positive");
  if (style == MD_PAIR_EAM_TAB && (!(params[0] > 0.0) || !(params[1] > 0.0))) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair: dr and drho must be positive");
  for (int d = 0; d < 3; ++d)
    if (s->box[d] < 3.0 * (rc + skin))
      return fail(s, MD_ERR_BOX_TOO_SMALL, "box edge %d = %g < 3 (rc+skin) = %g", d, s->box[d], 3.0 * (rc + skin));
  s->style = style;
  for (int k = 0; k < 5; ++k) s->params[k] = k < need ? params[k] : 0.0;
  s->rc = rc; s->skin = skin;
  s->pair_set = true; s->planned = false; s->list_valid = false; s->forces_valid = false; s->autotuned = false; s->tune_stage = 0; s->brick_forced = 0;
  return MD_OK;
}

int md_set_pair_coeff(md_system* s, int type_a, int type_b, const double* c, int n) {
  if (!s || !c) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair_coeff: NULL") : MD_ERR_BAD_ARGUMENT;
  if (type_a < 0 || type_b < 0 || type_a >= s->ntypes || type_b >= s->ntypes || type_a >= MAX_PAIR_TYPES || type_b >= MAX_PAIR_TYPES)
    return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair_coeff: types must lie in 0..min(ntypes, %d)-1", MAX_PAIR_TYPES);
  if (n != 3) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair_coeff: MD_PAIR_BUCK_COUL takes 3 coefficients {A, rho, C}, got %d", n);
  if (!std::isfinite(c[0]) || !std::isfinite(c[1]) || !std::isfinite(c[2]) || !(c[1] > 0.0))
    return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_pair_coeff: coefficients must be finite and rho positive");
  for (int k = 0; k < 3; ++k) s->pair_coef[type_a][type_b][k] = s->pair_coef[type_b][type_a][k] = c[k];
  s->pair_coef_set[type_a][type_b] = s->pair_coef_set[type_b][type_a] = true;
  s->planned = false; s->forces_valid = false;
  return MD_OK;
}

// per-interval cubic of a uniform table (reading s26): node slopes by centred differences (4th order inside, 2nd order next
// to the ends, one-sided at the ends), Hermite cubic c0 + c1 u + c2 u^2 + c3 u^3 on [k, k+1]
static void table_cubics(const double* y, int n, double h, std::vector<double>& c) {
  auto slope = [&](int k) {
    if (k <= 0) return (y[1] - y[0]) / h;
    if (k >= n - 1) return (y[n - 1] - y[n - 2]) / h;
    if (k == 1 || k == n - 2) return (y[k + 1] - y[k - 1]) / (2.0 * h);
    return (y[k - 2] - 8.0 * y[k - 1] + 8.0 * y[k + 1] - y[k + 2]) / (12.0 * h);
  };
  c.resize(4 * (size_t)(n - 1));
  for (int k = 0; k < n - 1; ++k) {
    const double D = y[k + 1] - y[k], m0 = h * slope(k), m1 = h * slope(k + 1);
    c[4 * k] = y[k]; c[4 * k + 1] = m0; c[4 * k + 2] = 3.0 * D - 2.0 * m0 - m1; c[4 * k + 3] = -2.0 * D + m0 + m1;
  }
}

int md_set_eam_tables(md_system* s, const double* rho_r, const double* phi_r, int nr, const double* F_rho, int nrho) {
  if (!s || !rho_r || !phi_r || !F_rho) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_eam_tables: NULL") : MD_ERR_BAD_ARGUMENT;
  if (nr < 5 || nrho < 5 || nr > (1 << 24) || nrho > (1 << 24)) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_eam_tables: tables need 5 .. 2^24 entries");
  if (s->style != MD_PAIR_EAM_TAB) return fail(s, MD_ERR_NOT_READY, "md_set_eam_tables: call md_set_pair(MD_PAIR_EAM_TAB, {dr, drho}, ...) first");
  for (int k = 0; k < nr; ++k) if (!std::isfinite(rho_r[k]) || !std::isfinite(phi_r[k])) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_eam_tables: non-finite entry");
  for (int k = 0; k < nrho; ++k) if (!std::isfinite(F_rho[k])) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_eam_tables: non-finite entry");
  std::vector<double> cr, cp, cF;
  table_cubics(rho_r, nr, s->params[0], cr);
  table_cubics(phi_r, nr, s->params[0], cp);
  table_cubics(F_rho, nrho, s->params[1], cF);
  std::vector<float> fr(cr.begin(), cr.end()), fpv(cp.begin(), cp.end());
  cudaFree(s->tab_rho_f); cudaFree(s->tab_phi_f); cudaFree(s->tab_rho_dd); cudaFree(s->tab_phi_dd); cudaFree(s->tab_F_dd);
  s->tab_rho_f = s->tab_phi_f = nullptr; s->tab_rho_dd = s->tab_phi_dd = s->tab_F_dd = nullptr;
  CK(dalloc(&s->tab_rho_f, (size_t)nr - 1)); CK(dalloc(&s->tab_phi_f, (size_t)nr - 1));
  CK(dalloc(&s->tab_rho_dd, (size_t)nr - 1)); CK(dalloc(&s->tab_phi_dd, (size_t)nr - 1)); CK(dalloc(&s->tab_F_dd, (size_t)nrho - 1));
  CK(cudaMemcpyAsync(s->tab_rho_f, fr.data(), fr.size() * sizeof(float), cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpyAsync(s->tab_phi_f, fpv.data(), fpv.size() * sizeof(float), cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpyAsync(s->tab_rho_dd, cr.data(), cr.size() * sizeof(double), cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpyAsync(s->tab_phi_dd, cp.data(), cp.size() * sizeof(double), cudaMemcpyHostToDevice, s->stream));
  CK(cudaMemcpyAsync(s->tab_F_dd, cF.data(), cF.size() * sizeof(double), cudaMemcpyHostToDevice, s->stream));
  CK(cudaStreamSynchronize(s->stream));   // the staging vectors are locals
  s->eam_nr = nr; s->eam_nrho = nrho;
  s->planned = false; s->forces_valid = false;
  return MD_OK;
}

int md_set_type_charges(md_system* s, const double* q, int n) {
  if (!s || !q) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_set_type_charges: NULL") : MD_ERR_BAD_ARGUMENT;
  if (n != s->ntypes || n > MAX_PAIR_TYPES) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_type_charges: wants ntypes (<= %d) charges", MAX_PAIR_TYPES);
  for (int k = 0; k < n; ++k) {
    if (!std::isfinite(q[k])) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_type_charges: non-finite charge");
    s->qtype[k] = q[k];
  }
  s->planned = false; s->forces_valid = false;
  return MD_OK;
}

int md_set_thermostat(md_system* s, int kind, double kT, double tau) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  if (kind != MD_THERMO_NONE && kind != MD_THERMO_NOSE_HOOVER) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_thermostat: unknown kind %d", kind);
  if (kind == MD_THERMO_NOSE_HOOVER && (!(kT > 0.0) || !(tau > 0.0) || !std::isfinite(kT) || !std::isfinite(tau) || s->N < 2))
    return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_thermostat: kT and tau must be positive (and N >= 2)");
  s->thermostat = kind; s->thermo_kT = kT; s->thermo_tau = tau; s->thermo_xi = 0.0; s->thermo_eta = 0.0;
  return MD_OK;
}

int md_get_thermostat(md_system* s, double out[3]) {
  if (!s || !out) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_get_thermostat: NULL") : MD_ERR_BAD_ARGUMENT;
  const double gkT = (3.0 * (double)s->N - 3.0) * s->thermo_kT, Q = gkT * s->thermo_tau * s->thermo_tau;
  out[0] = s->thermo_xi; out[1] = s->thermo_eta;
  out[2] = s->thermostat == MD_THERMO_NOSE_HOOVER ? 0.5 * Q * s->thermo_xi * s->thermo_xi + gkT * s->thermo_eta : 0.0;
  return MD_OK;
}

int md_set_neighbor(md_system* s, int list_kind, int kernel) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  if (list_kind != MD_LIST_FULL && list_kind != MD_LIST_HALF) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_neighbor: unknown list kind");
  if (kernel < MD_KERNEL_AUTO || kernel > MD_KERNEL_SUBWARP2) return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_neighbor: unknown kernel");
  if (list_kind == MD_LIST_HALF && !(kernel == MD_KERNEL_TPA || kernel == MD_KERNEL_AUTO))
    return fail(s, MD_ERR_BAD_ARGUMENT, "md_set_neighbor: a half list needs MD_KERNEL_TPA");
  s->list_kind = list_kind;
  s->kernel_req = kernel;
  s->kernel_eff = kernel == MD_KERNEL_AUTO ? MD_KERNEL_TPA : kernel;
  s->autotuned = false; s->tune_stage = 0; s->brick_forced = 0;
  s->planned = false; s->list_valid = false; s->forces_valid = false;
  return MD_OK;
}

int md_build_neighbors(md_system* s) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  if (s->kernel_req == MD_KERNEL_AUTO && !s->autotuned) {
    int rc = autotune(s, 5, nullptr);
    if (rc) return rc;
  }
  return build(s, false);
}

int md_autotune(md_system* s, int nrep, double ms_out[5]) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  return autotune(s, nrep, ms_out);
}

int md_compute_forces(md_system* s, double* f_out, double* energy_out, double virial_out[6]) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  int rc = ensure_list(s);
  if (rc) return rc;
  bool ev = energy_out || virial_out;
  CK(cudaEventRecord(s->ev0, s->stream));
  rc = compute_forces_device(s, ev);
  if (rc) return rc;
  CK(cudaEventRecord(s->ev1, s->stream));
  if (f_out) { rc = get_vec3(s, s->f, f_out); if (rc) return rc; }
  if (ev) {
    CK(cudaMemcpyAsync(s->scalars_h, s->scalars_d, 8 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    if (energy_out) *energy_out = s->scalars_h[0];
    if (virial_out) for (int k = 0; k < 6; ++k) virial_out[k] = s->scalars_h[1 + k];
  }
  s->force_timing_pending = true;   // read by md_get_stats once the stream has drained (the call may not have synchronised)
  return MD_OK;
}

int md_run(md_system* s, int64_t nsteps, double dt) {
  if (!s) return MD_ERR_BAD_ARGUMENT;
  if (nsteps < 0 || !std::isfinite(dt)) return fail(s, MD_ERR_BAD_ARGUMENT, "md_run: bad nsteps/dt");
  int64_t launches0 = s->launches, builds0 = s->nbuilds;
  s->force_timing_pending = false;   // ev0 / ev1 are reused below
  s->ms_build_in_run = 0;
  // ms_run covers the time stepping proper: variant selection (autotune, which reuses ev0 / ev1) and a first list
  // build that the call may have to do come before the first event; that build is reported in ms_build_in_run
  const bool had_list = s->list_valid;
  int rc = ensure_list(s);
  if (rc) return rc;
  if (!had_list) s->ms_build_in_run += s->ms_build;
  CK(cudaEventRecord(s->ev0, s->stream));
  if (!s->forces_valid) { rc = compute_forces_device(s, false); if (rc) return rc; }
  if (nsteps > 0) s->counts_valid = false;
  const int N = (int)s->N;
  const double trigger = 0.25 * s->skin * s->skin;
  const double hdtf = 0.5 * dt * s->ftm2v;
  auto upload_dtf = [&]() -> int {   // per-type kick factor of the fused epilogue (same expression as the integrator kernels: hdtf / m)
    std::vector<double> dtf(s->mass_h.size());
    for (size_t t = 0; t < dtf.size(); ++t) dtf[t] = hdtf / s->mass_h[t];
    CK(cudaMemcpyAsync(s->dtf_d, dtf.data(), dtf.size() * sizeof(double), cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));   // dtf is a stack object
    return MD_OK;
  };
  rc = upload_dtf();
  if (rc) return rc;
  const int64_t sample_every = (nsteps + md_system_impl::NSAMPLE - 1) / md_system_impl::NSAMPLE;
  int nsampled = 0;
  s->ms_force_sampled = 0; s->ms_pass1_sampled = 0;
  const bool eam = s->style == MD_PAIR_EAM_FS || s->style == MD_PAIR_EAM_TAB;
  const bool nvt = s->thermostat == MD_THERMO_NOSE_HOOVER;
  const bool fused = s->list_kind != MD_LIST_HALF && !nvt;
  if (nsteps > 0 && fused) {
    // Velocity Verlet with ONE launch per time step (two for EAM): the force kernel of step n also does the
    // second half kick of step n and the first half kick + drift of step n+1, writing the new positions to
    // the other x buffer and the max displacement to a device flag.  Steps are enqueued in batches without
    // host synchronisation; a step kernel that finds the list stale does nothing and raises `stop`, and so
    // do all later ones; the host then rebuilds and continues from the step that stopped.
    CK(cudaMemsetAsync(s->flags_d, 0, sizeof(Flags), s->stream));
    rc = initial_integrate(s, dt, hdtf);
    if (rc) return rc;
    s->forces_valid = false;
    int64_t remaining = nsteps;
    int parity = 0;
    // a rebuild is enqueued without waiting for it (pending): the next batch follows on the stream, its kernels judge
    // the build's flags themselves (list_is_stale) and the host does so with the flags it reads after that batch
    bool pending = false, pending_list = false;
    while (remaining > 0) {
      const int m = (int)std::min<int64_t>(s->batch, remaining);
      int sample_slot[64];
      for (int k = 0; k < m; ++k) {
        const bool last = (int64_t)k == remaining - 1;
        StepMode M;
        M.epi = last ? EPI_FINAL : EPI_KICK_DRIFT;
        M.in_run = 1; M.parity = (parity + k) & 1; M.dt = dt; M.hdtf = hdtf; M.trigger = trigger;
        M.xbuf = s->xcur ^ (k & 1);
        const int64_t step = nsteps - remaining + k;
        const bool sample = step % sample_every == 0 && nsampled < md_system_impl::NSAMPLE;
        sample_slot[k] = -1;
        if (sample) { sample_slot[k] = nsampled; CK(cudaEventRecord(s->pev[2 * nsampled], s->stream)); if (eam) s->mid_event = s->pev_mid[nsampled]; }
        rc = compute_forces_device(s, false, M);
        s->mid_event = nullptr;
        if (rc) return rc;
        if (sample) { CK(cudaEventRecord(s->pev[2 * nsampled + 1], s->stream)); ++nsampled; }
      }
      CK(cudaMemcpyAsync(s->flags_h, s->flags_d, sizeof(Flags), cudaMemcpyDeviceToHost, s->stream));
      CK(cudaStreamSynchronize(s->stream));
      const int done = s->flags_h->steps_done;
      const bool stopped = s->flags_h->stop != 0;
      if (done < 0 || done > m || (!stopped && done != m)) return fail(s, MD_ERR_CUDA, "md_run: inconsistent step count from the device (%d of %d)", done, m);
      if (pending) {
        bool again = false;
        rc = build_finish(s, *s->flags_h, pending_list, &again);
        if (rc) return rc;
        s->ms_build_in_run += s->ms_build;
        pending = false;
        // a capacity was too small: no step of this batch ran; the stopped branch below plans anew and builds again
        if (again && (done != 0 || !stopped)) return fail(s, MD_ERR_CUDA, "md_run: steps ran on an overflowed build");
      }
      for (int k = 0; k < m; ++k) {   // timings of the launches that really ran; a sampled launch that was skipped gives its slot back
        if (sample_slot[k] < 0) continue;
        if (k < done) {
          float t = 0;
          CK(cudaEventElapsedTime(&t, s->pev[2 * sample_slot[k]], s->pev[2 * sample_slot[k] + 1])); s->ms_force_sampled += t; s->nforce_sampled_acc++;
          if (eam) { CK(cudaEventElapsedTime(&t, s->pev[2 * sample_slot[k]], s->pev_mid[sample_slot[k]])); s->ms_pass1_sampled += t; }
        }
        else nsampled = std::min(nsampled, sample_slot[k]);
      }
      const bool final_ran = done == m && (int64_t)m == remaining;
      const int flips = final_ran ? done - 1 : done;   // kick+drift launches that ran
      s->xcur ^= (flips & 1);
      s->nsteps_total += done;
      s->steps_since_build += done;
      remaining -= done;
      parity = (parity + done) & 1;
      s->nforce -= (m - done);
      if (final_ran) s->forces_valid = true;
      if (stopped) {
        s->batch = std::min(32, std::max(2, done + 2));
        // MD_KERNEL_AUTO: the setup-time choice was made on the caller's positions, often a perfect
        // lattice, whose rows all have one length; it is confirmed ONCE on evolved positions, at the first rebuild
        // that comes 20 or more time steps later (the timing builds its own lists; the state is left as a build leaves it)
        if (s->kernel_req == MD_KERNEL_AUTO && s->tune_stage == 1 && s->nsteps_total - s->tune_step >= 20) {
          rc = autotune(s, 5, nullptr);
          if (rc) return rc;
          rc = upload_dtf();   // the timing ran dt = 0 steps
          if (rc) return rc;
        }
        if (s->balance_after <= 0) {   // tuning experiments only: balance right after every build
          rc = build(s, false);   // also clears the flags
          if (rc) return rc;
          s->ms_build_in_run += s->ms_build;
        } else {
          if (++s->build_attempts > 6) return fail(s, MD_ERR_OVERFLOW, "tile or neighbor-row capacity still exceeded after re-planning");
          s->list_valid = false; s->forces_valid = false; s->list_built_for_export = false; s->counts_valid = false;
          rc = build_enqueue(s, false, &pending_list, true);   // also clears the flags
          if (rc) return rc;
          pending = true;
        }
        parity = 0;
      } else if (remaining > 0) {
        if (s->steps_since_build >= s->balance_after && s->kernel_eff != MD_KERNEL_CELL) { rc = balance_rows(s); if (rc) return rc; }
        CK(cudaMemsetAsync(&s->flags_d->steps_done, 0, sizeof(int), s->stream));
        if (done == s->batch) s->batch = std::min(32, s->batch + 2);
      }
    }
  } else {
    // half list: the scatter kernel's forces are complete only when it has finished, so a time step is three launches
    // (kick + drift + displacement flag | forces | kick).  They are enqueued in batches like the fused path: the force
    // kernel reads the flag the integrator has just written and, if the list is stale, does nothing and raises `stop`;
    // every later kernel of the batch then does nothing either.  The host reads {steps_done, stop} once per batch; the
    // step that stopped has had its first half (kick + drift) applied, so the host rebuilds, evaluates the forces and
    // finishes it before it enqueues the next batch.
    // NVT (reading s25): TH(dt/2) before the first kick and after the second; the thermostat's scalar state lives on the
    // device (thermo_d), the kinetic energy it needs comes out of the second kick's kernel as per-block partials
    const unsigned nb256 = blocks_for(N, 256);
    auto final_integrate = [&](bool in_run) -> int {
      Flags* rf = in_run ? s->flags_d : (Flags*)nullptr;
      if (!nvt) {
        CK(launch(s, k_final_integrate, nb256, 256, 0, N, s->ld, s->v[s->cur], (const double*)s->f, (const int*)s->type[s->cur],
                  (const double*)s->mass_d, hdtf, rf));
        return MD_OK;
      }
      CK(launch(s, k_final_integrate_ke, nb256, 256, 0, N, s->ld, s->v[s->cur], (const double*)s->f, (const int*)s->type[s->cur],
                (const double*)s->mass_d, hdtf, s->ke_partial_d, rf));
      CK(launch(s, k_nh_reduce, 1, 256, 0, (int)nb256, (const double*)s->ke_partial_d, s->mvv2e, s->thermo_d, 0.5 * dt, (const Flags*)rf));
      CK(launch(s, k_scale_velocities, nb256, 256, 0, N, s->ld, s->v[s->cur], (const double*)(s->thermo_d + 3), (const Flags*)rf));
      return MD_OK;
    };
    auto first_half = [&](bool in_run) -> int {   // TH(dt/2) (NVT), then kick + drift + displacement flag
      if (nvt) CK(launch(s, k_nh_half, 1, 1, 0, s->thermo_d, 0.5 * dt, in_run ? (const Flags*)s->flags_d : (const Flags*)nullptr));
      return initial_integrate(s, dt, hdtf, in_run, nvt ? s->thermo_d + 3 : nullptr);
    };
    CK(cudaMemsetAsync(s->flags_d, 0, sizeof(Flags), s->stream));
    if (nvt && nsteps > 0) {
      // thermostat constants and state; the current kinetic energy (a kick by zero gives the partials)
      const double gkT = (3.0 * (double)s->N - 3.0) * s->thermo_kT;
      const double th[8] = {s->thermo_xi, s->thermo_eta, 0.0, 1.0, gkT, gkT * s->thermo_tau * s->thermo_tau, 0.0, 0.0};
      CK(cudaMemcpyAsync(s->thermo_d, th, sizeof th, cudaMemcpyHostToDevice, s->stream));
      CK(cudaStreamSynchronize(s->stream));   // th is a stack object
      CK(launch(s, k_final_integrate_ke, nb256, 256, 0, N, s->ld, s->v[s->cur], (const double*)s->f, (const int*)s->type[s->cur],
                (const double*)s->mass_d, 0.0, s->ke_partial_d, (Flags*)nullptr));
      CK(launch(s, k_nh_reduce, 1, 256, 0, (int)nb256, (const double*)s->ke_partial_d, s->mvv2e, s->thermo_d, 0.0, (const Flags*)nullptr));
    }
    int64_t remaining = nsteps;
    while (remaining > 0) {
      const int m = (int)std::min<int64_t>(s->batch, remaining);
      int sample_slot[64];
      for (int k = 0; k < m; ++k) {
        rc = first_half(true);
        if (rc) return rc;
        StepMode M;
        M.epi = EPI_FORCES; M.in_run = 1; M.parity = 0; M.trigger = trigger;
        const int64_t step = nsteps - remaining + k;
        const bool sample = step % sample_every == 0 && nsampled < md_system_impl::NSAMPLE;
        sample_slot[k] = -1;
        if (sample) { sample_slot[k] = nsampled; CK(cudaEventRecord(s->pev[2 * nsampled], s->stream)); if (eam) s->mid_event = s->pev_mid[nsampled]; }
        rc = compute_forces_device(s, false, M);
        s->mid_event = nullptr;
        if (rc) return rc;
        if (sample) { CK(cudaEventRecord(s->pev[2 * nsampled + 1], s->stream)); ++nsampled; }
        rc = final_integrate(true);
        if (rc) return rc;
      }
      CK(cudaMemcpyAsync(s->flags_h, s->flags_d, sizeof(Flags), cudaMemcpyDeviceToHost, s->stream));
      CK(cudaStreamSynchronize(s->stream));
      const int done = s->flags_h->steps_done;
      const bool stopped = s->flags_h->stop != 0;
      if (done < 0 || done > m || (!stopped && done != m)) return fail(s, MD_ERR_CUDA, "md_run: inconsistent step count from the device (%d of %d)", done, m);
      for (int k = 0; k < m; ++k) {
        if (sample_slot[k] < 0) continue;
        if (k < done) {
          float t = 0;
          CK(cudaEventElapsedTime(&t, s->pev[2 * sample_slot[k]], s->pev[2 * sample_slot[k] + 1])); s->ms_force_sampled += t; s->nforce_sampled_acc++;
          if (eam) { CK(cudaEventElapsedTime(&t, s->pev[2 * sample_slot[k]], s->pev_mid[sample_slot[k]])); s->ms_pass1_sampled += t; }
        }
        else nsampled = std::min(nsampled, sample_slot[k]);
      }
      s->nsteps_total += done;
      s->steps_since_build += done;
      remaining -= done;
      s->nforce -= (m - done);
      if (stopped) {
        s->batch = std::min(32, std::max(2, done + 2));
        rc = build(s, false);   // also clears the flags
        if (rc) return rc;
        s->ms_build_in_run += s->ms_build;
        rc = compute_forces_device(s, false);
        if (rc) return rc;
        rc = final_integrate(false);
        if (rc) return rc;
        s->nsteps_total++; s->steps_since_build++; remaining--;
      } else if (remaining > 0) {
        CK(cudaMemsetAsync(&s->flags_d->steps_done, 0, sizeof(int), s->stream));
        if (done == s->batch) s->batch = std::min(32, s->batch + 2);
      }
    }
    if (nvt && nsteps > 0) {   // thermostat state back to the handle
      CK(cudaMemcpyAsync(s->scalars_h + 9, s->thermo_d, 2 * sizeof(double), cudaMemcpyDeviceToHost, s->stream));
      CK(cudaStreamSynchronize(s->stream));
      s->thermo_xi = s->scalars_h[9]; s->thermo_eta = s->scalars_h[10];
    }
    s->forces_valid = true;
  }
  CK(cudaEventRecord(s->ev1, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  float ms = 0;
  cudaEventElapsedTime(&ms, s->ev0, s->ev1);
  s->ms_run = ms;
  s->nforce_sampled = s->nforce_sampled_acc;
  s->nforce_sampled_acc = 0;
  s->nbuilds_in_run = s->nbuilds - builds0;
  s->launches_last_run = s->launches - launches0;
  return MD_OK;
}

int md_get_positions(md_system* s, double* x) {
  if (!s || !x) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_get_positions: NULL") : MD_ERR_BAD_ARGUMENT;
  if (!s->have_x) return fail(s, MD_ERR_NOT_READY, "positions not set");
  return get_vec3(s, s->x[s->xcur], x);
}
int md_get_velocities(md_system* s, double* v) {
  if (!s || !v) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_get_velocities: NULL") : MD_ERR_BAD_ARGUMENT;
  return get_vec3(s, s->v[s->cur], v);
}
int md_get_forces(md_system* s, double* f) {
  if (!s || !f) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_get_forces: NULL") : MD_ERR_BAD_ARGUMENT;
  if (!s->forces_valid) return fail(s, MD_ERR_NOT_READY, "no valid forces: call md_compute_forces or md_run first");
  return get_vec3(s, s->f, f);
}

// one launch of k_export_list; device buffers only
static int export_launch(md_system* s, int mode, int* nn, int* neigh, int* owner, int64_t stride, int* stat) {
  const Geom& g = s->g;
  const double rl = s->rc + s->skin;
  ExportArgs E{};
  E.g = g; E.tab = s->tab; E.id = s->id[s->cur]; E.x = s->x[s->xcur]; E.ld = s->ld; E.list = s->list; E.numneigh = s->numneigh;
  E.rl2 = rl * rl; E.mode = mode; E.nn_out = nn; E.neigh_out = neigh; E.owner_out = owner; E.stride = (long long)stride; E.stat = stat;
  CK(launch(s, k_export_list, g.ntiles, BUILD_THREADS, export_smem(g), E));
  return MD_OK;
}

// Exact per-atom neighbor statistics of the current list (the stored rows are per pair of atoms and a superset):
// counted by the export kernel with the fp64 test, once per list.  Positions must be those of the build for the
// counts to be the build-time pair set; after time steps they describe the current positions.
static int exact_counts(md_system* s) {
  if (s->counts_valid) return MD_OK;
  if (!s->list_valid || !s->list_built_for_export) { s->max_nb_exact = 0; s->mean_nb_exact = 0; return MD_OK; }
  CK(cudaMemsetAsync(s->nstat_d, 0, 4 * sizeof(int), s->stream));
  int rc = export_launch(s, EXPORT_EXACT, s->io_i, nullptr, nullptr, 0, s->nstat_d);
  if (rc) return rc;
  int h[4];
  CK(cudaMemcpyAsync(h, s->nstat_d, sizeof h, cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  unsigned long long sum;
  memcpy(&sum, &h[2], sizeof sum);
  s->max_nb_exact = h[0];
  s->mean_nb_exact = (double)sum / (double)s->N;
  s->counts_valid = true;
  return MD_OK;
}

static int export_common(md_system* s, int mode, int32_t* numneigh, int32_t* neigh, int32_t* owner, int64_t stride) {
  int rc = ensure_list(s);
  if (rc) return rc;
  if (!s->list_built_for_export) { rc = build(s, true); if (rc) return rc; }
  const size_t N = (size_t)s->N;
  const bool dev_n = is_device_ptr(numneigh), dev_l = is_device_ptr(neigh), dev_o = owner ? is_device_ptr(owner) : true;
  // host buffers are filled through one staging buffer of the handle: [neigh N*stride][numneigh N][owner N]
  const size_t need = (dev_l ? 0 : N * (size_t)stride) + (dev_n ? 0 : N) + (dev_o ? 0 : N);
  if (need > s->export_alloc) {
    cudaFree(s->export_buf);
    s->export_buf = nullptr; s->export_alloc = 0;
    CK(dalloc(&s->export_buf, need));
    s->export_alloc = need;
  }
  int* p = s->export_buf;
  int* dl = dev_l ? neigh : p; if (!dev_l) p += N * (size_t)stride;
  int* dn = dev_n ? numneigh : p; if (!dev_n) p += N;
  int* dow = owner ? (dev_o ? owner : p) : nullptr;
  rc = export_launch(s, mode, dn, dl, dow, stride, nullptr);
  if (rc) return rc;
  if (!dev_n) CK(cudaMemcpyAsync(numneigh, dn, N * sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  if (!dev_l) CK(cudaMemcpyAsync(neigh, dl, N * (size_t)stride * sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  if (owner && !dev_o) CK(cudaMemcpyAsync(owner, dow, N * sizeof(int), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  return MD_OK;
}

int md_get_neighbors(md_system* s, int32_t* numneigh, int32_t* neigh, int64_t stride) {
  if (!s || !numneigh || !neigh || stride <= 0) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_get_neighbors: bad argument") : MD_ERR_BAD_ARGUMENT;
  return export_common(s, EXPORT_EXACT, numneigh, neigh, nullptr, stride);
}

int md_get_neighbor_rows(md_system* s, int32_t* row_owner, int32_t* numrow, int32_t* entries, int64_t stride) {
  if (!s || !row_owner || !numrow || !entries || stride <= 0)
    return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_get_neighbor_rows: bad argument") : MD_ERR_BAD_ARGUMENT;
  return export_common(s, EXPORT_RAW, numrow, entries, row_owner, stride);
}

int md_kinetic_energy(md_system* s, double* ke_out) {
  if (!s || !ke_out) return s ? fail(s, MD_ERR_BAD_ARGUMENT, "md_kinetic_energy: NULL") : MD_ERR_BAD_ARGUMENT;
  CK(cudaMemsetAsync(s->scalars_d + 8, 0, sizeof(double), s->stream));
  CK(launch(s, k_kinetic, std::min<unsigned>(blocks_for(s->N, 256), 1184u), 256, 0, (int)s->N, s->ld, (const double*)s->v[s->cur],
            (const int*)s->type[s->cur], (const double*)s->mass_d, s->scalars_d + 8));
  CK(cudaMemcpyAsync(s->scalars_h + 8, s->scalars_d + 8, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
  CK(cudaStreamSynchronize(s->stream));
  *ke_out = s->scalars_h[8] * s->mvv2e;
  return MD_OK;
}

int md_get_stats(md_system* s, md_stats* out) {
  if (!s || !out) return MD_ERR_BAD_ARGUMENT;
  memset(out, 0, sizeof *out);
  out->natoms = s->N; out->nsteps_total = s->nsteps_total; out->nbuilds = s->nbuilds; out->nforce_evals = s->nforce;
  out->kernel_variant = s->kernel_eff; out->list_kind = s->list_kind; out->precision = s->precision;
  out->lanes_per_atom = lanes_for(s->kernel_eff);
  if (s->planned) {
    for (int d = 0; d < 3; ++d) { out->ncells[d] = s->g.nc[d]; out->brick[d] = s->g.b[d]; }
    out->ntiles = s->g.ntiles; out->tile_capacity = s->g.tile_cap; out->row_capacity = s->g.row_cap;
  }
  out->list_balanced = s->list_balanced ? 1 : 0;
  {
    int rc = exact_counts(s);
    if (rc) return rc;
  }
  out->max_tile_atoms = s->max_tile_atoms; out->max_neighbors = s->max_nb_exact; out->mean_neighbors = s->mean_nb_exact;
  out->max_row = s->max_row; out->mean_row = s->mean_row;
  {
    int rc = md_kinetic_energy(s, &out->kinetic_energy);
    if (rc) return rc;
  }
  if (s->force_timing_pending) {
    float ms = 0;
    if (cudaEventElapsedTime(&ms, s->ev0, s->ev1) == cudaSuccess) s->ms_force = ms;
    s->force_timing_pending = false;
  }
  out->ms_build = s->ms_build; out->ms_force = s->ms_force; out->ms_run = s->ms_run;
  out->launches_last_run = s->launches_last_run; out->launches_total = s->launches;
  out->ms_force_sampled = s->ms_force_sampled; out->nforce_sampled = s->nforce_sampled;
  out->ms_build_in_run = s->ms_build_in_run; out->nbuilds_in_run = s->nbuilds_in_run; out->ms_force_pass1_sampled = s->ms_pass1_sampled;
  return MD_OK;
}

}  // extern "C"

// ---- md_kinetic_energy_noalloc: the kinetic-energy reduction for callers that cannot call cudaMalloc ---------------
// (see include/md_b200.h).  The per-block partials and the completion ticket live in a file-scope device array instead
// of handle memory: every GPU that loads the library holds these MD_NOALLOC_SCRATCH_BYTES until the process exits.
// In HOST code `g_noalloc_scratch` is only a stand-in for the symbol, not a device address: the address a kernel may
// dereference comes from cudaGetSymbolAddress, resolved once per device with that device current.

namespace {

constexpr int NOALLOC_BLOCK = 256;                    // atoms per block = atoms per partial
constexpr int NOALLOC_HEADER_BYTES = 256;             // [0] the ticket counter, rest of the first 256 bytes unused
constexpr int64_t NOALLOC_MAX_BLOCKS = (MD_NOALLOC_SCRATCH_BYTES - NOALLOC_HEADER_BYTES) / (int64_t)sizeof(double);
static_assert(NOALLOC_MAX_BLOCKS * NOALLOC_BLOCK == MD_NOALLOC_MAX_ATOMS, "header constant and scratch layout disagree");
constexpr int NOALLOC_MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_noalloc_scratch[MD_NOALLOC_SCRATCH_BYTES];

// One partial per block of 256 atoms (index order inside the block is fixed by block_sum); the block that draws the
// last ticket adds the partials in index order, so the result does not depend on the order the blocks finish in.
__global__ void __launch_bounds__(NOALLOC_BLOCK) k_kinetic_noalloc(int64_t N, const double* __restrict__ v, const int* __restrict__ type,
                                                                   const double* __restrict__ mass, double mvv2e,
                                                                   unsigned char* __restrict__ scratch, double* __restrict__ ke_out) {
  __shared__ double red[32];
  __shared__ bool last;
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
  double* partial = reinterpret_cast<double*>(scratch + NOALLOC_HEADER_BYTES);
  const int64_t n = (int64_t)blockIdx.x * NOALLOC_BLOCK + threadIdx.x;
  double ke[1] = {0.0};
  if (n < N) {
    const double vx = v[3 * n], vy = v[3 * n + 1], vz = v[3 * n + 2];
    ke[0] = 0.5 * mass[type[n]] * (vx * vx + vy * vy + vz * vz);
  }
  block_sum<1>(ke, red);
  if (threadIdx.x == 0) {
    partial[blockIdx.x] = ke[0];
    __threadfence();                                   // the partial is visible before the ticket is
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  double s[1] = {0.0};
  for (unsigned b = threadIdx.x; b < gridDim.x; b += NOALLOC_BLOCK) s[0] += __ldcg(partial + b);
  block_sum<1>(s, red);
  if (threadIdx.x == 0) {
    *ke_out = s[0] * mvv2e;
    *ticket = 0u;                                      // leave the counter as the next call expects it
  }
}

std::mutex g_noalloc_mutex;
unsigned char* g_noalloc_ptr[NOALLOC_MAX_DEVICES] = {};    // device address of g_noalloc_scratch, per device ordinal

}  // namespace

extern "C" int md_kinetic_energy_noalloc(const double* v_dev, const int32_t* type_dev, const double* mass_dev, int64_t N, double mvv2e,
                                         double* ke_out_dev, void* cuda_stream) {
  md_system* s = nullptr;   // errors go where a failed md_create's go: md_last_error(NULL) on this thread
  if (!v_dev || !type_dev || !mass_dev || !ke_out_dev) return fail(s, MD_ERR_BAD_ARGUMENT, "md_kinetic_energy_noalloc: NULL pointer");
  if (N <= 0) return fail(s, MD_ERR_BAD_ARGUMENT, "md_kinetic_energy_noalloc: N = %lld must be positive", (long long)N);
  if (N > MD_NOALLOC_MAX_ATOMS)
    return fail(s, MD_ERR_BAD_ARGUMENT,
                "md_kinetic_energy_noalloc: N = %lld exceeds MD_NOALLOC_MAX_ATOMS = %lld (the static scratch holds one partial per %d atoms "
                "in %d bytes); use md_kinetic_energy on a handle instead",
                (long long)N, (long long)MD_NOALLOC_MAX_ATOMS, NOALLOC_BLOCK, (int)MD_NOALLOC_SCRATCH_BYTES);
  int dev = 0;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(s, MD_ERR_BAD_ARGUMENT, "md_kinetic_energy_noalloc: device ordinal %d not supported", dev);
  unsigned char* scratch = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_ptr[dev]) {   // set-up, once per device, with that device current
      void* p = nullptr;
      CK(cudaGetSymbolAddress(&p, g_noalloc_scratch));
      if (!p) return fail(s, MD_ERR_CUDA, "md_kinetic_energy_noalloc: cudaGetSymbolAddress returned NULL");
      g_noalloc_ptr[dev] = static_cast<unsigned char*>(p);
    }
    scratch = g_noalloc_ptr[dev];
  }
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  // the ticket must start at zero: the last block of a completed call resets it, the memset covers a call that died
  CK(cudaMemsetAsync(scratch, 0, sizeof(unsigned int), stream));
  k_kinetic_noalloc<<<blocks_for(N, NOALLOC_BLOCK), NOALLOC_BLOCK, 0, stream>>>(N, v_dev, type_dev, mass_dev, mvv2e, scratch, ke_out_dev);
  CK(cudaGetLastError());
  return MD_OK;
}
