// md_kernels.cuh -- device code of the B200-native MD hot path (sm_100a).
//
// Design in one paragraph (details in DESIGN.md).  Atoms are counting-sorted into cells of edge
// >= rc+skin, the cells themselves ordered TILE-major: a tile ("brick") is a box of b^3 cells whose
// atoms are contiguous in memory.  Every heavy kernel is one thread block per tile: it stages the tile's
// interior cells plus a one-cell halo (periodic images resolved while staging) into shared memory as
// TILE-CENTRED coordinates -- fp32 in mixed mode, which is what makes fp32 pair math accurate enough in
// a 168-sigma box -- and then runs the paper's neighbor-list loop against shared
// memory: the "random access" load of atom j (L100) is an LDS, not a texture/L1 gather, and the list
// holds 16-bit tile-local indices, eight to a 128-bit word, so the index stream is half the classic
// 4 B/entry.  One template covers thread-per-atom (K=1), sub-warp (K=8) and warp-per-atom (K=32, the
// paper's BpA with a shuffle reduction instead of a block reduction).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace mdk {

constexpr int MAX_TILE_CELLS = 512;    // (b+2)^3 <= 512  =>  b <= 6
constexpr int BLOCK = 256;             // threads per tile block

struct Geom {
  double L[3];        // box
  double edge[3];     // cell edge = L / nc  (>= rc + skin)
  double inv_edge[3];
  int nc[3];          // cells per dimension (>= 3)
  int b[3];           // tile width in cells (interior)
  int nb[3];          // tiles per dimension
  int ncell;
  int ntiles;
  int tile_cap;       // staged atoms a tile can hold (excluding the dummy slot)
  int interior_cap;   // interior atoms a tile can hold (multiple of 32)
  int row_cap;        // list entries per atom (multiple of 8*K)
  int K;              // lanes per atom: 1, 8, 32
  int chunk_cap;      // row_cap / (8*K): 128-bit words per lane
  int half;           // 1: half list
};

// flags written by the device, read by the host after a build / at the end of a run
struct Flags {
  unsigned long long max_disp2_bits;  // max |x-x0|^2 as the bit pattern of a non-negative double
  int need_tile_cap;                  // > tile_cap     => staging overflow
  int need_interior_cap;              // > interior_cap => interior overflow
  int need_row_cap;                   // > row_cap      => a list row overflowed
  int nonfinite;                      // a non-finite coordinate was binned
  int max_tile_atoms;
  int max_row;
  unsigned long long sum_rows;
};

// ---------------------------------------------------------------------------------------------------
// cell order: tile-major.  Tiles are full (b cells) except the last one in each dimension.
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int tile_width(const Geom& g, int d, int bt) {
  int w = g.nc[d] - bt * g.b[d];
  return w < g.b[d] ? w : g.b[d];
}
__host__ __device__ inline int cell_order_id(const Geom& g, int cx, int cy, int cz) {
  int bx = cx / g.b[0], by = cy / g.b[1], bz = cz / g.b[2];
  int wx = tile_width(g, 0, bx), wy = tile_width(g, 1, by), wz = tile_width(g, 2, bz);
  int lx = cx - bx * g.b[0], ly = cy - by * g.b[1], lz = cz - bz * g.b[2];
  int base = g.nc[0] * g.nc[1] * (bz * g.b[2]) + g.nc[0] * (by * g.b[1]) * wz + (bx * g.b[0]) * wy * wz;
  return base + (lz * wy + ly) * wx + lx;
}

// ---------------------------------------------------------------------------------------------------
// small helpers
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 ld_stream(const uint4* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
template <int K>
__device__ __forceinline__ double group_sum(double v) {
#pragma unroll
  for (int o = K / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum(double v) { return group_sum<32>(v); }

// block-wide sum of NV doubles; result valid in thread 0.  red: shared scratch of NV*32 doubles.
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* red) {
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int k = 0; k < NV; ++k) v[k] = warp_sum(v[k]);
  __syncthreads();
  if (lane == 0)
#pragma unroll
    for (int k = 0; k < NV; ++k) red[k * 32 + wid] = v[k];
  __syncthreads();
  if (wid == 0) {
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      double t = lane < nw ? red[k * 32 + lane] : 0.0;
      v[k] = warp_sum(t);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// tile staging, shared by the list build, every force kernel and the list export
// ---------------------------------------------------------------------------------------------------
struct alignas(16) TileTables {   // lives in shared memory
  int start[MAX_TILE_CELLS];  // staged slot of the first atom of tile cell t
  int gstart[MAX_TILE_CELLS]; // global (sorted) index of the first atom of tile cell t
  int cnt[MAX_TILE_CELLS];    // atoms in tile cell t
  int scan_tmp[32];
  int c0[3], w[3], tc[3];     // first interior cell, interior width, tile width (w+2)
  int ntc;                    // tc[0]*tc[1]*tc[2]
  int n_int;                  // interior atoms (slots [0,n_int))
  int n_staged;               // interior + halo atoms; slot n_staged is the far-away dummy
  int brick_start;            // global index of interior slot 0
};

// Fills the tables for tile `tile`.  All threads of the block call it; ends with __syncthreads().
__device__ inline void tile_setup(const Geom& g, int tile, const int* __restrict__ cell_start, TileTables& tt) {
  const int tid = threadIdx.x;
  if (tid == 0) {
    int bx = tile % g.nb[0], by = (tile / g.nb[0]) % g.nb[1], bz = tile / (g.nb[0] * g.nb[1]);
    int bt[3] = {bx, by, bz};
    for (int d = 0; d < 3; ++d) {
      tt.c0[d] = bt[d] * g.b[d];
      tt.w[d] = tile_width(g, d, bt[d]);
      tt.tc[d] = tt.w[d] + 2;
    }
    tt.ntc = tt.tc[0] * tt.tc[1] * tt.tc[2];
    int first = cell_order_id(g, tt.c0[0], tt.c0[1], tt.c0[2]);
    int ncell_int = tt.w[0] * tt.w[1] * tt.w[2];
    tt.brick_start = cell_start[first];
    tt.n_int = cell_start[first + ncell_int] - tt.brick_start;
  }
  __syncthreads();
  const int ntc = tt.ntc;
  for (int t = tid; t < ntc; t += blockDim.x) {
    int tx = t % tt.tc[0], ty = (t / tt.tc[0]) % tt.tc[1], tz = t / (tt.tc[0] * tt.tc[1]);
    int cx = tt.c0[0] + tx - 1, cy = tt.c0[1] + ty - 1, cz = tt.c0[2] + tz - 1;
    cx += cx < 0 ? g.nc[0] : (cx >= g.nc[0] ? -g.nc[0] : 0);
    cy += cy < 0 ? g.nc[1] : (cy >= g.nc[1] ? -g.nc[1] : 0);
    cz += cz < 0 ? g.nc[2] : (cz >= g.nc[2] ? -g.nc[2] : 0);
    int oid = cell_order_id(g, cx, cy, cz);
    int s = cell_start[oid], c = cell_start[oid + 1] - s;
    bool interior = tx >= 1 && tx <= tt.w[0] && ty >= 1 && ty <= tt.w[1] && tz >= 1 && tz <= tt.w[2];
    tt.gstart[t] = s;
    tt.cnt[t] = c;
    tt.start[t] = interior ? -1 : c;   // halo: count, to be scanned; interior: marker
  }
  __syncthreads();
  // exclusive scan of the halo counts by warp 0
  if (tid < 32) {
    int per = (ntc + 31) / 32, lo = tid * per, hi = min(lo + per, ntc), sum = 0;
    for (int t = lo; t < hi; ++t) sum += tt.start[t] < 0 ? 0 : tt.start[t];
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int u = __shfl_up_sync(0xffffffffu, incl, o);
      if (tid >= o) incl += u;
    }
    int run = tt.n_int + incl - sum;
    for (int t = lo; t < hi; ++t) {
      int c = tt.start[t];
      if (c < 0) tt.start[t] = tt.gstart[t] - tt.brick_start;
      else { tt.start[t] = run; run += c; }
    }
    if (tid == 31) tt.n_staged = tt.n_int + incl;
  }
  __syncthreads();
}

// Periodic image shift minus tile centre for tile cell t, per dimension: staged = x + off.
__device__ __forceinline__ void tile_cell_offset(const Geom& g, const TileTables& tt, int t, double off[3]) {
  int tq[3] = {t % tt.tc[0], (t / tt.tc[0]) % tt.tc[1], t / (tt.tc[0] * tt.tc[1])};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    int u = tt.c0[d] + tq[d] - 1;
    double shift = u < 0 ? -g.L[d] : (u >= g.nc[d] ? g.L[d] : 0.0);
    double centre = (tt.c0[d] + 0.5 * tt.w[d]) * g.edge[d];
    off[d] = shift - centre;
  }
}

// Calls store(slot, global_index, off[3]) for every staged atom with slot < cap.  One warp per tile
// cell; two cells in flight per warp for memory-level parallelism.  Caller syncs afterwards.
template <class Store>
__device__ __forceinline__ void tile_stage(const Geom& g, const TileTables& tt, int cap, Store store) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int t = wid; t < tt.ntc; t += nw) {
    int c = tt.cnt[t];
    if (c == 0) continue;
    double off[3];
    tile_cell_offset(g, tt, t, off);
    int s0 = tt.start[t], g0 = tt.gstart[t];
    for (int k = lane; k < c; k += 32)
      if (s0 + k < cap) store(s0 + k, g0 + k, off);
  }
}

// ---------------------------------------------------------------------------------------------------
// a1: wrap + bin (north_star (1))
// ---------------------------------------------------------------------------------------------------
__global__ void k_bin(Geom g, int N, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,
                      int* __restrict__ cell_of, int* __restrict__ rank, int* __restrict__ cell_count, Flags* flags) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  double p[3] = {x[k], y[k], z[k]};
  int c[3];
  bool bad = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (!isfinite(p[d])) { bad = true; p[d] = 0.0; }
    double w = p[d] - g.L[d] * floor(p[d] / g.L[d]);
    if (w >= g.L[d]) w -= g.L[d];
    if (w < 0.0) w = 0.0;
    p[d] = w;
    int ci = (int)(w * g.inv_edge[d]);
    c[d] = ci >= g.nc[d] ? g.nc[d] - 1 : ci;
  }
  if (bad) atomicExch(&flags->nonfinite, 1);
  x[k] = p[0]; y[k] = p[1]; z[k] = p[2];
  int oid = cell_order_id(g, c[0], c[1], c[2]);
  cell_of[k] = oid;
  rank[k] = atomicAdd(&cell_count[oid], 1);
}

// a2: exclusive scan of the cell counts, one block (ncell is at most a few 1e5).
__global__ void k_scan_cells(int ncell, const int* __restrict__ cell_count, int* __restrict__ cell_start) {
  __shared__ int wsum[32];
  __shared__ int carry_s;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
  if (tid == 0) carry_s = 0;
  __syncthreads();
  for (int base = 0; base < ncell; base += blockDim.x) {
    int i = base + tid;
    int v = i < ncell ? cell_count[i] : 0;
    int incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int u = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += u;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      int s = lane < nw ? wsum[lane] : 0, si = s;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        int u = __shfl_up_sync(0xffffffffu, si, o);
        if (lane >= o) si += u;
      }
      wsum[lane] = si - s;   // exclusive
    }
    __syncthreads();
    int carry = carry_s;
    if (i < ncell) cell_start[i] = carry + wsum[wid] + incl - v;
    __syncthreads();
    if (tid == blockDim.x - 1) carry_s = carry + wsum[wid] + incl;
    __syncthreads();
  }
  if (tid == 0) cell_start[ncell] = carry_s;
}

__global__ void k_fill_perm(int N, const int* __restrict__ cell_of, const int* __restrict__ rank,
                            const int* __restrict__ cell_start, int* __restrict__ perm) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < N) perm[cell_start[cell_of[k]] + rank[k]] = k;
}

// The atomic ranks of k_bin are not reproducible; sorting each cell's slice of perm by previous index
// makes the whole order (and so every later summation order) deterministic.
__global__ void k_sort_cells(int ncell, const int* __restrict__ cell_start, int* __restrict__ perm) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= ncell) return;
  int lo = cell_start[c], hi = cell_start[c + 1];
  for (int a = lo + 1; a < hi; ++a) {
    int key = perm[a], b = a - 1;
    while (b >= lo && perm[b] > key) { perm[b + 1] = perm[b]; --b; }
    perm[b + 1] = key;
  }
}

// a2: spatial reorder of the per-atom arrays; x0 := x (reference for the displacement test)
__global__ void k_permute(int N, const int* __restrict__ perm, const double* __restrict__ xi, const double* __restrict__ vi,
                          const int* __restrict__ idi, const int* __restrict__ typei, double* __restrict__ xo,
                          double* __restrict__ vo, int* __restrict__ ido, int* __restrict__ typeo, double* __restrict__ x0,
                          size_t ld) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  int k = perm[n];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double p = xi[d * ld + k];
    xo[d * ld + n] = p;
    x0[d * ld + n] = p;
    vo[d * ld + n] = vi[d * ld + k];
  }
  ido[n] = idi[k];
  typeo[n] = typei[k];
}

// caller order <-> sorted order
__global__ void k_scatter_in(int N, const int* __restrict__ id, const double* __restrict__ in, double* __restrict__ out, size_t ld) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  size_t o = 3 * (size_t)id[n];
  out[n] = in[o]; out[ld + n] = in[o + 1]; out[2 * ld + n] = in[o + 2];
}
__global__ void k_gather_out(int N, const int* __restrict__ id, const double* __restrict__ in, double* __restrict__ out, size_t ld) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  size_t o = 3 * (size_t)id[n];
  out[o] = in[n]; out[o + 1] = in[ld + n]; out[o + 2] = in[2 * ld + n];
}
__global__ void k_iota(int N, int* __restrict__ a) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < N) a[n] = n;
}
__global__ void k_scatter_types(int N, const int* __restrict__ id, const int* __restrict__ in, int* __restrict__ out) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < N) out[n] = in[id[n]];
}

// ---------------------------------------------------------------------------------------------------
// a3: Verlet list build from the 27-cell stencil of the staged tile (north_star (2)); fp64 test.
// Shared memory: TileTables | sx[cap+1] sy[cap+1] sz[cap+1] doubles.
// List layout: 16-bit tile-local slots, 8 per uint4; entry e of interior atom a sits in word
//   q = e/8, lane s = q % K, chunk c = q / K  at  list[tile_base + c*slots_cap + a*K + s].
// Unused entries of the last word hold the dummy slot n_staged (a far-away point).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(BLOCK) k_build_list(Geom g, const int* __restrict__ cell_start, const double* __restrict__ x,
                                                      size_t ld, double rl2, uint4* __restrict__ list, int* __restrict__ numneigh,
                                                      Flags* flags) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  double* sx = reinterpret_cast<double*>(smem_raw + sizeof(TileTables));
  double* sy = sx + (g.tile_cap + 1);
  double* sz = sy + (g.tile_cap + 1);
  const int tile = blockIdx.x;
  tile_setup(g, tile, cell_start, tt);
  if (threadIdx.x == 0) {
    if (tt.n_staged > g.tile_cap) atomicMax(&flags->need_tile_cap, tt.n_staged);
    if (tt.n_int > g.interior_cap) atomicMax(&flags->need_interior_cap, tt.n_int);
    atomicMax(&flags->max_tile_atoms, tt.n_staged);
  }
  if (tt.n_staged > g.tile_cap || tt.n_int > g.interior_cap) return;   // host re-plans and rebuilds
  tile_stage(g, tt, g.tile_cap, [&](int slot, int gi, const double* off) {
    sx[slot] = x[gi] + off[0];
    sy[slot] = x[ld + gi] + off[1];
    sz[slot] = x[2 * ld + gi] + off[2];
  });
  __syncthreads();
  const int K = g.K;
  const size_t slots_cap = (size_t)g.interior_cap * K;
  uint4* tlist = list + (size_t)tile * g.chunk_cap * slots_cap;
  const unsigned dummy = (unsigned)tt.n_staged;
  int my_max = 0;
  unsigned long long my_sum = 0;
  // one thread per interior atom, walking the interior cells in staging order
  for (int a = threadIdx.x; a < tt.n_int; a += blockDim.x) {
    // which interior cell holds slot a?  interior cells are consecutive in order id; find by scanning
    // the tile-cell table (interior cells only); tiles hold at most a few hundred cells.
    int tx = 1, ty = 1, tz = 1;
    {
      int lo = 0, hi = tt.w[0] * tt.w[1] * tt.w[2] - 1;   // binary search over interior cells in order
      while (lo < hi) {
        int mid = (lo + hi + 1) >> 1;
        int mx = mid % tt.w[0], my = (mid / tt.w[0]) % tt.w[1], mz = mid / (tt.w[0] * tt.w[1]);
        int t = ((mz + 1) * tt.tc[1] + (my + 1)) * tt.tc[0] + (mx + 1);
        if (tt.start[t] <= a) lo = mid; else hi = mid - 1;
      }
      tx = lo % tt.w[0] + 1; ty = (lo / tt.w[0]) % tt.w[1] + 1; tz = lo / (tt.w[0] * tt.w[1]) + 1;
    }
    const double xi = sx[a], yi = sy[a], zi = sz[a];
    const int gi = tt.brick_start + a;
    unsigned long long lo64 = 0, hi64 = 0;
    int n = 0;
    auto flush = [&](int nn) {   // word q = (nn-1)/8 is complete (or final)
      int q = (nn - 1) >> 3;
      int s = q % K, c = q / K;
      uint4 w;
      w.x = (unsigned)lo64; w.y = (unsigned)(lo64 >> 32); w.z = (unsigned)hi64; w.w = (unsigned)(hi64 >> 32);
      tlist[(size_t)c * slots_cap + (size_t)a * K + s] = w;
    };
    for (int dz = -1; dz <= 1; ++dz)
      for (int dy = -1; dy <= 1; ++dy)
        for (int dx = -1; dx <= 1; ++dx) {
          int t = ((tz + dz) * tt.tc[1] + (ty + dy)) * tt.tc[0] + (tx + dx);
          int s0 = tt.start[t], c = tt.cnt[t], g0 = tt.gstart[t];
          for (int k = 0; k < c; ++k) {
            int j = s0 + k;
            double ddx = xi - sx[j], ddy = yi - sy[j], ddz = zi - sz[j];
            double r2 = ddx * ddx + ddy * ddy + ddz * ddz;
            bool take = r2 < rl2 && j != a;
            if (g.half) take = take && (g0 + k > gi);
            if (take) {
              if (n < g.row_cap) {
                int pos = n & 7;
                if (pos < 4) lo64 |= (unsigned long long)j << (16 * pos);
                else hi64 |= (unsigned long long)j << (16 * (pos - 4));
                if (pos == 7) { flush(n + 1); lo64 = 0; hi64 = 0; }
              }
              ++n;
            }
          }
        }
    int stored = n < g.row_cap ? n : g.row_cap;
    if (stored & 7) {   // pad the last word with the dummy slot
      for (int pos = stored & 7; pos < 8; ++pos) {
        if (pos < 4) lo64 |= (unsigned long long)dummy << (16 * pos);
        else hi64 |= (unsigned long long)dummy << (16 * (pos - 4));
      }
      flush(stored);
    }
    numneigh[gi] = stored;
    my_max = max(my_max, n);
    my_sum += (unsigned long long)stored;
  }
  // statistics
  for (int o = 16; o > 0; o >>= 1) {
    my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, o));
    my_sum += __shfl_xor_sync(0xffffffffu, my_sum, o);
  }
  if ((threadIdx.x & 31) == 0) {
    atomicMax(&flags->max_row, my_max);
    if (my_max > g.row_cap) atomicMax(&flags->need_row_cap, my_max);
    atomicAdd(&flags->sum_rows, my_sum);
  }
}

// list export in caller ids (pair-set parity).  Shared memory: TileTables | sid[cap+1] ints.
__global__ void __launch_bounds__(BLOCK) k_export_list(Geom g, const int* __restrict__ cell_start, const int* __restrict__ id,
                                                       const uint4* __restrict__ list, const int* __restrict__ numneigh,
                                                       int* __restrict__ nn_out, int* __restrict__ neigh_out, long long stride) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  int* sid = reinterpret_cast<int*>(smem_raw + sizeof(TileTables));
  const int tile = blockIdx.x;
  tile_setup(g, tile, cell_start, tt);
  tile_stage(g, tt, g.tile_cap, [&](int slot, int gi, const double*) { sid[slot] = id[gi]; });
  __syncthreads();
  const int K = g.K;
  const size_t slots_cap = (size_t)g.interior_cap * K;
  const uint4* tlist = list + (size_t)tile * g.chunk_cap * slots_cap;
  for (int a = threadIdx.x; a < tt.n_int; a += blockDim.x) {
    int gi = tt.brick_start + a, n = numneigh[gi], io = id[gi];
    nn_out[io] = n;
    for (int e = 0; e < n && e < stride; ++e) {
      int q = e >> 3, s = q % K, c = q / K;
      uint4 w = tlist[(size_t)c * slots_cap + (size_t)a * K + s];
      unsigned word = (&w.x)[(e & 7) >> 1];
      unsigned j = (e & 1) ? (word >> 16) : (word & 0xffffu);
      neigh_out[(long long)io * stride + e] = sid[j];
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// pair styles.  T = double (MD_FP64) or float (MD_MIXED pair math).
// A Body accumulates per-word partial sums in T and per-atom totals in double.
// ---------------------------------------------------------------------------------------------------
template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

struct PairParams {    // host-prepared constants, in double; kernels convert once
  double rc2;
  double lj1, lj2, lj3, lj4;             // 48 eps s^12, 24 eps s^6, 4 eps s^12, 4 eps s^6
  double A, p_r0, B, q_r0, inv_r0, p, q; // EAM: A, p/r0, B, q/r0, 1/r0, p, q
};

template <typename T> __device__ __forceinline__ T t_rcp(T x);
template <> __device__ __forceinline__ float t_rcp<float>(float x) { return rcp_approx(x); }
template <> __device__ __forceinline__ double t_rcp<double>(double x) { return 1.0 / x; }
template <typename T> __device__ __forceinline__ T t_rsqrt(T x);
template <> __device__ __forceinline__ float t_rsqrt<float>(float x) { return rsqrt_approx(x); }
template <> __device__ __forceinline__ double t_rsqrt<double>(double x) { return 1.0 / sqrt(x); }
// exp(-a) for a >= 0-ish arguments
template <typename T> __device__ __forceinline__ T t_exp(T x);
template <> __device__ __forceinline__ float t_exp<float>(float x) { return ex2_approx(x * 1.4426950408889634f); }
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }

// LJ 12-6 force (+ energy, virial when EV).  PAPER.md L102 calcPairForce, App. A L256.
template <typename T, bool EV>
struct LJBody {
  static constexpr int NT = EV ? 10 : 3;   // fx fy fz [e wxx wyy wzz wxy wxz wyz]
  T rc2, lj1, lj2, lj3, lj4;
  __device__ explicit LJBody(const PairParams& P) : rc2((T)P.rc2), lj1((T)P.lj1), lj2((T)P.lj2), lj3((T)P.lj3), lj4((T)P.lj4) {}
  __device__ __forceinline__ void pair(T dx, T dy, T dz, T r2, T, T, T (&p)[NT]) const {
    if (r2 < rc2) {
      T r2i = t_rcp<T>(r2);
      T r6 = r2i * r2i * r2i;
      T fp = r6 * (lj1 * r6 - lj2) * r2i;
      p[0] += fp * dx; p[1] += fp * dy; p[2] += fp * dz;
      if constexpr (EV) {
        p[3] += r6 * (lj3 * r6 - lj4);
        p[4] += dx * dx * fp; p[5] += dy * dy * fp; p[6] += dz * dz * fp;
        p[7] += dx * dy * fp; p[8] += dx * dz * fp; p[9] += dy * dz * fp;
      }
    }
  }
};

// EAM pass 1: rho_i = sum_j exp(-q (r/r0 - 1))            (a6)
template <typename T>
struct EamDensityBody {
  static constexpr int NT = 1;
  T rc2, q_r0, q;
  __device__ explicit EamDensityBody(const PairParams& P) : rc2((T)P.rc2), q_r0((T)P.q_r0), q((T)P.q) {}
  __device__ __forceinline__ void pair(T, T, T, T r2, T, T, T (&p)[NT]) const {
    if (r2 < rc2) {
      T r = r2 * t_rsqrt<T>(r2);
      p[0] += t_exp<T>(q - q_r0 * r);
    }
  }
};

// EAM pass 2: F_i = -sum_j [ (F'_i + F'_j) rho'(r) + phi'(r) ] D / r      (a7); w carries F'.
template <typename T, bool EV>
struct EamForceBody {
  static constexpr int NT = EV ? 10 : 3;
  T rc2, q_r0, q, p_r0, pp, A;
  __device__ explicit EamForceBody(const PairParams& P)
      : rc2((T)P.rc2), q_r0((T)P.q_r0), q((T)P.q), p_r0((T)P.p_r0), pp((T)P.p), A((T)P.A) {}
  __device__ __forceinline__ void pair(T dx, T dy, T dz, T r2, T wi, T wj, T (&p)[NT]) const {
    if (r2 < rc2) {
      T rinv = t_rsqrt<T>(r2);
      T r = r2 * rinv;
      T rho = t_exp<T>(q - q_r0 * r);
      T phi = A * t_exp<T>(pp - p_r0 * r);
      // rho' = -(q/r0) rho, phi' = -(p/r0) phi  =>  fpair = [ (F'_i+F'_j)(q/r0) rho + (p/r0) phi ] / r
      T fp = ((wi + wj) * q_r0 * rho + p_r0 * phi) * rinv;
      p[0] += fp * dx; p[1] += fp * dy; p[2] += fp * dz;
      if constexpr (EV) {
        p[3] += phi;
        p[4] += dx * dx * fp; p[5] += dy * dy * fp; p[6] += dz * dz * fp;
        p[7] += dx * dy * fp; p[8] += dx * dz * fp; p[9] += dy * dz * fp;
      }
    }
  }
};

// ---------------------------------------------------------------------------------------------------
// the neighbor-list loop of PAPER.md L88-122 for one (atom, lane): walks this lane's 128-bit words,
// 8 entries each, gathers from the shared-memory tile, accumulates word partials in T and totals in
// double.  `tile` holds n_staged+1 vec4 entries (x,y,z,w).
// ---------------------------------------------------------------------------------------------------
template <typename T, class Body>
__device__ __forceinline__ void list_loop(const Body& body, const typename Vec4<T>::type* __restrict__ tile,
                                          const uint4* __restrict__ words, size_t word_stride, int nwords,
                                          typename Vec4<T>::type pi, double (&tot)[Body::NT]) {
  constexpr int NT = Body::NT;
  if (nwords <= 0) return;
  uint4 w = ld_stream(words);
  for (int c = 0; c < nwords; ++c) {
    uint4 cur = w;
    if (c + 1 < nwords) w = ld_stream(words + (size_t)(c + 1) * word_stride);
    T p[NT];
#pragma unroll
    for (int k = 0; k < NT; ++k) p[k] = (T)0;
    const unsigned ww[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
    for (int h = 0; h < 4; ++h) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        unsigned j = u ? (ww[h] >> 16) : (ww[h] & 0xffffu);
        typename Vec4<T>::type pj = tile[j];
        T dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
        T r2 = dx * dx + dy * dy + dz * dz;
        body.pair(dx, dy, dz, r2, pi.w, pj.w, p);
      }
    }
#pragma unroll
    for (int k = 0; k < NT; ++k) tot[k] += (double)p[k];
  }
}

// the direct cell-list loop (reading s10): no list; atom a tests every staged atom of
// the 27 tile cells around its own cell.
template <typename T, class Body>
__device__ __forceinline__ void cell_loop(const Body& body, const typename Vec4<T>::type* __restrict__ tile, const TileTables& tt,
                                          int a, int tx, int ty, int tz, typename Vec4<T>::type pi, double (&tot)[Body::NT]) {
  constexpr int NT = Body::NT;
  for (int dz = -1; dz <= 1; ++dz)
    for (int dy = -1; dy <= 1; ++dy)
      for (int dx = -1; dx <= 1; ++dx) {
        int t = ((tz + dz) * tt.tc[1] + (ty + dy)) * tt.tc[0] + (tx + dx);
        int s0 = tt.start[t], c = tt.cnt[t];
        T p[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) p[k] = (T)0;
        for (int k = 0; k < c; ++k) {
          int j = s0 + k;
          if (j == a) continue;
          typename Vec4<T>::type pj = tile[j];
          T ex = pi.x - pj.x, ey = pi.y - pj.y, ez = pi.z - pj.z;
          T r2 = ex * ex + ey * ey + ez * ez;
          body.pair(ex, ey, ez, r2, pi.w, pj.w, p);
        }
#pragma unroll
        for (int k = 0; k < NT; ++k) tot[k] += (double)p[k];
      }
}

__device__ __forceinline__ void interior_cell_of(const TileTables& tt, int a, int& tx, int& ty, int& tz) {
  int lo = 0, hi = tt.w[0] * tt.w[1] * tt.w[2] - 1;
  while (lo < hi) {
    int mid = (lo + hi + 1) >> 1;
    int mx = mid % tt.w[0], my = (mid / tt.w[0]) % tt.w[1], mz = mid / (tt.w[0] * tt.w[1]);
    int t = ((mz + 1) * tt.tc[1] + (my + 1)) * tt.tc[0] + (mx + 1);
    if (tt.start[t] <= a) lo = mid; else hi = mid - 1;
  }
  tx = lo % tt.w[0] + 1; ty = (lo / tt.w[0]) % tt.w[1] + 1; tz = lo / (tt.w[0] * tt.w[1]) + 1;
}

// ---------------------------------------------------------------------------------------------------
// a5/a6/a7: the tile force kernel.
//   MODE 0: forces (LJ or EAM pass 2) -> f[3][N] (+ per-block energy/virial partials when EV)
//   MODE 1: EAM pass 1 -> rho[N], fp[N] = F'(rho) (+ per-block embedding energy partial)
//   HALF (MODE 0 only, K = 1): each pair once, -F scattered to f[j] with fp64 atomics (f zeroed before).
//   CELL: no list, direct cell loop.
// Shared memory: TileTables | vec4<T> tile[cap+1] | (HALF: int sgid[cap+1])
// w component of the staged atoms: F'(rho_j) for EAM pass 2, else 0.
// ---------------------------------------------------------------------------------------------------
struct ForceArgs {
  Geom g;
  PairParams P;
  const int* cell_start;
  const double* x; size_t ld;
  const uint4* list;
  const int* numneigh;
  const double* fp_in;     // EAM pass 2: F'(rho) per sorted atom (else NULL)
  double* f;               // MODE 0 out
  double* rho; double* fp_out;   // MODE 1 out
  double* ev_partials;     // [ntiles][8]: e, wxx, wyy, wzz, wxy, wxz, wyz, pad   (EV or MODE 1)
};

template <typename T, class Body, int K, int MODE, bool EV, bool HALF, bool CELL>
__global__ void __launch_bounds__(BLOCK) k_tile_force(ForceArgs A) {
  using V4 = typename Vec4<T>::type;
  constexpr int NT = Body::NT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  V4* tile = reinterpret_cast<V4*>(smem_raw + sizeof(TileTables));
  int* sgid = reinterpret_cast<int*>(tile + (A.g.tile_cap + 1));   // HALF only
  __shared__ double red[8 * 32];
  const Geom& g = A.g;
  const int tileid = blockIdx.x;
  tile_setup(g, tileid, A.cell_start, tt);
  const double* __restrict__ xs = A.x;
  const size_t ld = A.ld;
  const double* __restrict__ fpin = A.fp_in;
  tile_stage(g, tt, g.tile_cap, [&](int slot, int gi, const double* off) {
    V4 v;
    v.x = (T)(xs[gi] + off[0]);
    v.y = (T)(xs[ld + gi] + off[1]);
    v.z = (T)(xs[2 * ld + gi] + off[2]);
    v.w = fpin ? (T)fpin[gi] : (T)0;
    tile[slot] = v;
    if constexpr (HALF) sgid[slot] = gi;
  });
  if (threadIdx.x == 0) {
    V4 far;
    far.x = (T)1e15; far.y = (T)1e15; far.z = (T)1e15; far.w = (T)0;
    tile[tt.n_staged < g.tile_cap ? tt.n_staged : g.tile_cap] = far;
  }
  __syncthreads();
  const Body body(A.P);
  const size_t slots_cap = (size_t)g.interior_cap * K;
  const uint4* tlist = A.list + (size_t)tileid * g.chunk_cap * slots_cap;
  double ev[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const int nslots = tt.n_int * K;
  for (int base = 0; base < nslots; base += blockDim.x) {   // uniform trip count: shuffles below need full groups
    int sidx = base + threadIdx.x;
    bool active = sidx < nslots;
    int a = active ? sidx / K : 0, s = sidx % K;
    int gi = tt.brick_start + a;
    double tot[NT];
#pragma unroll
    for (int k = 0; k < NT; ++k) tot[k] = 0.0;
    if (active) {
      V4 pi = tile[a];
      if constexpr (CELL) {
        if (s == 0) {
          int tx, ty, tz;
          interior_cell_of(tt, a, tx, ty, tz);
          cell_loop<T, Body>(body, tile, tt, a, tx, ty, tz, pi, tot);
        }
      } else if constexpr (!HALF) {
        int n = A.numneigh[gi];
        int nq = (n + 7) >> 3;                       // words of this atom
        int mine = nq > s ? (nq - s + K - 1) / K : 0; // words q = s, s+K, ...
        list_loop<T, Body>(body, tile, tlist + sidx, slots_cap, mine, pi, tot);
      } else {
        // half list: each in-range pair once; +F to i (registers), -F to j (atomics)
        int n = A.numneigh[gi];
        int nq = (n + 7) >> 3;
        for (int c = 0; c < nq; ++c) {
          uint4 cur = tlist[(size_t)c * slots_cap + sidx];
          const unsigned ww[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
          for (int h = 0; h < 4; ++h)
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              unsigned j = u ? (ww[h] >> 16) : (ww[h] & 0xffffu);
              V4 pj = tile[j];
              T dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
              T r2 = dx * dx + dy * dy + dz * dz;
              T p[NT];
#pragma unroll
              for (int k = 0; k < NT; ++k) p[k] = (T)0;
              body.pair(dx, dy, dz, r2, pi.w, pj.w, p);
              if (p[0] != (T)0 || p[1] != (T)0 || p[2] != (T)0) {
                int gj = sgid[j];
                atomicAdd(&A.f[gj], -(double)p[0]);
                atomicAdd(&A.f[ld + gj], -(double)p[1]);
                atomicAdd(&A.f[2 * ld + gj], -(double)p[2]);
              }
#pragma unroll
              for (int k = 0; k < NT; ++k) tot[k] += (double)p[k];
            }
        }
      }
    }
    if constexpr (K > 1) {
#pragma unroll
      for (int k = 0; k < NT; ++k) tot[k] = group_sum<K>(tot[k]);
    }
    if (active && s == 0) {
      if constexpr (MODE == 0) {
        if constexpr (HALF) {
          atomicAdd(&A.f[gi], tot[0]); atomicAdd(&A.f[ld + gi], tot[1]); atomicAdd(&A.f[2 * ld + gi], tot[2]);
        } else {
          A.f[gi] = tot[0]; A.f[ld + gi] = tot[1]; A.f[2 * ld + gi] = tot[2];
        }
        if constexpr (EV) {
          const double wgt = HALF ? 1.0 : 0.5;   // a full list visits every pair twice
#pragma unroll
          for (int k = 0; k < 7; ++k) ev[k] += wgt * tot[3 + k];
        }
      } else {
        double rho = tot[0];
        double sq = sqrt(rho);
        A.rho[gi] = rho;
        A.fp_out[gi] = rho > 0.0 ? -A.P.B / (2.0 * sq) : 0.0;   // F'(0) := 0 (reading s13)
        ev[0] += -A.P.B * sq;                                    // embedding energy F(rho_i)
      }
    }
  }
  if constexpr (EV || MODE == 1) {
    block_sum<8>(ev, red);
    if (threadIdx.x == 0)
#pragma unroll
      for (int k = 0; k < 8; ++k) A.ev_partials[(size_t)tileid * 8 + k] = ev[k];
  }
}

// deterministic final reduction of the per-tile partials: out[k] (+)= sum_tiles partials[tile][k]
__global__ void k_reduce_ev(int ntiles, const double* __restrict__ partials, double* __restrict__ out, int accumulate) {
  __shared__ double red[8 * 32];
  double v[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  for (int t = threadIdx.x; t < ntiles; t += blockDim.x)
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] += partials[(size_t)t * 8 + k];
  block_sum<8>(v, red);
  if (threadIdx.x == 0)
#pragma unroll
    for (int k = 0; k < 8; ++k) out[k] = (accumulate ? out[k] : 0.0) + v[k];
}

// ---------------------------------------------------------------------------------------------------
// a8 + a4: velocity Verlet and the device-side displacement test
// ---------------------------------------------------------------------------------------------------
// v += dtf f ; x += dt v ; flag = max |x - x0|^2
__global__ void k_initial_integrate(int N, size_t ld, double* __restrict__ x, double* __restrict__ v, const double* __restrict__ f,
                                    const double* __restrict__ x0, const int* __restrict__ type, const double* __restrict__ mass,
                                    double dt, double half_dt_ftm2v, Flags* flags) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  double d2 = 0.0;
  if (n < N) {
    double dtf = half_dt_ftm2v / mass[type[n]];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double vv = v[d * ld + n] + dtf * f[d * ld + n];
      double xx = x[d * ld + n] + dt * vv;
      v[d * ld + n] = vv;
      x[d * ld + n] = xx;
      double dd = xx - x0[d * ld + n];
      d2 += dd * dd;
    }
  }
  for (int o = 16; o > 0; o >>= 1) d2 = fmax(d2, __shfl_xor_sync(0xffffffffu, d2, o));
  __shared__ double wmax[32];
  int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0) wmax[wid] = d2;
  __syncthreads();
  if (wid == 0) {
    d2 = lane < (blockDim.x >> 5) ? wmax[lane] : 0.0;
    for (int o = 16; o > 0; o >>= 1) d2 = fmax(d2, __shfl_xor_sync(0xffffffffu, d2, o));
    if (lane == 0 && d2 > 0.0) atomicMax(&flags->max_disp2_bits, (unsigned long long)__double_as_longlong(d2));
  }
}

__global__ void k_final_integrate(int N, size_t ld, double* __restrict__ v, const double* __restrict__ f,
                                  const int* __restrict__ type, const double* __restrict__ mass, double half_dt_ftm2v) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  double dtf = half_dt_ftm2v / mass[type[n]];
#pragma unroll
  for (int d = 0; d < 3; ++d) v[d * ld + n] += dtf * f[d * ld + n];
}

__global__ void k_kinetic(int N, size_t ld, const double* __restrict__ v, const int* __restrict__ type,
                          const double* __restrict__ mass, double* __restrict__ out) {
  __shared__ double red[32];
  double ke[1] = {0.0};
  for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < N; n += gridDim.x * blockDim.x) {
    double m = mass[type[n]];
    ke[0] += 0.5 * m * (v[n] * v[n] + v[ld + n] * v[ld + n] + v[2 * ld + n] * v[2 * ld + n]);
  }
  block_sum<1>(ke, red);
  if (threadIdx.x == 0) atomicAdd(out, ke[0]);
}

}  // namespace mdk
