// md_kernels.cuh -- device code of the B200-native MD hot path (sm_100a).
//
// Design in one paragraph (details in DESIGN.md).  Atoms are counting-sorted into cells of edge
// >= rc+skin, the cells themselves ordered TILE-major: a tile is a box of bx x by x bz cells whose atoms
// are contiguous in memory.  Every heavy kernel is one thread block per tile: it stages the tile's cells
// plus a one-cell halo (periodic images resolved while staging) into shared memory as TILE-CENTRED
// coordinates -- fp32 in mixed mode, which is what makes fp32 pair math accurate enough in a 168-sigma
// box -- and then runs the paper's neighbor-list loop against shared memory: the
// "random access" load of atom j (L100) is one 128-bit shared-memory load, not a texture/L1 gather, and
// the list holds 16-bit tile-local slot codes, eight to a 128-bit word, so the index stream is half the
// classic 4 B/entry.  One template covers thread-per-atom (K=1), sub-warp (K=4, 8) and warp-per-atom
// (K=32, the paper's BpA with a shuffle reduction instead of a block reduction).  The force kernel's
// epilogue also does the velocity-Verlet kick and drift, so a time step between rebuilds is ONE launch.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace mdk {

constexpr int MAX_TILE_CELLS = 216;    // (bx+2)(by+2)(bz+2) <= 216, each of bx, by, bz <= 4
constexpr int BUILD_THREADS = 256;     // threads per block of the list-build (when three blocks fit an SM) and cell-list kernels
constexpr int BUILD_MAX_THREADS = 384; // list build: block size when only two blocks fit an SM
constexpr int FORCE_MAX_THREADS = 1024;     // upper bound of the force kernels' block size (runtime choice): the mixed-precision
                                            // kernels are compiled for <= 56 registers (three 384-thread blocks per SM)
constexpr int FORCE_MAX_THREADS_WIDE = 640; // the same for the fp64 and the energy/virial instantiations (<= 96 registers)
#ifndef MDK_BUILD_MIN_BLOCKS
#define MDK_BUILD_MIN_BLOCKS 2
#endif
constexpr int BUILD_MIN_BLOCKS = MDK_BUILD_MIN_BLOCKS;    // with BUILD_MAX_THREADS: <= 85 registers, i.e. three 256-thread or two 384-thread blocks per SM
constexpr int RING = 48;               // list-build: pending entries a lane can hold in shared memory (>= 32 + 8)
constexpr int RING_STRIDE = RING * 2 + 16;   // bytes between the rings of neighbouring lanes (odd * 16)

struct Geom {
  double L[3];        // box
  double edge[3];     // cell edge = L / nc  (>= rc + skin)
  double inv_edge[3];
  double h[3];        // anchor spacing of the packed coordinates: edge rounded to so few bits that every
                      // (half-)integer multiple a tile needs is exact in fp32 (see tile_cell_offset_rel)
  int nc[3];          // cells per dimension (>= 3)
  int b[3];           // tile width in cells (interior)
  int nb[3];          // tiles per dimension
  int ncell;
  int ntiles;
  int tile_cap;       // staged slots a tile can hold (cells padded to multiples of 4; excluding the dummy slot)
  int interior_cap;   // interior slots (= list rows) a tile can hold (multiple of 32)
  int row_cap;        // list entries per atom (multiple of 8*K)
  int K;              // lanes per atom: 1, 8, 32
  int chunk_cap;      // row_cap / (8*K): 128-bit words per lane
  int half;           // 1: half list
  int code_shift;     // list entries hold slot << code_shift (3: fp32 tile, 4: fp64 tile)
};

// flags written by the device, read by the host after a build / after a batch of steps
struct Flags {
  unsigned long long max_disp2_bits[2];  // max |x-x0|^2 since the last build (bit pattern of a non-negative
                                         // double); slot p is written by steps of parity p, read by parity 1-p
  int stop;                           // a step kernel found the list stale and did nothing (sticky until the next build)
  int steps_done;                     // step kernels that ran since the host last cleared it
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
__device__ __forceinline__ void st_stream(uint4* p, uint4 v) {
  asm volatile("st.global.cs.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ float2 lds_f2(unsigned a) {
  float2 r;
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(r.x), "=f"(r.y) : "r"(a));
  return r;
}
__device__ __forceinline__ double2 lds_d2(unsigned a) {
  double2 r;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "r"(a));
  return r;
}
__device__ __forceinline__ uint4 lds_u4(unsigned a) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(a));
  return r;
}
__device__ __forceinline__ void sts_u4(unsigned a, uint4 v) {
  asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void sts_u16(unsigned a, unsigned v) {
  asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((unsigned short)v) : "memory");
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
template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };   // 32 B, 16-B aligned is all that is needed here
template <typename T> __device__ __forceinline__ typename Vec4<T>::type make_v4(T x, T y, T z, T w);
template <> __device__ __forceinline__ float4 make_v4<float>(float x, float y, float z, float w) { return make_float4(x, y, z, w); }
template <> __device__ __forceinline__ double4 make_v4<double>(double x, double y, double z, double w) { return make_double4(x, y, z, w); }

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
__device__ __forceinline__ void atomic_max_double_bits(unsigned long long* p, double v) {
  if (v > 0.0) atomicMax(p, (unsigned long long)__double_as_longlong(v));
}
// block-wide max of a non-negative double, then ONE atomicMax per block.  red: >= 32 doubles of shared scratch.
__device__ __forceinline__ void block_max_to_flag(double v, double* red, unsigned long long* flag) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  __syncthreads();
  if (lane == 0) red[wid] = v;
  __syncthreads();
  if (wid == 0) {
    v = lane < nw ? red[lane] : 0.0;
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if (lane == 0) atomic_max_double_bits(flag, v);
  }
}

// ---------------------------------------------------------------------------------------------------
// tile staging, shared by the list build, every force kernel and the list export.
// Staged slot order: the tile's cells (interior + halo) in tile scan order, x fastest; every cell is padded to a
// multiple of 4 slots (pad slots hold a far-away point), so that a cell's coordinates can be read four at a time
// with aligned 128-bit loads, and the three x-neighbours of a stencil row are ONE contiguous run of slots.
// List rows number the interior atoms only (same cell order, every cell padded to a multiple of 2: a list row
// belongs to a PAIR of atoms): interior slot = rstart[t] + k, pair row = (rstart[t] + k) / 2 for atom k of
// interior tile cell t, whose staged slot is start[t] + k.
// ---------------------------------------------------------------------------------------------------
struct alignas(16) TileTables {   // lives in shared memory
  int start[MAX_TILE_CELLS];  // staged slot of the first atom of tile cell t (multiple of 4)
  int gstart[MAX_TILE_CELLS]; // global (sorted) index of the first atom of tile cell t
  int cnt[MAX_TILE_CELLS];    // atoms in tile cell t
  int meta[MAX_TILE_CELLS];   // tx | ty << 8 | tz << 16 | interior << 24   (filled by tile_load only)
  int rstart[MAX_TILE_CELLS]; // interior cells: interior slot of the cell's first atom (multiple of 2); rows number the
                              // interior atoms only, in the same cell order
  int c0[3], w[3], tc[3];     // first interior cell, interior width, tile width (w+2)
  int ntc;                    // tc[0]*tc[1]*tc[2]
  int nic;                    // interior cells w[0]*w[1]*w[2]
  int n_int_slots;            // padded interior slots (list rows in use)
  int n_slots;                // all padded slots; slot n_slots is the far-away dummy
  int n_int_atoms;            // interior atoms
  int brick_start;            // global index of the first interior atom
};

__device__ __forceinline__ int pad4(int c) { return (c + 3) & ~3; }
__device__ __forceinline__ int pad2(int c) { return (c + 1) & ~1; }
__device__ __forceinline__ int interior_tile_cell(const TileTables& tt, int ic) {
  int lx = ic % tt.w[0], ly = (ic / tt.w[0]) % tt.w[1], lz = ic / (tt.w[0] * tt.w[1]);
  return ((lz + 1) * tt.tc[1] + (ly + 1)) * tt.tc[0] + (lx + 1);
}
__device__ __forceinline__ bool tile_cell_is_interior(const TileTables& tt, int t) {
  int tx = t % tt.tc[0], ty = (t / tt.tc[0]) % tt.tc[1], tz = t / (tt.tc[0] * tt.tc[1]);
  return tx >= 1 && tx <= tt.w[0] && ty >= 1 && ty <= tt.w[1] && tz >= 1 && tz <= tt.w[2];
}

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
    tt.nic = tt.w[0] * tt.w[1] * tt.w[2];
    int first = cell_order_id(g, tt.c0[0], tt.c0[1], tt.c0[2]);
    tt.brick_start = cell_start[first];
    tt.n_int_atoms = cell_start[first + tt.nic] - tt.brick_start;
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
    int s = cell_start[oid];
    tt.gstart[t] = s;
    tt.cnt[t] = cell_start[oid + 1] - s;
  }
  __syncthreads();
  // two exclusive scans of the padded counts by warp 0: all tile cells in scan order (slots), interior cells (rows)
  if (tid < 32) {
    int per = (ntc + 31) / 32, lo = tid * per, hi = min(lo + per, ntc), sum = 0, isum = 0;
    for (int t = lo; t < hi; ++t) {
      const int c4 = pad4(tt.cnt[t]);
      sum += c4;
      if (tile_cell_is_interior(tt, t)) isum += pad2(tt.cnt[t]);
    }
    int incl = sum, iincl = isum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int u = __shfl_up_sync(0xffffffffu, incl, o), v = __shfl_up_sync(0xffffffffu, iincl, o);
      if (tid >= o) { incl += u; iincl += v; }
    }
    int run = incl - sum, irun = iincl - isum;
    for (int t = lo; t < hi; ++t) {
      const int c4 = pad4(tt.cnt[t]);
      tt.start[t] = run;
      run += c4;
      if (tile_cell_is_interior(tt, t)) { tt.rstart[t] = irun; irun += pad2(tt.cnt[t]); } else tt.rstart[t] = 0;
    }
    if (tid == 31) { tt.n_int_slots = iincl; tt.n_slots = incl; }
  }
  __syncthreads();
}

// ---------------------------------------------------------------------------------------------------
// The tables above are computed ONCE per list build by k_tile_tables and kept in global memory
// (TILE_HDR ints of header + four ints {gstart, start<<16 | cnt, meta, rstart} per tile cell); every tile kernel
// launched between two builds only loads them (tile_load: one coalesced read, one barrier).
// ---------------------------------------------------------------------------------------------------
constexpr int TILE_CELL_INTS = 7;   // ints per tile cell in the table: gstart, start<<16|cnt, meta, rstart, and the fp32 offset
                                    // (x, y, z) of the cell's packed coordinates from the tile centre (tile_cell_offset_rel)
constexpr int TILE_HDR = 8;   // n_int_slots, n_slots, n_int_atoms, brick_start, n_staged_atoms, pad x3
__host__ __device__ inline int tile_tab_cells(const Geom& g) { return ((g.b[0] + 2) * (g.b[1] + 2) * (g.b[2] + 2) + 3) & ~3; }
// after the per-cell ints: one u16 per QUAD of staged slots (cells are padded to 4 slots, so a quad belongs to
// one tile cell) = the tile cell of that quad; lets the force kernel post-process the staged tile slot-parallel
__host__ __device__ inline int tile_tab_quads(const Geom& g) { return (g.tile_cap >> 2) + 2; }
__host__ __device__ inline int tile_tab_stride(const Geom& g) {
  return (TILE_HDR + TILE_CELL_INTS * tile_tab_cells(g) + ((tile_tab_quads(g) + 1) >> 1) + 3) & ~3;   // a multiple of 16 bytes: one bulk copy
}

__device__ __forceinline__ void tile_dims(const Geom& g, int tile, int c0[3], int w[3]) {
  int bt[3] = {tile % g.nb[0], (tile / g.nb[0]) % g.nb[1], tile / (g.nb[0] * g.nb[1])};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    c0[d] = bt[d] * g.b[d];
    w[d] = tile_width(g, d, bt[d]);
  }
}

// All threads of the block call it; ends with __syncthreads().
__device__ __forceinline__ void tile_load(const Geom& g, int tile, const int* __restrict__ tab, TileTables& tt) {
  const int* __restrict__ h = tab + (size_t)tile * tile_tab_stride(g);
  int c0[3], w[3];
  tile_dims(g, tile, c0, w);
  const int ntc = (w[0] + 2) * (w[1] + 2) * (w[2] + 2);
  if (threadIdx.x == 0) {
#pragma unroll
    for (int d = 0; d < 3; ++d) { tt.c0[d] = c0[d]; tt.w[d] = w[d]; tt.tc[d] = w[d] + 2; }
    tt.ntc = ntc;
    tt.nic = w[0] * w[1] * w[2];
    tt.n_int_slots = h[0]; tt.n_slots = h[1]; tt.n_int_atoms = h[2]; tt.brick_start = h[3];
  }
  const int tcs = tile_tab_cells(g);
  for (int t = threadIdx.x; t < ntc; t += blockDim.x) {
    const unsigned sc = (unsigned)h[TILE_HDR + tcs + t];
    tt.gstart[t] = h[TILE_HDR + t];
    tt.start[t] = (int)(sc >> 16);
    tt.cnt[t] = (int)(sc & 0xffffu);
    tt.meta[t] = h[TILE_HDR + 2 * tcs + t];
    tt.rstart[t] = h[TILE_HDR + 3 * tcs + t];
  }
  __syncthreads();
}

// one block per tile; also raises the capacity flags the host re-plans on
__global__ void __launch_bounds__(128) k_tile_tables(Geom g, const int* __restrict__ cell_start, int* __restrict__ tab, Flags* flags) {
  __shared__ TileTables tt;
  const int tile = blockIdx.x;
  tile_setup(g, tile, cell_start, tt);
  int* h = tab + (size_t)tile * tile_tab_stride(g);
  const int tcs = tile_tab_cells(g);
  int staged = 0;
  for (int t = threadIdx.x; t < tt.ntc; t += blockDim.x) {
    const int tx = t % tt.tc[0], ty = (t / tt.tc[0]) % tt.tc[1], tz = t / (tt.tc[0] * tt.tc[1]);
    h[TILE_HDR + t] = tt.gstart[t];
    h[TILE_HDR + tcs + t] = (int)(((unsigned)tt.start[t] << 16) | ((unsigned)tt.cnt[t] & 0xffffu));
    h[TILE_HDR + 2 * tcs + t] = tx | ty << 8 | tz << 16 | (tile_cell_is_interior(tt, t) ? 1 << 24 : 0);
    h[TILE_HDR + 3 * tcs + t] = tt.rstart[t];
    {
      const int tq[3] = {tx, ty, tz};
#pragma unroll
      for (int d = 0; d < 3; ++d) {   // the same expression as tile_cell_offset_rel
        const int u = tt.c0[d] + tq[d] - 1;
        const double wrap = u < 0 ? g.nc[d] * g.h[d] - g.L[d] : (u >= g.nc[d] ? g.L[d] - g.nc[d] * g.h[d] : 0.0);
        h[TILE_HDR + (4 + d) * tcs + t] = __float_as_int((float)((2 * (u - tt.c0[d]) + 1 - tt.w[d]) * (0.5 * g.h[d]) + wrap));
      }
    }
    staged += tt.cnt[t];
    unsigned short* qc = reinterpret_cast<unsigned short*>(h + TILE_HDR + TILE_CELL_INTS * tcs);
    const int q0 = tt.start[t] >> 2, q1 = min((tt.start[t] + pad4(tt.cnt[t])) >> 2, tile_tab_quads(g));
    for (int q = q0; q < q1; ++q) qc[q] = (unsigned short)t;
  }
  __shared__ int red[4];
  for (int o = 16; o > 0; o >>= 1) staged += __shfl_xor_sync(0xffffffffu, staged, o);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = staged;
  __syncthreads();
  if (threadIdx.x == 0) {
    h[0] = tt.n_int_slots; h[1] = tt.n_slots; h[2] = tt.n_int_atoms; h[3] = tt.brick_start;
    h[4] = red[0] + red[1] + red[2] + red[3]; h[5] = 0; h[6] = 0; h[7] = 0;
    if (tt.n_slots > g.tile_cap) atomicMax(&flags->need_tile_cap, tt.n_slots);
    if (tt.n_int_slots > g.interior_cap) atomicMax(&flags->need_interior_cap, tt.n_int_slots);
    atomicMax(&flags->max_tile_atoms, tt.n_slots);
  }
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

// The same for the PACKED coordinates xr = x - anchor(c), anchor(c) = (c + 1/2) h of the atom's storage cell c:
// staged = xr + off, off = anchor(unwrapped tile cell u) - (c0 + w/2) h  [+- (nc h - L) for a periodic image].
// h has so few significant bits that (2u + 1 - 2 c0 - w) (h/2) is EXACT in fp32: every atom of a tile is shifted
// by an exactly representable amount, so no rounding error is shared by all pairs of a cell pair (it would
// add up coherently in the virial); only cells seen through the periodic boundary carry one rounded term.
__device__ __forceinline__ void tile_cell_offset_rel(const Geom& g, const TileTables& tt, int t, double off[3]) {
  const int m = tt.meta[t];
  int tq[3] = {m & 0xff, (m >> 8) & 0xff, (m >> 16) & 0xff};
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int u = tt.c0[d] + tq[d] - 1;
    const double wrap = u < 0 ? g.nc[d] * g.h[d] - g.L[d] : (u >= g.nc[d] ? g.L[d] - g.nc[d] * g.h[d] : 0.0);
    off[d] = (2 * (u - tt.c0[d]) + 1 - tt.w[d]) * (0.5 * g.h[d]) + wrap;
  }
}
// cell index of a wrapped coordinate w in [0, L) -- the ONE definition used by binning and by everything
// that must agree with it about which cell an atom is stored in
__device__ __forceinline__ int cell_index_1d(const Geom& g, int d, double w) {
  int ci = (int)(w * g.inv_edge[d]);
  return ci >= g.nc[d] ? g.nc[d] - 1 : ci;
}
__device__ __forceinline__ double cell_anchor_1d(const Geom& g, int d, int ci) { return (ci + 0.5) * g.h[d]; }

// Calls store(slot, global_index, off[3], t) for every staged atom and pad(slot) for every pad slot and
// for the dummy slot, all with slot <= cap.  One warp per tile cell.  Caller syncs afterwards.
template <class Store, class Pad>
__device__ __forceinline__ void tile_stage(const Geom& g, const TileTables& tt, int cap, Store store, Pad pad) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int t = wid; t < tt.ntc; t += nw) {
    const int c = tt.cnt[t], c4 = pad4(c);
    if (c4 == 0) continue;
    double off[3];
    tile_cell_offset(g, tt, t, off);
    const int s0 = tt.start[t], g0 = tt.gstart[t];
    for (int k = lane; k < c4; k += 32) {
      if (s0 + k >= cap) continue;
      if (k < c) store(s0 + k, g0 + k, off, t);
      else pad(s0 + k);
    }
  }
  if (threadIdx.x == 0) pad(tt.n_slots < cap ? tt.n_slots : cap);
}

// ---------------------------------------------------------------------------------------------------
// a1: wrap + bin (north_star (1))
// ---------------------------------------------------------------------------------------------------
// It also packs, above the atom's arrival rank in its cell (bits 0..19), a 9-bit MORTON KEY of the atom's position
// within its cell (3 bits per dimension, bits 20..28): k_sort_cells orders a cell's atoms by it, so that
// consecutive atoms of a cell are spatial neighbours -- the list rows are per PAIR of consecutive atoms (below).
__device__ __forceinline__ int morton3(int a, int b, int c) {   // interleave three 3-bit numbers
  int m = 0;
#pragma unroll
  for (int k = 0; k < 3; ++k) m |= (((a >> k) & 1) << (3 * k)) | (((b >> k) & 1) << (3 * k + 1)) | (((c >> k) & 1) << (3 * k + 2));
  return m;
}
constexpr int RANK_BITS = 20;
__global__ void k_bin(Geom g, int N, double* __restrict__ x, double* __restrict__ y, double* __restrict__ z,
                      int* __restrict__ cell_of, int* __restrict__ rank, int* __restrict__ cell_count, Flags* flags) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  double p[3] = {x[k], y[k], z[k]};
  int c[3], sub[3];
  bool bad = false;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (!isfinite(p[d])) { bad = true; p[d] = 0.0; }
    double w = p[d] - g.L[d] * floor(p[d] / g.L[d]);
    if (w >= g.L[d]) w -= g.L[d];
    if (w < 0.0) w = 0.0;
    p[d] = w;
    c[d] = cell_index_1d(g, d, w);
    const int q = (int)((w * g.inv_edge[d] - (double)c[d]) * 8.0);
    sub[d] = q < 0 ? 0 : (q > 7 ? 7 : q);
  }
  if (bad) atomicExch(&flags->nonfinite, 1);
  else { x[k] = p[0]; y[k] = p[1]; z[k] = p[2]; }   // a non-finite coordinate is reported, not overwritten
  int oid = cell_order_id(g, c[0], c[1], c[2]);
  cell_of[k] = oid;
  rank[k] = atomicAdd(&cell_count[oid], 1) | (morton3(sub[0], sub[1], sub[2]) << RANK_BITS);
}

// a2: exclusive scan of the cell counts in two launches: per-block sums of SCAN_BLOCK cells, then every block
// adds up the sums of the blocks before it (there are few) and scans its own cells.
constexpr int SCAN_PER = 8;
constexpr int SCAN_BLOCK = 1024 * SCAN_PER;
__global__ void __launch_bounds__(1024) k_scan_block_sums(int ncell, const int* __restrict__ cell_count, int* __restrict__ block_sum) {
  __shared__ int wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int i0 = blockIdx.x * SCAN_BLOCK + tid * SCAN_PER;
  int sum = 0;
#pragma unroll
  for (int k = 0; k < SCAN_PER; ++k) sum += i0 + k < ncell ? cell_count[i0 + k] : 0;
  for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
  if (lane == 0) wsum[wid] = sum;
  __syncthreads();
  if (wid == 0) {
    int v = wsum[lane];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) block_sum[blockIdx.x] = v;
  }
}
__global__ void __launch_bounds__(1024) k_scan_cells(int ncell, const int* __restrict__ cell_count, const int* __restrict__ block_sum,
                                                     int* __restrict__ cell_start) {
  __shared__ int wsum[32];
  __shared__ int carry_s;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (wid == 0) {   // sum of the blocks before this one
    int v = 0;
    for (int b = lane; b < (int)blockIdx.x; b += 32) v += block_sum[b];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if (lane == 0) carry_s = v;
  }
  __syncthreads();
  const int i0 = blockIdx.x * SCAN_BLOCK + tid * SCAN_PER;
  int v[SCAN_PER], sum = 0;
#pragma unroll
  for (int k = 0; k < SCAN_PER; ++k) { v[k] = i0 + k < ncell ? cell_count[i0 + k] : 0; sum += v[k]; }
  int incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int u = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += u;
  }
  if (lane == 31) wsum[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    int s = wsum[lane], si = s;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int u = __shfl_up_sync(0xffffffffu, si, o);
      if (lane >= o) si += u;
    }
    wsum[lane] = si - s;   // exclusive
  }
  __syncthreads();
  int run = carry_s + wsum[wid] + incl - sum;
#pragma unroll
  for (int k = 0; k < SCAN_PER; ++k) {
    if (i0 + k < ncell) cell_start[i0 + k] = run;
    run += v[k];
  }
  if (i0 <= ncell - 1 && ncell - 1 < i0 + SCAN_PER) cell_start[ncell] = run;   // the thread that owns the last cell
}

__global__ void k_fill_perm(int N, const int* __restrict__ cell_of, const int* __restrict__ rank,
                            const int* __restrict__ cell_start, int* __restrict__ perm, int* __restrict__ mkey) {
  int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= N) return;
  const int r = rank[k], pos = cell_start[cell_of[k]] + (r & ((1 << RANK_BITS) - 1));
  perm[pos] = k;
  mkey[pos] = r >> RANK_BITS;
}

// The atomic ranks of k_bin are not reproducible; sorting each cell's slice of perm by (Morton key of the
// position within the cell, previous index) makes the whole order (and so every later summation order)
// deterministic AND spatially coherent within the cell.  One warp per cell, rank sort: every lane keeps up to
// SORT_PER of the cell's keys, each key's rank is the number of smaller keys (the keys of a cell are distinct),
// broadcast lane by lane with shuffles: c * ceil(c/32) steps instead of the c^2 of a serial insertion sort
// (a cell holds ~20 atoms at rc = 2.5 sigma, ~150 at rc = 5 sigma).
constexpr int SORT_PER = 16;   // cells of up to 512 atoms; larger ones fall back to a serial sort by lane 0
typedef unsigned long long sortkey_t;
__device__ __forceinline__ sortkey_t sort_key(int mk, int prev) { return ((sortkey_t)(unsigned)mk << 32) | (unsigned)prev; }
template <int PER>
__device__ __forceinline__ void sort_cell_by_warp(int lo, int n, int lane, int* __restrict__ perm, const int* __restrict__ mkey) {
  sortkey_t key[PER];
  int rank[PER];
#pragma unroll
  for (int i = 0; i < PER; ++i) {
    key[i] = lane + 32 * i < n ? sort_key(mkey[lo + lane + 32 * i], perm[lo + lane + 32 * i]) : ~0ull;
    rank[i] = 0;
  }
#pragma unroll
  for (int j = 0; j < PER; ++j) {          // the keys held in register j of every lane
    const int cnt = min(32, n - 32 * j);
    for (int l = 0; l < cnt; ++l) {
      const sortkey_t other = __shfl_sync(0xffffffffu, key[j], l);
#pragma unroll
      for (int i = 0; i < PER; ++i) rank[i] += other < key[i] ? 1 : 0;
    }
  }
  __syncwarp();
#pragma unroll
  for (int i = 0; i < PER; ++i)
    if (lane + 32 * i < n) perm[lo + rank[i]] = (int)(unsigned)key[i];
}
__global__ void __launch_bounds__(256) k_sort_cells(int ncell, const int* __restrict__ cell_start, int* __restrict__ perm,
                                                    int* __restrict__ mkey) {
  const int lane = threadIdx.x & 31;
  const int nwarps = gridDim.x * (blockDim.x >> 5);
  for (int c = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); c < ncell; c += nwarps) {   // a warp per cell, grid-stride
    const int lo = cell_start[c], n = cell_start[c + 1] - lo;
    if (n <= 1) continue;
    if (n <= 32) sort_cell_by_warp<1>(lo, n, lane, perm, mkey);
    else if (n <= 64) sort_cell_by_warp<2>(lo, n, lane, perm, mkey);
    else if (n <= 128) sort_cell_by_warp<4>(lo, n, lane, perm, mkey);
    else if (n <= 256) sort_cell_by_warp<8>(lo, n, lane, perm, mkey);
    else if (n <= 32 * SORT_PER) sort_cell_by_warp<SORT_PER>(lo, n, lane, perm, mkey);
    else if (lane == 0)
      for (int a = lo + 1; a < lo + n; ++a) {
        const int kp = perm[a], km = mkey[a];
        const sortkey_t key = sort_key(km, kp);
        int b = a - 1;
        while (b >= lo && sort_key(mkey[b], perm[b]) > key) { perm[b + 1] = perm[b]; mkey[b + 1] = mkey[b]; --b; }
        perm[b + 1] = kp; mkey[b + 1] = km;
      }
    __syncwarp();
  }
}

// a2: spatial reorder of the per-atom arrays; x0 := x (reference for the displacement test)
// It also writes the PACKED copy the force kernels stage from: xr[n] = (x - centre of its cell, 0) in T
// (fp32 in mixed mode), 16 or 32 B per atom, so that a tile cell is one contiguous bulk copy.
template <typename T>
__global__ void k_permute(Geom g, int N, const int* __restrict__ perm, const double* __restrict__ xi, const double* __restrict__ vi,
                          const int* __restrict__ idi, const int* __restrict__ typei, double* __restrict__ xo,
                          double* __restrict__ vo, int* __restrict__ ido, int* __restrict__ typeo, double* __restrict__ x0,
                          typename Vec4<T>::type* __restrict__ xr, size_t ld) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  int k = perm[n];
  T r[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double p = xi[d * ld + k];
    xo[d * ld + n] = p;
    x0[d * ld + n] = p;
    vo[d * ld + n] = vi[d * ld + k];
    r[d] = (T)(p - cell_anchor_1d(g, d, cell_index_1d(g, d, p)));
  }
  const int ty = typei[k];
  xr[n] = make_v4<T>(r[0], r[1], r[2], (T)ty);   // w: the atom's type (read by the multi-type pair styles; EAM overwrites it with -F')
  ido[n] = idi[k];
  typeo[n] = ty;
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
__global__ void k_check_types(int N, const int* __restrict__ type, int ntypes, int* __restrict__ bad) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < N && (type[n] < 0 || type[n] >= ntypes)) atomicExch(bad, 1);
}
__global__ void k_iota(int N, int* __restrict__ a) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n < N) a[n] = n;
}

// ---------------------------------------------------------------------------------------------------
// a3: Verlet list build from the 27-cell stencil of the staged tile (north_star (2)).
//
// PAIR ROWS.  A list row belongs to a PAIR of consecutive atoms of a cell (staged slots 2m, 2m+1; k_sort_cells
// orders a cell's atoms along a Morton curve, so the two are ~1.4 sigma apart in the LJ liquid) and holds the
// UNION of their neighbors: every staged atom j with |x_j - x_a|^2 < rl^2 for a = either atom of the pair,
// except the two atoms themselves (their mutual term is added by the force kernels directly).  The force
// kernel gathers each listed j ONCE and evaluates it against both atoms (packed f32x2 math), which cuts the
// gathers, the index stream and the list-loop instructions per atom to ~0.69 (measured union size: 1.38 rows).
//
// SUPERSET SEMANTICS.  The distance test runs in fp32 on tile-centred coordinates and accepts r2 < rl2_hi,
// rl2_hi = rl^2 (1 + band) with band four times the worst-case fp32 rounding of r2 (host: build_list_only), so a
// row never misses a pair the fp64 definition contains; it may hold a few pairs beyond rl (in the band, or
// within rl of the partner only), which the force kernels' r2 < rc2 test makes harmless.  The EXACT fp64 pair
// set of an atom (north_star (2)) is the row's entries that pass |x_i - x_j|^2 < rl^2 in fp64 from the global
// positions: md_get_neighbors (k_export_list) returns exactly that, md_get_neighbor_rows returns the raw rows.
//
// One LANE per pair row; a task = 32 consecutive pair rows, which may belong to different cells:
// the lanes of a warp then walk different candidate runs of about the same length, in lockstep (ragged pieces
// read a far-away dummy quad).  Four candidates per 128-bit broadcast load from SoA shared memory; accepted slot
// codes go to a small per-lane ring in shared memory (one predicated 16-bit store + pointer add each) and
// leave for global memory as complete 128-bit words.
// Shared memory: TileTables | offs[tile cells] float4 | rowcell[interior_cap/4 + 8] u16 | xs[capA] ys[capA] zs[capA] floats |
// rings[nwarps*32*RING_STRIDE].
// List layout: 16-bit codes (slot << code_shift), 8 per uint4; entry e of pair row r sits in word
//   q = e/8, lane s = q % K, chunk c = q / K  at  list[tile_base + c*slots_cap + r*K + s],  slots_cap = prow_cap * K.
// Unused entries of the last word hold the dummy slot n_slots (a far-away point).
// ---------------------------------------------------------------------------------------------------
struct BuildArgs {
  Geom g;
  const int* tab;          // per-tile tables (k_tile_tables)
  const void* xr;          // packed cell-relative positions (float4, or double4 when xr_double)
  int xr_double;
  float rl2_hi;            // fp32 accept test: r2 < rl2_hi = rl^2 (1 + band)
  uint4* list;
  int* numneigh;           // [ntiles][prow_cap]: entries of each pair row
  Flags* flags;
};

__host__ __device__ inline int prow_cap(const Geom& g) { return g.interior_cap >> 1; }   // pair rows a tile can hold
__device__ __forceinline__ int build_capA(const Geom& g) { return (g.tile_cap + 8) & ~3; }
__host__ __device__ inline int build_rowcell_len(const Geom& g) { return ((g.interior_cap >> 1) + 15) & ~7; }   // u16 entries (one per pair row), 16-byte multiple

// packed fp32 pairs (sm_100 FADD2 / FMUL2 / FFMA2: two lanes of math per issue slot)
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
// the same, never rematerialised: for loop invariants (ptxas otherwise rebuilds the pair with two moves at every use)
__device__ __forceinline__ f32x2 pack2_once(float lo, float hi) { f32x2 r; asm volatile("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// 128-bit shared load as two packed pairs {a0,a1} {a2,a3}: the pairs are ready for the f32x2 ops, no moves
__device__ __forceinline__ void lds_2x2(unsigned a, f32x2& p01, f32x2& p23) {
  asm volatile("ld.shared.v2.u64 {%0,%1}, [%2];" : "=l"(p01), "=l"(p23) : "r"(a));
}

// ring push of two candidates for a PAIR of atoms: qa = r2 of atom 0 to {candidate a, candidate b}, qb = the same
// for atom 1.  For each candidate: if (min(r2_0, r2_1) < hi) { ring[rp] = code (16 bit); rp += 2 }.  The compares
// live in the asm so that they feed the two predicated instructions directly (FSETP, FSETP.OR, @P STS.U16, @P IADD).
// SELF = 0: no exclusion (the candidates belong to another cell)
// SELF = 1: own cell, full list: skip the pair's own two slots: (code - self0) as unsigned must exceed one slot
// SELF = 2: own cell, half list: only slots after the pair's second atom: (code - self0) as signed must exceed one slot
template <int SELF, int SHIFT>
__device__ __forceinline__ void ring_push_pair(unsigned& rp, unsigned code_a, f32x2 qa, f32x2 qb, float hi, unsigned self0) {
  if constexpr (SELF == 0) {
    asm volatile(
        "{ .reg .pred p; .reg .f32 a0, a1, b0, b1; .reg .b16 c, d; .reg .b32 cb;\n"
        "  mov.b64 {a0, a1}, %2;\n"
        "  mov.b64 {b0, b1}, %3;\n"
        "  mov.b32 {c, d}, %1;\n"
        "  setp.lt.f32 p, a0, %4;\n"
        "  setp.lt.or.f32 p, b0, %4, p;\n"
        "  @p st.shared.u16 [%0], c;\n"
        "  @p add.u32 %0, %0, 2;\n"
        "  add.u32 cb, %1, %5;\n"
        "  mov.b32 {c, d}, cb;\n"
        "  setp.lt.f32 p, a1, %4;\n"
        "  setp.lt.or.f32 p, b1, %4, p;\n"
        "  @p st.shared.u16 [%0], c;\n"
        "  @p add.u32 %0, %0, 2; }"
        : "+r"(rp)
        : "r"(code_a), "l"(qa), "l"(qb), "f"(hi), "n"(1 << SHIFT)
        : "memory");
  } else if constexpr (SELF == 1) {
    asm volatile(
        "{ .reg .pred p; .reg .f32 a0, a1, b0, b1; .reg .b16 c, d; .reg .b32 cb, df;\n"
        "  mov.b64 {a0, a1}, %2;\n"
        "  mov.b64 {b0, b1}, %3;\n"
        "  mov.b32 {c, d}, %1;\n"
        "  sub.u32 df, %1, %6;\n"
        "  setp.lt.f32 p, a0, %4;\n"
        "  setp.lt.or.f32 p, b0, %4, p;\n"
        "  setp.gt.and.u32 p, df, %5, p;\n"
        "  @p st.shared.u16 [%0], c;\n"
        "  @p add.u32 %0, %0, 2;\n"
        "  add.u32 cb, %1, %5;\n"
        "  mov.b32 {c, d}, cb;\n"
        "  add.u32 df, df, %5;\n"
        "  setp.lt.f32 p, a1, %4;\n"
        "  setp.lt.or.f32 p, b1, %4, p;\n"
        "  setp.gt.and.u32 p, df, %5, p;\n"
        "  @p st.shared.u16 [%0], c;\n"
        "  @p add.u32 %0, %0, 2; }"
        : "+r"(rp)
        : "r"(code_a), "l"(qa), "l"(qb), "f"(hi), "n"(1 << SHIFT), "r"(self0)
        : "memory");
  } else {
    asm volatile(
        "{ .reg .pred p; .reg .f32 a0, a1, b0, b1; .reg .b16 c, d; .reg .b32 cb, df;\n"
        "  mov.b64 {a0, a1}, %2;\n"
        "  mov.b64 {b0, b1}, %3;\n"
        "  mov.b32 {c, d}, %1;\n"
        "  sub.u32 df, %1, %6;\n"
        "  setp.lt.f32 p, a0, %4;\n"
        "  setp.lt.or.f32 p, b0, %4, p;\n"
        "  setp.gt.and.s32 p, df, %5, p;\n"
        "  @p st.shared.u16 [%0], c;\n"
        "  @p add.u32 %0, %0, 2;\n"
        "  add.u32 cb, %1, %5;\n"
        "  mov.b32 {c, d}, cb;\n"
        "  add.u32 df, df, %5;\n"
        "  setp.lt.f32 p, a1, %4;\n"
        "  setp.lt.or.f32 p, b1, %4, p;\n"
        "  setp.gt.and.s32 p, df, %5, p;\n"
        "  @p st.shared.u16 [%0], c;\n"
        "  @p add.u32 %0, %0, 2; }"
        : "+r"(rp)
        : "r"(code_a), "l"(qa), "l"(qb), "f"(hi), "n"(1 << SHIFT), "r"(self0)
        : "memory");
  }
}

// The scan of nq quads of candidates (staged slots off/4 ..) for one lane = one pair of atoms: packed fp32 distance
// test of both atoms against four candidates per iteration, accepted codes to the lane's ring.
// FIXED > 0: the common full piece, a constant trip count.  RAGGED: the lanes of the warp hold different numbers of
// quads (their pairs belong to different cells): the warp runs nqmax rounds; a lane that has used up its nq quads
// reads the far-away dummy quad at off_dummy instead.
struct PairPos { f32x2 x0, y0, z0, x1, y1, z1; };   // each coordinate of an atom duplicated into both halves
template <int SELF, int SHIFT, int FIXED, bool RAGGED>
__device__ __forceinline__ void build_scan(unsigned& rp, unsigned xs_a, unsigned ys_a, unsigned zs_a, unsigned off, unsigned code, int nq,
                                           int nqmax, unsigned off_dummy, const PairPos& P, float hi, unsigned self0) {
  const int trips = FIXED > 0 ? FIXED : (RAGGED ? nqmax : nq);
#pragma unroll 2
  for (int q = 0; q < trips; ++q) {
    const unsigned o = (RAGGED && q >= nq) ? off_dummy : off;
    f32x2 X01, X23, Y01, Y23, Z01, Z23;
    lds_2x2(xs_a + o, X01, X23);
    lds_2x2(ys_a + o, Y01, Y23);
    lds_2x2(zs_a + o, Z01, Z23);
    f32x2 qa01, qa23, qb01, qb23;
    {
      const f32x2 dx01 = sub2(P.x0, X01), dx23 = sub2(P.x0, X23);
      const f32x2 dy01 = sub2(P.y0, Y01), dy23 = sub2(P.y0, Y23);
      const f32x2 dz01 = sub2(P.z0, Z01), dz23 = sub2(P.z0, Z23);
      qa01 = fma2(dz01, dz01, fma2(dy01, dy01, mul2(dx01, dx01)));
      qa23 = fma2(dz23, dz23, fma2(dy23, dy23, mul2(dx23, dx23)));
    }
    {
      const f32x2 dx01 = sub2(P.x1, X01), dx23 = sub2(P.x1, X23);
      const f32x2 dy01 = sub2(P.y1, Y01), dy23 = sub2(P.y1, Y23);
      const f32x2 dz01 = sub2(P.z1, Z01), dz23 = sub2(P.z1, Z23);
      qb01 = fma2(dz01, dz01, fma2(dy01, dy01, mul2(dx01, dx01)));
      qb23 = fma2(dz23, dz23, fma2(dy23, dy23, mul2(dx23, dx23)));
    }
    ring_push_pair<SELF, SHIFT>(rp, code, qa01, qb01, hi, self0);
    ring_push_pair<SELF, SHIFT>(rp, code + (2u << SHIFT), qa23, qb23, hi, self0);
    off += 16;
    code += 4u << SHIFT;
  }
}

template <bool HALF, int LOGK, int SHIFT>
__global__ void __launch_bounds__(BUILD_MAX_THREADS, BUILD_MIN_BLOCKS) k_build_list(BuildArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  const Geom& g = A.g;
  constexpr int K = 1 << LOGK;
  const int capA = build_capA(g);
  float4* offs = reinterpret_cast<float4*>(smem_raw + sizeof(TileTables));
  unsigned short* rowcell = reinterpret_cast<unsigned short*>(offs + tile_tab_cells(g));   // tile cell of every quad of interior slots
  float* xs = reinterpret_cast<float*>(rowcell + build_rowcell_len(g));
  float* ys = xs + capA;
  float* zs = ys + capA;
  unsigned char* rings = reinterpret_cast<unsigned char*>(zs + capA);
  const int tile = blockIdx.x;
  __shared__ int soff[27];   // tile-cell index offsets of the 27-cell stencil (the same for every cell of the tile)
  tile_load(g, tile, A.tab, tt);
  if (threadIdx.x < 27) {
    const int dx = (int)threadIdx.x % 3 - 1, dy = ((int)threadIdx.x / 3) % 3 - 1, dz = (int)threadIdx.x / 9 - 1;
    soff[threadIdx.x] = (dz * tt.tc[1] + dy) * tt.tc[0] + dx;
  }
  if (tt.n_slots > g.tile_cap || tt.n_int_slots > g.interior_cap) return;   // host re-plans and rebuilds
  for (int ic = threadIdx.x; ic < tt.nic; ic += blockDim.x) {
    const int t = interior_tile_cell(tt, ic);
    for (int i = 0; i < pad2(tt.cnt[t]) >> 1; ++i) rowcell[(tt.rstart[t] >> 1) + i] = (unsigned short)t;
  }
  // staging: tile-centred fp32 coordinates = packed cell-relative coordinate + the cell's offset (the same values the
  // force kernels stage), one thread per quad of slots, SoA so that four candidates are one broadcast 128-bit load
  for (int t = threadIdx.x; t < tt.ntc; t += blockDim.x) {
    double od[3];
    tile_cell_offset_rel(g, tt, t, od);
    offs[t] = make_float4((float)od[0], (float)od[1], (float)od[2], 0.f);
  }
  __syncthreads();
  {
    const unsigned short* __restrict__ qc =
        reinterpret_cast<const unsigned short*>(A.tab + (size_t)tile * tile_tab_stride(g) + TILE_HDR + TILE_CELL_INTS * tile_tab_cells(g));
    const int nq = tt.n_slots >> 2;
    for (int q = threadIdx.x; q < nq; q += blockDim.x) {
      const int t = qc[q];
      const int c = tt.cnt[t], k0 = 4 * q - tt.start[t], gb = tt.gstart[t] + k0;
      const float4 o = offs[t];
      float xv[4], yv[4], zv[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        if (k0 + u < c) {
          if (A.xr_double) {
            const double4 v = reinterpret_cast<const double4*>(A.xr)[gb + u];
            xv[u] = (float)v.x + o.x; yv[u] = (float)v.y + o.y; zv[u] = (float)v.z + o.z;
          } else {
            const float4 v = reinterpret_cast<const float4*>(A.xr)[gb + u];
            xv[u] = v.x + o.x; yv[u] = v.y + o.y; zv[u] = v.z + o.z;
          }
        } else {
          xv[u] = 1e15f; yv[u] = 1e15f; zv[u] = 1e15f;
        }
      }
      *reinterpret_cast<float4*>(xs + 4 * q) = make_float4(xv[0], xv[1], xv[2], xv[3]);
      *reinterpret_cast<float4*>(ys + 4 * q) = make_float4(yv[0], yv[1], yv[2], yv[3]);
      *reinterpret_cast<float4*>(zs + 4 * q) = make_float4(zv[0], zv[1], zv[2], zv[3]);
    }
    if (threadIdx.x < 4) {   // the dummy quad (its first slot is the dummy slot the list's padding names)
      xs[tt.n_slots + threadIdx.x] = 1e15f; ys[tt.n_slots + threadIdx.x] = 1e15f; zs[tt.n_slots + threadIdx.x] = 1e15f;
    }
  }
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const unsigned rbase = smem_addr(rings) + (unsigned)(wid * 32 + lane) * RING_STRIDE;
  const size_t slots_cap = (size_t)prow_cap(g) << LOGK;
  uint4* tlist = A.list + (size_t)tile * g.chunk_cap * slots_cap;
  const int max_words = g.chunk_cap << LOGK;
  const unsigned dummy = (unsigned)tt.n_slots << SHIFT;
  const float hi = A.rl2_hi;
  const unsigned xs_a = smem_addr(xs), ys_a = smem_addr(ys), zs_a = smem_addr(zs);
  int my_max = 0;
  unsigned long long my_sum = 0;

  const int nrp = tt.n_int_slots >> 1;                 // pair rows in use
  const unsigned off_dummy = 4u * (unsigned)tt.n_slots;
#pragma unroll 1
  for (int task = wid; task * 32 < nrp; task += nw) {
    const int prow = task * 32 + lane;                 // this lane's pair row
    const bool havep = prow < nrp;
    const int t = rowcell[havep ? prow : 0];           // its tile cell
    const int c = tt.cnt[t], g_lo = tt.gstart[t];
    const int kin0 = havep ? 2 * prow - tt.rstart[t] : c;   // index of the pair's first atom within its cell
    const bool act0 = kin0 < c, act1 = kin0 + 1 < c;
    const int aslot0 = tt.start[t] + (act0 ? kin0 : 0);                  // staged slot of the first atom
    PairPos P;
    {
      // an idle atom sits far away from everything, pad slots (+1e15) included: it accepts nothing
      const float x0 = act0 ? xs[aslot0] : -1e15f, y0 = act0 ? ys[aslot0] : -1e15f, z0 = act0 ? zs[aslot0] : -1e15f;
      const float x1 = act1 ? xs[aslot0 + 1] : -1e15f, y1 = act1 ? ys[aslot0 + 1] : -1e15f, z1 = act1 ? zs[aslot0 + 1] : -1e15f;
      P.x0 = pack2(x0, x0); P.y0 = pack2(y0, y0); P.z0 = pack2(z0, z0);
      P.x1 = pack2(x1, x1); P.y1 = pack2(y1, y1); P.z1 = pack2(z1, z1);
    }
    const unsigned self0 = (unsigned)aslot0 << SHIFT;
    unsigned rp = rbase;
    int nwords = 0;
    auto store_word = [&](uint4 v) {
      if (nwords < max_words) {
        const int s = nwords & (K - 1), cch = nwords >> LOGK;
        st_stream(tlist + (size_t)cch * slots_cap + ((size_t)prow << LOGK) + s, v);
      }
      ++nwords;
    };
    auto flush = [&]() {   // complete words leave; the remainder moves to the ring start
      const int pend = (int)(rp - rbase) >> 1, full = pend >> 3;
      for (int w = 0; w < full; ++w) store_word(lds_u4(rbase + 16 * w));
      if (full) sts_u4(rbase, lds_u4(rbase + 16 * full));
      rp = rbase + 2 * (pend & 7);
    };
    // Full list: 9 runs, one per (dy, dz): the cells x-1, x, x+1 are consecutive tile cells, hence one contiguous
    // range of staged slots (pad slots in between are far away and never taken).  Half list: 27 one-cell runs,
    // because a whole cell is kept or dropped (below).
    constexpr int NRUN = HALF ? 27 : 9;
#pragma unroll 1
    for (int sc = 0; sc < NRUN; ++sc) {
      int s0, s1;
      bool own;                                        // the run holds the pair's own cell (the same for all lanes)
      if constexpr (HALF) {
        const int tfirst = t + soff[sc];
        own = sc == 13;
        s0 = tt.start[tfirst];
        s1 = s0 + pad4(tt.cnt[tfirst]);
        // keep (i, j) iff j follows i in the sorted order; a cell is a contiguous range of that order, so for
        // another cell the answer is the same for all of its atoms; the own cell keeps the slots after the pair
        if (!own && tt.gstart[tfirst] < g_lo) s1 = s0;
      } else {
        const int tc = t + soff[3 * sc + 1];
        own = sc == 4;
        s0 = tt.start[tc - 1];
        s1 = tt.start[tc + 1] + pad4(tt.cnt[tc + 1]);
      }
      // (a lane without atoms scans its quad's runs like the others, so that full pieces stay uniform; it sits
      // far away and accepts nothing)
      const int npieces = (int)__reduce_max_sync(0xffffffffu, (unsigned)((s1 - s0 + 31) >> 5));
#pragma unroll 1
      for (int pc = 0; pc < npieces; ++pc) {   // pieces of <= 32 slots: what the ring is guaranteed to take
        const int j0 = s0 + 32 * pc;
        const int nq = max(0, min(8, (s1 - j0) >> 2));
        if ((int)(rp - rbase) > 2 * (RING - 32)) flush();
        const unsigned off = 4u * (unsigned)j0, code = (unsigned)j0 << SHIFT;
        constexpr int SELF = HALF ? 2 : 1;
        if (__all_sync(0xffffffffu, nq == 8)) {
          if (own) build_scan<SELF, SHIFT, 8, false>(rp, xs_a, ys_a, zs_a, off, code, 8, 8, off_dummy, P, hi, self0);
          else build_scan<0, SHIFT, 8, false>(rp, xs_a, ys_a, zs_a, off, code, 8, 8, off_dummy, P, hi, self0);
        } else {
          const int nqmax = (int)__reduce_max_sync(0xffffffffu, (unsigned)nq);
          if (own) build_scan<SELF, SHIFT, 0, true>(rp, xs_a, ys_a, zs_a, off, code, nq, nqmax, off_dummy, P, hi, self0);
          else build_scan<0, SHIFT, 0, true>(rp, xs_a, ys_a, zs_a, off, code, nq, nqmax, off_dummy, P, hi, self0);
        }
      }
    }
    // last words: complete ones, then the partial one padded with the dummy code
    flush();
    const int rem = (int)(rp - rbase) >> 1;   // 0..7
    if (rem) {
      for (int p = rem; p < 8; ++p) sts_u16(rbase + 2 * p, dummy);
      const int before = nwords;
      store_word(lds_u4(rbase));
      nwords = before;   // count below from complete words + rem
    }
    const int n = nwords * 8 + rem;
    if (havep) {
      const int stored = act0 ? (n < g.row_cap ? n : g.row_cap) : 0;
      A.numneigh[(size_t)tile * prow_cap(g) + prow] = stored;
      if (act0) {
        my_max = max(my_max, n);
        my_sum += (unsigned long long)stored;
      }
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, o));
    my_sum += __shfl_xor_sync(0xffffffffu, my_sum, o);
  }
  if (lane == 0) {
    atomicMax(&A.flags->max_row, my_max);
    if (my_max > g.row_cap) atomicMax(&A.flags->need_row_cap, my_max);
    atomicAdd(&A.flags->sum_rows, my_sum);
  }
}

// ---------------------------------------------------------------------------------------------------
// Row balancing (after every list build).  The force kernels fetch a neighbor with one 128-bit shared-memory load
// per lane; the hardware serves such a load a quarter warp (8 threads) at a time, and two of the 8 threads
// collide when their records fall into the same 16-byte bank group, i.e. when their slots agree mod 8 (measured:
// ~9 wavefronts per warp gather on random slots against 4 without collisions -- the force kernels' bound).
// The order of the entries within a row is free, so this kernel permutes every row such that, wherever
// possible, position u of word q holds an entry with  slot mod 8 == (u + thread index of (row, q)) mod 8:
// the 8 threads of a quarter warp, which walk their words in lockstep, then read 8 different bank groups.
// Residue classes are never perfectly even, so the surplus of the longer classes fills the holes of the
// shorter ones (those entries may collide), and the remaining holes name the dummy slot.
// One thread per (pair) row; its output row is assembled in a private stripe of shared memory (row_bytes).
// ---------------------------------------------------------------------------------------------------
struct BalanceArgs {
  Geom g;
  const int* tab;
  uint4* list;
  const int* numneigh;
  int row_bytes;      // shared-memory stripe per thread: row_cap * 2 + 16 (an odd number of 16-byte units)
};

template <int LOGK>
__global__ void __launch_bounds__(256) k_balance_rows(BalanceArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Geom& g = A.g;
  constexpr int K = 1 << LOGK;
  const int tile = blockIdx.x;
  const int* __restrict__ h = A.tab + (size_t)tile * tile_tab_stride(g);
  const int n_rows = h[0] >> 1, n_slots = h[1];   // pair rows
  if (n_slots > g.tile_cap || h[0] > g.interior_cap) return;
  const int shift = g.code_shift;
  const unsigned dummy = (unsigned)n_slots << shift;
  const size_t slots_cap = (size_t)prow_cap(g) << LOGK;
  uint4* tlist = A.list + (size_t)tile * g.chunk_cap * slots_cap;
  unsigned short* out = reinterpret_cast<unsigned short*>(smem_raw + (size_t)threadIdx.x * A.row_bytes);
  for (int a = threadIdx.x; a < n_rows; a += blockDim.x) {
    const int n = min(A.numneigh[(size_t)tile * prow_cap(g) + a], g.row_cap);
    if (n <= 0) continue;
    const int W = (n + 7) >> 3;
    auto word_ptr = [&](int q) { return tlist + (size_t)(q >> LOGK) * slots_cap + ((size_t)a << LOGK) + (q & (K - 1)); };
    auto tix = [&](int q) { return (a * K + (q & (K - 1))) & 7; };   // thread index mod 8 of the thread that reads word q
    // pass A: entries per residue class (16-bit counters, four to a 64-bit register)
    unsigned long long cnt[2] = {0ull, 0ull};
    for (int q = 0; q < W; ++q) {
      const uint4 w = *word_ptr(q);
      const unsigned ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const unsigned code = (e & 1) ? (ww[e >> 1] >> 16) : (ww[e >> 1] & 0xffffu);
        if (q * 8 + e < n) {            // the build leaves the real entries in the first n positions
          const unsigned rho = (code >> shift) & 7u;
          cnt[rho >> 2] += 1ull << (16 * (rho & 3u));
        }
      }
    }
    auto count_of = [&](unsigned rho) { return (int)((cnt[rho >> 2] >> (16 * (rho & 3u))) & 0xffffu); };
    // pass B: the k-th entry of class rho goes to word k, position (rho - tix(k)) & 7, while k < W; later ones fill holes
    unsigned long long cur[2] = {0ull, 0ull};
    int hr = 0, hk = min(count_of(0), W);     // hole cursor: class hr, word hk
    auto next_hole = [&]() {
      while (hr < 8 && hk >= W) { ++hr; hk = hr < 8 ? min(count_of((unsigned)hr), W) : 0; }
      const int pos = hk * 8 + ((hr - tix(hk)) & 7);
      ++hk;
      return pos;
    };
    for (int q = 0; q < W; ++q) {
      const uint4 w = *word_ptr(q);
      const unsigned ww[4] = {w.x, w.y, w.z, w.w};
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const unsigned code = (e & 1) ? (ww[e >> 1] >> 16) : (ww[e >> 1] & 0xffffu);
        if (q * 8 + e < n) {
          const unsigned rho = (code >> shift) & 7u;
          const int k = (int)((cur[rho >> 2] >> (16 * (rho & 3u))) & 0xffffu);
          cur[rho >> 2] += 1ull << (16 * (rho & 3u));
          const int pos = k < W ? k * 8 + (((int)rho - tix(k)) & 7) : next_hole();
          out[pos] = (unsigned short)code;
        }
      }
    }
    for (int left = 8 * W - n; left > 0; --left) out[next_hole()] = (unsigned short)dummy;
    for (int q = 0; q < W; ++q) *word_ptr(q) = *reinterpret_cast<const uint4*>(out + 8 * q);
  }
}

// fp64 decision of the pair-set definition (north_star (2)): |x_i - x_j|^2 < rl^2 from the global positions, atom gi
// of tile cell ti against atom gj of tile cell tj (their periodic images are the ones the tile stages).
__device__ __forceinline__ bool pair_in_list_fp64(const Geom& g, const TileTables& tt, const double* __restrict__ x, size_t ld,
                                                  int gi, int ti, int gj, int tj, double rl2) {
  double oi[3], oj[3];
  tile_cell_offset(g, tt, ti, oi);
  tile_cell_offset(g, tt, tj, oj);
  double r2 = 0.0;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double dd = (x[d * ld + gi] + oi[d]) - (x[d * ld + gj] + oj[d]);
    r2 += dd * dd;
  }
  return r2 < rl2;
}

// List export in caller ids (pair-set parity; test / diagnostic path, one thread per interior atom).
//   EXPORT_EXACT: nn_out[i], neigh_out[i][..] = the exact fp64 neighbor set of atom i: the entries of its pair's row
//                 (plus its partner) that pass the fp64 test; neigh_out may be NULL (counts only);
//                 stat[0] = max count (int), stat[2..3] = sum of counts (unsigned long long) when stat != NULL.
//   EXPORT_RAW:   the stored rows as they are: nn_out[i] = row length and neigh_out[i][..] = the row's entries for
//                 the FIRST atom of a pair (0 for the second); owner_out[i] = caller id of the pair's first atom.
// Shared memory: TileTables | sid[capA] | sgi[capA] ints | scl[capA] u16.
constexpr int EXPORT_EXACT = 0, EXPORT_RAW = 1;
struct ExportArgs {
  Geom g;
  const int* tab; const int* id; const double* x; size_t ld;
  const uint4* list; const int* numneigh;
  double rl2;
  int mode;
  int* nn_out; int* neigh_out; int* owner_out; long long stride;
  int* stat;
};
__global__ void __launch_bounds__(BUILD_THREADS) k_export_list(ExportArgs A) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  const Geom& g = A.g;
  const int capA = (g.tile_cap + 8) & ~3;
  int* sid = reinterpret_cast<int*>(smem_raw + sizeof(TileTables));
  int* sgi = sid + capA;
  unsigned short* scl = reinterpret_cast<unsigned short*>(sgi + capA);
  const int tile = blockIdx.x;
  tile_load(g, tile, A.tab, tt);
  tile_stage(g, tt, g.tile_cap, [&](int slot, int gi, const double*, int t) { sid[slot] = A.id[gi]; sgi[slot] = gi; scl[slot] = (unsigned short)t; },
             [&](int slot) { sid[slot] = -1; sgi[slot] = 0; scl[slot] = 0; });
  __syncthreads();
  const int K = g.K;
  const size_t slots_cap = (size_t)prow_cap(g) * K;
  const uint4* tlist = A.list + (size_t)tile * g.chunk_cap * slots_cap;
  int my_max = 0;
  unsigned long long my_sum = 0;
  for (int ic = 0; ic < tt.nic; ++ic) {
    const int t = interior_tile_cell(tt, ic);
    const int c = tt.cnt[t];
    for (int k = threadIdx.x; k < c; k += blockDim.x) {
      const int prow = (tt.rstart[t] + k) >> 1, which = k & 1;
      const int n = A.numneigh[(size_t)tile * prow_cap(g) + prow];
      const int slot = tt.start[t] + k, io = sid[slot], gi = sgi[slot];
      const int pslot = slot ^ 1;                      // the partner's slot (cells start at multiples of 4)
      const bool have_partner = (k ^ 1) < c;
      if (A.mode == EXPORT_RAW) {
        A.owner_out[io] = which ? sid[pslot] : io;
        if (which) { A.nn_out[io] = 0; continue; }
      }
      int m = 0;
      auto emit = [&](int jo) {
        if (A.neigh_out && m < A.stride) A.neigh_out[(long long)io * A.stride + m] = jo;
        ++m;
      };
      // the partner: never stored in the row (the force kernels add the pair's mutual term directly)
      if (A.mode == EXPORT_EXACT && have_partner && (!g.half || which == 0) &&
          pair_in_list_fp64(g, tt, A.x, A.ld, gi, t, sgi[pslot], t, A.rl2))
        emit(sid[pslot]);
      // the row's n entries sit somewhere in its ceil(n/8) words; the other positions name the dummy slot
      for (int e = 0; e < ((n + 7) & ~7); ++e) {
        const int q = e >> 3, sl = q % K, ch = q / K;
        const uint4 w = tlist[(size_t)ch * slots_cap + (size_t)prow * K + sl];
        const unsigned word = (&w.x)[(e & 7) >> 1];
        const unsigned code = (e & 1) ? (word >> 16) : (word & 0xffffu);
        const int js = (int)(code >> g.code_shift);
        if (js == tt.n_slots) continue;
        if (A.mode == EXPORT_RAW || pair_in_list_fp64(g, tt, A.x, A.ld, gi, t, sgi[js], scl[js], A.rl2)) emit(sid[js]);
      }
      A.nn_out[io] = m;
      my_max = max(my_max, m);
      my_sum += (unsigned long long)m;
    }
  }
  if (A.stat) {
    for (int o = 16; o > 0; o >>= 1) {
      my_max = max(my_max, __shfl_xor_sync(0xffffffffu, my_max, o));
      my_sum += __shfl_xor_sync(0xffffffffu, my_sum, o);
    }
    if ((threadIdx.x & 31) == 0) {
      atomicMax(&A.stat[0], my_max);
      atomicAdd(reinterpret_cast<unsigned long long*>(A.stat + 2), my_sum);
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// pair styles.  T = double (MD_FP64) or float (MD_MIXED pair math).
// A Body has two entry points:
//   pair  -- one (i, j) term on scalars (the direct cell-list kernel);
//   pair2 -- the terms (i0, j) and (i1, j) of the two atoms of a PAIR ROW against one gathered j, on two-wide
//            values Pk<T>: for float a packed f32x2 register pair (FADD2 / FMUL2 / FFMA2: two lanes of math per
//            issue slot), for double a plain struct of two doubles.
// Both accumulate per-word partial sums in T; the kernels add them to per-atom totals in double.
// Bodies are branch-free: out-of-range partners contribute an exact zero through a select.
// ---------------------------------------------------------------------------------------------------
template <typename T> struct Vec2;
template <> struct Vec2<float> { using type = float2; };
template <> struct Vec2<double> { using type = double2; };
template <typename T> __device__ __forceinline__ typename Vec2<T>::type lds_v2(unsigned a);
template <> __device__ __forceinline__ float2 lds_v2<float>(unsigned a) { return lds_f2(a); }
template <> __device__ __forceinline__ double2 lds_v2<double>(unsigned a) { return lds_d2(a); }

struct d64x2 { double a, b; };
template <typename T> struct Pk;
template <> struct Pk<float> { using type = f32x2; };
template <> struct Pk<double> { using type = d64x2; };
__device__ __forceinline__ f32x2 pk_make(float a, float b) { return pack2(a, b); }
__device__ __forceinline__ d64x2 pk_make(double a, double b) { return d64x2{a, b}; }
__device__ __forceinline__ f32x2 pk_make_once(float a, float b) { return pack2_once(a, b); }
__device__ __forceinline__ d64x2 pk_make_once(double a, double b) { return d64x2{a, b}; }
__device__ __forceinline__ float pk_lo(f32x2 v) { float a, b; unpack2(v, a, b); return a; }
__device__ __forceinline__ float pk_hi(f32x2 v) { float a, b; unpack2(v, a, b); return b; }
__device__ __forceinline__ double pk_lo(d64x2 v) { return v.a; }
__device__ __forceinline__ double pk_hi(d64x2 v) { return v.b; }
__device__ __forceinline__ f32x2 pk_add(f32x2 x, f32x2 y) { return add2(x, y); }
__device__ __forceinline__ f32x2 pk_sub(f32x2 x, f32x2 y) { return sub2(x, y); }
__device__ __forceinline__ f32x2 pk_mul(f32x2 x, f32x2 y) { return mul2(x, y); }
__device__ __forceinline__ f32x2 pk_fma(f32x2 x, f32x2 y, f32x2 z) { return fma2(x, y, z); }
__device__ __forceinline__ d64x2 pk_add(d64x2 x, d64x2 y) { return d64x2{x.a + y.a, x.b + y.b}; }
__device__ __forceinline__ d64x2 pk_sub(d64x2 x, d64x2 y) { return d64x2{x.a - y.a, x.b - y.b}; }
__device__ __forceinline__ d64x2 pk_mul(d64x2 x, d64x2 y) { return d64x2{x.a * y.a, x.b * y.b}; }
__device__ __forceinline__ d64x2 pk_fma(d64x2 x, d64x2 y, d64x2 z) { return d64x2{fma(x.a, y.a, z.a), fma(x.b, y.b, z.b)}; }
template <typename T> __device__ __forceinline__ typename Pk<T>::type pk_splat(T a) { return pk_make(a, a); }

constexpr int MAX_PAIR_TYPES = 4;   // types a multi-type pair style can tell apart (the staged record carries the type in w)
struct PairParams {    // host-prepared constants, in double; kernels convert once
  double rc2;
  double lj1, lj2, lj3, lj4;             // 48 eps s^12, 24 eps s^6, 4 eps s^12, 4 eps s^6
  double A, p_r0, B, q_r0, inv_r0, p, q; // EAM: A, p/r0, B, q/r0, 1/r0, p, q
  // the same rounded to fp32 once on the host (fill_float_copies): the mixed-precision bodies read these straight
  // from the constant bank instead of converting the doubles inside the list loop
  float f_rc2, f_lj1, f_lj2, f_lj3, f_lj4, f_A, f_p_r0, f_q_r0, f_p, f_q;
  // tabulated EAM (reading s26): per interval k of the uniform grids the cubic c0 + c1 u + c2 u^2 + c3 u^3, u = x/h - k
  // (host: md_set_eam_tables); rho(r) and phi(r) in the pair-math precision, F(rho) in double.  NULL: analytic EAM
  const void* tab_rho;     // [tab_nr - 1] Vec4<T>
  const void* tab_phi;     // [tab_nr - 1] Vec4<T>
  const double4* tab_F;    // [tab_nrho - 1]
  int tab_nr, tab_nrho;
  double inv_dr, inv_drho;
  // Buckingham + cutoff Coulomb: per type pair (ta, tb), entry 4 ta + tb: A, 1/rho, C, k q_a q_b
  double bc[MAX_PAIR_TYPES * MAX_PAIR_TYPES][4];
  __host__ void fill_float_copies() {
    f_rc2 = (float)rc2; f_lj1 = (float)lj1; f_lj2 = (float)lj2; f_lj3 = (float)lj3; f_lj4 = (float)lj4;
    f_A = (float)A; f_p_r0 = (float)p_r0; f_q_r0 = (float)q_r0; f_p = (float)p; f_q = (float)q;
  }
};
template <typename T> __device__ __forceinline__ T pp_pick(double d, float f);
template <> __device__ __forceinline__ float pp_pick<float>(double, float f) { return f; }
template <> __device__ __forceinline__ double pp_pick<double>(double d, float) { return d; }
#define MDK_PP(name) pp_pick<T>(P.name, P.f_##name)

template <typename T> __device__ __forceinline__ T t_rcp(T x);
template <> __device__ __forceinline__ float t_rcp<float>(float x) { return rcp_approx(x); }
template <> __device__ __forceinline__ double t_rcp<double>(double x) { return 1.0 / x; }
template <typename T> __device__ __forceinline__ T t_rsqrt(T x);
template <> __device__ __forceinline__ float t_rsqrt<float>(float x) { return rsqrt_approx(x); }
template <> __device__ __forceinline__ double t_rsqrt<double>(double x) { return 1.0 / sqrt(x); }
template <typename T> __device__ __forceinline__ T t_exp(T x);
template <> __device__ __forceinline__ float t_exp<float>(float x) { return ex2_approx(x * 1.4426950408889634f); }
template <> __device__ __forceinline__ double t_exp<double>(double x) { return exp(x); }

// the six virial products of one term, accumulated two-wide: p[4..9] += {dx dx, dy dy, dz dz, dx dy, dx dz, dy dz} fp
template <class PK>
__device__ __forceinline__ void virial2(PK dx, PK dy, PK dz, PK fp, PK* p) {
  const PK fx = pk_mul(fp, dx), fy = pk_mul(fp, dy), fz = pk_mul(fp, dz);
  p[4] = pk_fma(dx, fx, p[4]); p[5] = pk_fma(dy, fy, p[5]); p[6] = pk_fma(dz, fz, p[6]);
  p[7] = pk_fma(dx, fy, p[7]); p[8] = pk_fma(dx, fz, p[8]); p[9] = pk_fma(dy, fz, p[9]);
}

// LJ 12-6 force (+ energy, virial when EV).  PAPER.md L102 calcPairForce, App. A L256.
template <typename T, bool EV>
struct LJBody {
  // the w component of a staged record: the row's own atoms enter the list loop with own_w(w), every gathered atom j
  // with its staged w, and pair2 receives own_w(w_i) - w_j (the direct cell-list kernel: cell_own_w(w_i) + w_j)
  static __device__ __forceinline__ T own_w(T w) { return -w; }
  static __device__ __forceinline__ T mutual_w(T a, T b) { return a + b; }
  static __device__ __forceinline__ T cell_own_w(T w) { return w; }
  template <class TAB> __device__ __forceinline__ void attach(TAB*) {}
  static constexpr bool TABLE = false;
  static constexpr int SMEM_TABLES = 0;   // no coefficient tables to stage (tabulated EAM has)
  __device__ __forceinline__ void attach_tables(unsigned, unsigned) {}
  static constexpr int NT = EV ? 10 : 3;   // fx fy fz [e wxx wyy wzz wxy wxz wyz]
  using PK = typename Pk<T>::type;
  T rc2, lj1, lj2, lj3, lj4;
  __device__ explicit LJBody(const PairParams& P) : rc2(MDK_PP(rc2)), lj1(MDK_PP(lj1)), lj2(MDK_PP(lj2)), lj3(MDK_PP(lj3)), lj4(MDK_PP(lj4)) {}
  __device__ __forceinline__ void pair(T dx, T dy, T dz, T r2, T, bool ok, T (&p)[NT]) const {
    const bool in = ok && r2 < rc2;
    T r2i = t_rcp<T>(r2);
    T r6 = r2i * r2i * r2i;
    T fp = in ? r6 * (lj1 * r6 - lj2) * r2i : (T)0;
    p[0] += fp * dx; p[1] += fp * dy; p[2] += fp * dz;
    if constexpr (EV) {
      p[3] += in ? r6 * (lj3 * r6 - lj4) : (T)0;
      p[4] += dx * dx * fp; p[5] += dy * dy * fp; p[6] += dz * dz * fp;
      p[7] += dx * dy * fp; p[8] += dx * dz * fp; p[9] += dy * dz * fp;
    }
  }
  // 1/r^2 := 0 beyond the cutoff: r^-6, the force factor and the energy term are then exact zeros
  __device__ __forceinline__ void pair2(PK dx, PK dy, PK dz, PK r2, PK, PK (&p)[NT]) const {
    const T ra = pk_lo(r2), rb = pk_hi(r2);
    const T ia = ra < rc2 ? t_rcp<T>(ra) : (T)0, ib = rb < rc2 ? t_rcp<T>(rb) : (T)0;
    const PK r2i = pk_make(ia, ib);
    const PK r6 = pk_mul(pk_mul(r2i, r2i), r2i);
    const PK fp = pk_mul(pk_mul(r6, pk_fma(pk_splat<T>(lj1), r6, pk_splat<T>(-lj2))), r2i);
    p[0] = pk_fma(fp, dx, p[0]); p[1] = pk_fma(fp, dy, p[1]); p[2] = pk_fma(fp, dz, p[2]);
    if constexpr (EV) {
      p[3] = pk_fma(r6, pk_fma(pk_splat<T>(lj3), r6, pk_splat<T>(-lj4)), p[3]);
      virial2(dx, dy, dz, fp, p);
    }
  }
};

// EAM pass 1: rho_i = sum_j exp(-q (r/r0 - 1))            (a6)
template <typename T, bool EV>
struct EamDensityBody {
  // the w component of a staged record: the row's own atoms enter the list loop with own_w(w), every gathered atom j
  // with its staged w, and pair2 receives own_w(w_i) - w_j (the direct cell-list kernel: cell_own_w(w_i) + w_j)
  static __device__ __forceinline__ T own_w(T w) { return -w; }
  static __device__ __forceinline__ T mutual_w(T a, T b) { return a + b; }
  static __device__ __forceinline__ T cell_own_w(T w) { return w; }
  template <class TAB> __device__ __forceinline__ void attach(TAB*) {}
  static constexpr bool TABLE = false;
  static constexpr int SMEM_TABLES = 0;   // no coefficient tables to stage (tabulated EAM has)
  __device__ __forceinline__ void attach_tables(unsigned, unsigned) {}
  static constexpr int NT = 1;
  using PK = typename Pk<T>::type;
  T rc2, q_r0, q;
  __device__ explicit EamDensityBody(const PairParams& P) : rc2(MDK_PP(rc2)), q_r0(MDK_PP(q_r0)), q(MDK_PP(q)) {}
  __device__ __forceinline__ void pair(T, T, T, T r2, T, bool ok, T (&p)[NT]) const {
    const bool in = ok && r2 < rc2;
    T r = r2 * t_rsqrt<T>(r2);
    p[0] += in ? t_exp<T>(q - q_r0 * r) : (T)0;
  }
  __device__ __forceinline__ void pair2(PK, PK, PK, PK r2, PK, PK (&p)[NT]) const {
    const T ra = pk_lo(r2), rb = pk_hi(r2);
    const PK r = pk_mul(r2, pk_make(t_rsqrt<T>(ra), t_rsqrt<T>(rb)));
    const PK arg = pk_fma(pk_splat<T>(-q_r0), r, pk_splat<T>(q));
    const T ea = ra < rc2 ? t_exp<T>(pk_lo(arg)) : (T)0, eb = rb < rc2 ? t_exp<T>(pk_hi(arg)) : (T)0;
    p[0] = pk_add(p[0], pk_make(ea, eb));
  }
};

// EAM pass 2: F_i = -sum_j [ (F'_i + F'_j) rho'(r) + phi'(r) ] D / r      (a7); wsum = F'_i + F'_j.
template <typename T, bool EV>
struct EamForceBody {
  // the w component of a staged record: the row's own atoms enter the list loop with own_w(w), every gathered atom j
  // with its staged w, and pair2 receives own_w(w_i) - w_j (the direct cell-list kernel: cell_own_w(w_i) + w_j)
  static __device__ __forceinline__ T own_w(T w) { return -w; }
  static __device__ __forceinline__ T mutual_w(T a, T b) { return a + b; }
  static __device__ __forceinline__ T cell_own_w(T w) { return w; }
  template <class TAB> __device__ __forceinline__ void attach(TAB*) {}
  static constexpr bool TABLE = false;
  static constexpr int SMEM_TABLES = 0;   // no coefficient tables to stage (tabulated EAM has)
  __device__ __forceinline__ void attach_tables(unsigned, unsigned) {}
  static constexpr int NT = EV ? 10 : 3;
  using PK = typename Pk<T>::type;
  T rc2, q_r0, q, p_r0, pp, A;
  __device__ explicit EamForceBody(const PairParams& P)
      : rc2(MDK_PP(rc2)), q_r0(MDK_PP(q_r0)), q(MDK_PP(q)), p_r0(MDK_PP(p_r0)), pp(MDK_PP(p)), A(MDK_PP(A)) {}
  __device__ __forceinline__ void pair(T dx, T dy, T dz, T r2, T wsum, bool ok, T (&p)[NT]) const {
    const bool in = ok && r2 < rc2;
    T rinv = t_rsqrt<T>(r2);
    T r = r2 * rinv;
    T rho = t_exp<T>(q - q_r0 * r);
    T phi = A * t_exp<T>(pp - p_r0 * r);
    // rho' = -(q/r0) rho, phi' = -(p/r0) phi  =>  fpair = [ (F'_i+F'_j)(q/r0) rho + (p/r0) phi ] / r
    T fp = in ? (wsum * q_r0 * rho + p_r0 * phi) * rinv : (T)0;
    p[0] += fp * dx; p[1] += fp * dy; p[2] += fp * dz;
    if constexpr (EV) {
      p[3] += in ? phi : (T)0;
      p[4] += dx * dx * fp; p[5] += dy * dy * fp; p[6] += dz * dz * fp;
      p[7] += dx * dy * fp; p[8] += dx * dz * fp; p[9] += dy * dz * fp;
    }
  }
  // 1/r := 0 and phi := 0 beyond the cutoff zero the force factor and the energy term
  __device__ __forceinline__ void pair2(PK dx, PK dy, PK dz, PK r2, PK wsum, PK (&p)[NT]) const {
    const T ra = pk_lo(r2), rb = pk_hi(r2);
    const T ia = t_rsqrt<T>(ra), ib = t_rsqrt<T>(rb);
    const PK r = pk_mul(r2, pk_make(ia, ib));
    const PK arho = pk_fma(pk_splat<T>(-q_r0), r, pk_splat<T>(q));
    const PK aphi = pk_fma(pk_splat<T>(-p_r0), r, pk_splat<T>(pp));
    const bool ina = ra < rc2, inb = rb < rc2;
    const PK rho = pk_make(t_exp<T>(pk_lo(arho)), t_exp<T>(pk_hi(arho)));
    const PK phi = pk_make(ina ? A * t_exp<T>(pk_lo(aphi)) : (T)0, inb ? A * t_exp<T>(pk_hi(aphi)) : (T)0);
    const PK rinv = pk_make(ina ? ia : (T)0, inb ? ib : (T)0);
    const PK fp = pk_mul(pk_fma(pk_mul(wsum, pk_splat<T>(q_r0)), rho, pk_mul(pk_splat<T>(p_r0), phi)), rinv);
    p[0] = pk_fma(fp, dx, p[0]); p[1] = pk_fma(fp, dy, p[1]); p[2] = pk_fma(fp, dz, p[2]);
    if constexpr (EV) {
      p[3] = pk_add(p[3], phi);
      virial2(dx, dy, dz, fp, p);
    }
  }
};

// Embedding function of one atom: F(rho) and F'(rho).  Analytic (BASELINE.json cfg 4): F = -B sqrt(rho), F'(0) := 0
// (reading s13); tabulated (reading s26): the cubic of rho's interval and its derivative.
__device__ __forceinline__ void eam_embed(const PairParams& P, double rho, double& F, double& dF) {
  if (P.tab_F) {
    const double t = rho * P.inv_drho;
    int k = (int)floor(t);
    k = k < 0 ? 0 : (k > P.tab_nrho - 2 ? P.tab_nrho - 2 : k);
    const double u = t - (double)k;
    const double4 c = P.tab_F[k];
    F = c.x + u * (c.y + u * (c.z + u * c.w));
    dF = (c.y + u * (2.0 * c.z + 3.0 * c.w * u)) * P.inv_drho;
  } else {
    const double sq = sqrt(rho);
    F = -P.B * sq;
    dF = rho > 0.0 ? -P.B / (2.0 * sq) : 0.0;
  }
}

// Tabulated EAM (SURVEY.md 8(f)-2 second half; App. A: what the paper's EAM run used; reading s26).  The same
// two passes as the analytic style with rho(r), rho'(r), phi(r), phi'(r) from per-interval cubics: one 16-byte (fp64: 32)
// table load per function, atom of the row and list entry, through the read-only path (the tables are a few tens of KB).
template <typename T> __device__ __forceinline__ typename Vec4<T>::type lds_v4(unsigned a);   // defined with the force kernels' helpers
template <typename T>
struct TabLookup {
  using V4 = typename Vec4<T>::type;
  T inv_dr;
  int kmax;
  __device__ __forceinline__ int interval(T r, T& u) const {
    const T t = r * inv_dr;
    int k = (int)t;
    k = k > kmax ? kmax : (k < 0 ? 0 : k);   // (r = NaN for the self term r2 = 0 of the cell-list variant: any interval will do, the term is dropped)
    u = t - (T)k;
    return k;
  }
  // smem != 0: the table has been staged in shared memory at that address (k_tile_force_p); else the read-only path
  static __device__ __forceinline__ V4 load(const void* tab, unsigned smem, int k) {
    if constexpr (sizeof(T) == 4) {
      if (smem) return lds_v4<T>(smem + 16u * (unsigned)k);
    }
    return load(tab, k);
  }
  static __device__ __forceinline__ V4 load(const void* tab, int k) {
    if constexpr (sizeof(T) == 4) return __ldg(reinterpret_cast<const float4*>(tab) + k);
    else { const double2* q = reinterpret_cast<const double2*>(tab) + 2 * (size_t)k; const double2 a = __ldg(q), b = __ldg(q + 1); return make_double4(a.x, a.y, b.x, b.y); }
  }
  static __device__ __forceinline__ T value(const V4& c, T u) { return c.x + u * (c.y + u * (c.z + u * c.w)); }
  __device__ __forceinline__ T slope(const V4& c, T u) const { return (c.y + u * ((T)2 * c.z + (T)3 * c.w * u)) * inv_dr; }
};

template <typename T, bool EV>
struct EamTabDensityBody {
  static constexpr int NT = 1;
  using PK = typename Pk<T>::type;
  static __device__ __forceinline__ T own_w(T w) { return -w; }
  static __device__ __forceinline__ T mutual_w(T a, T b) { return a + b; }
  static __device__ __forceinline__ T cell_own_w(T w) { return w; }
  template <class TAB> __device__ __forceinline__ void attach(TAB*) {}
  static constexpr bool TABLE = false;
  T rc2;
  TabLookup<T> L;
  const void* tab_rho;
  unsigned s_rho = 0;   // shared-memory address of the staged table, 0: not staged
  static constexpr int SMEM_TABLES = 1;
  __device__ __forceinline__ void attach_tables(unsigned base, unsigned) { s_rho = base; }
  __device__ explicit EamTabDensityBody(const PairParams& P) : rc2(MDK_PP(rc2)), L{(T)P.inv_dr, P.tab_nr - 2}, tab_rho(P.tab_rho) {}
  __device__ __forceinline__ T rho_of(T r2) const {
    T u;
    const int k = L.interval(r2 * t_rsqrt<T>(r2), u);
    return TabLookup<T>::value(TabLookup<T>::load(tab_rho, s_rho, k), u);
  }
  __device__ __forceinline__ void pair(T, T, T, T r2, T, bool ok, T (&p)[NT]) const { p[0] += (ok && r2 < rc2) ? rho_of(r2) : (T)0; }
  __device__ __forceinline__ void pair2(PK, PK, PK, PK r2, PK, PK (&p)[NT]) const {
    const T ra = pk_lo(r2), rb = pk_hi(r2);
    // (an entry beyond the cutoff may lie beyond the table too: its interval is clamped and its value dropped)
    const T ea = ra < rc2 ? rho_of(ra) : (T)0, eb = rb < rc2 ? rho_of(rb) : (T)0;
    p[0] = pk_add(p[0], pk_make(ea, eb));
  }
};

template <typename T, bool EV>
struct EamTabForceBody {
  static constexpr int NT = EV ? 10 : 3;
  using PK = typename Pk<T>::type;
  using V4 = typename Vec4<T>::type;
  static __device__ __forceinline__ T own_w(T w) { return -w; }
  static __device__ __forceinline__ T mutual_w(T a, T b) { return a + b; }
  static __device__ __forceinline__ T cell_own_w(T w) { return w; }
  template <class TAB> __device__ __forceinline__ void attach(TAB*) {}
  static constexpr bool TABLE = false;
  T rc2;
  TabLookup<T> L;
  const void *tab_rho, *tab_phi;
  unsigned s_rho = 0, s_phi = 0;   // shared-memory addresses of the staged tables, 0: not staged
  static constexpr int SMEM_TABLES = 2;
  __device__ __forceinline__ void attach_tables(unsigned base, unsigned table_bytes) { s_rho = base; s_phi = base ? base + table_bytes : 0u; }
  __device__ explicit EamTabForceBody(const PairParams& P)
      : rc2(MDK_PP(rc2)), L{(T)P.inv_dr, P.tab_nr - 2}, tab_rho(P.tab_rho), tab_phi(P.tab_phi) {}
  // fpair = -[ (F'_i + F'_j) rho'(r) + phi'(r) ] / r and phi(r) of one term; zero beyond the cutoff
  __device__ __forceinline__ void term(T r2, T wsum, T& fp, T& phi) const {
    const bool in = r2 < rc2;
    const T rinv = t_rsqrt<T>(r2);
    T u;
    const int k = L.interval(r2 * rinv, u);
    const V4 cr = TabLookup<T>::load(tab_rho, s_rho, k), cp = TabLookup<T>::load(tab_phi, s_phi, k);
    fp = in ? -(wsum * L.slope(cr, u) + L.slope(cp, u)) * rinv : (T)0;
    phi = in ? TabLookup<T>::value(cp, u) : (T)0;
  }
  __device__ __forceinline__ void pair(T dx, T dy, T dz, T r2, T wsum, bool ok, T (&p)[NT]) const {
    T fp, phi;
    term(r2, wsum, fp, phi);
    if (!ok) { fp = (T)0; phi = (T)0; }
    p[0] += fp * dx; p[1] += fp * dy; p[2] += fp * dz;
    if constexpr (EV) {
      p[3] += phi;
      p[4] += dx * dx * fp; p[5] += dy * dy * fp; p[6] += dz * dz * fp;
      p[7] += dx * dy * fp; p[8] += dx * dz * fp; p[9] += dy * dz * fp;
    }
  }
  __device__ __forceinline__ void pair2(PK dx, PK dy, PK dz, PK r2, PK wsum, PK (&p)[NT]) const {
    T fa, fb, pa, pb;
    term(pk_lo(r2), pk_lo(wsum), fa, pa);
    term(pk_hi(r2), pk_hi(wsum), fb, pb);
    const PK fp = pk_make(fa, fb);
    p[0] = pk_fma(fp, dx, p[0]); p[1] = pk_fma(fp, dy, p[1]); p[2] = pk_fma(fp, dz, p[2]);
    if constexpr (EV) {
      p[3] = pk_add(p[3], pk_make(pa, pb));
      virial2(dx, dy, dz, fp, p);
    }
  }
};

// Buckingham + cutoff Coulomb (App. A, LAMMPS style buck/coul/cut):
//   u_ab(r) = A_ab exp(-r/rho_ab) - C_ab / r^6 + k q_a q_b / r,  r^2 < rc^2;  F_i = fpair D,
//   fpair = [ (A/rho) r exp(-r/rho) - 6 C / r^6 + k q_a q_b / r ] / r^2.
// The type of an atom travels in the w component of its staged record; the row's own atoms carry -4 t_i, so the
// list loop hands pair2 the value -(4 t_i + t_j): the index of the type pair's coefficients in a 16-entry table
// in shared memory (one 128-bit load per atom of the row and list entry; 256 bits in fp64).
template <typename T, bool EV>
struct BuckCoulBody {
  static constexpr int NT = EV ? 10 : 3;
  using PK = typename Pk<T>::type;
  using V4 = typename Vec4<T>::type;
  static constexpr bool TABLE = true;
  static constexpr int SMEM_TABLES = 0;   // no coefficient tables to stage (tabulated EAM has)
  __device__ __forceinline__ void attach_tables(unsigned, unsigned) {}
  static __device__ __forceinline__ T own_w(T w) { return (T)(-MAX_PAIR_TYPES) * w; }
  static __device__ __forceinline__ T mutual_w(T a, T b) { return a + b * (T)(1.0 / MAX_PAIR_TYPES); }   // -(4 t0 + t1)
  static __device__ __forceinline__ T cell_own_w(T w) { return (T)MAX_PAIR_TYPES * w; }
  T rc2;
  const V4* tab = nullptr;
  __device__ explicit BuckCoulBody(const PairParams& P) : rc2(MDK_PP(rc2)) {}
  // fills the shared-memory table (all threads of the block call it; the caller synchronises before the first use)
  __device__ __forceinline__ void attach(V4* t) { tab = t; }
  static __device__ __forceinline__ void fill(const PairParams& P, V4* t) {
    for (int k = threadIdx.x; k < MAX_PAIR_TYPES * MAX_PAIR_TYPES; k += blockDim.x)
      t[k] = make_v4<T>((T)P.bc[k][0], (T)P.bc[k][1], (T)P.bc[k][2], (T)P.bc[k][3]);
  }
  __device__ __forceinline__ V4 coef(T w) const {
    int k = (int)((w < (T)0 ? -w : w) + (T)0.25);                      // |w| = 4 t_i + t_j exactly; the quarter guards the cast
    k = k < MAX_PAIR_TYPES * MAX_PAIR_TYPES ? k : 0;                   // pad and dummy entries carry any w: they are out of range anyway
    return tab[k];
  }
  __device__ __forceinline__ void pair(T dx, T dy, T dz, T r2, T wsum, bool ok, T (&p)[NT]) const {
    const bool in = ok && r2 < rc2;
    const V4 c = coef(wsum);
    const T rinv = t_rsqrt<T>(r2), r = r2 * rinv, r2i = rinv * rinv, r6i = r2i * r2i * r2i;
    const T ex = c.x * t_exp<T>(-r * c.y);
    const T fp = in ? (ex * r * c.y - (T)6 * c.z * r6i + c.w * rinv) * r2i : (T)0;
    p[0] += fp * dx; p[1] += fp * dy; p[2] += fp * dz;
    if constexpr (EV) {
      p[3] += in ? ex - c.z * r6i + c.w * rinv : (T)0;
      p[4] += dx * dx * fp; p[5] += dy * dy * fp; p[6] += dz * dz * fp;
      p[7] += dx * dy * fp; p[8] += dx * dz * fp; p[9] += dy * dz * fp;
    }
  }
  // 1/r := 0 beyond the cutoff zeroes the Coulomb term and, through 1/r^2, the whole force factor; the energy is masked
  __device__ __forceinline__ void pair2(PK dx, PK dy, PK dz, PK r2, PK wsum, PK (&p)[NT]) const {
    const T ra = pk_lo(r2), rb = pk_hi(r2);
    const V4 ca = coef(pk_lo(wsum)), cb = coef(pk_hi(wsum));
    const bool ina = ra < rc2, inb = rb < rc2;
    const T ia = t_rsqrt<T>(ra), ib = t_rsqrt<T>(rb);
    const PK r = pk_mul(r2, pk_make(ia, ib));
    const PK irho = pk_make(ca.y, cb.y);
    const PK arg = pk_mul(r, irho);
    const PK ex = pk_mul(pk_make(ca.x, cb.x), pk_make(t_exp<T>(-pk_lo(arg)), t_exp<T>(-pk_hi(arg))));
    const PK rinv = pk_make(ina ? ia : (T)0, inb ? ib : (T)0);
    const PK r2i = pk_mul(rinv, rinv);
    const PK r6i = pk_mul(pk_mul(r2i, r2i), r2i);
    const PK c6 = pk_mul(pk_make(ca.z, cb.z), r6i), coul = pk_mul(pk_make(ca.w, cb.w), rinv);
    // (A/rho) r e^{-r/rho} - 6 C/r^6 + kqq/r, times 1/r^2 (zero beyond the cutoff)
    const PK fp = pk_mul(pk_fma(pk_mul(ex, arg), pk_splat<T>((T)1), pk_fma(pk_splat<T>((T)-6), c6, coul)), r2i);
    p[0] = pk_fma(fp, dx, p[0]); p[1] = pk_fma(fp, dy, p[1]); p[2] = pk_fma(fp, dz, p[2]);
    if constexpr (EV) {
      const PK m = pk_make(ina ? (T)1 : (T)0, inb ? (T)1 : (T)0);
      p[3] = pk_fma(m, pk_add(pk_sub(ex, c6), coul), p[3]);
      virial2(dx, dy, dz, fp, p);
    }
  }
};

// ---------------------------------------------------------------------------------------------------
// a5/a6/a7 (+ a8, a4 fused): arguments shared by the force kernels
// ---------------------------------------------------------------------------------------------------
constexpr int EPI_FORCES = 0;      // write f[i] (md_compute_forces; first evaluation of a run)
constexpr int EPI_KICK_DRIFT = 1;  // v += dtf f; then next step's first half: v += dtf f; x' = x + dt v; max |x'-x0|^2
constexpr int EPI_FINAL = 2;       // v += dtf f; write f[i] (last step of a run)

struct ForceArgs {
  Geom g;
  PairParams P;
  const int* cell_start;
  const int* tab;          // per-tile tables of the last build (k_tile_tables)
  const double* x; size_t ld;
  const void* xr;          // packed cell-relative positions (Vec4<T>) of the positions in x; .w = -F'(rho) for EAM pass 2
  void* xr_new;            // EPI_KICK_DRIFT: packed copy of x_new
  const uint4* list;
  const int* numneigh;
  const double* fp_in;     // EAM pass 2, cell-list variant only: F'(rho) per sorted atom (else NULL)
  double* f;               // forces out
  double* rho; double* fp_out;   // EAM pass 1 out
  double* ev_partials;     // [ntiles][8]: e, wxx, wyy, wzz, wxy, wxz, wyz, pad
  // time stepping (a8) and the displacement test (a4), fused into the epilogue
  int epi;                 // EPI_*
  int in_run;              // 1: the launch belongs to a batch of steps: do nothing if the list is stale
  int parity;              // reads max_disp2_bits[parity], writes max_disp2_bits[1-parity]
  double* v; double* x_new; const double* x0;
  const int* type; const double* mass;
  const double* dtf_type;  // [ntypes]: half_dt_ftm2v / mass[t] (host-prepared per md_run)
  int tab_smem_bytes;      // tabulated EAM in k_tile_force_p: bytes of ONE coefficient table staged behind the tile buffers (0: none)
  double dt, half_dt_ftm2v, trigger;
  Flags* flags;
};

// Programmatic dependent launch (step kernels inside md_run are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization): the next launch of the stream may be set up and its blocks
// scheduled while this grid is still running; nothing the previous grid wrote may be read before pdl_wait().  Both are
// no-ops in a launch without the attribute.
__device__ __forceinline__ void pdl_wait_then_release() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

// true if this launch must do nothing: an earlier step of the batch moved some atom farther than
// skin/2 from its position at the last build, so the host has to rebuild first (reading s4).
__device__ __forceinline__ bool list_is_stale(const ForceArgs& A) {
  if (!A.in_run) return false;
  const double d2 = __longlong_as_double((long long)A.flags->max_disp2_bits[A.parity]);
  // the build before this batch is judged here too (md_run does not wait for it): a tile or row that outgrew its
  // capacity, or a non-finite coordinate, stops the batch before its first step
  const bool bad_build = A.flags->need_tile_cap > A.g.tile_cap || A.flags->need_interior_cap > A.g.interior_cap ||
                         A.flags->need_row_cap > A.g.row_cap || A.flags->nonfinite != 0;
  const bool stale = A.flags->stop != 0 || d2 > A.trigger || bad_build;
  if (stale && threadIdx.x == 0 && blockIdx.x == 0) atomicExch(&A.flags->stop, 1);
  return stale;
}

// per-atom epilogue; returns |x'-x0|^2 for EPI_KICK_DRIFT (else 0).  cc[3]: centre of the cell the atom is
// stored in (for the packed copy of the new position).
template <typename T>
__device__ __forceinline__ double atom_epilogue(const ForceArgs& A, int gi, const double (&tot)[3], const double (&cc)[3]) {
  const size_t ld = A.ld;
  if (A.epi == EPI_FORCES) {
    A.f[gi] = tot[0]; A.f[ld + gi] = tot[1]; A.f[2 * ld + gi] = tot[2];
    return 0.0;
  }
  // all loads first: the arrays may alias as far as the compiler knows, so a store between two loads would
  // serialise three memory round trips
  double vv[3], xx[3] = {0.0, 0.0, 0.0}, x0v[3] = {0.0, 0.0, 0.0};
#pragma unroll
  for (int d = 0; d < 3; ++d) vv[d] = A.v[d * ld + gi];
  if (A.epi == EPI_KICK_DRIFT) {
#pragma unroll
    for (int d = 0; d < 3; ++d) { xx[d] = A.x[d * ld + gi]; x0v[d] = A.x0[d * ld + gi]; }
  }
  const int ty = A.type[gi];
  const double dtf = A.dtf_type[ty];   // dt/2 ftm2v / m of the atom's type (a tiny table, L1-resident)
  double d2 = 0.0;
  T r[3];
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    vv[d] += dtf * tot[d];                                  // second half kick of this step
    if (A.epi == EPI_KICK_DRIFT) {
      vv[d] += dtf * tot[d];                                // first half kick of the next step
      xx[d] += A.dt * vv[d];                                // drift
      r[d] = (T)(xx[d] - cc[d]);
      const double dd = xx[d] - x0v[d];
      d2 += dd * dd;
    }
  }
  if (A.epi == EPI_KICK_DRIFT) {
#pragma unroll
    for (int d = 0; d < 3; ++d) { A.x_new[d * ld + gi] = xx[d]; A.v[d * ld + gi] = vv[d]; }
    reinterpret_cast<typename Vec4<T>::type*>(A.xr_new)[gi] = make_v4<T>(r[0], r[1], r[2], (T)ty);
  } else {
#pragma unroll
    for (int d = 0; d < 3; ++d) { A.f[d * ld + gi] = tot[d]; A.v[d * ld + gi] = vv[d]; }
  }
  return d2;
}

// per-pair epilogue: the two atoms gi and gi + 1 (the second only if act1); returns max |x'-x0|^2 for
// EPI_KICK_DRIFT (else 0).  WIDE = false: one atom after the other (both at once would need 36 more live registers
// than the 56-register kernels have); WIDE = true (k_tile_force_p, 72 registers): all loads of both atoms first.
template <typename T, bool WIDE>
__device__ __forceinline__ double atom_epilogue2(const ForceArgs& A, int gi, bool act1, const double (&ta)[3], const double (&tb)[3],
                                                 const double (&cc)[3]) {
  if constexpr (!WIDE) {
    double d2 = atom_epilogue<T>(A, gi, ta, cc);
    if (act1) d2 = fmax(d2, atom_epilogue<T>(A, gi + 1, tb, cc));
    return d2;
  } else {
    const size_t ld = A.ld;
    if (A.epi == EPI_FORCES) {
      A.f[gi] = ta[0]; A.f[ld + gi] = ta[1]; A.f[2 * ld + gi] = ta[2];
      if (act1) { A.f[gi + 1] = tb[0]; A.f[ld + gi + 1] = tb[1]; A.f[2 * ld + gi + 1] = tb[2]; }
      return 0.0;
    }
    const int g1 = act1 ? gi + 1 : gi;
    double va[3], vb[3], xa[3] = {0.0, 0.0, 0.0}, xb[3] = {0.0, 0.0, 0.0}, x0a[3] = {0.0, 0.0, 0.0}, x0b[3] = {0.0, 0.0, 0.0};
    const int tya = A.type[gi], tyb = A.type[g1];
#pragma unroll
    for (int d = 0; d < 3; ++d) { va[d] = A.v[d * ld + gi]; vb[d] = A.v[d * ld + g1]; }
    if (A.epi == EPI_KICK_DRIFT) {
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        xa[d] = A.x[d * ld + gi]; xb[d] = A.x[d * ld + g1];
        x0a[d] = A.x0[d * ld + gi]; x0b[d] = A.x0[d * ld + g1];
      }
    }
    const double dtfa = A.dtf_type[tya], dtfb = A.dtf_type[tyb];
    double d2a = 0.0, d2b = 0.0;
    T ra[3], rb[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      va[d] += dtfa * ta[d];                                  // second half kick of this step
      vb[d] += dtfb * tb[d];
      if (A.epi == EPI_KICK_DRIFT) {
        va[d] += dtfa * ta[d];                                // first half kick of the next step
        vb[d] += dtfb * tb[d];
        xa[d] += A.dt * va[d];                                // drift
        xb[d] += A.dt * vb[d];
        ra[d] = (T)(xa[d] - cc[d]);
        rb[d] = (T)(xb[d] - cc[d]);
        const double da = xa[d] - x0a[d], db = xb[d] - x0b[d];
        d2a += da * da;
        d2b += db * db;
      }
    }
    if (A.epi == EPI_KICK_DRIFT) {
#pragma unroll
      for (int d = 0; d < 3; ++d) { A.x_new[d * ld + gi] = xa[d]; A.v[d * ld + gi] = va[d]; }
      reinterpret_cast<typename Vec4<T>::type*>(A.xr_new)[gi] = make_v4<T>(ra[0], ra[1], ra[2], (T)tya);
      if (act1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) { A.x_new[d * ld + gi + 1] = xb[d]; A.v[d * ld + gi + 1] = vb[d]; }
        reinterpret_cast<typename Vec4<T>::type*>(A.xr_new)[gi + 1] = make_v4<T>(rb[0], rb[1], rb[2], (T)tyb);
      }
    } else {
#pragma unroll
      for (int d = 0; d < 3; ++d) { A.f[d * ld + gi] = ta[d]; A.v[d * ld + gi] = va[d]; }
      if (act1) {
#pragma unroll
        for (int d = 0; d < 3; ++d) { A.f[d * ld + gi + 1] = tb[d]; A.v[d * ld + gi + 1] = vb[d]; }
      }
    }
    return act1 ? fmax(d2a, d2b) : d2a;
  }
}

// ---------------------------------------------------------------------------------------------------
// staged-tile gathers: the "random access" load of atom j is ONE 128-bit shared-memory
// load (two for fp64) of {x, y, z, w} in tile-centred coordinates; w holds -F'(rho_j) in EAM pass 2.
// Measured on B200 (random slots, 32 lanes): LDS.128 from AoS 11.0 SM-cycles per warp-gather, two
// LDS.64 from split arrays 12.9, two LDS.64 from AoS 17.0.
// ---------------------------------------------------------------------------------------------------
template <typename T> __device__ __forceinline__ typename Vec4<T>::type lds_v4(unsigned a);
template <> __device__ __forceinline__ float4 lds_v4<float>(unsigned a) {
  float4 r;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "r"(a));
  return r;
}
template <> __device__ __forceinline__ double4 lds_v4<double>(unsigned a) {
  double4 r;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(r.x), "=d"(r.y) : "r"(a));
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2+16];" : "=d"(r.z), "=d"(r.w) : "r"(a));
  return r;
}

// One staged record loaded component by component (four scalar loads): for the row's OWN two atoms, whose
// coordinates are then free to sit in whatever registers the packed pairs {x0, x1}, {y0, y1}, {z0, z1} need
// (after a 128-bit load they are pinned to an aligned quad, and ptxas rebuilds each pair with two moves per use).
template <typename T> __device__ __forceinline__ typename Vec4<T>::type lds_v4_scalars(unsigned a);
template <> __device__ __forceinline__ float4 lds_v4_scalars<float>(unsigned a) {
  float4 r;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r.x) : "r"(a));
  asm volatile("ld.shared.f32 %0, [%1+4];" : "=f"(r.y) : "r"(a));
  asm volatile("ld.shared.f32 %0, [%1+8];" : "=f"(r.z) : "r"(a));
  asm volatile("ld.shared.f32 %0, [%1+12];" : "=f"(r.w) : "r"(a));
  return r;
}
template <> __device__ __forceinline__ double4 lds_v4_scalars<double>(unsigned a) { return lds_v4<double>(a); }

// TMA 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void mbar_init(unsigned mbar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned mbar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(unsigned dst, const void* src, unsigned bytes, unsigned mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src), "r"(bytes),
               "r"(mbar)
               : "memory");
}
__device__ __forceinline__ bool mbar_test(unsigned mbar, unsigned parity) {   // has the phase of this parity completed? (does not block)
  unsigned ok = 0;
  asm volatile("{ .reg .pred p; mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
               : "=r"(ok)
               : "r"(mbar), "r"(parity)
               : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned mbar, unsigned parity) {
  unsigned ok = 0;
  while (!ok)
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok)
                 : "r"(mbar), "r"(parity)
                 : "memory");
}

// ---------------------------------------------------------------------------------------------------
// the neighbor-list loop of PAPER.md L88-122 for one (pair row, lane): walks this lane's 128-bit words,
// 8 entries each; each entry is a slot code (slot << code_shift; the staged record sits at
// st_base + 2 * code) and is evaluated against BOTH atoms of the pair (pi0, pi1) with two-wide math.
// w of the staged atoms holds -F'(rho_j) for EAM pass 2, so pw - jw = F'_i + F'_j.
// ---------------------------------------------------------------------------------------------------
template <typename T, class Body>
__device__ __forceinline__ void list_loop(const Body& body, unsigned st_base, const uint4* __restrict__ words, size_t word_stride,
                                          int nwords, typename Vec4<T>::type pi0, typename Vec4<T>::type pi1, double (&tot0)[Body::NT],
                                          double (&tot1)[Body::NT], uint4 w0, bool have_w0) {
  constexpr int NT = Body::NT;
  using PK = typename Pk<T>::type;
  if (nwords <= 0) return;
  // two words in flight ahead of the one being processed: a word is 8 gathers x 2 atoms = ~230 issue slots of work
  // for the warp, but with only a few of the SM's warps inside this loop at a time that is less than a DRAM round
  // trip (measured: with one word ahead, 16 % of the loop's stall samples wait for the next word)
  uint4 w = have_w0 ? w0 : ld_stream(words);
  uint4 wn = w;
  if (nwords > 1) wn = ld_stream(words + word_stride);
  const PK xi = pk_make_once(pi0.x, pi1.x), yi = pk_make_once(pi0.y, pi1.y), zi = pk_make_once(pi0.z, pi1.z), wi = pk_make(pi0.w, pi1.w);
  for (int c = 0; c < nwords; ++c) {
    const uint4 cur = w;
    w = wn;
    if (c + 2 < nwords) wn = ld_stream(words + (size_t)(c + 2) * word_stride);
    PK p[NT];
#pragma unroll
    for (int k = 0; k < NT; ++k) p[k] = pk_splat<T>((T)0);
    const unsigned ww[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
    for (int h = 0; h < 4; ++h) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const unsigned code = u ? (ww[h] >> 16) : (ww[h] & 0xffffu);
        const typename Vec4<T>::type pj = lds_v4<T>(st_base + 2u * code);
        const PK dx = pk_sub(xi, pk_splat<T>(pj.x)), dy = pk_sub(yi, pk_splat<T>(pj.y)), dz = pk_sub(zi, pk_splat<T>(pj.z));
        const PK r2 = pk_fma(dz, dz, pk_fma(dy, dy, pk_mul(dx, dx)));
        body.pair2(dx, dy, dz, r2, pk_sub(wi, pk_splat<T>(pj.w)), p);
      }
    }
#pragma unroll
    for (int k = 0; k < NT; ++k) { tot0[k] += (double)pk_lo(p[k]); tot1[k] += (double)pk_hi(p[k]); }
  }
}

// ---------------------------------------------------------------------------------------------------
// a5/a6/a7: the tile force kernel over the Verlet list of PAIR ROWS.
//   MODE 0: forces (LJ or EAM pass 2) + epilogue A.epi (+ per-block energy/virial partials when EV)
//   MODE 1: EAM pass 1 -> rho[N], fp[N] = F'(rho), packed w = -F'(rho) (+ embedding energy partial when EV)
//   HALF (K = 1): each pair once, the term on j scattered with fp64 atomics (forces -F; density: the same rho term);
//         EPI_FORCES only, the unfused integrator kernels do the time stepping.
// Thread <-> (pair row r = interior slots 2r, 2r+1; lane s of K).  Block size is chosen by the host so that the
// tile's rows fill whole rounds of the block.
// Staging: the tile's cells (interior + one-cell halo) are contiguous runs of the packed array, so each
// is ONE TMA bulk copy (cp.async.bulk, <= 216 per tile, all in flight at once, one mbarrier); a second
// pass in shared memory adds each cell's offset from the tile centre (periodic image included).
// Shared memory: TileTables | st[capA] Vec4<T> | offs[tile cells] Vec4<T> | scell[interior_cap] u16 | qcell[quads] u16 | (HALF: sgid[capA] int)
// ---------------------------------------------------------------------------------------------------
__host__ __device__ inline int force_capA(const Geom& g) { return (g.tile_cap + 8) & ~3; }
constexpr int FORCE_MAX_REGS = 56;   // three 384-thread blocks (or one 1024-thread block) per SM

template <typename T, class Body, int K, int MODE, bool EV, bool HALF>
__global__ void __maxnreg__((EV || sizeof(T) == 8) ? 96 : FORCE_MAX_REGS) k_tile_force(ForceArgs A) {
  using V4 = typename Vec4<T>::type;
  using PK = typename Pk<T>::type;
  constexpr int NT = Body::NT;
  pdl_wait_then_release();
  if (list_is_stale(A)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  const Geom& g = A.g;
  const int capA = force_capA(g);
  V4* st = reinterpret_cast<V4*>(smem_raw + sizeof(TileTables));
  V4* offs = st + capA;                                           // per tile cell: offset of its atoms from the tile centre
  unsigned short* scell = reinterpret_cast<unsigned short*>(offs + tile_tab_cells(g));
  unsigned short* qcell = scell + g.interior_cap;                 // per quad of staged slots: its tile cell
  int* sgid = reinterpret_cast<int*>(qcell + ((tile_tab_quads(g) + 7) & ~7));   // HALF only
  __shared__ double red[8 * 32];
  __shared__ __align__(8) unsigned long long mbar_storage;
  const unsigned mbar = smem_addr(&mbar_storage);
  const int tileid = blockIdx.x;
  if (threadIdx.x == 0) mbar_init(mbar, 1);
  __shared__ __align__(16) unsigned char pair_tab[Body::TABLE ? MAX_PAIR_TYPES * MAX_PAIR_TYPES * sizeof(V4) : 16];   // per-type-pair coefficients
  if constexpr (Body::TABLE) Body::fill(A.P, reinterpret_cast<V4*>(pair_tab));
  tile_load(g, tileid, A.tab, tt);
  const int pcap = prow_cap(g);
  const unsigned st_base = smem_addr(st);
  int n_first = 0;
  uint4 w_first = make_uint4(0, 0, 0, 0);
  {
    const V4* __restrict__ xr = reinterpret_cast<const V4*>(A.xr);
    const int* __restrict__ htab = A.tab + (size_t)tileid * tile_tab_stride(g);
    if (threadIdx.x == 0) mbar_expect_tx(mbar, (unsigned)htab[4] * (unsigned)sizeof(V4));
    for (int t = threadIdx.x; t < tt.ntc; t += blockDim.x) {
      const int c = tt.cnt[t];
      if (c > 0) bulk_g2s(st_base + (unsigned)tt.start[t] * (unsigned)sizeof(V4), xr + tt.gstart[t], (unsigned)c * (unsigned)sizeof(V4), mbar);
      double offd[3];
      tile_cell_offset_rel(g, tt, t, offd);
      offs[t] = make_v4<T>((T)offd[0], (T)offd[1], (T)offd[2], (T)0);
    }
    // while the bulk copies fly: this thread's row length and first list word of the first round, ...
    if constexpr (!HALF) {
      if ((int)threadIdx.x < pcap * K) {
        n_first = A.numneigh[(size_t)tileid * pcap + threadIdx.x / K];
        w_first = ld_stream(A.list + (size_t)tileid * g.chunk_cap * ((size_t)pcap * K) + threadIdx.x);
      }
    }
    // ... and the quad -> tile cell map of this tile
    const int nq = tt.n_slots >> 2;
    {
      const unsigned* __restrict__ qsrc = reinterpret_cast<const unsigned*>(htab + TILE_HDR + TILE_CELL_INTS * tile_tab_cells(g));
      unsigned* qdst = reinterpret_cast<unsigned*>(qcell);
      for (int k = threadIdx.x; k < (nq + 1) >> 1; k += blockDim.x) qdst[k] = qsrc[k];
    }
    __syncthreads();
    mbar_wait(mbar, 0);
    // offsets, pad slots, slot -> cell map: one thread per quad of slots
    for (int q = threadIdx.x; q < nq; q += blockDim.x) {
      const int t = qcell[q];
      const int c = tt.cnt[t], k0 = 4 * q - tt.start[t];
      const V4 o = offs[t];
      const bool interior = (tt.meta[t] >> 24) != 0;
      unsigned sc[2] = {0xffffffffu, 0xffffffffu};
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int slot = 4 * q + u;
        if (k0 + u < c) {
          V4 v = st[slot];
          v.x += o.x; v.y += o.y; v.z += o.z;
          st[slot] = v;
          sc[u >> 1] = (u & 1) ? ((sc[u >> 1] & 0xffffu) | ((unsigned)t << 16)) : ((sc[u >> 1] & 0xffff0000u) | (unsigned)t);
        } else {
          st[slot] = make_v4<T>((T)1e15, (T)1e15, (T)1e15, (T)0);
        }
        if constexpr (HALF) sgid[slot] = k0 + u < c ? tt.gstart[t] + k0 + u : 0;
      }
      if (interior) {   // indexed by interior slot; a pair of slots is one list row (the cell's rows are padded to 2, not 4)
        unsigned* sp = reinterpret_cast<unsigned*>(scell + tt.rstart[t] + k0);
        if (k0 < c) sp[0] = sc[0];
        if (k0 + 2 < c) sp[1] = sc[1];
      }
    }
    if (threadIdx.x == 0) st[tt.n_slots] = make_v4<T>((T)1e15, (T)1e15, (T)1e15, (T)0);   // the dummy slot
  }
  __syncthreads();
  Body body(A.P);
  body.attach(reinterpret_cast<V4*>(pair_tab));
  const size_t ld = A.ld;
  const size_t slots_cap = (size_t)pcap * K;
  const uint4* tlist = A.list + (size_t)tileid * g.chunk_cap * slots_cap;
  double ev[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  double d2max = 0.0;
  const int nlanes = (tt.n_int_slots >> 1) * K;
  for (int base = 0; base < nlanes; base += blockDim.x) {   // uniform trip count: the shuffles below need full groups
    const int sidx = base + threadIdx.x;
    const int r = sidx / K, s = sidx % K;                   // pair row, lane of the row
    unsigned cells = 0xffffffffu;
    if (sidx < nlanes) cells = reinterpret_cast<const unsigned*>(scell)[r];
    const unsigned cell = cells & 0xffffu;
    const bool act0 = cell != 0xffffu, act1 = (cells >> 16) != 0xffffu;   // the pair's atoms (act1 implies act0)
    const int kin = act0 ? 2 * r - tt.rstart[cell] : 0;     // index of the first atom within its cell
    const int gi = act0 ? tt.gstart[cell] + kin : 0;        // the second atom is gi + 1
    double tot0[NT], tot1[NT];
#pragma unroll
    for (int k = 0; k < NT; ++k) { tot0[k] = 0.0; tot1[k] = 0.0; }
    if (act0) {
      const int slot0 = tt.start[cell] + kin;
      V4 pi0 = lds_v4_scalars<T>(st_base + (unsigned)slot0 * (unsigned)sizeof(V4));
      V4 pi1 = lds_v4_scalars<T>(st_base + (unsigned)(slot0 + 1) * (unsigned)sizeof(V4));   // a pad slot if there is no partner: far from everything
      if (!act1) { pi1.x = (T)-1e15; pi1.y = (T)-1e15; pi1.z = (T)-1e15; pi1.w = (T)0; }    // ... and from the dummy slot too
      pi0.w = Body::own_w(pi0.w); pi1.w = Body::own_w(pi1.w);
      const int n = (!HALF && base == 0) ? n_first : A.numneigh[(size_t)tileid * pcap + r];
      const int nq = (n + 7) >> 3;                          // words of this row
      if (act1 && s == 0) {
        // the pair's mutual term (the two atoms are never entries of their own row)
        PK p[NT];
#pragma unroll
        for (int k = 0; k < NT; ++k) p[k] = pk_splat<T>((T)0);
        const T ex = pi0.x - pi1.x, ey = pi0.y - pi1.y, ez = pi0.z - pi1.z;
        const T r2 = ex * ex + ey * ey + ez * ez;
        body.pair2(pk_make(ex, -ex), pk_make(ey, -ey), pk_make(ez, -ez), pk_splat<T>(r2), pk_splat<T>(Body::mutual_w(pi0.w, pi1.w)), p);
#pragma unroll
        for (int k = 0; k < NT; ++k) {
          tot0[k] += (double)pk_lo(p[k]);
          if (!(HALF && MODE == 0 && k >= 3)) tot1[k] += (double)pk_hi(p[k]);   // a half list counts the pair's energy and virial once
        }
      }
      if constexpr (!HALF) {
        if constexpr (MODE == 0) {
          if (A.epi != EPI_FORCES) {   // the epilogue's operands: start them towards L2 now (a 32-byte sector holds both atoms')
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.type + gi));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.v + gi));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.v + ld + gi));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.v + 2 * ld + gi));
            if (A.epi == EPI_KICK_DRIFT) {
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x + ld + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x + 2 * ld + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x0 + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x0 + ld + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x0 + 2 * ld + gi));
            }
          }
        }
#ifdef MDK_SKIP_LOOP   // timing experiment: everything but the list loop
        const int mine = 0;
#else
        const int mine = nq > s ? (nq - s + K - 1) / K : 0;   // words q = s, s+K, ...
#endif
        list_loop<T, Body>(body, st_base, tlist + sidx, slots_cap, mine, pi0, pi1, tot0, tot1, w_first, base == 0);
      } else {
        // half list: each in-range pair once; the term of i (registers), the term of j (atomics)
        for (int c = 0; c < nq; ++c) {
          const uint4 cur = tlist[(size_t)c * slots_cap + sidx];
          const unsigned ww[4] = {cur.x, cur.y, cur.z, cur.w};
#pragma unroll
          for (int h = 0; h < 4; ++h)
#pragma unroll
            for (int u = 0; u < 2; ++u) {
              const unsigned code = u ? (ww[h] >> 16) : (ww[h] & 0xffffu);
              const V4 pj = lds_v4<T>(st_base + 2u * code);
              const PK dx = pk_make(pi0.x - pj.x, pi1.x - pj.x), dy = pk_make(pi0.y - pj.y, pi1.y - pj.y), dz = pk_make(pi0.z - pj.z, pi1.z - pj.z);
              const PK r2 = pk_fma(dz, dz, pk_fma(dy, dy, pk_mul(dx, dx)));
              PK p[NT];
#pragma unroll
              for (int k = 0; k < NT; ++k) p[k] = pk_splat<T>((T)0);
              body.pair2(dx, dy, dz, r2, pk_make(pi0.w - pj.w, pi1.w - pj.w), p);
              const int gj = sgid[code >> g.code_shift];
              if constexpr (MODE == 0) {
                const T sx = pk_lo(p[0]) + pk_hi(p[0]), sy = pk_lo(p[1]) + pk_hi(p[1]), sz = pk_lo(p[2]) + pk_hi(p[2]);
                if (sx != (T)0 || sy != (T)0 || sz != (T)0) {
                  atomicAdd(&A.f[gj], -(double)sx);
                  atomicAdd(&A.f[ld + gj], -(double)sy);
                  atomicAdd(&A.f[2 * ld + gj], -(double)sz);
                }
              } else {
                const T sr = pk_lo(p[0]) + pk_hi(p[0]);     // rho is symmetric: j receives what i0 and i1 receive
                if (sr != (T)0) atomicAdd(&A.rho[gj], (double)sr);
              }
#pragma unroll
              for (int k = 0; k < NT; ++k) { tot0[k] += (double)pk_lo(p[k]); tot1[k] += (double)pk_hi(p[k]); }
            }
        }
      }
    }
    if constexpr (K > 1) {
#pragma unroll
      for (int k = 0; k < NT; ++k) { tot0[k] = group_sum<K>(tot0[k]); tot1[k] = group_sum<K>(tot1[k]); }
    }
    if (act0 && s == 0) {
      if constexpr (MODE == 0) {
        if constexpr (HALF) {
          atomicAdd(&A.f[gi], tot0[0]); atomicAdd(&A.f[ld + gi], tot0[1]); atomicAdd(&A.f[2 * ld + gi], tot0[2]);
          if (act1) { atomicAdd(&A.f[gi + 1], tot1[0]); atomicAdd(&A.f[ld + gi + 1], tot1[1]); atomicAdd(&A.f[2 * ld + gi + 1], tot1[2]); }
        } else {
          double cc[3] = {0.0, 0.0, 0.0};
          if (A.epi == EPI_KICK_DRIFT) {
            const int m = tt.meta[cell];
            const int tq[3] = {m & 0xff, (m >> 8) & 0xff, (m >> 16) & 0xff};
#pragma unroll
            for (int d = 0; d < 3; ++d) cc[d] = cell_anchor_1d(g, d, tt.c0[d] + tq[d] - 1);
          }
          const double ta[3] = {tot0[0], tot0[1], tot0[2]}, tb[3] = {tot1[0], tot1[1], tot1[2]};
          d2max = fmax(d2max, atom_epilogue2<T, false>(A, gi, act1, ta, tb, cc));
        }
        if constexpr (EV) {
          const double wgt = HALF ? 1.0 : 0.5;   // a full list visits every pair twice
#pragma unroll
          for (int k = 0; k < 7; ++k) ev[k] += wgt * (tot0[3 + k] + (act1 ? tot1[3 + k] : 0.0));
        }
      } else {
        if constexpr (HALF) {
          atomicAdd(&A.rho[gi], tot0[0]);
          if (act1) atomicAdd(&A.rho[gi + 1], tot1[0]);
        } else {
#pragma unroll
          for (int a = 0; a < 2; ++a) {
            if (a == 1 && !act1) break;
            const double rho = a ? tot1[0] : tot0[0];
            double Fv, fpv;
            eam_embed(A.P, rho, Fv, fpv);
            A.rho[gi + a] = rho;
            A.fp_out[gi + a] = fpv;
            reinterpret_cast<T*>(const_cast<void*>(A.xr))[4 * (size_t)(gi + a) + 3] = (T)(-fpv);   // read back as pj.w by pass 2
            if constexpr (EV) ev[0] += Fv;                           // embedding energy F(rho_i)
          }
        }
      }
    }
  }
  if constexpr (EV) {
    block_sum<8>(ev, red);
    if (threadIdx.x == 0)
#pragma unroll
      for (int k = 0; k < 8; ++k) A.ev_partials[(size_t)tileid * 8 + k] = ev[k];
  }
  if constexpr (MODE == 0 && !HALF) {
    if (A.epi == EPI_KICK_DRIFT) {   // a4: device-side max-displacement reduction
      // only a displacement beyond the trigger matters to the next step (list_is_stale), so a warp reports its
      // maximum only then: no block barrier at the end of the kernel, and in most steps no atomic at all
      for (int o = 16; o > 0; o >>= 1) d2max = fmax(d2max, __shfl_xor_sync(0xffffffffu, d2max, o));
      if ((threadIdx.x & 31) == 0 && d2max > A.trigger) atomic_max_double_bits(&A.flags->max_disp2_bits[1 - A.parity], d2max);
    }
    if (A.in_run && A.epi != EPI_FORCES && blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(&A.flags->steps_done, 1);   // fused steps only: the unfused paths count in their last kernel
  }
}

// EAM with a half list, between the two passes: rho (accumulated with atomics by pass 1) -> F'(rho), the packed
// w = -F'(rho) that pass 2 gathers, and the embedding energy (one partial per block, added to ev_partials[.][0]).
template <typename T>
__global__ void __launch_bounds__(256) k_eam_embed(int N, PairParams P, const double* __restrict__ rho, double* __restrict__ fp, T* __restrict__ xr4,
                                                   double* __restrict__ ev_out) {
  __shared__ double red[32];
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  double e[1] = {0.0};
  if (n < N) {
    double Fv, fpv;
    eam_embed(P, rho[n], Fv, fpv);
    fp[n] = fpv;
    xr4[4 * (size_t)n + 3] = (T)(-fpv);
    e[0] = Fv;
  }
  if (ev_out) {
    block_sum<1>(e, red);
    if (threadIdx.x == 0) atomicAdd(ev_out, e[0]);
  }
}

// ---------------------------------------------------------------------------------------------------
// a5/a6/a7, the mixed-precision production path: the SAME list loop, bodies and epilogue as k_tile_force, in a
// PERSISTENT, warp-specialised kernel (one block per SM) that takes the tile prologue off the critical path.
// Measured on B200 at cfg 5: the prologue of k_tile_force (table loads -> barrier -> ~140 small bulk copies ->
// mbarrier wait -> offset pass -> barrier) is a chain of dependent round trips worth 0.16 ms of a 0.51 ms
// launch, with a third of the resident warps waiting in it at any time.  Here
//   * four PRODUCER warps walk the block's tiles ahead of the others: one bulk copy brings the tile's table
//     (k_tile_tables: cell starts, counts, offsets, quad map) into shared memory, then one bulk copy per tile
//     cell stages the packed coordinates, all counted on the buffer's `full` mbarrier; then they add the cell
//     offsets in place in chunks of 128 slots, each chunk counted on the buffer's `ready` mbarrier;
//   * 24 CONSUMER warps take 32-lane tasks (32 / K pair rows of one tile) from a shared counter, in tile order: a warp
//     waits for its tile (helping with the tile's chunks meanwhile), runs the list loop and the fused epilogue, and
//     counts the task on the buffer's `empty` mbarrier, which the producers wait for before they refill the buffer;
//   * three tile buffers (two where three do not fit).
// Tiles of a block: blockIdx.x + k gridDim.x; tile k uses buffer k % NB.
// Shared memory: header (128 B: mbarriers, task counter, finished-task counts) | NB x { table[tile_tab_stride] ints |
// st[capA] float4 | scell[interior_cap] u16 | claim words } | (tabulated EAM: the coefficient tables).
// ---------------------------------------------------------------------------------------------------
constexpr int FORCE_P_MAX_NBUF = 3;               // tile buffers
constexpr int FORCE_P_MAX_REGS = 72;              // registers per thread at launch: up to 896 threads per block
constexpr int FORCE_P_MAX_THREADS = 896;          // consumer threads + the producer warps
constexpr int FORCE_P_CONSUMER_REGS = 80;         // after the register split below: (896 x 72 - 128 x 24) / 768
constexpr int FORCE_P_NPROD = 4;                  // producer warps
constexpr int FORCE_P_CLAIM_BYTES = 512;          // per buffer: one claim word per post-processing chunk (tile_cap < 16384: <= 128 chunks)
__host__ __device__ inline size_t force_p_buf_bytes(const Geom& g) {
  return (size_t)tile_tab_stride(g) * 4 + (size_t)force_capA(g) * 16 + (((size_t)g.interior_cap * 2 + 15) & ~(size_t)15) + FORCE_P_CLAIM_BYTES;
}
__host__ __device__ inline size_t force_p_smem(const Geom& g, int nbuf) { return 128 + (size_t)nbuf * force_p_buf_bytes(g); }
__host__ __device__ inline int force_p_chunks(const Geom& g) { return ((g.tile_cap >> 2) + 1 + 31) >> 5; }   // chunks of 32 quads of slots

__device__ __forceinline__ void mbar_arrive(unsigned mbar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void group_barrier(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// the per-tile table as it lies in shared memory (k_tile_tables' layout)
struct TileView {
  const int* h;
  int tcs;
  __device__ __forceinline__ int n_int_slots() const { return h[0]; }
  __device__ __forceinline__ int n_slots() const { return h[1]; }
  __device__ __forceinline__ int n_staged() const { return h[4]; }
  __device__ __forceinline__ int gstart(int t) const { return h[TILE_HDR + t]; }
  __device__ __forceinline__ int start(int t) const { return (int)((unsigned)h[TILE_HDR + tcs + t] >> 16); }
  __device__ __forceinline__ int cnt(int t) const { return h[TILE_HDR + tcs + t] & 0xffff; }
  __device__ __forceinline__ int meta(int t) const { return h[TILE_HDR + 2 * tcs + t]; }
  __device__ __forceinline__ int rstart(int t) const { return h[TILE_HDR + 3 * tcs + t]; }
  __device__ __forceinline__ float off(int d, int t) const { return __int_as_float(h[TILE_HDR + (4 + d) * tcs + t]); }
  __device__ __forceinline__ const unsigned short* qc() const { return reinterpret_cast<const unsigned short*>(h + TILE_HDR + TILE_CELL_INTS * tcs); }
};

// post-processing of one chunk (32 quads = 128 staged slots) of a landed tile: cell offsets added in place, pad slots and
// the dummy slot set far away, pair row -> cells map.  One warp per chunk; consecutive lanes take consecutive slots, so
// every 128-bit access of the warp is four conflict-free wavefronts (a quad of slots per lane made it sixteen, and the
// tile's post-processing cost 2 us of the shared-memory pipe that the gathers of the list loop live on).
__device__ __forceinline__ void force_p_post_chunk(const TileView& tv, float4* st, unsigned short* scell, int ch, int lane) {
  const int ns = tv.n_slots();
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int slot = ch * 128 + u * 32 + lane;
    if (slot < ns) {
      const int t = tv.qc()[slot >> 2];
      const int c = tv.cnt(t), kk = slot - tv.start(t);       // index within the cell (cells are padded to quads of slots)
      if (kk < c) {
        float4 v = st[slot];
        v.x += tv.off(0, t); v.y += tv.off(1, t); v.z += tv.off(2, t);
        st[slot] = v;
      } else {
        st[slot] = make_float4(1e15f, 1e15f, 1e15f, 0.f);
      }
      // indexed by interior slot; a pair of slots is one list row (the cell's rows are padded to 2, not 4)
      if ((tv.meta(t) >> 24) != 0 && (kk & ~1) < c) scell[tv.rstart(t) + kk] = kk < c ? (unsigned short)t : (unsigned short)0xffffu;
    } else if (slot == ns) {
      st[ns] = make_float4(1e15f, 1e15f, 1e15f, 0.f);   // the dummy slot
    }
  }
}

// The post-processing chunks of a landed tile are shared between the producer warps, which walk them from the front, and
// the consumer warps that would otherwise wait for the tile (at the start of a launch all of them do), which walk them
// from the back.  A chunk belongs to whoever first moves its claim word from the tile's generation `gen` to gen + 1:
// one word per chunk, because two dozen warps hammering ONE shared counter serialise (measured: 1.8 us for 28 chunks).
__device__ __forceinline__ void force_p_post_share(const TileView& tv, float4* st, unsigned short* scell, int* claim, int gen, int nchunks,
                                                   unsigned ready_b, int lane, int first, int step, bool from_back) {
  for (int i = first; i < nchunks; i += step) {
    const int ch = from_back ? nchunks - 1 - i : i;
    int won = 0;
    if (lane == 0 && *reinterpret_cast<volatile int*>(claim + ch) == gen) won = atomicCAS(claim + ch, gen, gen + 1) == gen;
    won = __shfl_sync(0xffffffffu, won, 0);
    if (!won) continue;
    force_p_post_chunk(tv, st, scell, ch, lane);
    __syncwarp();
    if (lane == 0) mbar_arrive(ready_b);   // release: the consumers' wait acquires the chunk
  }
}

template <class Body, int K, int MODE>
__global__ void __maxnreg__(FORCE_P_MAX_REGS) k_tile_force_p(ForceArgs A, int gthreads, int NG, int NB) {
  constexpr int NP = FORCE_P_NPROD;
  using T = float;
  using V4 = float4;
  constexpr int NT = Body::NT;
  pdl_wait_then_release();
  if (list_is_stale(A)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Geom& g = A.g;
  const int capA = force_capA(g), tcs = tile_tab_cells(g), tab_ints = tile_tab_stride(g);
  const unsigned buf_bytes = (unsigned)force_p_buf_bytes(g);
  const unsigned smem0 = smem_addr(smem_raw);
  // per buffer: `tabfull` (the table has landed), `full` (the coordinates have landed), `ready` (the cell offsets
  // have been added: the list loop may start), `empty` (all tasks of the tile are done: the producer may refill);
  // behind the mbarriers, in the 128-byte header: the consumers' task counter and the per-buffer finished-task counts
  constexpr int MB = FORCE_P_MAX_NBUF;
  auto full = [&](int b) { return smem0 + 8u * (unsigned)b; };
  auto tabfull = [&](int b) { return smem0 + 8u * (unsigned)(MB + b); };
  auto empty = [&](int b) { return smem0 + 8u * (unsigned)(2 * MB + b); };
  auto ready = [&](int b) { return smem0 + 8u * (unsigned)(3 * MB + b); };
  int* next_task = reinterpret_cast<int*>(smem_raw + 8 * 4 * MB);   // the consumers' task counter
  volatile int* fin = next_task + 1;   // per buffer: tasks finished in it since the launch began (never reset)
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const int gwarps = gthreads >> 5;
  const int nchunks = force_p_chunks(g);
  constexpr int ROUNDS = K >= 32 ? 4 : 1;   // 32-lane rounds per task: a warp per row takes four rows at a time (the dealing costs as much as a short row)
  const int tasks_per_tile = (prow_cap(g) * K + 32 * ROUNDS - 1) / (32 * ROUNDS);
  if (threadIdx.x == 0) {
    for (int b = 0; b < NB; ++b) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(full(b)), "r"(1) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(tabfull(b)), "r"(1) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(empty(b)), "r"(tasks_per_tile) : "memory");
      asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(ready(b)), "r"(nchunks) : "memory");
    }
    *next_task = 0;
    for (int b = 0; b < MB; ++b) fin[b] = 0;
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __shared__ __align__(16) unsigned char pair_tab[Body::TABLE ? MAX_PAIR_TYPES * MAX_PAIR_TYPES * sizeof(V4) : 16];   // per-type-pair coefficients
  if constexpr (Body::TABLE) Body::fill(A.P, reinterpret_cast<V4*>(pair_tab));
  // tabulated EAM (reading s26): the per-interval cubics of rho(r) (and phi(r) in pass 2) are copied behind the tile
  // buffers once per launch; the bodies then look them up with one 128-bit shared-memory load instead of a global one
  if constexpr (Body::SMEM_TABLES > 0) {
    if (A.tab_smem_bytes) {
      float4* dst = reinterpret_cast<float4*>(smem_raw + 128 + (size_t)NB * buf_bytes);
      const int n4 = A.tab_smem_bytes / 16;
      const float4* src0 = reinterpret_cast<const float4*>(A.P.tab_rho);
      const float4* src1 = reinterpret_cast<const float4*>(A.P.tab_phi);
      for (int i = threadIdx.x; i < n4; i += blockDim.x) {
        dst[i] = __ldg(src0 + i);
        if (Body::SMEM_TABLES > 1) dst[n4 + i] = __ldg(src1 + i);
      }
    }
  }
  auto claims = [&](int b) { return reinterpret_cast<int*>(smem_raw + 128 + (size_t)(b + 1) * buf_bytes - FORCE_P_CLAIM_BYTES); };
  for (int i = threadIdx.x; i < NB * (FORCE_P_CLAIM_BYTES / 4); i += blockDim.x) claims(i / (FORCE_P_CLAIM_BYTES / 4))[i % (FORCE_P_CLAIM_BYTES / 4)] = 0;
  __syncthreads();
  const int ntl = ((int)g.ntiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // tiles of this block
  const int pcap = prow_cap(g);

  // Register split (setmaxnreg): the block is launched with FORCE_P_MAX_REGS registers per thread; the producer
  // warpgroup keeps 24 and hands the rest to the consumer warpgroups, which grow to FORCE_P_CONSUMER_REGS (the list
  // loop spills 68 bytes at 72 registers, 16 at 80; measured -3 % at cfg 5).  Hence groups are whole warpgroups
  // (gthreads % 128 == 0) and the producers are the last four warps of the block.
  if (wid >= NG * gwarps) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 24;");
    // ---------------- producer warps: they walk ALL tiles of the block in order, sharing each tile's copies ----------------
    // (issuing ~150 small bulk copies takes one warp several microseconds; measured with one producer warp, the
    // staging pipeline alone took 0.2 ms per launch at cfg 5 and the consumers waited for it)
    const int pw = wid - NG * gwarps;
    if (pw >= NP) return;
    const V4* __restrict__ xr = reinterpret_cast<const V4*>(A.xr);
    // the table of tile k is requested as early as its buffer is free: by the first producer thread, either ahead of time
    // (while the cells of tile k - 1 are in flight, if the buffer is free by then) or at the top of iteration k
    auto request_table = [&](int k) {
      const int b = k % NB;
      mbar_expect_tx(tabfull(b), (unsigned)tab_ints * 4u);
      bulk_g2s(smem0 + 128u + (unsigned)b * buf_bytes, A.tab + (size_t)((int)blockIdx.x + k * (int)gridDim.x) * tab_ints, (unsigned)tab_ints * 4u,
               tabfull(b));
    };
    int requested = 0;   // tables requested so far (meaningful in the first producer thread only)
    for (int k = 0; k < ntl; ++k) {
      const int b = k % NB, j = k / NB;
      const int tile = (int)blockIdx.x + k * (int)gridDim.x;
      unsigned char* bufp = smem_raw + 128 + (size_t)b * buf_bytes;
      const unsigned buf = smem0 + 128u + (unsigned)b * buf_bytes;
      TileView tv{reinterpret_cast<const int*>(bufp), tcs};
      if (pw == 0 && lane == 0 && requested <= k) {
        if (j > 0) mbar_wait(empty(b), (unsigned)((j - 1) & 1));
        request_table(k);
        requested = k + 1;
      }
      mbar_wait(tabfull(b), (unsigned)(j & 1));
      int c0[3], w[3];
      tile_dims(g, tile, c0, w);
      const int ntc = (w[0] + 2) * (w[1] + 2) * (w[2] + 2);
      if (pw == 0 && lane == 0) mbar_expect_tx(full(b), (unsigned)tv.n_staged() * 16u);
      group_barrier(3, 32 * NP);   // the byte count is posted before any of the tile's copies can complete
      const unsigned st_a = buf + (unsigned)tab_ints * 4u;
      for (int t = pw * 32 + lane; t < ntc; t += 32 * NP) {
        const int c = tv.cnt(t);
        if (c > 0) bulk_g2s(st_a + (unsigned)tv.start(t) * 16u, xr + tv.gstart(t), (unsigned)c * 16u, full(b));
      }
      if (pw == 0 && lane == 0 && k + 1 < ntl) {   // the next tile's table, if its buffer is free already
        const int b1 = (k + 1) % NB, j1 = (k + 1) / NB;
        if (j1 == 0 || mbar_test(empty(b1), (unsigned)((j1 - 1) & 1))) { request_table(k + 1); requested = k + 2; }
      }
      // the tile's post-processing, off the consumers' critical path (7 % of their time when they did all of it themselves):
      // the producers run a tile ahead of the consumers in the steady state, so they can afford to wait for the copies here
      mbar_wait(full(b), (unsigned)(j & 1));
      {
        float4* stp = reinterpret_cast<float4*>(bufp + (size_t)tab_ints * 4);
        unsigned short* scp = reinterpret_cast<unsigned short*>(stp + capA);
        force_p_post_share(tv, stp, scp, claims(b), j, nchunks, ready(b), lane, pw, NP, false);
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // these generic stores precede the buffer's next bulk copies
      }
    }
    return;
  }

  // ---------------- consumer warps ----------------
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(FORCE_P_CONSUMER_REGS));
  Body body(A.P);
  body.attach(reinterpret_cast<V4*>(pair_tab));
  body.attach_tables(A.tab_smem_bytes ? smem0 + 128u + (unsigned)NB * buf_bytes : 0u, (unsigned)A.tab_smem_bytes);
  const size_t ld = A.ld;
  const size_t slots_cap = (size_t)pcap * K;
  // Work is dealt to the consumer WARPS, not to groups: a task is 32 consecutive lane slots (32 / K pair rows) of one
  // tile, handed out in tile order from a shared counter.  A block's tiles rarely divide evenly among two groups (cfg 4:
  // three tiles per SM left one group idle for a third of the launch), and a tile's rows rarely fill a group.
  const int tpt = tasks_per_tile;               // (the trailing tasks of a tile are empty: pcap is a capacity)
  const int ntasks = ntl * tpt;
  double d2max = 0.0;
  for (;;) {
    int task = 0;
    if (lane == 0) task = atomicAdd(next_task, 1);
    task = __shfl_sync(0xffffffffu, task, 0);
    if (task >= ntasks) break;
    const int k = task / tpt, tc = task - k * tpt;
    const int b = k % NB, j = k / NB;
    const int tile = (int)blockIdx.x + k * (int)gridDim.x;
    const uint4* tlist = A.list + (size_t)tile * g.chunk_cap * slots_cap;
    int sidx = tc * (32 * ROUNDS) + lane;
    int r = sidx / K;                                       // pair row
    const int s = sidx % K;                                 // lane of the row (the same in every round)
    // while the tile lands: this lane's row length and first list word
    int n_first = 0;
    uint4 w_first = make_uint4(0, 0, 0, 0);
    if (sidx < (int)slots_cap) {
      n_first = A.numneigh[(size_t)tile * pcap + r];
      w_first = ld_stream(tlist + sidx);
    }
    unsigned char* bufp = smem_raw + 128 + (size_t)b * buf_bytes;
    TileView tv{reinterpret_cast<const int*>(bufp), tcs};
    V4* st = reinterpret_cast<V4*>(bufp + (size_t)tab_ints * 4);
    unsigned short* scell = reinterpret_cast<unsigned short*>(st + capA);
    const unsigned st_base = smem_addr(st);
    // A parity wait is only right for a waiter at most one phase ahead of the barrier, and tasks are dealt without regard
    // to what has landed (with few tasks per tile a free warp can be handed a tile whose buffer still holds the tile
    // NB before it, or the one 2 NB before): first make sure the buffer's previous tile is finished, by count
    while (fin[b] < j * tpt) __nanosleep(32);
    if (!mbar_test(ready(b), (unsigned)(j & 1))) {   // the tile is not ready: help with its post-processing instead of waiting
      mbar_wait(tabfull(b), (unsigned)(j & 1));
      mbar_wait(full(b), (unsigned)(j & 1));
      force_p_post_share(tv, st, scell, claims(b), j, nchunks, ready(b), lane, tc, tpt, true);
      mbar_wait(ready(b), (unsigned)(j & 1));
    }
    int c0[3], wdt[3];
    tile_dims(g, tile, c0, wdt);
    const int nlanes = (tv.n_int_slots() >> 1) * K;
#pragma unroll 1
    for (int rr = 0; rr < ROUNDS; ++rr) {
      if (rr > 0) {
        sidx += 32;
        r = sidx / K;
        n_first = 0;
        if (sidx < (int)slots_cap) {
          n_first = A.numneigh[(size_t)tile * pcap + r];
          w_first = ld_stream(tlist + sidx);
        }
      }
      unsigned cells = 0xffffffffu;
      if (sidx < nlanes) cells = reinterpret_cast<const unsigned*>(scell)[r];
      const unsigned cell = cells & 0xffffu;
      const bool act0 = cell != 0xffffu, act1 = (cells >> 16) != 0xffffu;   // the pair's atoms (act1 implies act0)
      const int kin = act0 ? 2 * r - tv.rstart(cell) : 0;     // index of the first atom within its cell
      const int gi = act0 ? tv.gstart(cell) + kin : 0;        // the second atom is gi + 1
      double tot0[NT], tot1[NT];
#pragma unroll
      for (int q = 0; q < NT; ++q) { tot0[q] = 0.0; tot1[q] = 0.0; }
      if (act0) {
        const int slot0 = tv.start(cell) + kin;
        V4 pi0 = lds_v4_scalars<T>(st_base + (unsigned)slot0 * 16u);
        V4 pi1 = lds_v4_scalars<T>(st_base + (unsigned)(slot0 + 1) * 16u);   // a pad slot if there is no partner
        if (!act1) { pi1.x = -1e15f; pi1.y = -1e15f; pi1.z = -1e15f; pi1.w = 0.f; }
        pi0.w = Body::own_w(pi0.w); pi1.w = Body::own_w(pi1.w);
        const int nq = (n_first + 7) >> 3;                    // words of this row
        if (act1 && s == 0) {
          // the pair's mutual term (the two atoms are never entries of their own row)
          typename Pk<T>::type p[NT];
#pragma unroll
          for (int q = 0; q < NT; ++q) p[q] = pk_splat<T>(0.f);
          const T ex = pi0.x - pi1.x, ey = pi0.y - pi1.y, ez = pi0.z - pi1.z;
          const T r2 = ex * ex + ey * ey + ez * ez;
          body.pair2(pk_make(ex, -ex), pk_make(ey, -ey), pk_make(ez, -ez), pk_splat<T>(r2), pk_splat<T>(Body::mutual_w(pi0.w, pi1.w)), p);
#pragma unroll
          for (int q = 0; q < NT; ++q) { tot0[q] += (double)pk_lo(p[q]); tot1[q] += (double)pk_hi(p[q]); }
        }
        if constexpr (MODE == 0) {
          if (A.epi != EPI_FORCES) {   // the epilogue's operands: start them towards L2 now (a 32-byte sector holds both atoms')
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.type + gi));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.v + gi));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.v + ld + gi));
            asm volatile("prefetch.global.L2 [%0];" ::"l"(A.v + 2 * ld + gi));
            if (A.epi == EPI_KICK_DRIFT) {
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x + ld + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x + 2 * ld + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x0 + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x0 + ld + gi));
              asm volatile("prefetch.global.L2 [%0];" ::"l"(A.x0 + 2 * ld + gi));
            }
          }
        }
#ifdef MDK_SKIP_LOOP   // timing experiment: everything but the list loop
        const int mine = 0;
#else
        const int mine = nq > s ? (nq - s + K - 1) / K : 0;   // words q = s, s+K, ...
#endif
        list_loop<T, Body>(body, st_base, tlist + sidx, slots_cap, mine, pi0, pi1, tot0, tot1, w_first, true);
      }
      if constexpr (K > 1) {
#pragma unroll
        for (int q = 0; q < NT; ++q) { tot0[q] = group_sum<K>(tot0[q]); tot1[q] = group_sum<K>(tot1[q]); }
      }
      if (act0 && s == 0) {
        if constexpr (MODE == 0) {
          double cc[3] = {0.0, 0.0, 0.0};
          if (A.epi == EPI_KICK_DRIFT) {
            const int m = tv.meta(cell);
            const int tq[3] = {m & 0xff, (m >> 8) & 0xff, (m >> 16) & 0xff};
#pragma unroll
            for (int d = 0; d < 3; ++d) cc[d] = cell_anchor_1d(g, d, c0[d] + tq[d] - 1);
          }
          const double ta[3] = {tot0[0], tot0[1], tot0[2]}, tb[3] = {tot1[0], tot1[1], tot1[2]};
          d2max = fmax(d2max, atom_epilogue2<T, false>(A, gi, act1, ta, tb, cc));
        } else {
#pragma unroll
          for (int a = 0; a < 2; ++a) {
            if (a == 1 && !act1) break;
            const double rho = a ? tot1[0] : tot0[0];
            double Fv, fpv;
            eam_embed(A.P, rho, Fv, fpv);
            A.rho[gi + a] = rho;
            A.fp_out[gi + a] = fpv;
            reinterpret_cast<T*>(const_cast<void*>(A.xr))[4 * (size_t)(gi + a) + 3] = (T)(-fpv);   // read back as pj.w by pass 2
          }
        }
      }
    }
    // this task is done with the buffer: the producer may refill it when all tasks of the tile have said so (its next
    // writes are bulk copies)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (lane == 0) {
      mbar_arrive(empty(b));
      atomicAdd(const_cast<int*>(fin) + b, 1);
    }
  }
  if constexpr (MODE == 0) {
    if (A.epi == EPI_KICK_DRIFT) {   // a4: device-side max-displacement reduction (see k_tile_force)
      for (int o = 16; o > 0; o >>= 1) d2max = fmax(d2max, __shfl_xor_sync(0xffffffffu, d2max, o));
      if (lane == 0 && d2max > A.trigger) atomic_max_double_bits(&A.flags->max_disp2_bits[1 - A.parity], d2max);
    }
    if (A.in_run && A.epi != EPI_FORCES && blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(&A.flags->steps_done, 1);   // fused steps only: the unfused paths count in their last kernel
  }
}

// ---------------------------------------------------------------------------------------------------
// a5' direct cell-list variant (reading s10): no list.  One warp per interior cell, one
// lane per atom; every lane tests every staged atom of the 27 tile cells around its cell, four
// candidates per broadcast 128-bit load from SoA shared memory (the same walk as the list build).
// Shared memory: TileTables | xs ys zs ws [capA] of T.
// ---------------------------------------------------------------------------------------------------
template <typename T, class Body, int MODE, bool EV>
__global__ void __launch_bounds__(BUILD_THREADS) k_cell_force(ForceArgs A) {
  using V4 = typename Vec4<T>::type;
  constexpr int NT = Body::NT;
  if (list_is_stale(A)) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  TileTables& tt = *reinterpret_cast<TileTables*>(smem_raw);
  const Geom& g = A.g;
  const int capA = force_capA(g);
  T* xs = reinterpret_cast<T*>(smem_raw + sizeof(TileTables));
  T* ys = xs + capA;
  T* zs = ys + capA;
  T* ws = zs + capA;
  __shared__ double red[8 * 32];
  const int tileid = blockIdx.x;
  tile_load(g, tileid, A.tab, tt);
  const double* __restrict__ x = A.x;
  const size_t ld = A.ld;
  const double* __restrict__ fpin = A.fp_in;
  tile_stage(g, tt, g.tile_cap,
             [&](int slot, int gi, const double* off, int) {
               xs[slot] = (T)(x[gi] + off[0]);
               ys[slot] = (T)(x[ld + gi] + off[1]);
               zs[slot] = (T)(x[2 * ld + gi] + off[2]);
               ws[slot] = fpin ? (T)fpin[gi] : (T)A.type[gi];   // F'(rho_j) in EAM pass 2, else the atom's type
             },
             [&](int slot) { xs[slot] = (T)1e15; ys[slot] = (T)1e15; zs[slot] = (T)1e15; ws[slot] = (T)0; });
  __shared__ __align__(16) unsigned char pair_tab[Body::TABLE ? MAX_PAIR_TYPES * MAX_PAIR_TYPES * sizeof(V4) : 16];   // per-type-pair coefficients
  if constexpr (Body::TABLE) Body::fill(A.P, reinterpret_cast<V4*>(pair_tab));
  __syncthreads();
  Body body(A.P);
  body.attach(reinterpret_cast<V4*>(pair_tab));
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  double ev[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  double d2max = 0.0;
  for (int ic = wid; ic < tt.nic; ic += nw) {
    const int t = interior_tile_cell(tt, ic);
    const int s_lo = tt.start[t], c = tt.cnt[t], g_lo = tt.gstart[t];
    const int tx = t % tt.tc[0], ty = (t / tt.tc[0]) % tt.tc[1], tz = t / (tt.tc[0] * tt.tc[1]);
    for (int r0 = 0; r0 < c; r0 += 32) {
      const bool act = r0 + lane < c;
      const int a = act ? s_lo + r0 + lane : s_lo;
      const int gi = g_lo + r0 + lane;
      const T xi = xs[a], yi = ys[a], zi = zs[a], wi = Body::cell_own_w(ws[a]);
      double tot[NT];
#pragma unroll
      for (int k = 0; k < NT; ++k) tot[k] = 0.0;
      for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
          for (int dx = -1; dx <= 1; ++dx) {
            const int t2 = ((tz + dz) * tt.tc[1] + (ty + dy)) * tt.tc[0] + (tx + dx);
            const int s0 = tt.start[t2], c2 = tt.cnt[t2];
            const int aself = t2 == t ? a : -1;
            T p[NT];
#pragma unroll
            for (int k = 0; k < NT; ++k) p[k] = (T)0;
            for (int q = 0; q < (c2 + 3) >> 2; ++q) {
              const int j0 = s0 + 4 * q;
              const V4 X = *reinterpret_cast<const V4*>(xs + j0), Y = *reinterpret_cast<const V4*>(ys + j0);
              const V4 Z = *reinterpret_cast<const V4*>(zs + j0), W = *reinterpret_cast<const V4*>(ws + j0);
              const T xx[4] = {X.x, X.y, X.z, X.w}, yy[4] = {Y.x, Y.y, Y.z, Y.w}, zz[4] = {Z.x, Z.y, Z.z, Z.w};
              const T wj[4] = {W.x, W.y, W.z, W.w};
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const T ex = xi - xx[u], ey = yi - yy[u], ez = zi - zz[u];
                const T r2 = ex * ex + ey * ey + ez * ez;
                body.pair(ex, ey, ez, r2, wi + wj[u], j0 + u != aself, p);
              }
            }
#pragma unroll
            for (int k = 0; k < NT; ++k) tot[k] += (double)p[k];
          }
      if (act) {
        if constexpr (MODE == 0) {
          const double t3[3] = {tot[0], tot[1], tot[2]};
          const double cc[3] = {cell_anchor_1d(g, 0, tt.c0[0] + tx - 1), cell_anchor_1d(g, 1, tt.c0[1] + ty - 1),
                                cell_anchor_1d(g, 2, tt.c0[2] + tz - 1)};
          d2max = fmax(d2max, atom_epilogue<T>(A, gi, t3, cc));
          if constexpr (EV)
#pragma unroll
            for (int k = 0; k < 7; ++k) ev[k] += 0.5 * tot[3 + k];
        } else {
          const double rho = tot[0];
          double Fv, fpv;
          eam_embed(A.P, rho, Fv, fpv);
          A.rho[gi] = rho;
          A.fp_out[gi] = fpv;
          if constexpr (EV) ev[0] += Fv;
        }
      }
    }
  }
  if constexpr (EV) {
    block_sum<8>(ev, red);
    if (threadIdx.x == 0)
#pragma unroll
      for (int k = 0; k < 8; ++k) A.ev_partials[(size_t)tileid * 8 + k] = ev[k];
  }
  if constexpr (MODE == 0) {
    if (A.epi == EPI_KICK_DRIFT) block_max_to_flag(d2max, red, &A.flags->max_disp2_bits[1 - A.parity]);
    if (A.in_run && A.epi != EPI_FORCES && blockIdx.x == 0 && threadIdx.x == 0) atomicAdd(&A.flags->steps_done, 1);   // fused steps only: the unfused paths count in their last kernel
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
// a8 + a4 unfused: velocity Verlet and the device-side displacement test.  Used for
// the first half step of every md_run and by the half-list path (whose forces are complete only when
// the scatter kernel has finished).
// ---------------------------------------------------------------------------------------------------
// v += dtf f ; x += dt v ; flag = max |x - x0|^2
// The atom's storage cell is the cell of x0 (its wrapped position at the last build); the packed copy xr is
// kept in step with x.
template <typename T>
__global__ void k_initial_integrate(Geom g, int N, size_t ld, double* __restrict__ x, double* __restrict__ v, const double* __restrict__ f,
                                    const double* __restrict__ x0, const int* __restrict__ type, const double* __restrict__ mass,
                                    typename Vec4<T>::type* __restrict__ xr, double dt, double half_dt_ftm2v, unsigned long long* flag,
                                    const Flags* run_flags, const double* __restrict__ vscale) {
  __shared__ double red[32];
  if (run_flags && run_flags->stop) return;   // a batched step after the one that found the list stale: do nothing
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  double d2 = 0.0;
  const double sc = vscale ? *vscale : 1.0;   // NVT: the thermostat's velocity scale of this half step (k_nh_half)
  if (n < N) {
    const int ty = type[n];
    double dtf = half_dt_ftm2v / mass[ty];
    T r[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double vv = sc * v[d * ld + n] + dtf * f[d * ld + n];
      double xx = x[d * ld + n] + dt * vv;
      v[d * ld + n] = vv;
      x[d * ld + n] = xx;
      const double p0 = x0[d * ld + n];
      double dd = xx - p0;
      d2 += dd * dd;
      r[d] = (T)(xx - cell_anchor_1d(g, d, cell_index_1d(g, d, p0)));
    }
    xr[n] = make_v4<T>(r[0], r[1], r[2], (T)ty);
  }
  block_max_to_flag(d2, red, flag);
}

__global__ void k_final_integrate(int N, size_t ld, double* __restrict__ v, const double* __restrict__ f,
                                  const int* __restrict__ type, const double* __restrict__ mass, double half_dt_ftm2v, Flags* run_flags) {
  int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (run_flags) {   // batched stepping (half-list path): skipped once the list is stale; the step's last kernel counts it
    if (run_flags->stop) return;
    if (n == 0) atomicAdd(&run_flags->steps_done, 1);
  }
  if (n >= N) return;
  double dtf = half_dt_ftm2v / mass[type[n]];
#pragma unroll
  for (int d = 0; d < 3; ++d) v[d * ld + n] += dtf * f[d * ld + n];
}

// ---------------------------------------------------------------------------------------------------
// NVT (reading s25): one Nose-Hoover thermostat, TH(dt/2) kick drift force kick TH(dt/2),
//   TH(h): xi += h/2 G(KE); s = exp(-xi h); v *= s; KE *= s^2; eta += xi h; xi += h/2 G(KE),  G = (2 KE - g kT)/Q.
// Thermostat state on the device: th[0] xi, th[1] eta, th[2] KE (energy units), th[3] velocity scale of the last TH,
// th[4] g kT, th[5] Q.  The per-atom work fuses into the integrator kernels; the scalar update is one thread.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void nh_half(double* th, double h) {
  double xi = th[0], ke = th[2];
  const double gkT = th[4], Q = th[5];
  xi += 0.5 * h * (2.0 * ke - gkT) / Q;
  const double sc = exp(-xi * h);
  ke *= sc * sc;
  th[1] += xi * h;
  xi += 0.5 * h * (2.0 * ke - gkT) / Q;
  th[0] = xi; th[2] = ke; th[3] = sc;
}
__global__ void k_nh_half(double* th, double h, const Flags* run_flags) {
  if (run_flags && run_flags->stop) return;
  nh_half(th, h);
}
// second kick + this block's share of the kinetic energy after it (deterministic: one partial per block, no atomics)
__global__ void __launch_bounds__(256) k_final_integrate_ke(int N, size_t ld, double* __restrict__ v, const double* __restrict__ f,
                                                            const int* __restrict__ type, const double* __restrict__ mass, double half_dt_ftm2v,
                                                            double* __restrict__ partial, Flags* run_flags) {
  __shared__ double red[32];
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (run_flags) {
    if (run_flags->stop) return;
    if (n == 0) atomicAdd(&run_flags->steps_done, 1);
  }
  double ke[1] = {0.0};
  if (n < N) {
    const double m = mass[type[n]], dtf = half_dt_ftm2v / m;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double vv = v[d * ld + n] + dtf * f[d * ld + n];
      v[d * ld + n] = vv;
      ke[0] += 0.5 * m * vv * vv;
    }
  }
  block_sum<1>(ke, red);
  if (threadIdx.x == 0) partial[blockIdx.x] = ke[0];
}
// one block: KE = mvv2e * sum of the partials in index order; then TH(h) if h > 0
__global__ void __launch_bounds__(256) k_nh_reduce(int nblocks, const double* __restrict__ partial, double mvv2e, double* th, double h,
                                                   const Flags* run_flags) {
  __shared__ double red[32];
  if (run_flags && run_flags->stop) return;
  double s[1] = {0.0};
  for (int b = threadIdx.x; b < nblocks; b += blockDim.x) s[0] += partial[b];
  block_sum<1>(s, red);
  if (threadIdx.x == 0) {
    th[2] = s[0] * mvv2e;
    th[3] = 1.0;
    if (h > 0.0) nh_half(th, h);
  }
}
__global__ void k_scale_velocities(int N, size_t ld, double* __restrict__ v, const double* __restrict__ vscale, const Flags* run_flags) {
  if (run_flags && run_flags->stop) return;
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  const double sc = *vscale;
#pragma unroll
  for (int d = 0; d < 3; ++d) v[d * ld + n] *= sc;
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
