// Internal context of libjefi (not part of the C-ABI; see include/jefi.h for the boundary).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "jefi.h"

// ---- ring geometry -------------------------------------------------------------------------------------
// Source tile: tsx*tsy*tsz = 64 cells (4x4x4; 1x8x8 on grids with nx <= 3, where a 4-wide tile would be 3/4 padding).
// The ring is stored tile by tile and, inside a tile, slot by slot, so that the slot window of one source tile is ONE
// contiguous run of rows (two when the ring wraps) = one TMA bulk copy:
//   ring[tile][slot] = row of JEFI_ROW_QUADS float4:  [0,64)    S(cell) = (Jx/c, Jz/c, rho, Jy/c) of that step
//                                                     [64,128)  D(cell) = S(step) - S(step-1)   (backward difference)
//                                                     [128]     pad: makes the row pitch 2064 B, so that the same cell
//                                                               in consecutive slots falls in consecutive 16-byte bank
//                                                               groups of shared memory (pitch mod 128 = 16)
// with slot = step mod H, tile = tx + ntx*(ty + nty*tz), cell = lx + tsx*(ly + tsy*lz).  The component order
// (Jx, Jz | rho, Jy) puts the operands of the packed FP32 instructions (FFMA2) in aligned register pairs.
// The grid is padded to a multiple of the tile per axis; padded cells stay zero for ever (they are never written).
constexpr int JEFI_TCELLS = 64;
constexpr int JEFI_NEVENTS = 64;
constexpr int JEFI_ROW_QUADS = 2 * JEFI_TCELLS + 1;        // float4 per (tile, slot) row
constexpr int JEFI_ROW_BYTES = JEFI_ROW_QUADS * 16;        // 2064

// Tile geometries the field kernel is compiled for (template parameter of k_field_tiled / k_build_perm).
// A consumer thread owns one UNIT of the observation tile: CX cells that are neighbours along x.  With CX = 2 the pairs
// (o, s) and (o + ex, s + ex) have the same offset, i.e. the same distance, delay and geometric factors, which are then
// evaluated once for both (translation invariance of the uniform grid).
template <int OBX_, int OBY_, int OBZ_, int TSX_, int TSY_, int TSZ_, int CX_ = 1>
struct jefi_tile_geom {
  static constexpr int OBX = OBX_, OBY = OBY_, OBZ = OBZ_;  // observation tile in cells
  static constexpr int TSX = TSX_, TSY = TSY_, TSZ = TSZ_;  // source tile (64 cells = one ring row)
  static constexpr int CX = CX_;                            // cells per thread (along x)
  static constexpr int UX = OBX_ / CX_;                     // units per axis: UX x OBY x OBZ = 512 = one per consumer thread
  static constexpr int CELLS = OBX_ * OBY_ * OBZ_;
  static_assert(UX * CX_ == OBX_ && UX * OBY_ * OBZ_ == 512 && TSX_ * TSY_ * TSZ_ == JEFI_TCELLS, "tile sizes");
  static_assert(OBX_ % TSX_ == 0 && OBY_ % TSY_ == 0 && OBZ_ % TSZ_ == 0, "observation tile = whole source tiles");
  static_assert(CX_ == 1 || (CX_ == 2 && TSX_ == 4), "CX = 2 is written for 4-wide source rows");
  // Where unit u (home order, x fastest) keeps its second-level accumulators in shared memory: a rotation of the low index bits
  // by the high ones.  The 32 units a warp evaluates for one source tile are (nearly) equidistant from it, i.e. they lie on a
  // plane through the observation tile, and neighbours in the evaluation order are neighbours on that plane; in home order a
  // plane x = const puts them all in one or two of the 8 bank groups a quarter-warp's 16-byte accesses spread over (CX = 2,
  // 48 bytes per unit) or in 4 of the 32 banks (CX = 1, 4-byte accesses), so the read-modify-write of every item was replayed
  // ~4 times.  With the rotation the units of a plane of any axis orientation fall evenly on all banks.
  __host__ __device__ static constexpr int acc_slot(int u) {
    if (CX_ == 2) return (u & ~7) | ((u + (u >> 3) + 2 * (u >> 6)) & 7);                // u = ux + 8 cy + 64 cz: low bits (ux + cy + 2 cz) mod 8
    if (OBX_ == 8) return (u & ~31) | ((u + 9 * (u >> 6) + 4 * ((u >> 5) & 1)) & 31);   // u = cx + 8 cy + 64 cz: + 9 cz + 4 (cy >> 2)
    return u;
  }
};
using jefi_geom_cube = jefi_tile_geom<8, 8, 8, 4, 4, 4>;
using jefi_geom_slabx = jefi_tile_geom<1, 16, 32, 1, 8, 8>;
using jefi_geom_dyad = jefi_tile_geom<16, 8, 8, 4, 4, 4, 2>;
enum { JEFI_GEOM_CUBE = 0, JEFI_GEOM_SLABX = 1, JEFI_GEOM_DYAD = 2 };

struct jefi_dims {
  int nx, ny, nz;     // real cells
  int tsx, tsy, tsz;  // source tile
  int obx, oby, obz;  // observation tile
  int ntx, nty, ntz;  // source tiles per axis
  int H;              // ring depth
  long N;             // nx*ny*nz
  long ncell_pad;     // ntx*nty*ntz*TCELLS
};

// tile index and cell-in-tile of grid cell (i, j, k)
__host__ __device__ inline void jefi_tile_cell(const jefi_dims& d, int i, int j, int k, long& tile, int& cell) {
  int tx = i / d.tsx, ty = j / d.tsy, tz = k / d.tsz;
  int lx = i - tx * d.tsx, ly = j - ty * d.tsy, lz = k - tz * d.tsz;
  tile = tx + (long)d.ntx * (ty + (long)d.nty * tz);
  cell = lx + d.tsx * (ly + d.tsy * lz);
}
// float4 index of S(cell) in ring row (tile, slot); D(cell) sits JEFI_TCELLS quads further
__host__ __device__ inline size_t jefi_ring_quad(const jefi_dims& d, long tile, int slot, int cell) {
  return ((size_t)tile * d.H + (size_t)slot) * JEFI_ROW_QUADS + (size_t)cell;
}

// Extent of the delay table per axis: it covers every offset the tiled kernel can form, including offsets that
// involve zero-padded cells (the grid padded to whole observation tiles, plus one tile of slack).
inline int jefi_table_extent(int n, int ob) { return ((n + ob - 1) / ob) * ob + ob; }

// Scaled geometry used by the field kernels: d' = d/(c dt) so that |d'| = s is the delay in steps (Eq. 2.6).
struct jefi_geom {
  float kx, ky, kz;   // dx/(c dt), dy/(c dt), dz/(c dt)
  float prefE;        // dV/(4 pi eps0) / (c dt)^2            -> E = prefE * sum[ d'(rho rs^3 + Drho rs^2) - DJt rs ]
  float prefB;        // -mu0 dV/(4 pi) * c / (c dt)^2        -> B = prefB * sum[ d' x (Jt rs^3 + DJt rs^2) ],  Jt = J/c
};

struct jefi_ctx {
  jefi_config cfg;
  jefi_dims dims;
  jefi_geom geom;
  double c, eps0, mu0;
  int ndt;
  int shape_order;      // resolved: 1 or 2
  int field_impl;       // resolved: JEFI_FIELD_REFERENCE or JEFI_FIELD_TILED
  int tile_geom;        // JEFI_GEOM_*
  long step;            // n; -1 before the first push
  cudaStream_t stream;
  float4* ring;         // [tile][slot][JEFI_ROW_QUADS]
  long ring_bytes;
  int* mtab_dev;        // [ez][ey][ex] delay table (fp64-built on the host)
  int* mtab_host;
  int tex, tey, tez;    // its extents
  // tiled-kernel launch parameters
  int wmax;             // largest slot window over all (obs tile, source tile) pairs
  int wpitch;           // compiled shared-memory pitch (rows per stage) it is served from
  size_t tiled_smem;
  int chunk;            // source tiles per CTA (blockIdx.y splits the source range)
  int nsplit;           // pieces of the source range; > 1: partial sums go to `partial` and k_reduce_partials adds them
  float* partial;       // [nsplit][6][N]
  unsigned short* perm; // evaluation order of the 512 cells of an observation tile per relative tile offset
  int *tile_first, *tile_last;  // per source tile: first and last step whose ring row (S or D) was not all zero (INT-ish max / -1: never)
  int ndx, ndy, ndz;
  // cell-sorted deposit scratch (jefi_particles.cu)
  unsigned *sort_count, *sort_offset, *sort_sums;  // per-bin counts, exclusive offsets, scan tile sums (+ grand total)
  int *sort_key, *sort_rank, *sort_order;          // per particle
  long sort_cap;
  long sort_gen;                                   // bumped whenever the per-particle scratch is reallocated (part of jefi_pic_step's graph key)
  long sorted_np;                                  // np of the last jefi_sort_particles call (-1: none): the caller's list is
  int deposits_since_sort;                         // (nearly) cell-sorted for the next few steps, which decides the run-deposit kernel
  float4* eb_pack;                                 // jefi_push_particles: E, B packed two float4 per node
  void* sort_buf;                                  // jefi_sort_particles: permuted copies of the caller's arrays
  // jefi_pic_step: one whole PIC step as a CUDA graph.  The step-dependent kernel arguments (n, ring slot, previous slot) are
  // read from step_dev, which the graph's first kernel advances, so that the same executable graph replays every step.
  int* step_dev;            // device int[4]: n, n mod H, (n-1) mod H or -1
  long step_dev_value;      // the step step_dev currently holds (-2: nothing uploaded yet)
  bool capturing;           // a graph capture is in progress: kernels take the step from step_dev, no event records
  cudaGraphExec_t pic_exec;
  unsigned long long pic_key[24];
  long pic_launches;        // kernels per replay
  // host-variant staging
  float* src_stage;     // 4N floats, device staging of jefi_field_step_host
  float* eb_stage;      // 6N floats
  // bookkeeping
  long launches;
  cudaEvent_t ev0[JEFI_NEVENTS], ev1[JEFI_NEVENTS];  // around the field kernel(s) of the last JEFI_NEVENTS field steps
  long field_calls;
  std::string err;
  std::string impl_reason;
};

// Every entry point runs on the context's device whatever the calling thread's current device is, and restores it.
struct jefi_device_guard {
  int prev = -1;
  bool switched = false;
  explicit jefi_device_guard(const jefi_ctx* c) {
    if (c && cudaGetDevice(&prev) == cudaSuccess && prev != c->cfg.device) switched = cudaSetDevice(c->cfg.device) == cudaSuccess;
  }
  ~jefi_device_guard() {
    if (switched) cudaSetDevice(prev);
  }
};

#define JEFI_CUDA_TRY(ctx, call)                                                                   \
  do {                                                                                             \
    cudaError_t e__ = (call);                                                                      \
    if (e__ != cudaSuccess) {                                                                      \
      (ctx)->err = std::string(#call) + ": " + cudaGetErrorString(e__);                            \
      return JEFI_ECUDA;                                                                           \
    }                                                                                              \
  } while (0)

// the nearest-step delay from the squared scaled distance, in the tiled kernel's own fp32 arithmetic.
// rs = rsqrt(q); s = q*rs; m = round-to-nearest(s) via the 1.5*2^23 magic constant (no F2I on the hot path).
// jefi_create proves on the device that this equals the fp64 table for every offset of the grid.
#define JEFI_MAGIC 12582912.0f
__device__ __forceinline__ float jefi_rsqrt(float x) {  // one MUFU.RSQ, no denormal fix-up code
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ int jefi_delay_fp32(float q) {
  float rs = jefi_rsqrt(q);
  float t = fmaf(q, rs, JEFI_MAGIC);
  return __float_as_int(t) - 0x4B400000;
}
__device__ __forceinline__ float jefi_q_fp32(float kx, float ky, float kz, float fi, float fj, float fk) {
  float ax = kx * fi, ay = ky * fj, az = kz * fk;
  return fmaf(ax, ax, fmaf(ay, ay, az * az));
}

// implemented in the .cu files
int jefi_launch_push_sources(jefi_ctx* c, const float* rho, const float* jx, const float* jy, const float* jz);
int jefi_field_step_impl(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz, float* eb_packed);
int jefi_deposit_impl(jefi_ctx* c, long np, const float* x, const float* y, const float* z, const float* ux, const float* uy,
                      const float* uz, const float* qw, const unsigned char* alive, float* rho, float* jx, float* jy, float* jz);
int jefi_push_packed_impl(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz, const float* q_over_m,
                          unsigned char* alive, const float* eb_packed);
int jefi_prepare_deposit_scratch(jefi_ctx* c, long np);  // allocations a captured deposit must not make
int jefi_launch_field_reference(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz,
                                float* eb_packed);
int jefi_launch_field_tiled(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz,
                            float* eb_packed);
int jefi_tiled_prepare(jefi_ctx* c);   // window size + smem opt-in; returns JEFI_ESTATE if it cannot run
int jefi_verify_delay_fp32(jefi_ctx* c, long* mismatches, long* offsets);
cudaError_t jefi_field_check_errors(unsigned long long out[2]);     // -DJEFI_CHECKED counters (zero in normal builds)
cudaError_t jefi_particle_check_errors(unsigned long long out[2]);
