// Internal context of libjefi (not part of the C-ABI; see include/jefi.h for the boundary).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>

#include "jefi.h"

// ---- ring geometry -------------------------------------------------------------------------------------
// Source tile: TS^3 cells.  The ring is stored tile by tile and, inside a tile, slot by slot, so that the slot window
// of one source tile is ONE contiguous run of rows (two when the ring wraps) = one TMA bulk copy:
//   ring[tile][slot] = row of JEFI_ROW_QUADS float4:  [0,64)    S(cell) = (Jx/c, Jz/c, rho, Jy/c) of that step
//                                                     [64,128)  D(cell) = S(step) - S(step-1)   (backward difference)
//                                                     [128]     pad: makes the row pitch 2064 B, so that the same cell
//                                                               in consecutive slots falls in consecutive 16-byte bank
//                                                               groups of shared memory (pitch mod 128 = 16)
// with slot = step mod H, tile = tx + ntx*(ty + nty*tz), cell = lx + TS*(ly + TS*lz).  The component order
// (Jx, Jz | rho, Jy) puts the operands of the packed FP32 instructions (FFMA2) in aligned register pairs.
// The grid is padded to a multiple of TS per axis; padded cells stay zero for ever (they are never written).
constexpr int JEFI_TS = 4;
constexpr int JEFI_TCELLS = JEFI_TS * JEFI_TS * JEFI_TS;
constexpr int JEFI_ROW_QUADS = 2 * JEFI_TCELLS + 1;        // float4 per (tile, slot) row
constexpr int JEFI_ROW_BYTES = JEFI_ROW_QUADS * 16;        // 2064

struct jefi_dims {
  int nx, ny, nz;     // real cells
  int ntx, nty, ntz;  // source tiles per axis
  int H;              // ring depth
  long N;             // nx*ny*nz
  long ncell_pad;     // ntx*nty*ntz*TCELLS
};

// tile index and cell-in-tile of grid cell (i, j, k)
__host__ __device__ inline void jefi_tile_cell(const jefi_dims& d, int i, int j, int k, long& tile, int& cell) {
  int tx = i / JEFI_TS, ty = j / JEFI_TS, tz = k / JEFI_TS;
  int lx = i - tx * JEFI_TS, ly = j - ty * JEFI_TS, lz = k - tz * JEFI_TS;
  tile = tx + (long)d.ntx * (ty + (long)d.nty * tz);
  cell = lx + JEFI_TS * (ly + JEFI_TS * lz);
}
// float4 index of S(cell) in ring row (tile, slot); D(cell) sits JEFI_TCELLS quads further
__host__ __device__ inline size_t jefi_ring_quad(const jefi_dims& d, long tile, int slot, int cell) {
  return ((size_t)tile * d.H + (size_t)slot) * JEFI_ROW_QUADS + (size_t)cell;
}

// Extent of the delay table per axis: it covers every offset the tiled kernel can form, including offsets that
// involve zero-padded cells (observation tiles are 8 cells, source tiles 4 cells wide).
inline int jefi_table_extent(int n) { return ((n + 7) / 8) * 8 + 8; }

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
  int field_impl;       // resolved: JEFI_FIELD_REFERENCE or JEFI_FIELD_TILED
  long step;            // n; -1 before the first push
  cudaStream_t stream;
  float4* ring;         // [tile][slot][JEFI_ROW_QUADS]
  long ring_bytes;
  int* mtab_dev;        // [nz][ny][nx] delay table (fp64-built on the host)
  int* mtab_host;
  // tiled-kernel launch parameters
  int wmax;             // largest slot window over all (obs tile, source tile) pairs
  int wpitch;           // compiled shared-memory pitch chosen for it
  size_t tiled_smem;
  int chunk;            // source tiles per CTA (blockIdx.y splits the source range; > 1 split -> atomic output)
  unsigned short* perm; // evaluation order of the 512 cells of an observation tile per relative tile offset
  int ndx, ndy, ndz;
  // cell-sorted deposit scratch (jefi_particles.cu)
  unsigned *sort_count, *sort_offset, *sort_sums;  // per-bin counts, exclusive offsets, scan tile sums (+ grand total)
  int *sort_key, *sort_rank, *sort_order;          // per particle
  long sort_cap;
  float4* eb_pack;                                 // jefi_push_particles: E, B packed two float4 per node
  void* sort_buf;                                  // jefi_sort_particles: permuted copies of the caller's arrays
  // host-variant staging
  float* src_stage;     // 4N floats, device staging of jefi_field_step_host
  float* eb_stage;      // 6N floats
  // bookkeeping
  long launches;
  cudaEvent_t ev0, ev1;
  bool ev_valid;
  std::string err;
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
int jefi_launch_field_reference(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz);
int jefi_launch_field_tiled(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz);
int jefi_tiled_prepare(jefi_ctx* c);   // window size + smem opt-in; returns JEFI_ESTATE if it cannot run
int jefi_verify_delay_fp32(jefi_ctx* c, long* mismatches);
