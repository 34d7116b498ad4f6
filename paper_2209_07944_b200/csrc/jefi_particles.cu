// libjefi: CIC deposit (Eqs. 2.15-2.19) and field interpolation +
// relativistic Boris push + kill (row a5; PAPER.md:117-127 Eqs. 2.7-2.11, :193-205 Eq. 2.20).
#include <string.h>

#include <mutex>
#include <string>

#include "jefi_ctx.h"

// Eq. (2.15)/(2.17) in grid units: node index i = floor(xi - 1/2), fraction alpha = xi - 1/2 - i.  xi - 0.5 is exact
// in fp32 for 0.25 <= xi < 2^23, so the index equals the fp64 oracle's bit for bit (DESIGN.md §3 A9).  Positions far
// outside any grid (a caller's stale alive flag) are clamped before the float -> int conversion; they stay outside.
__device__ __forceinline__ void cic_cell(float xi, int& i, float& alpha) {
  float s = fminf(fmaxf(xi, -16.f), 2.0e9f) - 0.5f;
  float f = floorf(s);
  i = (int)f;
  alpha = s - f;
}

// The nodes one axis of a particle touches and their weights, for the two shape functions (jefi_config.shape_order):
//   ORDER 1  S^(1), Eqs. (2.13), (2.16): nodes i0 = floor(xi - 1/2) and i0 + 1 with weights 1 - alpha, alpha;
//   ORDER 2  S^(2), Eq. (2.14) (reading A11: the quadratic B-spline): centre node ic = floor(xi), nodes ic-1, ic, ic+1 with
//            weights (1/2)(1/2 - d)^2, 3/4 - d^2, (1/2)(1/2 + d)^2, d = xi - (ic + 1/2) in [-1/2, 1/2) (xi - ic and the
//            subtraction of 1/2 are exact in fp32, so d equals the fp64 oracle's).
template <int ORDER>
struct axis_stencil {
  static constexpr int NN = ORDER + 1;
  int i0;       // first node
  float w[NN];
  __device__ __forceinline__ void set(float xi) {
    if (ORDER == 1) {
      float al;
      cic_cell(xi, i0, al);
      w[0] = 1.f - al;
      w[ORDER] = al;
    } else {
      const float xc = fminf(fmaxf(xi, -16.f), 2.0e9f);
      const float f = floorf(xc);
      const float dlt = (xc - f) - 0.5f;
      i0 = (int)f - 1;
      w[0] = 0.5f * (0.5f - dlt) * (0.5f - dlt);
      w[1] = 0.75f - dlt * dlt;
      w[ORDER] = 0.5f * (0.5f + dlt) * (0.5f + dlt);
    }
  }
};
// bins of the cell sort per axis and the key of a base node: i0 in [-(NN-1), n-1] <=> at least one node inside the grid
template <int ORDER>
__device__ __forceinline__ bool base_key(int nx, int ny, int nz, int i0, int j0, int k0, int& key) {
  constexpr int S = ORDER;  // NN - 1
  key = (i0 + S) + (nx + S) * ((j0 + S) + (ny + S) * (k0 + S));
  return i0 >= -S && i0 < nx && j0 >= -S && j0 < ny && k0 >= -S && k0 < nz;
}

// ------------------------------------------------------------------------------------------------------------
// deposit: one thread per particle; the 8 node contributions of the 4 quantities go out as fp32 reductions.
// Lanes of a warp whose particles fall on the same node first combine their contributions with a match-any
// segmented shuffle reduction, so a cell-sorted particle list issues one atomic per (warp, node) instead of one per
// particle (warp-aggregated atomics).
// ------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void warp_aggregated_add4(float* __restrict__ rho, float* __restrict__ jx, float* __restrict__ jy,
                                                     float* __restrict__ jz, long node, float r, float vx, float vy, float vz) {
  // Called by all 32 lanes.  node < 0 marks "nothing to add" (virtual node or dead particle); such keys are unique
  // per lane so they never form a group.
  const unsigned FULL = 0xffffffffu;
  const unsigned lane = threadIdx.x & 31;
  const unsigned peers = __match_any_sync(FULL, node);  // lanes that target the same node
  float a0 = r, a1 = r * vx, a2 = r * vy, a3 = r * vz;
  const unsigned cnt = __popc(peers);
  const unsigned maxcnt = __reduce_max_sync(FULL, cnt);
  if (maxcnt > 1) {
    // tree reduction inside every peer group: at stride s the lanes of rank 0, 2s, 4s.. add the lane of rank + s
    const unsigned rank = __popc(peers & ((1u << lane) - 1u));
    for (unsigned stride = 1; stride < maxcnt; stride <<= 1) {
      const bool has = rank + stride < cnt;
      const int partner = has ? (int)__fns(peers, 0, (int)(rank + stride + 1)) : (int)lane;
      const float b0 = __shfl_sync(FULL, a0, partner), b1 = __shfl_sync(FULL, a1, partner);
      const float b2 = __shfl_sync(FULL, a2, partner), b3 = __shfl_sync(FULL, a3, partner);
      if (has && (rank & (2u * stride - 1u)) == 0u) { a0 += b0; a1 += b1; a2 += b2; a3 += b3; }
    }
    if (rank != 0) return;  // only the lowest lane of a group issues the atomics (after the last shuffle)
  }
  if (node >= 0) {
    atomicAdd(rho + node, a0); atomicAdd(jx + node, a1); atomicAdd(jy + node, a2); atomicAdd(jz + node, a3);
  }
}

template <int ORDER>
__global__ void __launch_bounds__(256) k_deposit(int nx, int ny, int nz, float inv_dV, float cc, long np,
                                                 const float* __restrict__ x, const float* __restrict__ y,
                                                 const float* __restrict__ z, const float* __restrict__ ux,
                                                 const float* __restrict__ uy, const float* __restrict__ uz,
                                                 const float* __restrict__ qw, const unsigned char* __restrict__ alive,
                                                 float* __restrict__ rho, float* __restrict__ jx, float* __restrict__ jy,
                                                 float* __restrict__ jz) {
  constexpr int NN = ORDER + 1;
  long p = (long)blockIdx.x * blockDim.x + threadIdx.x;
  bool live = p < np && (alive == nullptr || alive[p] != 0);
  axis_stencil<ORDER> sx, sy, sz;
  sx.set(0.f); sy.set(0.f); sz.set(0.f);
  float r0 = 0, vx = 0, vy = 0, vz = 0;
  if (live) {
    sx.set(x[p]); sy.set(y[p]); sz.set(z[p]);
    float u0 = ux[p], u1 = uy[p], u2 = uz[p];
    float ig = rsqrtf(1.f + u0 * u0 + u1 * u1 + u2 * u2);  // 1/gamma
    vx = cc * u0 * ig; vy = cc * u1 * ig; vz = cc * u2 * ig;  // v = c u / gamma
    r0 = qw[p] * inv_dV;                                     // Eq. (2.18)
  }
#pragma unroll
  for (int c = 0; c < NN; c++)
#pragma unroll
    for (int b = 0; b < NN; b++)
#pragma unroll
      for (int a = 0; a < NN; a++) {
        int ii = sx.i0 + a, jj = sy.i0 + b, kk = sz.i0 + c;
        bool ok = live && ii >= 0 && ii < nx && jj >= 0 && jj < ny && kk >= 0 && kk < nz;  // virtual nodes dropped
        float w = sx.w[a] * sy.w[b] * sz.w[c];                                               // Eq. (2.16)
        long node = ok ? (long)ii + (long)nx * ((long)jj + (long)ny * kk) : -1 - (long)(threadIdx.x & 31);
        warp_aggregated_add4(rho, jx, jy, jz, node, r0 * w, vx, vy, vz);
      }
}

// ------------------------------------------------------------------------------------------------------------
// cell-sorted deposit (internal order; the caller's arrays are never permuted).
//
//   k_sort_keys     key = base node (i+1, j+1, k+1) of Eq. (2.15) linearised over (nx+1)(ny+1)(nz+1) bins; an atomic
//                   counter per bin hands every alive particle its rank inside the bin
//   exclusive scan  of the bin counts (three small kernels)
//   k_sort_scatter  order[offset[key] + rank] = particle
//   k_deposit_sorted  thread t takes particle order[t]; lanes with equal keys are contiguous, so the 8 x 4 node
//                   contributions are combined with a segmented shuffle reduction (5 steps) and only the first lane
//                   of every run issues the fp32 reductions: one per (warp, cell, node, quantity).
// ------------------------------------------------------------------------------------------------------------
template <int ORDER>
__global__ void __launch_bounds__(256) k_sort_keys(int nx, int ny, int nz, int nbins, long np, const float* __restrict__ x,
                                                   const float* __restrict__ y, const float* __restrict__ z,
                                                   const unsigned char* __restrict__ alive, int* __restrict__ key,
                                                   int* __restrict__ rank, unsigned* __restrict__ count) {
  long p = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  int kk = nbins, r = 0;  // extra last bin: dead particles and particles with no node inside the grid
  if (alive == nullptr || alive[p] != 0) {
    axis_stencil<ORDER> sx, sy, sz;
    sx.set(x[p]); sy.set(y[p]); sz.set(z[p]);
    // A particle whose base node is outside [-(NN-1), n) has all its nodes outside the grid (virtual): it
    // deposits nothing and is left out of the order.
    int k2;
    if (base_key<ORDER>(nx, ny, nz, sx.i0, sy.i0, sz.i0, k2)) kk = k2;
  }
  r = (int)atomicAdd(count + kk, 1u);
  key[p] = kk;
  rank[p] = r;
}

constexpr int SCAN_ITEMS = 8, SCAN_THREADS = 256, SCAN_TILE = SCAN_ITEMS * SCAN_THREADS;

// exclusive scan of one tile of SCAN_TILE counts; tile total -> sums[blockIdx.x]
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tiles(const unsigned* __restrict__ in, unsigned* __restrict__ out, long n,
                                                             unsigned* __restrict__ sums) {
  __shared__ unsigned warp_tot[SCAN_THREADS / 32];
  const long base = (long)blockIdx.x * SCAN_TILE + (long)threadIdx.x * SCAN_ITEMS;
  unsigned v[SCAN_ITEMS], t = 0;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) { v[i] = base + i < n ? in[base + i] : 0u; t += v[i]; }
  const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  unsigned inc = t;
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) { unsigned o = __shfl_up_sync(0xffffffffu, inc, s); if (lane >= (unsigned)s) inc += o; }
  if (lane == 31) warp_tot[warp] = inc;
  __syncthreads();
  unsigned woff = 0;
  for (unsigned w = 0; w < warp; w++) woff += warp_tot[w];
  unsigned run = woff + inc - t;
#pragma unroll
  for (int i = 0; i < SCAN_ITEMS; i++) { if (base + i < n) out[base + i] = run; run += v[i]; }
  if (threadIdx.x == SCAN_THREADS - 1) sums[blockIdx.x] = woff + inc;
}
// exclusive scan of the tile totals in one block (ntiles <= a few thousand); grand total -> sums[ntiles]
__global__ void __launch_bounds__(1024) k_scan_sums(unsigned* __restrict__ sums, int ntiles) {
  __shared__ unsigned warp_tot[32];
  __shared__ unsigned carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int b0 = 0; b0 < ntiles; b0 += 1024) {
    const int i = b0 + threadIdx.x;
    const unsigned t = i < ntiles ? sums[i] : 0u;
    unsigned inc = t;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) { unsigned o = __shfl_up_sync(0xffffffffu, inc, s); if (lane >= (unsigned)s) inc += o; }
    if (lane == 31) warp_tot[warp] = inc;
    __syncthreads();
    unsigned woff = 0;
    for (unsigned w = 0; w < warp; w++) woff += warp_tot[w];
    const unsigned c0 = carry;
    if (i < ntiles) sums[i] = c0 + woff + inc - t;
    __syncthreads();
    if (threadIdx.x == 1023) carry = c0 + woff + inc;
    __syncthreads();
  }
  if (threadIdx.x == 0) sums[ntiles] = carry;
}
__global__ void __launch_bounds__(256) k_scan_add(unsigned* __restrict__ out, long n, const unsigned* __restrict__ sums) {
  long i = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] += sums[i / SCAN_TILE];
}

__device__ unsigned long long g_jefi_part_errors[2];  // -DJEFI_CHECKED: [0] scatter index outside the list
cudaError_t jefi_particle_check_errors(unsigned long long out[2]) { return cudaMemcpyFromSymbol(out, g_jefi_part_errors, 2 * sizeof(unsigned long long)); }

__global__ void __launch_bounds__(256) k_sort_scatter(long np, const int* __restrict__ key, const int* __restrict__ rank,
                                                      const unsigned* __restrict__ offset, int* __restrict__ order) {
  long p = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  const unsigned dst = offset[key[p]] + (unsigned)rank[p];
#ifdef JEFI_CHECKED
  if ((long)dst >= np) { atomicAdd(&g_jefi_part_errors[0], 1ull); return; }
#endif
  order[dst] = (int)p;
}

template <int ORDER>
__global__ void __launch_bounds__(256) k_deposit_sorted(int nx, int ny, int nz, float inv_dV, float cc, long np,
                                                        const unsigned* __restrict__ n_alive, const int* __restrict__ order,
                                                        const unsigned char* __restrict__ alive, const float* __restrict__ x,
                                                        const float* __restrict__ y, const float* __restrict__ z,
                                                        const float* __restrict__ ux, const float* __restrict__ uy,
                                                        const float* __restrict__ uz, const float* __restrict__ qw,
                                                        float* __restrict__ rho, float* __restrict__ jx,
                                                        float* __restrict__ jy, float* __restrict__ jz) {
  constexpr int NN = ORDER + 1;
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  const long na = order ? (long)*n_alive : np;
  if (((long)blockIdx.x * blockDim.x + (threadIdx.x & ~31)) >= na) return;  // whole warp beyond the last particle
  bool live = t < na;
  const unsigned FULL = 0xffffffffu, lane = threadIdx.x & 31;
  int kk = -2 - (int)lane;  // padding lanes and non-depositing particles: unique keys, never merged
  axis_stencil<ORDER> sx, sy, sz;
  sx.set(0.f); sy.set(0.f); sz.set(0.f);
  float r0 = 0, vx = 0, vy = 0, vz = 0;
  long p = t;
  if (live) {
    if (order) p = order[t];
    else live = alive == nullptr || alive[p] != 0;
  }
  if (live) {
    sx.set(x[p]); sy.set(y[p]); sz.set(z[p]);
    // distinct base nodes in [-(NN-1), n) give distinct keys.  A particle outside that range (possible with alive == NULL or
    // a stale flag) has no node in the grid: it keeps its unique negative key, so that it can neither alias the key of an
    // in-grid cell nor be merged into a neighbour's run.
    int k2;
    if (base_key<ORDER>(nx, ny, nz, sx.i0, sy.i0, sz.i0, k2)) kk = k2;
    else live = false;
  }
  if (live) {
    float u0 = ux[p], u1 = uy[p], u2 = uz[p];
    float ig = rsqrtf(1.f + u0 * u0 + u1 * u1 + u2 * u2);
    vx = cc * u0 * ig; vy = cc * u1 * ig; vz = cc * u2 * ig;
    r0 = qw[p] * inv_dV;
  }
  // run structure of the warp: a run = maximal stretch of neighbouring lanes with the same key (in a cell-sorted list, all
  // particles of the cell that fall in this warp; in an unsorted list mostly single lanes)
  const int kprev = __shfl_up_sync(FULL, kk, 1);
  const bool head = lane == 0 || kprev != kk;
  const unsigned heads = __ballot_sync(FULL, head);
  const unsigned above = heads & ~((2u << lane) - 1u);         // run heads strictly above this lane
  const unsigned run_end = above ? (unsigned)__ffs(above) - 2u : 31u;  // last lane of this lane's run
  bool same[5];
  unsigned any_same = 0;  // bit s: some lane of the warp still has a partner at stride 2^s (skips the idle reduction steps of
                          // short runs: with 4 particles per cell only strides 1 and 2 do any work)
#pragma unroll
  for (int s = 0; s < 5; s++) {
    same[s] = lane + (1u << s) <= run_end;
    any_same |= (__ballot_sync(FULL, same[s]) != 0u ? 1u : 0u) << s;
  }
#pragma unroll
  for (int c = 0; c < NN; c++)
#pragma unroll
    for (int b = 0; b < NN; b++)
#pragma unroll
      for (int a = 0; a < NN; a++) {
        const float w = sx.w[a] * sy.w[b] * sz.w[c];
        float a0 = r0 * w, a1 = a0 * vx, a2 = a0 * vy, a3 = a0 * vz;
#pragma unroll
        for (int s = 0; s < 5; s++) {  // segmented suffix sum: the head of a run ends up with the run total
          if (!((any_same >> s) & 1u)) continue;  // warp-uniform
          const float b0 = __shfl_down_sync(FULL, a0, 1u << s), b1 = __shfl_down_sync(FULL, a1, 1u << s);
          const float b2 = __shfl_down_sync(FULL, a2, 1u << s), b3 = __shfl_down_sync(FULL, a3, 1u << s);
          if (same[s]) { a0 += b0; a1 += b1; a2 += b2; a3 += b3; }
        }
        const int ii = sx.i0 + a, jj = sy.i0 + b, kz = sz.i0 + c;
        if (live && head && ii >= 0 && ii < nx && jj >= 0 && jj < ny && kz >= 0 && kz < nz) {  // virtual nodes dropped
          const long node = (long)ii + (long)nx * ((long)jj + (long)ny * kz);
          atomicAdd(rho + node, a0); atomicAdd(jx + node, a1); atomicAdd(jy + node, a2); atomicAdd(jz + node, a3);
        }
      }
}

// ------------------------------------------------------------------------------------------------------------
// Run deposit for S^(1), transposed through shared memory (JEFI_DEPOSIT_RUNS on lists the context does not know to be sorted).
//
// Phase 1, lane = particle: the 8 node weights x (rho, Jx, Jy, Jz) = 32 contributions of the particle go to the warp's
// shared-memory tile V[value][particle] (pitch 33 floats: conflict-free both ways), with the particle's base node as a linear
// index and the 8-bit mask of its nodes that lie inside the grid.
// Phase 2, lane = value (node = lane / 4, quantity = lane % 4): the lane adds its value over the particles of the warp in
// order and, at the end of every run of equal base nodes (warp-uniform: the ballot of run heads), issues ONE reduction for
// (run, node, quantity).  So a run costs one 32-lane RED instruction whose lanes hit the 8 nodes of one cell in the four
// grids (x-neighbour nodes share a sector), instead of 32 RED instructions with one active lane per run, and the
// 32 x 5 segmented shuffle steps of k_deposit_sorted become 32 conflict-free LDS + FADD.  Correct for any particle order
// (an unsorted list simply has 32 runs per warp).  Sums inside a run are taken in lane order.
// ------------------------------------------------------------------------------------------------------------
constexpr int DEP_WARPS = 8, DEP_PITCH = 33, DEP_TILE = 32 * DEP_PITCH + 64;  // floats per warp: V[32][33], base[32], mask[32]
__global__ void __launch_bounds__(32 * DEP_WARPS) k_deposit_runs(int nx, int ny, int nz, float inv_dV, float cc, long np,
                                                                 const unsigned* __restrict__ n_alive, const int* __restrict__ order,
                                                                 const unsigned char* __restrict__ alive, const float* __restrict__ x,
                                                                 const float* __restrict__ y, const float* __restrict__ z,
                                                                 const float* __restrict__ ux, const float* __restrict__ uy,
                                                                 const float* __restrict__ uz, const float* __restrict__ qw,
                                                                 float* __restrict__ rho, float* __restrict__ jx,
                                                                 float* __restrict__ jy, float* __restrict__ jz) {
  __shared__ float tile[DEP_WARPS][DEP_TILE];
  const long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  const long na = order ? (long)*n_alive : np;
  if (((long)blockIdx.x * blockDim.x + (threadIdx.x & ~31)) >= na) return;  // whole warp beyond the last particle
  const unsigned FULL = 0xffffffffu, lane = threadIdx.x & 31;
  float* V = tile[threadIdx.x >> 5];
  int* Bs = reinterpret_cast<int*>(V + 32 * DEP_PITCH);
  unsigned* Ms = reinterpret_cast<unsigned*>(Bs + 32);
  bool live = t < na;
  int kk = -2 - (int)lane;  // padding lanes and non-depositing particles: unique keys, never merged
  axis_stencil<1> sx, sy, sz;
  sx.set(0.f); sy.set(0.f); sz.set(0.f);
  float r0 = 0, vx = 0, vy = 0, vz = 0;
  long p = t;
  if (live) {
    if (order) p = order[t];
    else live = alive == nullptr || alive[p] != 0;
  }
  if (live) {
    sx.set(x[p]); sy.set(y[p]); sz.set(z[p]);
    int k2;  // a particle with no node inside the grid keeps its unique negative key (see k_deposit_sorted)
    if (base_key<1>(nx, ny, nz, sx.i0, sy.i0, sz.i0, k2)) kk = k2;
    else live = false;
  }
  if (live) {
    float u0 = ux[p], u1 = uy[p], u2 = uz[p];
    float ig = rsqrtf(1.f + u0 * u0 + u1 * u1 + u2 * u2);
    vx = cc * u0 * ig; vy = cc * u1 * ig; vz = cc * u2 * ig;
    r0 = qw[p] * inv_dV;
  }
  const int kprev = __shfl_up_sync(FULL, kk, 1);
  const unsigned heads = __ballot_sync(FULL, lane == 0 || kprev != kk);  // bit l: lane l starts a run
  unsigned inside = 0;
#pragma unroll
  for (int c = 0; c < 2; c++)
#pragma unroll
    for (int b = 0; b < 2; b++)
#pragma unroll
      for (int a = 0; a < 2; a++) {
        const int node = a + 2 * b + 4 * c;
        const float a0 = r0 * (sx.w[a] * sy.w[b] * sz.w[c]);  // Eq. (2.16), (2.18)
        V[(4 * node + 0) * DEP_PITCH + lane] = a0;
        V[(4 * node + 1) * DEP_PITCH + lane] = a0 * vx;         // Eq. (2.19)
        V[(4 * node + 2) * DEP_PITCH + lane] = a0 * vy;
        V[(4 * node + 3) * DEP_PITCH + lane] = a0 * vz;
        const int ii = sx.i0 + a, jj = sy.i0 + b, kz = sz.i0 + c;
        inside |= (live && ii >= 0 && ii < nx && jj >= 0 && jj < ny && kz >= 0 && kz < nz ? 1u : 0u) << node;  // virtual nodes dropped
      }
  Bs[lane] = sx.i0 + nx * (sy.i0 + ny * sz.i0);  // linear index of the base node; exact for every node that is inside
  Ms[lane] = inside;
  __syncwarp();
  // phase 2: this lane owns value (node, quantity) of every run
  const int node = (int)lane >> 2;
  const int off = (node & 1) + nx * (((node >> 1) & 1) + ny * (node >> 2));
  float* const arr = (lane & 3) == 0 ? rho : (lane & 3) == 1 ? jx : (lane & 3) == 2 ? jy : jz;
  const float* Vl = V + lane * DEP_PITCH;
  float acc = 0.f;
#pragma unroll
  for (int q = 0; q < 32; q++) {
    acc += Vl[q];
    if (q == 31 || ((heads >> (q + 1)) & 1u)) {  // warp-uniform: particle q ends a run
      if ((Ms[q] >> node) & 1u) atomicAdd(arr + (Bs[q] + off), acc);
      acc = 0.f;
    }
  }
}

static inline long sort_bins(const jefi_ctx* c) {
  const jefi_dims& d = c->dims;
  const int s = c->shape_order;  // nodes per axis - 1
  return (long)(d.nx + s) * (d.ny + s) * (d.nz + s);
}

static int ensure_sort_scratch(jefi_ctx* c, long np) {
  const long nb = sort_bins(c) + 1;  // + the bin of the non-depositing particles
  const long ntiles = (nb + SCAN_TILE - 1) / SCAN_TILE;
  if (!c->sort_count) {
    JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_count, (size_t)nb * sizeof(unsigned)));
    JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_offset, (size_t)nb * sizeof(unsigned)));
    JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_sums, (size_t)(ntiles + 1) * sizeof(unsigned)));
  }
  if (np > c->sort_cap) {
    if (c->sort_key) { cudaFree(c->sort_key); cudaFree(c->sort_rank); cudaFree(c->sort_order); }
    if (c->sort_buf) cudaFree(c->sort_buf);
    c->sort_key = c->sort_rank = c->sort_order = nullptr;
    c->sort_buf = nullptr;
    c->sort_cap = 0;
    JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_key, (size_t)np * sizeof(int)));
    JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_rank, (size_t)np * sizeof(int)));
    JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_order, (size_t)np * sizeof(int)));
    c->sort_cap = np;
    c->sort_gen++;  // a captured PIC-step graph that scatters into the old buffers must not be replayed (jefi_pic_step compares this)
  }
  return JEFI_OK;
}

// Builds c->sort_order: the depositing particles grouped by base node, then everything else (dead, or with no node in
// the grid).  The number of depositing particles is the offset of the last bin, c->sort_offset[sort_bins].
static int build_cell_order(jefi_ctx* c, long np, const float* x, const float* y, const float* z, const unsigned char* alive) {
  const jefi_dims& d = c->dims;
  int rc = ensure_sort_scratch(c, np);
  if (rc != JEFI_OK) return rc;
  const long nbins = sort_bins(c), nb = nbins + 1;
  const int ntiles = (int)((nb + SCAN_TILE - 1) / SCAN_TILE);
  const unsigned pb = (unsigned)((np + 255) / 256);
  JEFI_CUDA_TRY(c, cudaMemsetAsync(c->sort_count, 0, (size_t)nb * sizeof(unsigned), c->stream));
  if (c->shape_order == 2)
    k_sort_keys<2><<<pb, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, (int)nbins, np, x, y, z, alive, c->sort_key, c->sort_rank, c->sort_count);
  else
    k_sort_keys<1><<<pb, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, (int)nbins, np, x, y, z, alive, c->sort_key, c->sort_rank, c->sort_count);
  k_scan_tiles<<<ntiles, SCAN_THREADS, 0, c->stream>>>(c->sort_count, c->sort_offset, nb, c->sort_sums);
  k_scan_sums<<<1, 1024, 0, c->stream>>>(c->sort_sums, ntiles);
  k_scan_add<<<(unsigned)((nb + 255) / 256), 256, 0, c->stream>>>(c->sort_offset, nb, c->sort_sums);
  k_sort_scatter<<<pb, 256, 0, c->stream>>>(np, c->sort_key, c->sort_rank, c->sort_offset, c->sort_order);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches += 5;
  return JEFI_OK;
}

extern "C" int jefi_deposit(jefi_ctx* c, long np, const float* x, const float* y, const float* z, const float* ux,
                            const float* uy, const float* uz, const float* qw, const unsigned char* alive, float* rho,
                            float* jx, float* jy, float* jz) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (np < 0 || np > 0x7fffffffL || !rho || !jx || !jy || !jz || (np > 0 && (!x || !y || !z || !ux || !uy || !uz || !qw))) {
    c->err = "jefi_deposit: NULL array or np out of range";
    return JEFI_EINVAL;
  }
  return jefi_deposit_impl(c, np, x, y, z, ux, uy, uz, qw, alive, rho, jx, jy, jz);
}

int jefi_prepare_deposit_scratch(jefi_ctx* c, long np) {
  int mode = c->cfg.deposit_mode;
  return (mode == JEFI_DEPOSIT_SORTED && np > 0) ? ensure_sort_scratch(c, np) : JEFI_OK;
}

int jefi_deposit_impl(jefi_ctx* c, long np, const float* x, const float* y, const float* z, const float* ux, const float* uy,
                      const float* uz, const float* qw, const unsigned char* alive, float* rho, float* jx, float* jy, float* jz) {
  const jefi_dims& d = c->dims;
  if (jx == rho + d.N && jy == jx + d.N && jz == jy + d.N) {  // one [4][N] block (the usual case): one memset node
    JEFI_CUDA_TRY(c, cudaMemsetAsync(rho, 0, 4 * d.N * sizeof(float), c->stream));
  } else {
    JEFI_CUDA_TRY(c, cudaMemsetAsync(rho, 0, d.N * sizeof(float), c->stream));
    JEFI_CUDA_TRY(c, cudaMemsetAsync(jx, 0, d.N * sizeof(float), c->stream));
    JEFI_CUDA_TRY(c, cudaMemsetAsync(jy, 0, d.N * sizeof(float), c->stream));
    JEFI_CUDA_TRY(c, cudaMemsetAsync(jz, 0, d.N * sizeof(float), c->stream));
  }
  if (np == 0) return JEFI_OK;
  float inv_dV = (float)(1.0 / (c->cfg.dx * c->cfg.dy * c->cfg.dz));
  static_assert(32 * DEP_WARPS == 256, "one block size for every deposit kernel");
  unsigned blocks = (unsigned)((np + 255) / 256);
  int mode = c->cfg.deposit_mode;
  if (mode == JEFI_DEPOSIT_AUTO) mode = JEFI_DEPOSIT_RUNS;  // cheapest on sorted and unsorted lists alike
  const float cc = (float)c->c;
  const bool s2 = c->shape_order == 2;
  // Two kernels combine runs of equal cells (both correct for any order).  On a cell-sorted list (a few particles per cell,
  // most runs short) the segmented shuffle reduction of k_deposit_sorted is the cheaper one (config-5 set: 0.214 ms against
  // 0.253 ms); on a list in arbitrary order, where every lane is its own run and the L2 reductions bind, k_deposit_runs issues one
  // 32-lane reduction per particle covering its 8 nodes x 4 grids (half the L2 sectors: 0.82 ms against 1.44 ms).  The context
  // takes the first when the caller's list was put in cell order by jefi_sort_particles within the last 64 deposits.
  const bool sorted_hint = c->sorted_np == np && c->deposits_since_sort < 64;
  if (c->deposits_since_sort < (1 << 30)) c->deposits_since_sort++;
  if (mode == JEFI_DEPOSIT_SORTED) {
    int rc = build_cell_order(c, np, x, y, z, alive);
    if (rc != JEFI_OK) return rc;
    const unsigned* na = c->sort_offset + sort_bins(c);
    if (s2) k_deposit_sorted<2><<<blocks, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, na, c->sort_order, alive, x, y, z, ux, uy, uz, qw, rho, jx, jy, jz);
    else k_deposit_sorted<1><<<blocks, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, na, c->sort_order, alive, x, y, z, ux, uy, uz, qw, rho, jx, jy, jz);
  } else if (mode == JEFI_DEPOSIT_RUNS) {
    if (s2) k_deposit_sorted<2><<<blocks, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, nullptr, nullptr, alive, x, y, z, ux, uy, uz, qw, rho, jx, jy, jz);
    else if (sorted_hint) k_deposit_sorted<1><<<blocks, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, nullptr, nullptr, alive, x, y, z, ux, uy, uz, qw, rho, jx, jy, jz);
    else k_deposit_runs<<<blocks, 32 * DEP_WARPS, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, nullptr, nullptr, alive, x, y, z, ux, uy, uz, qw, rho, jx, jy, jz);
  } else {
    if (s2) k_deposit<2><<<blocks, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, x, y, z, ux, uy, uz, qw, alive, rho, jx, jy, jz);
    else k_deposit<1><<<blocks, 256, 0, c->stream>>>(d.nx, d.ny, d.nz, inv_dV, cc, np, x, y, z, ux, uy, uz, qw, alive, rho, jx, jy, jz);
  }
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  return JEFI_OK;
}

// The internal cell order for these positions (debug/parity export; synchronises).
extern "C" int jefi_debug_cell_order(jefi_ctx* c, long np, const float* x, const float* y, const float* z,
                                     const unsigned char* alive, int* order_out, long* n_alive_host) {
  if (!c || np < 0 || np > 0x7fffffffL || !n_alive_host || (np > 0 && (!x || !y || !z || !order_out))) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  *n_alive_host = 0;
  if (np == 0) return JEFI_OK;
  int rc = build_cell_order(c, np, x, y, z, alive);
  if (rc != JEFI_OK) return rc;
  unsigned na = 0;
  JEFI_CUDA_TRY(c, cudaMemcpyAsync(&na, c->sort_offset + sort_bins(c), sizeof na, cudaMemcpyDeviceToHost, c->stream));
  JEFI_CUDA_TRY(c, cudaMemcpyAsync(order_out, c->sort_order, (size_t)np * sizeof(int), cudaMemcpyDeviceToDevice, c->stream));
  JEFI_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  *n_alive_host = (long)na;
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// jefi_sort_particles: the caller asks for its own arrays to be put in cell order (gather through the order into
// context scratch with coalesced writes, then a coalesced copy back).
// ------------------------------------------------------------------------------------------------------------
struct perm_arrays {
  float* f[8];          // x y z ux uy uz qw qm
  unsigned char* alive;
  int* tag;             // may be NULL
};
__global__ void __launch_bounds__(256) k_permute_gather(long np, const int* __restrict__ order, perm_arrays A, float* __restrict__ buf,
                                                        unsigned char* __restrict__ abuf, int* __restrict__ tbuf) {
  long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= np) return;
  const int p = order[t];
#pragma unroll
  for (int a = 0; a < 8; a++) buf[(size_t)a * np + t] = A.f[a][p];
  abuf[t] = A.alive[p];
  if (A.tag) tbuf[t] = A.tag[p];
}
__global__ void __launch_bounds__(256) k_permute_copyback(long np, perm_arrays A, const float* __restrict__ buf,
                                                          const unsigned char* __restrict__ abuf, const int* __restrict__ tbuf) {
  long t = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= np) return;
#pragma unroll
  for (int a = 0; a < 8; a++) A.f[a][t] = buf[(size_t)a * np + t];
  A.alive[t] = abuf[t];
  if (A.tag) A.tag[t] = tbuf[t];
}

extern "C" int jefi_sort_particles(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz, float* qw,
                                   float* q_over_m, unsigned char* alive, int* tag) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (np < 0 || np > 0x7fffffffL || (np > 0 && (!x || !y || !z || !ux || !uy || !uz || !qw || !q_over_m || !alive))) {
    c->err = "jefi_sort_particles: NULL array or np out of range";
    return JEFI_EINVAL;
  }
  if (np == 0) return JEFI_OK;
  int rc = build_cell_order(c, np, x, y, z, alive);
  if (rc != JEFI_OK) return rc;
  if (!c->sort_buf) JEFI_CUDA_TRY(c, cudaMalloc(&c->sort_buf, (size_t)c->sort_cap * (8 * sizeof(float) + sizeof(int) + 1) + 64));
  float* buf = (float*)c->sort_buf;
  int* tbuf = (int*)(buf + (size_t)8 * c->sort_cap);
  unsigned char* abuf = (unsigned char*)(tbuf + c->sort_cap);
  perm_arrays A;
  A.f[0] = x; A.f[1] = y; A.f[2] = z; A.f[3] = ux; A.f[4] = uy; A.f[5] = uz; A.f[6] = qw; A.f[7] = q_over_m;
  A.alive = alive; A.tag = tag;
  const unsigned pb = (unsigned)((np + 255) / 256);
  k_permute_gather<<<pb, 256, 0, c->stream>>>(np, c->sort_order, A, buf, abuf, tbuf);
  k_permute_copyback<<<pb, 256, 0, c->stream>>>(np, A, buf, abuf, tbuf);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches += 2;
  c->sorted_np = np;
  c->deposits_since_sort = 0;
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// interpolation + Boris + kill: one thread per particle
// ------------------------------------------------------------------------------------------------------------
struct push_consts {
  int nx, ny, nz;
  float half_dt_over_c;  // dt/(2c): u += (q/m) * this * E
  float half_dt;         // dt/2:    t = (q/m) * this * B / gamma
  float sx, sy, sz;      // c dt / dx ...: grid-unit displacement = (u/gamma) * s
  float Eext[3], Bext[3];
};

// E, B of a node packed into two float4 (Ex, Ey, Ez, Bx | By, Bz, 0, 0): the push then gathers 16 quads per particle instead
// of 48 words (one sector per node when the lanes of a warp sit in the same cell).  24 N bytes in, 32 N out per step.
__global__ void __launch_bounds__(256) k_pack_fields(long N, const float* __restrict__ ex, const float* __restrict__ ey,
                                                     const float* __restrict__ ez, const float* __restrict__ bx,
                                                     const float* __restrict__ by, const float* __restrict__ bz,
                                                     float4* __restrict__ pack) {
  long n = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  pack[2 * n] = make_float4(ex[n], ey[n], ez[n], bx[n]);
  pack[2 * n + 1] = make_float4(by[n], bz[n], 0.f, 0.f);
}

#ifndef JEFI_PUSH_MINBLOCKS
#define JEFI_PUSH_MINBLOCKS 8  /* 32 registers: 100 % occupancy; measured 0.239 -> 0.183 ms on the sorted config-5 list */
#endif
template <bool PACKED, int ORDER>
__global__ void __launch_bounds__(256, ORDER == 1 ? JEFI_PUSH_MINBLOCKS : 4) k_push(push_consts K, long np, float* __restrict__ x, float* __restrict__ y,
                                              float* __restrict__ z, float* __restrict__ ux, float* __restrict__ uy,
                                              float* __restrict__ uz, const float* __restrict__ qm,
                                              unsigned char* __restrict__ alive, const float* __restrict__ ex,
                                              const float* __restrict__ ey, const float* __restrict__ ez,
                                              const float* __restrict__ bx, const float* __restrict__ by,
                                              const float* __restrict__ bz, const float4* __restrict__ pack) {
  constexpr int NN = ORDER + 1;
  long p = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np || alive[p] == 0) return;
  float xp = x[p], yp = y[p], zp = z[p];
  axis_stencil<ORDER> nx_, ny_, nz_;
  nx_.set(xp); ny_.set(yp); nz_.set(zp);
  float E0 = 0, E1 = 0, E2 = 0, B0 = 0, B1 = 0, B2 = 0;
#pragma unroll
  for (int c = 0; c < NN; c++)
#pragma unroll
    for (int b = 0; b < NN; b++)
#pragma unroll
      for (int a = 0; a < NN; a++) {  // Eq. (2.20); virtual nodes count as zero
        int ii = nx_.i0 + a, jj = ny_.i0 + b, kk = nz_.i0 + c;
        if (ii >= 0 && ii < K.nx && jj >= 0 && jj < K.ny && kk >= 0 && kk < K.nz) {
          float w = nx_.w[a] * ny_.w[b] * nz_.w[c];
          long node = (long)ii + (long)K.nx * ((long)jj + (long)K.ny * kk);
          if (PACKED) {
            const float4 f0 = __ldg(pack + 2 * node), f1 = __ldg(pack + 2 * node + 1);
            E0 = fmaf(w, f0.x, E0); E1 = fmaf(w, f0.y, E1); E2 = fmaf(w, f0.z, E2);
            B0 = fmaf(w, f0.w, B0); B1 = fmaf(w, f1.x, B1); B2 = fmaf(w, f1.y, B2);
          } else {
            E0 = fmaf(w, __ldg(ex + node), E0); E1 = fmaf(w, __ldg(ey + node), E1); E2 = fmaf(w, __ldg(ez + node), E2);
            B0 = fmaf(w, __ldg(bx + node), B0); B1 = fmaf(w, __ldg(by + node), B1); B2 = fmaf(w, __ldg(bz + node), B2);
          }
        }
      }
  E0 += K.Eext[0]; E1 += K.Eext[1]; E2 += K.Eext[2];
  B0 += K.Bext[0]; B1 += K.Bext[1]; B2 += K.Bext[2];
  const float qom = qm[p];
  const float he = qom * K.half_dt_over_c, hb = qom * K.half_dt;
  // Eq. (2.9): half electric kick
  float umx = fmaf(he, E0, ux[p]), umy = fmaf(he, E1, uy[p]), umz = fmaf(he, E2, uz[p]);
  // Eq. (2.10): rotation, gamma taken at u^-
  float igm = 1.0f / sqrtf(1.f + umx * umx + umy * umy + umz * umz);
  float tx = hb * B0 * igm, ty = hb * B1 * igm, tz = hb * B2 * igm;
  float upx = umx + (umy * tz - umz * ty);
  float upy = umy + (umz * tx - umx * tz);
  float upz = umz + (umx * ty - umy * tx);
  float sc = 2.f / (1.f + tx * tx + ty * ty + tz * tz);
  float sx = tx * sc, sy = ty * sc, sz = tz * sc;
  float uqx = umx + (upy * sz - upz * sy);
  float uqy = umy + (upz * sx - upx * sz);
  float uqz = umz + (upx * sy - upy * sx);
  // Eq. (2.11): second half kick
  float unx = fmaf(he, E0, uqx), uny = fmaf(he, E1, uqy), unz = fmaf(he, E2, uqz);
  float ign = 1.0f / sqrtf(1.f + unx * unx + uny * uny + unz * unz);
  // Eq. (2.8) in grid units
  float xn = fmaf(unx * ign, K.sx, xp), yn = fmaf(uny * ign, K.sy, yp), zn = fmaf(unz * ign, K.sz, zp);
  ux[p] = unx; uy[p] = uny; uz[p] = unz;
  x[p] = xn; y[p] = yn; z[p] = zn;
  if (xn < 0.f || xn >= (float)K.nx || yn < 0.f || yn >= (float)K.ny || zn < 0.f || zn >= (float)K.nz) alive[p] = 0;
}

static push_consts make_push_consts(const jefi_ctx* c) {
  const jefi_dims& d = c->dims;
  push_consts K;
  K.nx = d.nx; K.ny = d.ny; K.nz = d.nz;
  K.half_dt_over_c = (float)(c->cfg.dt / (2.0 * c->c));
  K.half_dt = (float)(c->cfg.dt / 2.0);
  K.sx = (float)(c->c * c->cfg.dt / c->cfg.dx); K.sy = (float)(c->c * c->cfg.dt / c->cfg.dy); K.sz = (float)(c->c * c->cfg.dt / c->cfg.dz);
  for (int a = 0; a < 3; a++) { K.Eext[a] = (float)c->cfg.Eext[a]; K.Bext[a] = (float)c->cfg.Bext[a]; }
  return K;
}

template <bool PACKED>
static void launch_push(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz, const float* q_over_m,
                        unsigned char* alive, const float* ex, const float* ey, const float* ez, const float* bx, const float* by,
                        const float* bz, const float4* pack) {
  const push_consts K = make_push_consts(c);
  const unsigned blocks = (unsigned)((np + 255) / 256);
  if (c->shape_order == 2)
    k_push<PACKED, 2><<<blocks, 256, 0, c->stream>>>(K, np, x, y, z, ux, uy, uz, q_over_m, alive, ex, ey, ez, bx, by, bz, pack);
  else
    k_push<PACKED, 1><<<blocks, 256, 0, c->stream>>>(K, np, x, y, z, ux, uy, uz, q_over_m, alive, ex, ey, ez, bx, by, bz, pack);
  c->launches++;
}

extern "C" int jefi_push_particles(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz,
                                   const float* q_over_m, unsigned char* alive, const float* ex, const float* ey,
                                   const float* ez, const float* bx, const float* by, const float* bz) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (np < 0 || !ex || !ey || !ez || !bx || !by || !bz || (np > 0 && (!x || !y || !z || !ux || !uy || !uz || !q_over_m || !alive))) {
    c->err = "jefi_push_particles: NULL array or negative np";
    return JEFI_EINVAL;
  }
  if (np == 0) return JEFI_OK;
  const jefi_dims& d = c->dims;
  if (np >= d.N) {  // enough particles per node for a packed copy of the fields to pay for itself (jefi_field_step_packed +
                    // jefi_push_particles_packed avoid this pass altogether)
    if (!c->eb_pack) JEFI_CUDA_TRY(c, cudaMalloc(&c->eb_pack, (size_t)d.N * 2 * sizeof(float4)));
    k_pack_fields<<<(unsigned)((d.N + 255) / 256), 256, 0, c->stream>>>(d.N, ex, ey, ez, bx, by, bz, c->eb_pack);
    c->launches++;
    launch_push<true>(c, np, x, y, z, ux, uy, uz, q_over_m, alive, ex, ey, ez, bx, by, bz, c->eb_pack);
  } else {
    launch_push<false>(c, np, x, y, z, ux, uy, uz, q_over_m, alive, ex, ey, ez, bx, by, bz, nullptr);
  }
  JEFI_CUDA_TRY(c, cudaGetLastError());
  return JEFI_OK;
}

extern "C" int jefi_push_particles_packed(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz,
                                          const float* q_over_m, unsigned char* alive, const float* eb_packed) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (np < 0 || !eb_packed || ((uintptr_t)eb_packed & 15u) || (np > 0 && (!x || !y || !z || !ux || !uy || !uz || !q_over_m || !alive))) {
    c->err = "jefi_push_particles_packed: NULL or misaligned array, or negative np";
    return JEFI_EINVAL;
  }
  return jefi_push_packed_impl(c, np, x, y, z, ux, uy, uz, q_over_m, alive, eb_packed);
}

int jefi_push_packed_impl(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz, const float* q_over_m,
                          unsigned char* alive, const float* eb_packed) {
  if (np == 0) return JEFI_OK;
  launch_push<true>(c, np, x, y, z, ux, uy, uz, q_over_m, alive, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr,
                    reinterpret_cast<const float4*>(eb_packed));
  JEFI_CUDA_TRY(c, cudaGetLastError());
  return JEFI_OK;
}

template <int ORDER>
__global__ void __launch_bounds__(256) k_cell_index(long np, const float* __restrict__ x, const float* __restrict__ y,
                                                    const float* __restrict__ z, int* __restrict__ ijk) {
  long p = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= np) return;
  axis_stencil<ORDER> sx, sy, sz;
  sx.set(x[p]); sy.set(y[p]); sz.set(z[p]);
  constexpr int C = ORDER - 1;  // order 2: report the centre node i0 + 1
  ijk[3 * p] = sx.i0 + C; ijk[3 * p + 1] = sy.i0 + C; ijk[3 * p + 2] = sz.i0 + C;
}

extern "C" int jefi_debug_cell_index(jefi_ctx* c, long np, const float* x, const float* y, const float* z, int* ijk_out) {
  if (!c || np < 0 || (np > 0 && (!x || !y || !z || !ijk_out))) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (np == 0) return JEFI_OK;
  if (c->shape_order == 2) k_cell_index<2><<<(unsigned)((np + 255) / 256), 256, 0, c->stream>>>(np, x, y, z, ijk_out);
  else k_cell_index<1><<<(unsigned)((np + 255) / 256), 256, 0, c->stream>>>(np, x, y, z, ijk_out);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  JEFI_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// jefi_deposit_static: the cell-sorted CIC deposit for callers that must not allocate (include/jefi.h has the contract).
//
// Who needs this.  Some programs that link libjefi are not free to call cudaMalloc at the moment they want a deposit: a host
// application that gave the whole device to its own memory pool at start-up and allows no driver allocation afterwards (a
// second allocator would overrun or fragment its budget, and a late cudaMalloc may simply fail there), or a step loop with a
// latency bound (cudaMalloc and cudaFree can synchronise the whole device and take an unbounded time).
// jefi_deposit with JEFI_DEPOSIT_SORTED grows context scratch with cudaMalloc on first use and whenever np grows; this entry
// point does the same arithmetic with the same kernels, but every byte of its scratch (sort keys, ranks, the cell order, bin
// counts, bin offsets, scan sums) lives in the fixed array below, which the library's CUDA module carries: each GPU the
// library is loaded on reserves it when that module is loaded there, and holds it until the process exits.  No context is needed either.
//
// The array is shared by all calls on a device and is NOT cleared between them.  Only the bin counters have to start at zero
// (one cudaMemsetAsync on the caller's stream per call); keys, ranks, order, offsets and scan sums are fully rewritten for
// the first np particles / the bins of this grid before any kernel of the same call reads them, so whatever an earlier call
// on another grid or a longer list left behind is never looked at.  Two calls that run on the GPU at the same time (different
// streams, or two host threads) would sort into the same memory and corrupt each other: callers serialise them.
// ------------------------------------------------------------------------------------------------------------
namespace {
constexpr long ST_MAX_NP = JEFI_STATIC_MAX_PARTICLES;
constexpr long ST_MAX_BINS = JEFI_STATIC_MAX_BINS;                                  // (nx+1)(ny+1)(nz+1) + 1 must fit
constexpr long ST_MAX_SCAN_TILES = (ST_MAX_BINS + SCAN_TILE - 1) / SCAN_TILE;
constexpr size_t st_round(size_t b) { return (b + 255) & ~(size_t)255; }
constexpr size_t ST_OFF_KEY = 0;
constexpr size_t ST_OFF_RANK = ST_OFF_KEY + st_round(ST_MAX_NP * sizeof(int));
constexpr size_t ST_OFF_ORDER = ST_OFF_RANK + st_round(ST_MAX_NP * sizeof(int));
constexpr size_t ST_OFF_COUNT = ST_OFF_ORDER + st_round(ST_MAX_NP * sizeof(int));
constexpr size_t ST_OFF_OFFSET = ST_OFF_COUNT + st_round(ST_MAX_BINS * sizeof(unsigned));
constexpr size_t ST_OFF_SUMS = ST_OFF_OFFSET + st_round(ST_MAX_BINS * sizeof(unsigned));
constexpr size_t ST_BYTES = ST_OFF_SUMS + st_round((ST_MAX_SCAN_TILES + 1) * sizeof(unsigned));
static_assert(ST_BYTES <= JEFI_STATIC_SCRATCH_BYTES, "include/jefi.h states the size of the static scratch");
constexpr int ST_MAX_DEVICES = 64;
}  // namespace

// The scratch itself.  In host code this name is only a handle for the runtime (a host-side shadow symbol), not a device
// address: kernels get the address cudaGetSymbolAddress returns for the device that is current (static_scratch_base).
static __device__ __align__(256) unsigned char g_jefi_static_scratch[JEFI_STATIC_SCRATCH_BYTES];

static std::mutex g_static_mu;
static unsigned char* g_static_base[ST_MAX_DEVICES];  // per device ordinal; NULL until the first call on that device

// Device address of the scratch on `device`, which must be the current device.  Looked up once per device.
static cudaError_t static_scratch_base(int device, unsigned char** base) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_base[device]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_jefi_static_scratch);
    if (e != cudaSuccess) return e;
    g_static_base[device] = static_cast<unsigned char*>(p);
  }
  *base = g_static_base[device];
  return cudaSuccess;
}

static int static_fail(char* errbuf, int errbuf_len, int code, const std::string& msg) {
  if (errbuf && errbuf_len > 0) {
    const size_t n = msg.size() < (size_t)errbuf_len - 1 ? msg.size() : (size_t)errbuf_len - 1;
    memcpy(errbuf, msg.data(), n);
    errbuf[n] = 0;
  }
  return code;
}

extern "C" int jefi_deposit_static(int device, void* stream, int nx, int ny, int nz, double dx, double dy, double dz, double c,
                                   long np, const float* x, const float* y, const float* z, const float* ux, const float* uy,
                                   const float* uz, const float* qw, const unsigned char* alive, float* rho, float* jx,
                                   float* jy, float* jz, char* errbuf, int errbuf_len) {
  if (errbuf && errbuf_len > 0) errbuf[0] = 0;
  // ---- argument checks: before any CUDA call ----
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || c < 0)
    return static_fail(errbuf, errbuf_len, JEFI_EINVAL, "jefi_deposit_static: nx, ny, nz >= 1 and dx, dy, dz > 0 are required");
  if (np < 0 || !rho || !jx || !jy || !jz || (np > 0 && (!x || !y || !z || !ux || !uy || !uz || !qw)))
    return static_fail(errbuf, errbuf_len, JEFI_EINVAL, "jefi_deposit_static: NULL array or negative np");
  if (np > ST_MAX_NP)
    return static_fail(errbuf, errbuf_len, JEFI_EINVAL,
                       "jefi_deposit_static: np = " + std::to_string(np) + " exceeds JEFI_STATIC_MAX_PARTICLES = " +
                           std::to_string(ST_MAX_NP) + " (the static scratch is fixed; use jefi_deposit for longer lists)");
  const long nbins = (long)(nx + 1) * (ny + 1) * (nz + 1), nb = nbins + 1;
  if (nb > ST_MAX_BINS)
    return static_fail(errbuf, errbuf_len, JEFI_EINVAL,
                       "jefi_deposit_static: (nx+1)(ny+1)(nz+1)+1 = " + std::to_string(nb) + " sort bins exceed JEFI_STATIC_MAX_BINS = " +
                           std::to_string(ST_MAX_BINS) + " (the static scratch is fixed; use jefi_deposit for larger grids)");
  if (device < 0 || device >= ST_MAX_DEVICES)
    return static_fail(errbuf, errbuf_len, JEFI_EINVAL, "jefi_deposit_static: device ordinal out of range");
  // ---- make `device` current for the rest of the call ----
  struct guard_t {
    int prev = -1;
    bool switched = false;
    ~guard_t() { if (switched) cudaSetDevice(prev); }
  } guard;
  cudaError_t e = cudaGetDevice(&guard.prev);
  if (e == cudaSuccess && guard.prev != device) {
    e = cudaSetDevice(device);
    guard.switched = e == cudaSuccess;
  }
  unsigned char* base = nullptr;
  if (e == cudaSuccess) e = static_scratch_base(device, &base);
  if (e != cudaSuccess) return static_fail(errbuf, errbuf_len, JEFI_ECUDA, std::string("jefi_deposit_static: set-up: ") + cudaGetErrorString(e));
  int* key = reinterpret_cast<int*>(base + ST_OFF_KEY);
  int* rank = reinterpret_cast<int*>(base + ST_OFF_RANK);
  int* order = reinterpret_cast<int*>(base + ST_OFF_ORDER);
  unsigned* count = reinterpret_cast<unsigned*>(base + ST_OFF_COUNT);
  unsigned* offset = reinterpret_cast<unsigned*>(base + ST_OFF_OFFSET);
  unsigned* sums = reinterpret_cast<unsigned*>(base + ST_OFF_SUMS);
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  const size_t N = (size_t)nx * ny * nz;
#define ST_TRY(call)                                                                                                       \
  do {                                                                                                                     \
    cudaError_t e__ = (call);                                                                                              \
    if (e__ != cudaSuccess) return static_fail(errbuf, errbuf_len, JEFI_ECUDA, std::string("jefi_deposit_static: " #call ": ") + cudaGetErrorString(e__)); \
  } while (0)
  // outputs are overwritten, as in jefi_deposit
  ST_TRY(cudaMemsetAsync(rho, 0, N * sizeof(float), st));
  ST_TRY(cudaMemsetAsync(jx, 0, N * sizeof(float), st));
  ST_TRY(cudaMemsetAsync(jy, 0, N * sizeof(float), st));
  ST_TRY(cudaMemsetAsync(jz, 0, N * sizeof(float), st));
  if (np == 0) return JEFI_OK;
  // the one part of the shared scratch that must start at zero: this grid's bin counters (the previous call's are stale)
  ST_TRY(cudaMemsetAsync(count, 0, (size_t)nb * sizeof(unsigned), st));
  const int ntiles = (int)((nb + SCAN_TILE - 1) / SCAN_TILE);
  const unsigned pb = (unsigned)((np + 255) / 256);
  k_sort_keys<1><<<pb, 256, 0, st>>>(nx, ny, nz, (int)nbins, np, x, y, z, alive, key, rank, count);
  k_scan_tiles<<<ntiles, SCAN_THREADS, 0, st>>>(count, offset, nb, sums);
  k_scan_sums<<<1, 1024, 0, st>>>(sums, ntiles);
  k_scan_add<<<(unsigned)((nb + 255) / 256), 256, 0, st>>>(offset, nb, sums);
  k_sort_scatter<<<pb, 256, 0, st>>>(np, key, rank, offset, order);
  const float inv_dV = (float)(1.0 / (dx * dy * dz));
  const float cc = (float)(c > 0 ? c : 299792458.0);
  k_deposit_sorted<1><<<pb, 256, 0, st>>>(nx, ny, nz, inv_dV, cc, np, offset + nbins, order, alive, x, y, z, ux, uy, uz, qw, rho, jx, jy, jz);
  ST_TRY(cudaGetLastError());
#undef ST_TRY
  return JEFI_OK;
}
