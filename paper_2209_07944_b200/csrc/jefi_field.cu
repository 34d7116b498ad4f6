// libjefi: the Jefimenko field gather (SURVEY.md §8 row a3; PAPER.md:103-109 Eqs. 2.4-2.6, :221 self cell).
//
// In scaled units d' = d/(c dt), s = |d'|, rs = 1/s, Jt = J/c, D* = backward difference over one step:
//   E = prefE * sum [ d' (rho rs^3 + Drho rs^2) - DJt rs ]          (Eq. 2.4)
//   B = prefB * sum [ d' x (Jt rs^3 + DJt rs^2) ]                    (Eq. 2.5)
// sources taken from ring slot (n - m) mod H with m = round(s) (Eq. 2.6, nearest-step reading).
//
// Two kernels:
//   k_field_reference  one thread per observation cell, all sources, delays from the fp64-built table.
//   k_field_tiled      256-thread CTA owns an 8x8x8 observation tile (2 cells per thread), walks the 4x4x4 source
//                      tiles, stages each tile's slot window [m_lo, m_hi] in shared memory with cp.async and
//                      evaluates pairs with the source cell warp-uniform and the delay per lane.
#include <stdio.h>

#include "jefi_ctx.h"

// ------------------------------------------------------------------------------------------------------------
// reference kernel
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_field_reference(jefi_dims d, jefi_geom g, int ex_, int ey_, long n,
                                                         const int* __restrict__ mtab, const float4* __restrict__ ringS,
                                                         const float4* __restrict__ ringD, float* __restrict__ ex,
                                                         float* __restrict__ ey, float* __restrict__ ez,
                                                         float* __restrict__ bx, float* __restrict__ by,
                                                         float* __restrict__ bz) {
  long oc = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (oc >= d.N) return;
  const int I = (int)(oc % d.nx), J = (int)((oc / d.nx) % d.ny), K = (int)(oc / ((long)d.nx * d.ny));
  float aex = 0, aey = 0, aez = 0, abx = 0, aby = 0, abz = 0;
  for (int k = 0; k < d.nz; k++) {
    float lex = 0, ley = 0, lez = 0, lbx = 0, lby = 0, lbz = 0;  // per-plane partial sums (two-level accumulation)
    for (int j = 0; j < d.ny; j++)
      for (int i = 0; i < d.nx; i++) {
        if (i == I && j == J && k == K) continue;
        int di = I - i, dj = J - j, dk = K - k;
        int m = mtab[abs(di) + (long)ex_ * (abs(dj) + (long)ey_ * abs(dk))];
        long t = n - m;
        if (m > d.H - 2 || t < 0) continue;  // A15; zero before t0
        size_t idx = (size_t)jefi_ring_cell(d, i, j, k) * d.H + (size_t)(t % d.H);
        float4 S = ringS[idx], D = ringD[idx];
        float ax = g.kx * (float)di, ay = g.ky * (float)dj, az = g.kz * (float)dk;
        float q = fmaf(ax, ax, fmaf(ay, ay, az * az));
        float rs = rsqrtf(q), rs2 = rs * rs, rs3 = rs2 * rs;
        float qq = fmaf(rs2, D.x, rs3 * S.x);
        lex = fmaf(ax, qq, lex); ley = fmaf(ay, qq, ley); lez = fmaf(az, qq, lez);
        lex = fmaf(-rs, D.y, lex); ley = fmaf(-rs, D.z, ley); lez = fmaf(-rs, D.w, lez);
        float wx = fmaf(rs2, D.y, rs3 * S.y), wy = fmaf(rs2, D.z, rs3 * S.z), wz = fmaf(rs2, D.w, rs3 * S.w);
        lbx = fmaf(ay, wz, lbx); lbx = fmaf(-az, wy, lbx);
        lby = fmaf(az, wx, lby); lby = fmaf(-ax, wz, lby);
        lbz = fmaf(ax, wy, lbz); lbz = fmaf(-ay, wx, lbz);
      }
    aex += lex; aey += ley; aez += lez; abx += lbx; aby += lby; abz += lbz;
  }
  ex[oc] = g.prefE * aex; ey[oc] = g.prefE * aey; ez[oc] = g.prefE * aez;
  bx[oc] = g.prefB * abx; by[oc] = g.prefB * aby; bz[oc] = g.prefB * abz;
}

int jefi_launch_field_reference(jefi_ctx* c, float* ex, float* ey, float* ez, float* bx, float* by, float* bz) {
  const jefi_dims& d = c->dims;
  unsigned blocks = (unsigned)((d.N + 127) / 128);
  k_field_reference<<<blocks, 128, 0, c->stream>>>(d, c->geom, jefi_table_extent(d.nx), jefi_table_extent(d.ny), c->step,
                                                   c->mtab_dev, c->ringS, c->ringD, ex, ey, ez, bx, by, bz);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// tiled kernel
//
// CTA = 256 threads = one 8x8x8 observation tile (512 cells, two per thread); 2 CTAs per SM.
// For every 4x4x4 source tile the CTA stages, per source cell, the window of ring slots [m_lo, m_hi] that the tile
// pair can address (m from the extreme offsets), S window and D window, with one TMA bulk copy per (cell, array)
// (cp.async.bulk + mbarrier; the ring layout [tile][cell][slot] makes each window one contiguous run, two when the
// ring wraps).  Shared-memory index j = m_hi - m, so that memory order equals slot order.
//
// Pair evaluation: the source cell is warp-uniform, the delay per lane:
//   q = |d'|^2 (1 FFMA), rs = rsqrt(q) (MUFU), t = q*rs + 1.5*2^23 (1 FFMA, integer m in the mantissa),
//   address = K - 16*bits(t) (1 IMAD), 2 x LDS.128, then 20 FP32 ops:
//   u = rs*S + D (4), r2 = rs^2 (1), a' = r2*d' (3), E += a'*u.x - rs*D.yzw (6), B += a' x u.yzw (6).
//
// Shared-memory delivery is the scarce resource: measured on B200, an LDS.128 takes 2 cycles when every quarter-warp
// (8 lanes) touches at most 2 distinct 16-byte words and 4 cycles otherwise.  Which lane evaluates which observation
// cell is free (any assignment gives the same sums), so for every source tile the 512 cells are taken in the order of
// their distance to the tile (half-slot buckets): 8 consecutive lanes are then almost equidistant from every source
// cell of the tile and ~95% of the loads run at the 2-cycle rate.  The order depends only on the relative tile
// offset; jefi_tiled_prepare tabulates it once (k_build_perm) and the kernel fetches the 1 KB row with the same
// mbarrier as the windows.  Per-tile partial sums are added to a shared-memory accumulator [6][512] (second level of
// the two-level accumulation), because a cell is evaluated by a different thread in every tile.
// ------------------------------------------------------------------------------------------------------------
constexpr int OB = 8;            // observation tile edge
constexpr int OBCELLS = OB * OB * OB;
constexpr int TILED_THREADS = 256;
constexpr int P_OBS = OBCELLS / TILED_THREADS;  // observation cells per thread

struct tiled_params {
  jefi_dims d;
  jefi_geom g;
  int n;           // current step
  int nslot;       // n mod H
  int nobx, noby, nobz;
  int ndx, ndy;    // extents of the permutation table in relative-offset space
  const float4* ringS;
  const float4* ringD;
  const unsigned short* perm;  // [ndz][ndy][ndx][512]
  float *ex, *ey, *ez, *bx, *by, *bz;
};

// ---- mbarrier / TMA bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk) ----
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// min / max of |a| over the integer interval [lo, hi]
__device__ __forceinline__ void abs_range(int lo, int hi, int& mn, int& mx) {
  int alo = abs(lo), ahi = abs(hi);
  mx = max(alo, ahi);
  mn = (lo <= 0 && hi >= 0) ? 0 : min(alo, ahi);
}

template <int IMM>
__device__ __forceinline__ float4 lds128_imm(uint32_t addr) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4+%5];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr), "n"(IMM));
  return v;
}

// One observation cell against one source cell.  K = shared address of the cell's S window + 16*(m_hi + MAGICBITS).
template <int WP, bool SELF, int CELL>
__device__ __forceinline__ void one_pair(uint32_t K, float ax, float ay, float az, float qyz, float (&loc)[6]) {
  constexpr int SOFF = CELL * WP * 16;
  constexpr int DOFF = SOFF + JEFI_TCELLS * WP * 16;
  float q = fmaf(ax, ax, qyz);
  float rs = jefi_rsqrt(q);
  if (SELF) rs = q > 0.f ? rs : 0.f;        // the self cell contributes exactly zero
  float t = fmaf(q, rs, JEFI_MAGIC);        // MAGIC + round(s): m sits in the mantissa
  uint32_t addr = K - (uint32_t)__float_as_int(t) * 16u;   // window entry j = m_hi - m
  const float4 S = lds128_imm<SOFF>(addr);
  const float4 D = lds128_imm<DOFF>(addr);
  float r2 = rs * rs;
  float u0 = fmaf(rs, S.x, D.x), u1 = fmaf(rs, S.y, D.y), u2 = fmaf(rs, S.z, D.z), u3 = fmaf(rs, S.w, D.w);
  float bxr = ax * r2, byr = ay * r2, bzr = az * r2;      // d' rs^2
  loc[0] = fmaf(bxr, u0, loc[0]); loc[1] = fmaf(byr, u0, loc[1]); loc[2] = fmaf(bzr, u0, loc[2]);
  loc[0] = fmaf(-rs, D.y, loc[0]); loc[1] = fmaf(-rs, D.z, loc[1]); loc[2] = fmaf(-rs, D.w, loc[2]);
  loc[3] = fmaf(byr, u3, loc[3]); loc[3] = fmaf(-bzr, u2, loc[3]);
  loc[4] = fmaf(bzr, u1, loc[4]); loc[4] = fmaf(-bxr, u3, loc[4]);
  loc[5] = fmaf(bxr, u2, loc[5]); loc[5] = fmaf(-byr, u1, loc[5]);
}

template <int WP, bool SELF, int LY>
__device__ __forceinline__ void one_row(uint32_t Kz, const float (&ax)[JEFI_TS], float ay, float az, float az2, float (&loc)[6]) {
  float qyz = fmaf(ay, ay, az2);
  one_pair<WP, SELF, JEFI_TS * LY + 0>(Kz, ax[0], ay, az, qyz, loc);
  one_pair<WP, SELF, JEFI_TS * LY + 1>(Kz, ax[1], ay, az, qyz, loc);
  one_pair<WP, SELF, JEFI_TS * LY + 2>(Kz, ax[2], ay, az, qyz, loc);
  one_pair<WP, SELF, JEFI_TS * LY + 3>(Kz, ax[3], ay, az, qyz, loc);
}

// one observation cell against the 64 cells of the staged source tile
template <int WP, bool SELF>
__device__ __forceinline__ void tile_pairs(uint32_t K, float kz, const float (&ax)[JEFI_TS], const float (&ay)[JEFI_TS], float fz0,
                                           float (&loc)[6]) {
#pragma unroll 1
  for (int lz = 0; lz < JEFI_TS; lz++) {
    const float az = kz * (fz0 - (float)lz);
    const float az2 = az * az;
    const uint32_t Kz = K + (uint32_t)(lz * JEFI_TS * JEFI_TS * WP * 16);
    one_row<WP, SELF, 0>(Kz, ax, ay[0], az, az2, loc);
    one_row<WP, SELF, 1>(Kz, ax, ay[1], az, az2, loc);
    one_row<WP, SELF, 2>(Kz, ax, ay[2], az, az2, loc);
    one_row<WP, SELF, 3>(Kz, ax, ay[3], az, az2, loc);
  }
}

template <int WP>
__global__ void __launch_bounds__(TILED_THREADS, 2) k_field_tiled(tiled_params P) {
  extern __shared__ __align__(128) unsigned char smem[];
  // dynamic shared memory: [S windows][D windows][accumulators 6 x 512 floats][permutation 512 x u16]
  constexpr uint32_t PITCHB = WP * 16;
  constexpr uint32_t DOFFB = JEFI_TCELLS * PITCHB;  // D window follows the S window
  float* accS = reinterpret_cast<float*>(smem + 2 * DOFFB);
  unsigned short* permS = reinterpret_cast<unsigned short*>(smem + 2 * DOFFB + 6 * OBCELLS * sizeof(float));
  __shared__ __align__(8) unsigned long long mbar_storage;
  const jefi_dims& d = P.d;
  const int tid = threadIdx.x;
  // observation tile of this CTA
  const int obx = blockIdx.x % P.nobx, oby = (blockIdx.x / P.nobx) % P.noby, obz = blockIdx.x / (P.nobx * P.noby);
  const int ox0 = obx * OB, oy0 = oby * OB, oz0 = obz * OB;

  for (int i = tid; i < 6 * OBCELLS; i += TILED_THREADS) accS[i] = 0.f;
  const uint32_t smS = (uint32_t)__cvta_generic_to_shared(smem);
  const uint32_t permA = (uint32_t)__cvta_generic_to_shared(permS);
  const uint32_t bar = (uint32_t)__cvta_generic_to_shared(&mbar_storage);
  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  uint32_t phase = 0;
  // thread -> (cell, array) of the bulk copies it issues
  const int cp_cell = tid & (JEFI_TCELLS - 1);
  const int cp_arr = tid >> 6;  // 0: S, 1: D, 2: permutation row (thread 128), 3: none

  int st = 0;
  for (int stz = 0; stz < d.ntz; stz++)
    for (int sty = 0; sty < d.nty; sty++)
      for (int stx = 0; stx < d.ntx; stx++, st++) {
        const int sx0 = stx * JEFI_TS, sy0 = sty * JEFI_TS, sz0 = stz * JEFI_TS;
        // slot window of this (observation tile, source tile) pair from the extreme offsets
        int mnx, mxx, mny, mxy, mnz, mxz;
        abs_range(ox0 - (sx0 + JEFI_TS - 1), ox0 + OB - 1 - sx0, mnx, mxx);
        abs_range(oy0 - (sy0 + JEFI_TS - 1), oy0 + OB - 1 - sy0, mny, mxy);
        abs_range(oz0 - (sz0 + JEFI_TS - 1), oz0 + OB - 1 - sz0, mnz, mxz);
        const bool self = (mnx == 0 && mny == 0 && mnz == 0);
        const int m_lo = self ? 0 : jefi_delay_fp32(jefi_q_fp32(P.g.kx, P.g.ky, P.g.kz, (float)mnx, (float)mny, (float)mnz));
        const int m_hi = jefi_delay_fp32(jefi_q_fp32(P.g.kx, P.g.ky, P.g.kz, (float)mxx, (float)mxy, (float)mxz));
        const int W = m_hi - m_lo + 1;  // <= WP (jefi_tiled_prepare)
        // window entry j <-> delay m = m_hi - j <-> absolute step t = n - m_hi + j.  Entries with t < 0 (before t0,
        // PAPER.md:217) or m > H-2 (not stored, reading A15) are zero: j < jv.
        int jv = max(m_hi - P.n, m_hi - (d.H - 2));
        jv = jv < 0 ? 0 : (jv > W ? W : jv);
        const int nvalid = W - jv;          // <= H - 1
        int s0 = P.nslot - (m_hi - jv);     // ring slot of entry jv; m_hi - jv <= H - 2
        s0 += s0 < 0 ? d.H : 0;
        const int lenA = min(nvalid, d.H - s0), lenB = nvalid - lenA;  // ring wrap: at most two runs

        fence_proxy_async();  // order this thread's generic-proxy accesses of the window before the async-proxy writes
        __syncthreads();      // everyone is done with the previous tile (window, permutation, accumulator updates)
        if (jv > 0) {         // zero part of the window (only in the first steps of a run or with a shallow ring)
          for (int idx = tid; idx < 2 * JEFI_TCELLS * jv; idx += TILED_THREADS) {
            int row = idx / jv, j = idx - row * jv;
            *reinterpret_cast<float4*>(smem + (size_t)row * PITCHB + (size_t)j * 16) = make_float4(0.f, 0.f, 0.f, 0.f);
          }
        }
        if (tid == 0) mbar_expect_tx(bar, (uint32_t)(2 * JEFI_TCELLS * nvalid * 16 + OBCELLS * 2));
        if (cp_arr < 2) {
          if (nvalid > 0) {
            const float4* ring = cp_arr == 0 ? P.ringS : P.ringD;
            const float4* src = ring + ((size_t)st * JEFI_TCELLS + cp_cell) * d.H;
            const uint32_t dst = smS + (uint32_t)cp_arr * DOFFB + (uint32_t)cp_cell * PITCHB + (uint32_t)jv * 16u;
            bulk_g2s(dst, src + s0, (uint32_t)lenA * 16u, bar);
            if (lenB > 0) bulk_g2s(dst + (uint32_t)lenA * 16u, src, (uint32_t)lenB * 16u, bar);
          }
        } else if (tid == 2 * JEFI_TCELLS) {
          const int ix = 2 * obx - stx + (d.ntx - 1), iy = 2 * oby - sty + (d.nty - 1), iz = 2 * obz - stz + (d.ntz - 1);
          const size_t row = (size_t)ix + (size_t)P.ndx * ((size_t)iy + (size_t)P.ndy * iz);
          bulk_g2s(permA, P.perm + row * OBCELLS, OBCELLS * 2, bar);
        }
        const uint32_t K = smS + ((uint32_t)m_hi + 0x4B400000u) * 16u;  // wraps mod 2^32 together with bits*16

        mbar_wait(bar, phase);
        phase ^= 1u;
        if (jv > 0) __syncthreads();  // the zero fill is generic-proxy: make it visible to all warps

#pragma unroll 1
        for (int p = 0; p < P_OBS; p++) {
          // the cell this lane evaluates for this source tile: 8 consecutive lanes are (almost) equidistant from it
          const int c = permS[p * TILED_THREADS + tid];
          const int cx = c & 7, cy = (c >> 3) & 7, cz = c >> 6;
          float ax[JEFI_TS], ay[JEFI_TS];
#pragma unroll
          for (int l = 0; l < JEFI_TS; l++) {
            ax[l] = P.g.kx * (float)(ox0 + cx - sx0 - l);
            ay[l] = P.g.ky * (float)(oy0 + cy - sy0 - l);
          }
          const float fz0 = (float)(oz0 + cz - sz0);
          float loc[6];
#pragma unroll
          for (int a = 0; a < 6; a++) loc[a] = 0.f;
          if (self)
            tile_pairs<WP, true>(K, P.g.kz, ax, ay, fz0, loc);
          else
            tile_pairs<WP, false>(K, P.g.kz, ax, ay, fz0, loc);
          // second accumulation level; this tile, cell c belongs to this thread alone
#pragma unroll
          for (int a = 0; a < 6; a++) accS[a * OBCELLS + c] += loc[a];
        }
      }

  __syncthreads();
#pragma unroll
  for (int p = 0; p < P_OBS; p++) {
    const int c = p * TILED_THREADS + tid;  // home order: x fastest inside the tile
    const int oi = ox0 + (c & 7), oj = oy0 + ((c >> 3) & 7), ok = oz0 + (c >> 6);
    if (oi < d.nx && oj < d.ny && ok < d.nz) {
      const size_t o = (size_t)oi + (size_t)d.nx * ((size_t)oj + (size_t)d.ny * ok);
      P.ex[o] = P.g.prefE * accS[c]; P.ey[o] = P.g.prefE * accS[OBCELLS + c]; P.ez[o] = P.g.prefE * accS[2 * OBCELLS + c];
      P.bx[o] = P.g.prefB * accS[3 * OBCELLS + c]; P.by[o] = P.g.prefB * accS[4 * OBCELLS + c];
      P.bz[o] = P.g.prefB * accS[5 * OBCELLS + c];
    }
  }
}

// Evaluation order of the 512 cells of an observation tile for one relative tile offset D = (ox0 - sx0, ..):
// ascending distance to the centre of the source tile in half-slot buckets, ties in home order (x fastest).
// One CTA of 512 threads per offset; rank by counting (a one-off O(512^2) per offset at create time).
__global__ void __launch_bounds__(OBCELLS) k_build_perm(int ndx, int ndy, int ntx, int nty, int ntz, jefi_geom g,
                                                        unsigned short* __restrict__ perm) {
  __shared__ int keys[OBCELLS];
  const int c = threadIdx.x;
  const int ix = blockIdx.x % ndx, iy = (blockIdx.x / ndx) % ndy, iz = blockIdx.x / (ndx * ndy);
  const float Dx = (float)(JEFI_TS * (ix - (ntx - 1))), Dy = (float)(JEFI_TS * (iy - (nty - 1))), Dz = (float)(JEFI_TS * (iz - (ntz - 1)));
  const float half = 0.5f * (float)(JEFI_TS - 1);
  const float rx = g.kx * (Dx + (float)(c & 7) - half), ry = g.ky * (Dy + (float)((c >> 3) & 7) - half),
              rz = g.kz * (Dz + (float)(c >> 6) - half);
  const int key = (int)(2.f * sqrtf(rx * rx + ry * ry + rz * rz));
  keys[c] = key;
  __syncthreads();
  int pos = 0;
  for (int j = 0; j < OBCELLS; j++) {
    int kj = keys[j];
    pos += (kj < key) || (kj == key && j < c);
  }
  perm[(size_t)blockIdx.x * OBCELLS + pos] = (unsigned short)c;
}

// window pitches the kernel is compiled for (float4 entries per source-cell row)
static const int kPitches[] = {36, 64, 96};
typedef void (*tiled_fn)(tiled_params);
static tiled_fn tiled_kernel_for(int wp) {
  switch (wp) {
    case 36: return k_field_tiled<36>;
    case 64: return k_field_tiled<64>;
    case 96: return k_field_tiled<96>;
  }
  return nullptr;
}

// Largest slot window over all relative placements of an 8^3 observation tile and a 4^3 source tile (host, fp64),
// shared-memory opt-in, and the evaluation-order table.
int jefi_tiled_prepare(jefi_ctx* c) {
  const jefi_dims& d = c->dims;
  const double L0 = c->c * c->cfg.dt;
  const int nobx = (d.nx + OB - 1) / OB, noby = (d.ny + OB - 1) / OB, nobz = (d.nz + OB - 1) / OB;
  int wmax = 1;
  auto rng = [](int lo, int hi, int& mn, int& mx) {
    int alo = abs(lo), ahi = abs(hi);
    mx = alo > ahi ? alo : ahi;
    mn = (lo <= 0 && hi >= 0) ? 0 : (alo < ahi ? alo : ahi);
  };
  // the window depends only on the per-axis difference D = ox0 - sx0 (a multiple of 4)
  for (int Dz = -(d.ntz - 1) * JEFI_TS; Dz <= (nobz - 1) * OB; Dz += JEFI_TS)
    for (int Dy = -(d.nty - 1) * JEFI_TS; Dy <= (noby - 1) * OB; Dy += JEFI_TS)
      for (int Dx = -(d.ntx - 1) * JEFI_TS; Dx <= (nobx - 1) * OB; Dx += JEFI_TS) {
        int mnx, mxx, mny, mxy, mnz, mxz;
        rng(Dx - (JEFI_TS - 1), Dx + OB - 1, mnx, mxx);
        rng(Dy - (JEFI_TS - 1), Dy + OB - 1, mny, mxy);
        rng(Dz - (JEFI_TS - 1), Dz + OB - 1, mnz, mxz);
        double rlo = sqrt(pow(mnx * c->cfg.dx, 2) + pow(mny * c->cfg.dy, 2) + pow(mnz * c->cfg.dz, 2));
        double rhi = sqrt(pow(mxx * c->cfg.dx, 2) + pow(mxy * c->cfg.dy, 2) + pow(mxz * c->cfg.dz, 2));
        int w = (int)floor(rhi / L0 + 0.5) - (int)floor(rlo / L0 + 0.5) + 1;
        if (w > wmax) wmax = w;
      }
  c->wmax = wmax;
  int wp = 0;
  for (int cand : kPitches)
    if (cand >= wmax) { wp = cand; break; }
  if (wp == 0) {
    char buf[160];
    snprintf(buf, sizeof buf, "tiled kernel: slot window of %d exceeds the largest compiled pitch %d", wmax, kPitches[2]);
    c->err = buf;
    return JEFI_ESTATE;
  }
  c->wpitch = wp;
  c->tiled_smem = (size_t)2 * JEFI_TCELLS * wp * sizeof(float4) + 6 * OBCELLS * sizeof(float) + OBCELLS * sizeof(unsigned short);
  int dev = c->cfg.device, max_optin = 0;
  cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (c->tiled_smem + 64 > (size_t)max_optin) {
    char buf[160];
    snprintf(buf, sizeof buf, "tiled kernel needs %zu B of shared memory (window %d slots), device allows %d", c->tiled_smem, wmax, max_optin);
    c->err = buf;
    return JEFI_ESTATE;
  }
  cudaError_t e = cudaFuncSetAttribute(tiled_kernel_for(wp), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->tiled_smem);
  if (e != cudaSuccess) { c->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
  // evaluation-order table over all relative tile offsets
  c->ndx = d.ntx + 2 * nobx - 2; c->ndy = d.nty + 2 * noby - 2; c->ndz = d.ntz + 2 * nobz - 2;
  size_t rows = (size_t)c->ndx * c->ndy * c->ndz;
  if ((e = cudaMalloc(&c->perm, rows * OBCELLS * sizeof(unsigned short))) != cudaSuccess) {
    c->err = std::string("permutation table allocation: ") + cudaGetErrorString(e);
    return JEFI_ENOMEM;
  }
  k_build_perm<<<(unsigned)rows, OBCELLS, 0, c->stream>>>(c->ndx, c->ndy, d.ntx, d.nty, d.ntz, c->geom, c->perm);
  if ((e = cudaGetLastError()) != cudaSuccess) { c->err = std::string("k_build_perm: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
  c->launches++;
  return JEFI_OK;
}

int jefi_launch_field_tiled(jefi_ctx* c, float* ex, float* ey, float* ez, float* bx, float* by, float* bz) {
  const jefi_dims& d = c->dims;
  tiled_params P;
  P.d = d; P.g = c->geom; P.n = (int)c->step; P.nslot = (int)(c->step % d.H);
  P.nobx = (d.nx + OB - 1) / OB; P.noby = (d.ny + OB - 1) / OB; P.nobz = (d.nz + OB - 1) / OB;
  P.ndx = c->ndx; P.ndy = c->ndy;
  P.ringS = c->ringS; P.ringD = c->ringD; P.perm = c->perm;
  P.ex = ex; P.ey = ey; P.ez = ez; P.bx = bx; P.by = by; P.bz = bz;
  unsigned blocks = (unsigned)(P.nobx * P.noby * P.nobz);
  tiled_kernel_for(c->wpitch)<<<blocks, TILED_THREADS, c->tiled_smem, c->stream>>>(P);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  return JEFI_OK;
}
