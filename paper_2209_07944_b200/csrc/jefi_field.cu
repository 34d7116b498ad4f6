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
// ------------------------------------------------------------------------------------------------------------
constexpr int OB = 8;            // observation tile edge
constexpr int TILED_THREADS = 256;
constexpr int P_OBS = 2;         // observation cells per thread (z and z+4)

struct tiled_params {
  jefi_dims d;
  jefi_geom g;
  long n;          // current step
  int nslot;       // n mod H
  int wpitch;      // float4 entries per cell row in shared memory (>= largest window)
  int nobx, noby, nobz;
  const float4* ringS;
  const float4* ringD;
  float *ex, *ey, *ez, *bx, *by, *bz;
};

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, bool valid) {
  int sz = valid ? 16 : 0;  // src-size 0 -> the 16 destination bytes are zero-filled
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

// min / max of |a| over the integer interval [lo, hi]
__device__ __forceinline__ void abs_range(int lo, int hi, int& mn, int& mx) {
  int alo = abs(lo), ahi = abs(hi);
  mx = max(alo, ahi);
  mn = (lo <= 0 && hi >= 0) ? 0 : min(alo, ahi);
}

template <bool SELF>
__device__ __forceinline__ void tile_pairs(const unsigned char* __restrict__ smS, uint32_t dOff, uint32_t pitchB, float kx,
                                           float ky, float kz, const float (&fx0)[P_OBS], const float (&fy0)[P_OBS],
                                           const float (&fz0)[P_OBS], uint32_t cconst, float (&acc)[P_OBS][6]) {
  float loc[P_OBS][6];
#pragma unroll
  for (int p = 0; p < P_OBS; p++)
#pragma unroll
    for (int a = 0; a < 6; a++) loc[p][a] = 0.f;

#pragma unroll 1
  for (int lz = 0; lz < JEFI_TS; lz++) {
#pragma unroll 2
    for (int ly = 0; ly < JEFI_TS; ly++) {
      float ay[P_OBS], az[P_OBS], qyz[P_OBS];
#pragma unroll
      for (int p = 0; p < P_OBS; p++) {
        ay[p] = ky * (fy0[p] - (float)ly);
        az[p] = kz * (fz0[p] - (float)lz);
        qyz[p] = fmaf(ay[p], ay[p], az[p] * az[p]);
      }
      const unsigned char* row = smS + (uint32_t)(JEFI_TS * (ly + JEFI_TS * lz)) * pitchB;
#pragma unroll
      for (int lx = 0; lx < JEFI_TS; lx++) {
        const unsigned char* cellp = row + (uint32_t)lx * pitchB;
#pragma unroll
        for (int p = 0; p < P_OBS; p++) {
          float ax = kx * (fx0[p] - (float)lx);
          float q = fmaf(ax, ax, qyz[p]);
          float rs = jefi_rsqrt(q);
          if (SELF) rs = q > 0.f ? rs : 0.f;  // the self cell contributes exactly zero
          float t = fmaf(q, rs, JEFI_MAGIC);   // MAGIC + round(s)
          uint32_t off = (uint32_t)__float_as_int(t) * 16u + cconst;  // byte offset of slot m - m_lo in the cell's window
          if (SELF) off = q > 0.f ? off : 0u;
          const float4 S = *reinterpret_cast<const float4*>(cellp + off);
          const float4 D = *reinterpret_cast<const float4*>(cellp + off + dOff);
          float rs2 = rs * rs, rs3 = rs2 * rs;
          float qq = fmaf(rs2, D.x, rs3 * S.x);
          loc[p][0] = fmaf(ax, qq, loc[p][0]);
          loc[p][1] = fmaf(ay[p], qq, loc[p][1]);
          loc[p][2] = fmaf(az[p], qq, loc[p][2]);
          loc[p][0] = fmaf(-rs, D.y, loc[p][0]);
          loc[p][1] = fmaf(-rs, D.z, loc[p][1]);
          loc[p][2] = fmaf(-rs, D.w, loc[p][2]);
          float wx = fmaf(rs2, D.y, rs3 * S.y);
          float wy = fmaf(rs2, D.z, rs3 * S.z);
          float wz = fmaf(rs2, D.w, rs3 * S.w);
          loc[p][3] = fmaf(ay[p], wz, loc[p][3]);
          loc[p][3] = fmaf(-az[p], wy, loc[p][3]);
          loc[p][4] = fmaf(az[p], wx, loc[p][4]);
          loc[p][4] = fmaf(-ax, wz, loc[p][4]);
          loc[p][5] = fmaf(ax, wy, loc[p][5]);
          loc[p][5] = fmaf(-ay[p], wx, loc[p][5]);
        }
      }
    }
  }
#pragma unroll
  for (int p = 0; p < P_OBS; p++)
#pragma unroll
    for (int a = 0; a < 6; a++) acc[p][a] += loc[p][a];  // second accumulation level: one add per tile
}

__global__ void __launch_bounds__(TILED_THREADS, 2) k_field_tiled(tiled_params P) {
  extern __shared__ __align__(16) unsigned char smem[];
  const jefi_dims& d = P.d;
  const int tid = threadIdx.x;
  const int lane = tid & 31, warp = tid >> 5;
  // observation tile of this CTA
  const int obx = blockIdx.x % P.nobx, oby = (blockIdx.x / P.nobx) % P.noby, obz = blockIdx.x / (P.nobx * P.noby);
  const int ox0 = obx * OB, oy0 = oby * OB, oz0 = obz * OB;
  // lane -> cell of a 4x4x2 warp box; every quarter-warp (8 lanes) is a compact 2x2x2 sub-box so that one
  // LDS.128 phase touches few distinct slots of the same source cell
  const int lxo = (lane & 1) + 2 * ((lane >> 3) & 1);
  const int lyo = ((lane >> 1) & 1) + 2 * ((lane >> 4) & 1);
  const int lzo = (lane >> 2) & 1;
  const int oi = ox0 + 4 * (warp & 1) + lxo;
  const int oj = oy0 + 4 * ((warp >> 1) & 1) + lyo;
  const int ok0 = oz0 + 2 * (warp >> 2) + lzo;  // second cell at ok0 + 4

  float acc[P_OBS][6];
#pragma unroll
  for (int p = 0; p < P_OBS; p++)
#pragma unroll
    for (int a = 0; a < 6; a++) acc[p][a] = 0.f;

  const uint32_t pitchB = (uint32_t)P.wpitch * 16u;
  const uint32_t dOff = (uint32_t)JEFI_TCELLS * pitchB;  // D window follows the S window
  const uint32_t smS_addr = (uint32_t)__cvta_generic_to_shared(smem);
  const int ntiles = d.ntx * d.nty * d.ntz;

  for (int st = 0; st < ntiles; st++) {
    const int stx = st % d.ntx, sty = (st / d.ntx) % d.nty, stz = st / (d.ntx * d.nty);
    const int sx0 = stx * JEFI_TS, sy0 = sty * JEFI_TS, sz0 = stz * JEFI_TS;
    // slot window of this (observation tile, source tile) pair from the extreme offsets
    int mnx, mxx, mny, mxy, mnz, mxz;
    abs_range(ox0 - (sx0 + JEFI_TS - 1), ox0 + OB - 1 - sx0, mnx, mxx);
    abs_range(oy0 - (sy0 + JEFI_TS - 1), oy0 + OB - 1 - sy0, mny, mxy);
    abs_range(oz0 - (sz0 + JEFI_TS - 1), oz0 + OB - 1 - sz0, mnz, mxz);
    const bool self = (mnx == 0 && mny == 0 && mnz == 0);
    const int m_lo = self ? 0 : jefi_delay_fp32(jefi_q_fp32(P.g.kx, P.g.ky, P.g.kz, (float)mnx, (float)mny, (float)mnz));
    const int m_hi = jefi_delay_fp32(jefi_q_fp32(P.g.kx, P.g.ky, P.g.kz, (float)mxx, (float)mxy, (float)mxz));
    const int W = m_hi - m_lo + 1;

    __syncthreads();  // everyone is done reading the previous tile
    {
      const size_t tile_base = (size_t)st * JEFI_TCELLS * d.H;
      const unsigned rcp = 0xFFFFFFFFu / (unsigned)W + 1u;  // ceil(2^32 / W): exact quotient for idx < 2^16
      const int total = JEFI_TCELLS * W;
      for (int idx = tid; idx < total; idx += TILED_THREADS) {
        int cell = W == 1 ? idx : (int)__umulhi((unsigned)idx, rcp);
        int w = idx - cell * W;
        int m = m_lo + w;
        long t = P.n - m;
        bool valid = (t >= 0) && (m <= d.H - 2);
        int slot = P.nslot - m;
        slot += slot < 0 ? d.H : 0;
        slot = valid ? slot : 0;
        size_t g = tile_base + (size_t)cell * d.H + slot;
        uint32_t dst = smS_addr + (uint32_t)cell * pitchB + (uint32_t)w * 16u;
        cp_async16(dst, P.ringS + g, valid);
        cp_async16(dst + dOff, P.ringD + g, valid);
      }
      cp_async_wait_all();
    }
    __syncthreads();

    float fx0[P_OBS], fy0[P_OBS], fz0[P_OBS];
#pragma unroll
    for (int p = 0; p < P_OBS; p++) {
      fx0[p] = (float)(oi - sx0);
      fy0[p] = (float)(oj - sy0);
      fz0[p] = (float)(ok0 + 4 * p - sz0);
    }
    const uint32_t cconst = 0u - (0x4B400000u + (uint32_t)m_lo) * 16u;  // wraps mod 2^32 together with bits*16
    if (self)
      tile_pairs<true>(smem, dOff, pitchB, P.g.kx, P.g.ky, P.g.kz, fx0, fy0, fz0, cconst, acc);
    else
      tile_pairs<false>(smem, dOff, pitchB, P.g.kx, P.g.ky, P.g.kz, fx0, fy0, fz0, cconst, acc);
  }

#pragma unroll
  for (int p = 0; p < P_OBS; p++) {
    const int ok = ok0 + 4 * p;
    if (oi < d.nx && oj < d.ny && ok < d.nz) {
      const size_t o = (size_t)oi + (size_t)d.nx * ((size_t)oj + (size_t)d.ny * ok);
      P.ex[o] = P.g.prefE * acc[p][0]; P.ey[o] = P.g.prefE * acc[p][1]; P.ez[o] = P.g.prefE * acc[p][2];
      P.bx[o] = P.g.prefB * acc[p][3]; P.by[o] = P.g.prefB * acc[p][4]; P.bz[o] = P.g.prefB * acc[p][5];
    }
  }
}

// Largest slot window over all relative placements of an 8^3 observation tile and a 4^3 source tile (host, fp64).
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
  c->tiled_smem = (size_t)2 * JEFI_TCELLS * wmax * sizeof(float4);
  int dev = c->cfg.device, max_optin = 0;
  cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (c->tiled_smem > (size_t)max_optin) {
    char buf[160];
    snprintf(buf, sizeof buf, "tiled kernel needs %zu B of shared memory (window %d slots), device allows %d", c->tiled_smem, wmax, max_optin);
    c->err = buf;
    return JEFI_ESTATE;
  }
  cudaError_t e = cudaFuncSetAttribute(k_field_tiled, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->tiled_smem);
  if (e != cudaSuccess) { c->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
  return JEFI_OK;
}

int jefi_launch_field_tiled(jefi_ctx* c, float* ex, float* ey, float* ez, float* bx, float* by, float* bz) {
  const jefi_dims& d = c->dims;
  tiled_params P;
  P.d = d; P.g = c->geom; P.n = c->step; P.nslot = (int)(c->step % d.H); P.wpitch = c->wmax;
  P.nobx = (d.nx + OB - 1) / OB; P.noby = (d.ny + OB - 1) / OB; P.nobz = (d.nz + OB - 1) / OB;
  P.ringS = c->ringS; P.ringD = c->ringD;
  P.ex = ex; P.ey = ey; P.ez = ez; P.bx = bx; P.by = by; P.bz = bz;
  unsigned blocks = (unsigned)(P.nobx * P.noby * P.nobz);
  k_field_tiled<<<blocks, TILED_THREADS, c->tiled_smem, c->stream>>>(P);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  return JEFI_OK;
}
