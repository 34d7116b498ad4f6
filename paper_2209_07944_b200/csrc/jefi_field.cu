// libjefi: the Jefimenko field gather (SURVEY.md §8 row a3; PAPER.md:103-109 Eqs. 2.4-2.6, :221 self cell).
//
// In scaled units d' = d/(c dt), s = |d'|, rs = 1/s, Jt = J/c, D* = backward difference over one step:
//   E = prefE * sum [ d' (rho rs^3 + Drho rs^2) - DJt rs ]          (Eq. 2.4)
//   B = prefB * sum [ d' x (Jt rs^3 + DJt rs^2) ]                    (Eq. 2.5)
// sources taken from ring slot (n - m) mod H with m = round(s) (Eq. 2.6, nearest-step reading).
//
// Kernels:
//   k_field_reference  one thread per observation cell, all sources, delays from the fp64-built table (the paper's K1 in
//                      fp32; used on request or when the fp32 delay arithmetic cannot be proven for a grid).
//   k_field_tiled      warp-specialised CTA: 16 consumer warps own one observation tile of 512 units (a unit = one cell, or a
//                      dyad of two x-neighbour cells that share distance, delay and geometric factors) and walk the 64-cell
//                      source tiles; a producer warp stages each tile's slot window [m_lo, m_hi] in a two-stage
//                      shared-memory ring with TMA bulk copies (mbarrier full/done pipeline).  Compiled for three tile
//                      geometries (8x8x8 / 4x4x4 cubes, one cell per thread; 16x8x8 / 4x4x4 dyads, two cells per thread:
//                      the benchmark's; 1x16x32 / 1x8x8 for nx <= 3 slabs), two window pitches and the two retarded-time
//                      rules.  A window wider than the pitch is served in several passes.
//   k_reduce_partials  adds, in a fixed order, the partial sums of a launch that split the source range over CTAs.
//   k_build_perm       once per context: the evaluation order of the 512 cells per relative tile offset.
#include <stdio.h>
#include <stdlib.h>

#include "jefi_ctx.h"

// ------------------------------------------------------------------------------------------------------------
// reference kernel
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_field_reference(jefi_dims d, jefi_geom g, int ex_, int ey_, long n, const int* __restrict__ step_dev,
                                                         int linear, long oc0, long oc1,
                                                         const int* __restrict__ mtab, const float4* __restrict__ ring,
                                                         float* __restrict__ ex, float* __restrict__ ey,
                                                         float* __restrict__ ez, float* __restrict__ bx,
                                                         float* __restrict__ by, float* __restrict__ bz, float4* __restrict__ pack) {
  long oc = oc0 + (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (oc >= oc1) return;
  if (step_dev) n = step_dev[0];  // jefi_pic_step's graph
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
        long tile; int cell;
        jefi_tile_cell(d, i, j, k, tile, cell);
        size_t idx = jefi_ring_quad(d, tile, (int)(t % d.H), cell);
        float4 S = ring[idx];
        const float4 D = ring[idx + JEFI_TCELLS];  // (Jx, Jz, rho, Jy)/scaled, see jefi_ctx.h
        float ax = g.kx * (float)di, ay = g.ky * (float)dj, az = g.kz * (float)dk;
        float q = fmaf(ax, ax, fmaf(ay, ay, az * az));
        float rs = rsqrtf(q), rs2 = rs * rs, rs3 = rs2 * rs;
        if (linear) {  // JEFI_DELAY_LINEAR: values on the line through the two samples, S(t_r) = S - phi D, phi = s - m
          const float phi = fmaf(q, rs, -(float)m);
          S.x = fmaf(-phi, D.x, S.x); S.y = fmaf(-phi, D.y, S.y); S.z = fmaf(-phi, D.z, S.z); S.w = fmaf(-phi, D.w, S.w);
        }
        float qq = fmaf(rs2, D.z, rs3 * S.z);
        lex = fmaf(ax, qq, lex); ley = fmaf(ay, qq, ley); lez = fmaf(az, qq, lez);
        lex = fmaf(-rs, D.x, lex); ley = fmaf(-rs, D.w, ley); lez = fmaf(-rs, D.y, lez);
        float wx = fmaf(rs2, D.x, rs3 * S.x), wy = fmaf(rs2, D.w, rs3 * S.w), wz = fmaf(rs2, D.y, rs3 * S.y);
        lbx = fmaf(ay, wz, lbx); lbx = fmaf(-az, wy, lbx);
        lby = fmaf(az, wx, lby); lby = fmaf(-ax, wz, lby);
        lbz = fmaf(ax, wy, lbz); lbz = fmaf(-ay, wx, lbz);
      }
    aex += lex; aey += ley; aez += lez; abx += lbx; aby += lby; abz += lbz;
  }
  const float vex = g.prefE * aex, vey = g.prefE * aey, vez = g.prefE * aez;
  const float vbx = g.prefB * abx, vby = g.prefB * aby, vbz = g.prefB * abz;
  ex[oc] = vex; ey[oc] = vey; ez[oc] = vez;
  bx[oc] = vbx; by[oc] = vby; bz[oc] = vbz;
  if (pack) {
    pack[2 * oc] = make_float4(vex, vey, vez, vbx);
    pack[2 * oc + 1] = make_float4(vby, vbz, 0.f, 0.f);
  }
}

int jefi_launch_field_reference(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz,
                                float* eb_packed) {
  const jefi_dims& d = c->dims;
  const long oc0 = (long)k0 * d.nx * d.ny, oc1 = (long)k1 * d.nx * d.ny;  // observation cells of the z-planes [k0, k1)
  unsigned blocks = (unsigned)((oc1 - oc0 + 127) / 128);
  k_field_reference<<<blocks, 128, 0, c->stream>>>(d, c->geom, c->tex, c->tey, c->step, c->capturing ? c->step_dev : nullptr,
                                                   c->cfg.delay_rule == JEFI_DELAY_LINEAR ? 1 : 0, oc0, oc1,
                                                   c->mtab_dev, c->ring, ex, ey, ez, bx, by, bz, reinterpret_cast<float4*>(eb_packed));
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// tiled kernel
//
// CTA = 16 consumer warps + 1 producer warp (544 threads), one CTA per SM.  The consumers own one observation tile
// (G::OBX x G::OBY x G::OBZ cells = 512 units of G::CX cells, one unit per thread) against the source tiles [t0, t1) of the linear tile order (the
// whole grid, or one chunk of it when the launch splits the source range over blockIdx.y; the pieces' partial sums are
// then written to a [piece][6][N] buffer and added in a fixed order by k_reduce_partials).
//
// Staging.  For an (observation tile, source tile) pair the delays lie in [m_lo, m_hi] (from the extreme offsets), and
// the ring stores a source tile slot by slot (jefi_ctx.h), so the window is one contiguous run of W = m_hi-m_lo+1 ring
// rows (two runs when the ring wraps).  The producer warp's lane 0 issues it as one or two TMA bulk copies
// (cp.async.bulk, SASS UBLKCP) into stage `item & 1`, together with the 1 KB evaluation-order row, on the stage's `full`
// mbarrier; consumers release a stage by arriving (one lane per warp) on its `done` mbarrier.  Row j of a stage
// holds delay m = m_top - j.  A window wider than the compiled pitch WP (large dx/(c dt), e.g. the paper's kappa = 6
// example) is served in ceil(W/WP) passes over the same source tile: pass p stages the delays
// [m_hi - p WP - (R-1), m_hi - p WP] and every lane whose delay falls outside contributes exactly zero (MODE_MULTI).
// The pipeline runs over (tile, pass) items; the stage header tells the consumers what an item is, and a terminal item
// (MODE_END) that nothing follows.  An item whose rows would ALL be zero - every delay of the tile pair reaches back before t0
// or beyond the stored depth (reading A15) - is not staged: its pairs add exactly nothing.  In the first steps of
// a run the kernel therefore evaluates only the sources inside the light cone of t0 of each observation tile.
//
// Pair evaluation: the source cell is warp-uniform, the delay per lane:
//   q = |d'|^2 (FFMA), rs = rsqrt(q) (MUFU), t = q*rs + 1.5*2^23 (FFMA; the integer m sits in the mantissa),
//   address = K - 2064*bits(t) (IMAD), 2 x LDS.128 (S and D quads), then with packed FP32 (fma.rn.f32x2 = SASS FFMA2,
//   scalar operands broadcast, halves swapped for free):
//     (wx,wz) = rs*(Jx,Jz) + (DJx,DJz)      (u0,wy) = rs*(rho,Jy) + (Drho,DJy)             2 FFMA2
//     r2 = rs^2, (a_x,a_z) = (ax,az)*r2, a_y = ay*r2                                       4 FMUL
//     Exz += (a_x,a_z)*u0   Fxz += rs*(DJx,DJz)   Ey += a_y*u0   Fy += rs*DJy              2 FFMA2 + 2 FFMA
//     Bxz += a_y*(wz,wx)    Cxz += wy*(a_z,a_x)   By12 += (a_z,a_x)*(wx,wz)                3 FFMA2
//   E = (Exz - Fxz, Ey - Fy), B = (Bxz.lo - Cxz.lo, By12.lo - By12.hi, Cxz.hi - Bxz.hi):   19 issue slots per pair
//   (9 scalar FMA-pipe, 7 packed, 1 MUFU, 2 LDS) against 26 for the scalar form.
//
// Shared-memory delivery is the scarce resource (measured, profiles/): an LDS.128 takes 4 data-pipe cycles, 2 when
// every lane l reads the same address as lane l^1.  Which lane evaluates which observation cell is free (any assignment
// gives the same sums), so for every source tile the 512 cells are taken in an order tabulated per relative tile offset
// (k_build_perm): neighbouring lanes then mostly share a slot.  Per-tile partial sums are added to a shared-memory
// accumulator (6 sums per cell: [6][512] for one-cell units, [512][12] for dyads; second level of the two-level accumulation),
// because a cell is evaluated by a different thread in every tile; the `done` barrier of item-1 orders these updates between items.
// ------------------------------------------------------------------------------------------------------------
constexpr int OBCELLS = 512;
constexpr int NCONS = 512;  // consumer threads = observation cells of a tile
constexpr int NCWARPS = NCONS / 32;
constexpr int TILED_THREADS = NCONS + 32;  // + producer warp
constexpr int HDR_BYTES = 32;
enum { MODE_PLAIN = 0, MODE_SELF = 1, MODE_MULTI = 2, MODE_END = 3 };

struct tiled_params {
  jefi_dims d;
  jefi_geom g;
  int n;           // current step
  int nslot;       // n mod H
  int nobx, noby;
  int ndx, ndy;    // extents of the permutation table in relative-offset space
  int obz0;        // first observation tile layer of this launch (jefi_field_step_slab)
  int k1;          // observation planes k >= k1 are not written
  int chunk;       // source tiles per blockIdx.y
  int to_partial;  // 1: write this piece's sums to partial[blockIdx.y][6][N] (source range split over blockIdx.y)
  const int* step_dev;  // non-NULL (jefi_pic_step's graph): n and nslot are read from the device-side step state
  const float4* ring;
  const unsigned short* perm;  // [ndz][ndy][ndx][512]
  const int *tile_first, *tile_last;  // per source tile: span of steps whose ring row is not all zero (k_push_sources)
  float *ex, *ey, *ez, *bx, *by, *bz;
  float4* pack;    // optional interleaved output (jefi_field_step_packed)
  float* partial;
};

struct stage_hdr {  // written by the producer before it arms the stage's full barrier
  uint32_t K;       // shared address of the stage's row 0 + 2064*(m_top + 0x4B400000)  (mod 2^32)
  int mode;         // MODE_PLAIN / MODE_SELF (the source tile contains r' = r) / MODE_MULTI (one of several passes) / MODE_END
  int dx0, dy0, dz0;  // ox0 - sx0, oy0 - sy0, oz0 - sz0
  uint32_t Mtop;    // m_top + 0x4B400000 (MODE_MULTI)
  uint32_t R;       // rows staged in this item (MODE_MULTI)
  int last;         // bit 0: terminal item (MODE_END), nothing follows; JEFI_CHECKED: bits 1.. = sequence number of the item
};
static_assert(sizeof(stage_hdr) == HDR_BYTES, "stage header");

template <int WP, int CELLS>
struct stage_layout {
  static constexpr uint32_t ROWS = WP * JEFI_ROW_BYTES;
  static constexpr uint32_t PERM = ROWS;                       // u16[512]
  static constexpr uint32_t HDR = PERM + OBCELLS * 2;
  static constexpr uint32_t BYTES = ((HDR + HDR_BYTES + 127) / 128) * 128;
  static constexpr uint32_t ACC = 2 * BYTES;                   // float[6][CELLS]
  static constexpr uint32_t BAR = ACC + 6 * CELLS * 4;         // full[2], done[2]
  static constexpr uint32_t TOTAL = BAR + 4 * 8;
};

// ---- mbarrier / TMA bulk-copy primitives (PTX ISA: mbarrier, cp.async.bulk) ----
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
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

// ---- packed FP32 (sm_100: fma/mul .f32x2 on 64-bit register pairs) ----
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ float lo32(f32x2 v) {
  float a;
  asm("{ .reg .b32 jf_unused; mov.b64 {%0, jf_unused}, %1; }" : "=f"(a) : "l"(v));
  return a;
}
__device__ __forceinline__ float hi32(f32x2 v) {
  float b;
  asm("{ .reg .b32 jf_unused; mov.b64 {jf_unused, %0}, %1; }" : "=f"(b) : "l"(v));
  return b;
}
__device__ __forceinline__ f32x2 swap2(f32x2 v) { return pk(hi32(v), lo32(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
// min / max of |a| over the integer interval [lo, hi]
__host__ __device__ __forceinline__ void abs_range(int lo, int hi, int& mn, int& mx) {
  int alo = lo < 0 ? -lo : lo, ahi = hi < 0 ? -hi : hi;
  mx = alo > ahi ? alo : ahi;
  mn = (lo <= 0 && hi >= 0) ? 0 : (alo < ahi ? alo : ahi);
}

struct quad2 {  // one LDS.128 as two aligned register pairs
  f32x2 xy, zw;
};
template <int IMM>
__device__ __forceinline__ quad2 lds128_imm(uint32_t addr) {
  quad2 v;
  asm volatile("ld.shared.v2.b64 {%0, %1}, [%2+%3];" : "=l"(v.xy), "=l"(v.zw) : "r"(addr), "n"(IMM));
  return v;
}

struct pair_acc {  // per-tile partial sums of one observation cell (first accumulation level)
  f32x2 Exz, Fxz, Bxz, Cxz, By12;
  float Ey, Fy;
};

// what a consumer thread needs to address the stage of one item
struct item_addr {
  uint32_t K;     // MODE_PLAIN / MODE_SELF: row 0 + 2064*(m_top + 0x4B400000);  MODE_MULTI: row 0
  uint32_t Mtop;  // MODE_MULTI
  uint32_t R;     // MODE_MULTI
#ifdef JEFI_CHECKED
  uint32_t lo, hi;  // shared-memory byte range of the rows staged for this item (both + the z-layer offset)
#endif
};

// -DJEFI_CHECKED (libjefi_checked.so, paper_2209_07944_b200/build.py --checked): the library's own memory checks, run under the
// whole GPU test-suite in place of compute-sanitizer (closed on this pool): every shared-memory address a consumer lane forms
// must lie inside the rows staged for its item [0]; every item a consumer reads must carry the sequence number it expects,
// i.e. the stage was neither refilled early nor read before it was filled [1]; the producer poisons a stage with NaN before
// refilling it, so a row that no copy or zero fill covered shows up as NaN in E, B and fails parity; the cell sort's scatter
// index must be inside the list [2].  jefi_debug_check_errors() returns the counters (all zero = clean).
__device__ unsigned long long g_jefi_check_errors[2];
#ifdef JEFI_CHECKED
#define JEFI_CHECK_FAIL(kind) atomicAdd(&g_jefi_check_errors[kind], 1ull)
#endif
cudaError_t jefi_field_check_errors(unsigned long long out[2]) { return cudaMemcpyFromSymbol(out, g_jefi_check_errors, 2 * sizeof(unsigned long long)); }

// The part of a pair evaluation that depends only on the offset r - r' (and, through the address, on the staged item): with
// G::CX = 2 it is shared by the pairs (o, s) and (o + ex, s + ex).  Az = item address + byte offset of the z layer.
template <bool LINEAR>
struct pair_geom {
  uint32_t addr;  // shared address of the ring row of this offset's delay
  float rs, a_y, nphi;
  f32x2 Axz;      // (a_x, a_z) = d' rs^2
};
template <int MODE, bool LINEAR>
__device__ __forceinline__ void make_geom(const item_addr& Az, float ax, float ay, float az, float qyz, pair_geom<LINEAR>& g) {
  const float q = fmaf(ax, ax, qyz);
  float rs = jefi_rsqrt(q);
  if (MODE != MODE_PLAIN) rs = q > 0.f ? rs : 0.f;  // the self cell contributes exactly zero
  const float t = fmaf(q, rs, JEFI_MAGIC);          // MAGIC + round(s): m sits in the mantissa
  uint32_t addr;
  if (MODE == MODE_MULTI) {
    const uint32_t j = Az.Mtop - (uint32_t)__float_as_int(t);  // m_top - m: the row of this lane's delay
    const bool in = j < Az.R;                                 // else the delay belongs to another pass: contributes zero
    rs = in ? rs : 0.f;
    addr = Az.K + (in ? j : 0u) * (uint32_t)JEFI_ROW_BYTES;
  } else {
    addr = Az.K - (uint32_t)__float_as_int(t) * (uint32_t)JEFI_ROW_BYTES;  // row j = m_top - m
  }
#ifdef JEFI_CHECKED
  if (addr < Az.lo || addr + (uint32_t)JEFI_ROW_BYTES > Az.hi) {  // the row of this delay lies outside the rows staged for this item
    JEFI_CHECK_FAIL(0);
    addr = Az.lo;
  }
#endif
  g.addr = addr;
  g.rs = rs;
  if (LINEAR) g.nphi = fmaf(-q, rs, t - JEFI_MAGIC);  // m - s
  const float r2 = rs * rs;
  g.Axz = pk(ax * r2, az * r2);   // (a_x, a_z) = d' rs^2: two scalar multiplies, so that no (ax, az) register pair
  g.a_y = ay * r2;                // has to be kept alive (measured 1.3 % faster than one FMUL2 on kept pairs)
}
// One observation cell against source cell CELL of the staged tile, with the geometry of their offset.
template <bool LINEAR, int CELL>
__device__ __forceinline__ void acc_pair(const pair_geom<LINEAR>& g, pair_acc& A) {
  constexpr int SOFF = CELL * 16;
  constexpr int DOFF = SOFF + JEFI_TCELLS * 16;
  quad2 S = lds128_imm<SOFF>(g.addr);         // (Jx, Jz | rho, Jy)
  const quad2 D = lds128_imm<DOFF>(g.addr);   // (DJx, DJz | Drho, DJy)
  if (LINEAR) {  // JEFI_DELAY_LINEAR: S(t_r) = S - phi D with phi = s - m in [-1/2, 1/2) (3 scalar + 2 packed instructions)
    const f32x2 nphi2 = pk(g.nphi, g.nphi);
    S.xy = fma2(nphi2, D.xy, S.xy);
    S.zw = fma2(nphi2, D.zw, S.zw);
  }
  const float rs = g.rs, a_y = g.a_y;
  const f32x2 rs2 = pk(rs, rs);
  const f32x2 wxz = fma2(rs2, S.xy, D.xy);  // (wx, wz)
  const f32x2 u0wy = fma2(rs2, S.zw, D.zw); // (u0, wy)
  const f32x2 Axz = g.Axz;
  const float u0 = lo32(u0wy), wy = hi32(u0wy);
  const f32x2 Azx = swap2(Axz);
  // The order of the seven accumulations (and 32 pairs per loop iteration, tile_pairs) was chosen by measurement on B200:
  // ten orders of these independent statements ran between 741 and 767 ms per 96^3 step (register-bank conflicts and operand
  // reuse between neighbouring FFMA2 depend on it); this one is the fastest.
  A.Exz = fma2(Axz, pk(u0, u0), A.Exz);
  A.Bxz = fma2(pk(a_y, a_y), swap2(wxz), A.Bxz);  // (a_y wz, a_y wx)
  A.Ey = fmaf(a_y, u0, A.Ey);
  A.Cxz = fma2(pk(wy, wy), Azx, A.Cxz);           // (wy a_z, wy a_x)
  A.Fy = fmaf(rs, hi32(D.zw), A.Fy);
  A.By12 = fma2(Azx, wxz, A.By12);                // (a_z wx, a_x wz)
  A.Fxz = fma2(rs2, D.xy, A.Fxz);
}

// Two observation cells against two source cells with ONE geometry (G::CX = 2: (cell 1, source CELL1) and (cell 0, source
// CELL0) have the same offset).  The statements of the two pairs alternate so that the shared operands (rs, a_y, Axz, Azx) sit
// in the same operand slot of neighbouring instructions (a register operand repeated there can be served by the operand
// reuse cache); the order was chosen by A/B on B200 like the one of acc_pair.
template <bool LINEAR, int CELL1, int CELL0>
__device__ __forceinline__ void acc_pair2(const pair_geom<LINEAR>& g, pair_acc& A1, pair_acc& A0) {
  quad2 S1 = lds128_imm<CELL1 * 16>(g.addr);
  const quad2 D1 = lds128_imm<CELL1 * 16 + JEFI_TCELLS * 16>(g.addr);
  quad2 S0 = lds128_imm<CELL0 * 16>(g.addr);
  const quad2 D0 = lds128_imm<CELL0 * 16 + JEFI_TCELLS * 16>(g.addr);
  if (LINEAR) {
    const f32x2 nphi2 = pk(g.nphi, g.nphi);
    S1.xy = fma2(nphi2, D1.xy, S1.xy);
    S0.xy = fma2(nphi2, D0.xy, S0.xy);
    S1.zw = fma2(nphi2, D1.zw, S1.zw);
    S0.zw = fma2(nphi2, D0.zw, S0.zw);
  }
  const float rs = g.rs, a_y = g.a_y;
  const f32x2 rs2 = pk(rs, rs);
  const f32x2 wxz1 = fma2(rs2, S1.xy, D1.xy);
  const f32x2 wxz0 = fma2(rs2, S0.xy, D0.xy);
  const f32x2 u0wy1 = fma2(rs2, S1.zw, D1.zw);
  const f32x2 u0wy0 = fma2(rs2, S0.zw, D0.zw);
  A1.Fxz = fma2(rs2, D1.xy, A1.Fxz);
  A0.Fxz = fma2(rs2, D0.xy, A0.Fxz);
  A1.Fy = fmaf(rs, hi32(D1.zw), A1.Fy);
  A0.Fy = fmaf(rs, hi32(D0.zw), A0.Fy);
  const f32x2 Axz = g.Axz;
  const f32x2 Azx = swap2(Axz);
  const f32x2 ay2 = pk(a_y, a_y);
  const float u01 = lo32(u0wy1), wy1 = hi32(u0wy1), u00 = lo32(u0wy0), wy0 = hi32(u0wy0);
  A1.Exz = fma2(Axz, pk(u01, u01), A1.Exz);
  A0.Exz = fma2(Axz, pk(u00, u00), A0.Exz);
  A1.Bxz = fma2(ay2, swap2(wxz1), A1.Bxz);
  A0.Bxz = fma2(ay2, swap2(wxz0), A0.Bxz);
  A1.Ey = fmaf(a_y, u01, A1.Ey);
  A0.Ey = fmaf(a_y, u00, A0.Ey);
  A1.Cxz = fma2(Azx, pk(wy1, wy1), A1.Cxz);
  A0.Cxz = fma2(Azx, pk(wy0, wy0), A0.Cxz);
  A1.By12 = fma2(Azx, wxz1, A1.By12);
  A0.By12 = fma2(Azx, wxz0, A0.By12);
}

// compile-time loops over the cells of the staged source tile (the LDS offsets of one_pair are immediates)
// G::CX == 1: ax[l] = kx (dx0 + cx - l), one geometry per pair.
// G::CX == 2: the thread's cells are x and x + 1; ax[jj] = kx (dx0 + x + 1 - jj), jj = 0..4, is the offset of the pairs
//             (cell 1, source l = jj) and (cell 0, source l = jj - 1): 5 geometries serve the 8 pairs of a source row.
template <class G, int MODE, bool LINEAR, int CELL0, int LX>
__device__ __forceinline__ void row_pairs(const item_addr& Az, const float (&ax)[G::TSX + G::CX - 1], float ay, float az, float qyz,
                                          pair_acc (&A)[G::CX]) {
  if constexpr (LX < G::TSX + G::CX - 1) {
    pair_geom<LINEAR> g;
    make_geom<MODE, LINEAR>(Az, ax[LX], ay, az, qyz, g);
    if constexpr (G::CX == 1) {
      acc_pair<LINEAR, CELL0 + LX>(g, A[0]);
    } else {
      if constexpr (LX >= 1 && LX < G::TSX) acc_pair2<LINEAR, CELL0 + LX, CELL0 + LX - 1>(g, A[1], A[0]);
      else if constexpr (LX < G::TSX) acc_pair<LINEAR, CELL0 + LX>(g, A[1]);
      else acc_pair<LINEAR, CELL0 + LX - 1>(g, A[0]);
    }
    row_pairs<G, MODE, LINEAR, CELL0, LX + 1>(Az, ax, ay, az, qyz, A);
  }
}
template <class G, int MODE, bool LINEAR, int CELL0, int LY>
__device__ __forceinline__ void layer_rows(const item_addr& Az, const float (&ax)[G::TSX + G::CX - 1], const float (&ay)[G::TSY], float az, float az2,
                                           pair_acc (&A)[G::CX]) {
  if constexpr (LY < G::TSY) {
    const float qyz = fmaf(ay[LY], ay[LY], az2);
    row_pairs<G, MODE, LINEAR, CELL0 + G::TSX * LY, 0>(Az, ax, ay[LY], az, qyz, A);
    layer_rows<G, MODE, LINEAR, CELL0, LY + 1>(Az, ax, ay, az, az2, A);
  }
}
template <class G, int MODE, bool LINEAR, int ZU, int ZO>
__device__ __forceinline__ void z_layers(const item_addr& Az, float kz, const float (&ax)[G::TSX + G::CX - 1], const float (&ay)[G::TSY], float fz,
                                         pair_acc (&A)[G::CX]) {
  if constexpr (ZO < ZU) {
    const float az = kz * (fz - (float)ZO);
    const float az2 = az * az;
    layer_rows<G, MODE, LINEAR, ZO * G::TSX * G::TSY, 0>(Az, ax, ay, az, az2, A);
    z_layers<G, MODE, LINEAR, ZU, ZO + 1>(Az, kz, ax, ay, fz, A);
  }
}

// the thread's G::CX observation cells against the 64 cells of the staged source tile; the z loop is unrolled to 32 pairs per
// iteration
template <class G, int MODE, bool LINEAR>
__device__ __forceinline__ void tile_pairs(const item_addr& A0, float kz, const float (&ax)[G::TSX + G::CX - 1], const float (&ay)[G::TSY], float fz0,
                                           pair_acc (&A)[G::CX]) {
  constexpr int LAYER = G::TSX * G::TSY;            // cells per z layer of the source tile
  constexpr int PAIRS_PER_ITER = 32;                                        // straight-line pairs per loop iteration (measured: 16, 32, 64)
  constexpr int ZU = LAYER * G::CX >= PAIRS_PER_ITER ? 1 : PAIRS_PER_ITER / (LAYER * G::CX);  // layers per loop iteration
#pragma unroll 1
  for (int lz = 0; lz < G::TSZ; lz += ZU) {
    item_addr Az = A0;
    Az.K = A0.K + (uint32_t)(lz * LAYER * 16);
#ifdef JEFI_CHECKED
    Az.lo = A0.lo + (uint32_t)(lz * LAYER * 16);
    Az.hi = A0.hi + (uint32_t)(lz * LAYER * 16);
#endif
    z_layers<G, MODE, LINEAR, ZU, 0>(Az, kz, ax, ay, fz0 - (float)lz, A);
  }
}

// MULTI: the grid has tile pairs whose window exceeds WP (compiled in only then: the common single-pass kernels carry neither
// the third evaluation mode nor its registers)
template <class G, int WP, bool LINEAR, bool MULTI>
__global__ void __launch_bounds__(TILED_THREADS, 1) k_field_tiled(tiled_params P) {
  using L = stage_layout<WP, G::CELLS>;
  extern __shared__ __align__(128) unsigned char smem[];
  const jefi_dims& d = P.d;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t sm0 = (uint32_t)__cvta_generic_to_shared(smem);
  float* accS = reinterpret_cast<float*>(smem + L::ACC);
  const uint32_t barFull = sm0 + L::BAR, barDone = barFull + 16;
  // observation tile and source-tile range of this CTA
  const int obx = blockIdx.x % P.nobx, oby = (blockIdx.x / P.nobx) % P.noby, obz = P.obz0 + blockIdx.x / (P.nobx * P.noby);
  const int ox0 = obx * G::OBX, oy0 = oby * G::OBY, oz0 = obz * G::OBZ;
  const int ntiles = d.ntx * d.nty * d.ntz;
  const int t0 = blockIdx.y * P.chunk;
  const int nt = min(P.chunk, ntiles - t0);

  if (tid < NCONS)
    for (int i = tid; i < 6 * G::CELLS; i += NCONS) accS[i] = 0.f;
  if (tid == 0) {
    mbar_init(barFull, 1); mbar_init(barFull + 8, 1);
    mbar_init(barDone, NCWARPS); mbar_init(barDone + 8, NCWARPS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp == NCWARPS) {
    // ------------------------------------------------ producer warp ------------------------------------------------
    const int n_now = P.step_dev ? P.step_dev[0] : P.n, nslot_now = P.step_dev ? P.step_dev[1] : P.nslot;
    // delays of the tile pair (observation tile, source tile tt) from the extreme offsets
    auto tile_window = [&](int tt, int& stx, int& sty, int& stz, int& m_lo, int& m_hi, bool& self) {
      stx = tt % d.ntx; sty = (tt / d.ntx) % d.nty; stz = tt / (d.ntx * d.nty);
      const int sx0 = stx * G::TSX, sy0 = sty * G::TSY, sz0 = stz * G::TSZ;
      int mnx, mxx, mny, mxy, mnz, mxz;
      abs_range(ox0 - (sx0 + G::TSX - 1), ox0 + G::OBX - 1 - sx0, mnx, mxx);
      abs_range(oy0 - (sy0 + G::TSY - 1), oy0 + G::OBY - 1 - sy0, mny, mxy);
      abs_range(oz0 - (sz0 + G::TSZ - 1), oz0 + G::OBZ - 1 - sz0, mnz, mxz);
      self = (mnx == 0 && mny == 0 && mnz == 0);
      m_lo = self ? 0 : jefi_delay_fp32(jefi_q_fp32(P.g.kx, P.g.ky, P.g.kz, (float)mnx, (float)mny, (float)mnz));
      m_hi = jefi_delay_fp32(jefi_q_fp32(P.g.kx, P.g.ky, P.g.kz, (float)mxx, (float)mxy, (float)mxz));
    };
    int item = 0;
    for (int base = 0; base < nt; base += 32) {
      // 32 source tiles at a time, one per lane: which of them has anything to contribute at this step?  Its window must reach a
      // stored step >= 0 (light cone of t0; depth, reading A15) and overlap the span of steps in which the tile's ring
      // row was not all zero (k_push_sources).  In the first steps of a run and on mostly empty grids nearly every tile drops out
      // here, 32 per round trip.
      int occ_first = 0x7f7f7f7f, occ_last = -1;
      int l_stx = 0, l_sty = 0, l_stz = 0, l_mlo = 0, l_mhi = 0;
      bool l_self = false, keep = false;
      if (base + lane < nt) {
        tile_window(t0 + base + lane, l_stx, l_sty, l_stz, l_mlo, l_mhi, l_self);
        occ_first = P.tile_first[t0 + base + lane];
        occ_last = P.tile_last[t0 + base + lane];
        const int mcap = min(n_now, d.H - 2);                        // largest delay with a stored, emitted step
        keep = l_mlo <= mcap && n_now - l_mlo >= occ_first && n_now - min(l_mhi, mcap) <= occ_last;
      }
      unsigned todo = __ballot_sync(0xffffffffu, keep);
      while (todo) {
      const int lsel = __ffs(todo) - 1;
      todo &= todo - 1;
      const int it = base + lsel;
      const unsigned FULLW = 0xffffffffu;
      const int t_first = __shfl_sync(FULLW, occ_first, lsel), t_last = __shfl_sync(FULLW, occ_last, lsel);
      const int stx = __shfl_sync(FULLW, l_stx, lsel), sty = __shfl_sync(FULLW, l_sty, lsel), stz = __shfl_sync(FULLW, l_stz, lsel);
      const int m_lo = __shfl_sync(FULLW, l_mlo, lsel), m_hi = __shfl_sync(FULLW, l_mhi, lsel);
      const bool self = __shfl_sync(FULLW, (int)l_self, lsel) != 0;
      const int sx0 = stx * G::TSX, sy0 = sty * G::TSY, sz0 = stz * G::TSZ;
      const int W = m_hi - m_lo + 1;
      const int npass = MULTI ? (W + WP - 1) / WP : 1;  // 1 unless the window exceeds the compiled pitch
      const size_t tile = (size_t)(t0 + it);
      const float4* rows = P.ring + tile * d.H * JEFI_ROW_QUADS;
      const int ix = (G::OBX / G::TSX) * obx - stx + (d.ntx - 1), iy = (G::OBY / G::TSY) * oby - sty + (d.nty - 1),
                iz = (G::OBZ / G::TSZ) * obz - stz + (d.ntz - 1);
      const size_t prow = (size_t)ix + (size_t)P.ndx * ((size_t)iy + (size_t)P.ndy * iz);
      for (int p = 0; p < npass; p++) {
        const int m_top = m_hi - p * WP;
        const int R = min(WP, m_top - m_lo + 1);
        // row j <-> delay m = m_top - j <-> absolute step t = n - m_top + j.  Rows with t < 0 (before t0)
        // or m > H-2 (not stored, reading A15) are zero: j < jv.
        int jv = max(m_top - n_now, m_top - (d.H - 2));
        jv = jv < 0 ? 0 : (jv > R ? R : jv);
        const int nvalid = R - jv;          // <= H - 1
        // Nothing of this window has been emitted yet (every delay of the tile pair reaches back before t0) or is stored: all
        // its sources are exactly zero, so the pairs add exactly nothing and the item is not staged at all.  In the first
        // n steps of a run only sources within n c dt of an observation tile are evaluated (the light cone of t0).
        if (nvalid == 0) continue;
        // the same for a source tile that held nothing but zeros during the steps this window reads, n - m_top + jv .. n - m_top +
        // R - 1 (an empty region of the grid, or one the charge has not reached or has left): skipped exactly as well
        if (n_now - m_top + R - 1 < t_first || n_now - m_top + jv > t_last) continue;
        const int s = item & 1;
        if (item >= 2) mbar_wait(barDone + 8 * s, ((item - 2) >> 1) & 1);  // consumers are done with item-2 (same stage)
        int s0 = nslot_now - (m_top - jv);  // ring slot of row jv; m_top - jv <= H - 2
        s0 += s0 < 0 ? d.H : 0;
        const int lenA = min(nvalid, d.H - s0), lenB = nvalid - lenA;  // ring wrap: at most two runs
        const uint32_t sb = sm0 + (uint32_t)s * L::BYTES;
#ifdef JEFI_CHECKED
        {  // poison the whole stage: a row that neither a copy nor the zero fill covers reads as NaN
          uint32_t* zz = reinterpret_cast<uint32_t*>(smem + (size_t)s * L::BYTES);
          for (int i = lane; i < (int)(L::ROWS / 4); i += 32) zz[i] = 0x7fc00000u;
          __syncwarp();
        }
#endif
        if (jv > 0) {  // zero rows (only in the first steps of a run or with a shallow ring)
          float4* z = reinterpret_cast<float4*>(smem + (size_t)s * L::BYTES);
          for (int i = lane; i < jv * JEFI_ROW_QUADS; i += 32) z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        __syncwarp();
        if (lane == 0) {
          stage_hdr h;
          h.Mtop = (uint32_t)m_top + 0x4B400000u;
          h.K = npass > 1 ? sb : sb + h.Mtop * (uint32_t)JEFI_ROW_BYTES;  // wraps mod 2^32 together with bits*2064
          h.mode = npass > 1 ? MODE_MULTI : (self ? MODE_SELF : MODE_PLAIN);
          h.dx0 = ox0 - sx0; h.dy0 = oy0 - sy0; h.dz0 = oz0 - sz0;
          h.R = (uint32_t)R;
          h.last = 0;
#ifdef JEFI_CHECKED
          h.last |= item << 1;  // sequence number of the item, checked by every consumer thread
#endif
          *reinterpret_cast<stage_hdr*>(smem + (size_t)s * L::BYTES + L::HDR) = h;
          fence_proxy_async();  // generic-proxy accesses of this stage (zero fill, earlier reads) before the async-proxy writes
          const uint32_t bar = barFull + 8 * s;
          mbar_expect_tx(bar, (uint32_t)(nvalid * JEFI_ROW_BYTES + OBCELLS * 2));
          if (lenA > 0) bulk_g2s(sb + (uint32_t)(jv * JEFI_ROW_BYTES), rows + (size_t)s0 * JEFI_ROW_QUADS, (uint32_t)(lenA * JEFI_ROW_BYTES), bar);
          if (lenB > 0) bulk_g2s(sb + (uint32_t)((jv + lenA) * JEFI_ROW_BYTES), rows, (uint32_t)(lenB * JEFI_ROW_BYTES), bar);
          bulk_g2s(sb + L::PERM, P.perm + prow * OBCELLS, OBCELLS * 2, bar);
        }
        item++;
      }
      }  // tiles of this round with something to contribute
    }
    {  // terminal item: tells the consumers that nothing follows (how many items were staged depends on the light cone)
      const int s = item & 1;
      if (item >= 2) mbar_wait(barDone + 8 * s, ((item - 2) >> 1) & 1);
      if (lane == 0) {
        stage_hdr h;
        h.K = 0; h.mode = MODE_END; h.dx0 = h.dy0 = h.dz0 = 0; h.Mtop = 0; h.R = 0;
        h.last = 1;
#ifdef JEFI_CHECKED
        h.last |= item << 1;
#endif
        *reinterpret_cast<stage_hdr*>(smem + (size_t)s * L::BYTES + L::HDR) = h;
        mbar_expect_tx(barFull + 8 * s, 0u);  // no bytes follow: the phase completes with this arrival
      }
    }
    return;
  }

  // -------------------------------------------------- consumer warps --------------------------------------------------
  // the consumers take items until the terminal one (MODE_END): how many were staged depends on the step (light cone of t0)
  for (int item = 0;; item++) {
    const int s = item & 1;
    const unsigned char* st = smem + (size_t)s * L::BYTES;
    mbar_wait(barFull + 8 * s, (item >> 1) & 1);
    const stage_hdr h = *reinterpret_cast<const stage_hdr*>(st + L::HDR);
#ifdef JEFI_CHECKED
    if ((h.last >> 1) != item) JEFI_CHECK_FAIL(1);
#endif
    if (h.mode == MODE_END) break;
    // the unit (G::CX cells along x) this lane evaluates for this source tile: neighbouring lanes are (almost) equidistant from it
    const int c = reinterpret_cast<const unsigned short*>(st + L::PERM)[tid];
    const int cx = G::CX * (c % G::UX), cy = (c / G::UX) % G::OBY, cz = c / (G::UX * G::OBY);
    float ax[G::TSX + G::CX - 1], ay[G::TSY];
#pragma unroll
    for (int l = 0; l < G::TSX + G::CX - 1; l++) ax[l] = P.g.kx * (float)(h.dx0 + cx + (G::CX - 1) - l);
#pragma unroll
    for (int l = 0; l < G::TSY; l++) ay[l] = P.g.ky * (float)(h.dy0 + cy - l);
    const float fz0 = (float)(h.dz0 + cz);
    pair_acc A[G::CX];
#pragma unroll
    for (int i = 0; i < G::CX; i++) {
      A[i].Exz = A[i].Fxz = A[i].Bxz = A[i].Cxz = A[i].By12 = pk(0.f, 0.f);
      A[i].Ey = A[i].Fy = 0.f;
    }
    item_addr I0;
    I0.K = h.K; I0.Mtop = h.Mtop; I0.R = h.R;
#ifdef JEFI_CHECKED
    I0.lo = sm0 + (uint32_t)s * L::BYTES;
    I0.hi = I0.lo + h.R * (uint32_t)JEFI_ROW_BYTES;
    if (h.R > (uint32_t)WP) JEFI_CHECK_FAIL(0);
#endif
    if (h.mode == MODE_PLAIN)
      tile_pairs<G, MODE_PLAIN, LINEAR>(I0, P.g.kz, ax, ay, fz0, A);
    else if (!MULTI || h.mode == MODE_SELF)
      tile_pairs<G, MODE_SELF, LINEAR>(I0, P.g.kz, ax, ay, fz0, A);
    else
      tile_pairs<G, MODE_MULTI, LINEAR>(I0, P.g.kz, ax, ay, fz0, A);
    // second accumulation level.  Unit c belongs to this thread alone in this item; the previous item's updates
    // (by other threads) are complete once every consumer warp has arrived on that item's done barrier.
    if (item > 0) mbar_wait(barDone + 8 * ((item - 1) & 1), ((item - 1) >> 1) & 1);
    const int sc = G::acc_slot(c);  // bank-spreading home of unit c's accumulators (jefi_ctx.h)
    if constexpr (G::CX == 1) {
      accS[sc] += lo32(A[0].Exz) - lo32(A[0].Fxz);
      accS[G::CELLS + sc] += A[0].Ey - A[0].Fy;
      accS[2 * G::CELLS + sc] += hi32(A[0].Exz) - hi32(A[0].Fxz);
      accS[3 * G::CELLS + sc] += lo32(A[0].Bxz) - lo32(A[0].Cxz);
      accS[4 * G::CELLS + sc] += lo32(A[0].By12) - hi32(A[0].By12);
      accS[5 * G::CELLS + sc] += hi32(A[0].Cxz) - hi32(A[0].Bxz);
    } else {
      // dyads keep their 12 sums together (48 bytes per unit: Ex0 Ex1 Ey0 Ey1 | Ez0 Ez1 Bx0 Bx1 | By0 By1 Bz0 Bz1): three
      // 16-byte read-modify-writes.  A 16-byte access is served per quarter-warp, and 8 permuted units collide on fewer of the 8
      // bank groups ((3 sc + k) mod 8) than 16 units do on the 16 bank pairs of an 8-byte access.
      float4* a4 = reinterpret_cast<float4*>(accS) + 3 * sc;
      float4 v;
      v = a4[0];
      v.x += lo32(A[0].Exz) - lo32(A[0].Fxz); v.y += lo32(A[1].Exz) - lo32(A[1].Fxz);
      v.z += A[0].Ey - A[0].Fy; v.w += A[1].Ey - A[1].Fy;
      a4[0] = v;
      v = a4[1];
      v.x += hi32(A[0].Exz) - hi32(A[0].Fxz); v.y += hi32(A[1].Exz) - hi32(A[1].Fxz);
      v.z += lo32(A[0].Bxz) - lo32(A[0].Cxz); v.w += lo32(A[1].Bxz) - lo32(A[1].Cxz);
      a4[1] = v;
      v = a4[2];
      v.x += lo32(A[0].By12) - hi32(A[0].By12); v.y += lo32(A[1].By12) - hi32(A[1].By12);
      v.z += hi32(A[0].Cxz) - hi32(A[0].Bxz); v.w += hi32(A[1].Cxz) - hi32(A[1].Bxz);
      a4[2] = v;
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(barDone + 8 * s);  // stage s may be refilled; this warp's accumulator updates are done
  }

  asm volatile("bar.sync 1, %0;" ::"n"(NCONS) : "memory");  // consumers only: all accumulator updates are visible
#pragma unroll
  for (int c = tid; c < G::CELLS; c += NCONS) {  // home order: x fastest inside the tile
    const int oi = ox0 + c % G::OBX, oj = oy0 + (c / G::OBX) % G::OBY, ok = oz0 + c / (G::OBX * G::OBY);
    if (oi < d.nx && oj < d.ny && ok < P.k1) {
      const size_t o = (size_t)oi + (size_t)d.nx * ((size_t)oj + (size_t)d.ny * ok);
      // cell c belongs to unit c / CX (x fastest).  CX = 1: component-major [6][cells]; CX = 2: 12 sums per unit (see above)
      const int a = G::CX == 1 ? G::acc_slot(c) : 12 * G::acc_slot(c / G::CX) + c % G::CX;
      constexpr int CS = G::CX == 1 ? G::CELLS : 2;  // stride between the components of a cell
      const float vex = P.g.prefE * accS[a], vey = P.g.prefE * accS[CS + a], vez = P.g.prefE * accS[2 * CS + a];
      const float vbx = P.g.prefB * accS[3 * CS + a], vby = P.g.prefB * accS[4 * CS + a], vbz = P.g.prefB * accS[5 * CS + a];
      if (P.to_partial) {
        float* q = P.partial + (size_t)blockIdx.y * 6 * (size_t)d.N + o;
        q[0] = vex; q[d.N] = vey; q[2 * d.N] = vez; q[3 * d.N] = vbx; q[4 * d.N] = vby; q[5 * d.N] = vbz;
      } else {
        P.ex[o] = vex; P.ey[o] = vey; P.ez[o] = vez;
        P.bx[o] = vbx; P.by[o] = vby; P.bz[o] = vbz;
        if (P.pack) {
          P.pack[2 * o] = make_float4(vex, vey, vez, vbx);
          P.pack[2 * o + 1] = make_float4(vby, vbz, 0.f, 0.f);
        }
      }
    }
  }
}

// Sum of the `nsplit` partial results of a launch that split the source range over blockIdx.y, piece 0 first: the same
// order on every run, so E and B are bit-reproducible (and observation slabs assemble the full step bit for bit).
__global__ void __launch_bounds__(256) k_reduce_partials(long N, int nsplit, long c0, long c1, const float* __restrict__ partial,
                                                         float* __restrict__ ex, float* __restrict__ ey, float* __restrict__ ez,
                                                         float* __restrict__ bx, float* __restrict__ by, float* __restrict__ bz,
                                                         float4* __restrict__ pack) {
  const long o = c0 + (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (o >= c1) return;
  float v[6];
#pragma unroll
  for (int a = 0; a < 6; a++) v[a] = partial[(size_t)a * N + o];
  for (int s = 1; s < nsplit; s++) {
    const float* q = partial + (size_t)s * 6 * (size_t)N + o;
#pragma unroll
    for (int a = 0; a < 6; a++) v[a] += q[(size_t)a * N];
  }
  ex[o] = v[0]; ey[o] = v[1]; ez[o] = v[2]; bx[o] = v[3]; by[o] = v[4]; bz[o] = v[5];
  if (pack) {
    pack[2 * o] = make_float4(v[0], v[1], v[2], v[3]);
    pack[2 * o + 1] = make_float4(v[4], v[5], 0.f, 0.f);
  }
}

// Evaluation order of the 512 cells of an observation tile for one relative tile offset D = (ox0 - sx0, ..).
// What it is for: an LDS.128 costs 2 data-pipe cycles instead of 4 when EVERY lane pair (2k, 2k+1) of the warp reads one
// quad, i.e. when the two observation cells of every pair have the same delay to the source cell being evaluated.
//   1. rank the cells by their distance to the centre of the source tile (ties in home order, x fastest); going down this order,
//      the first free cell takes as partner the one of the next 8 free cells that agrees with it on the delay to the most source
//      cells (equidistant AND close together): these are the 256 lane pairs;
//   2. per pair, the 64-bit set of source cells for which its two delays differ (same fp32 delay arithmetic as the kernel);
//   3. deal the pairs to the 16 warps greedily: a warp starts from the first free pair of the distance order and then takes,
//      15 times, the free pair among the next `band` pairs that adds the fewest new cells to the union of its pairs' sets
//      (a source cell outside the union takes the fast path for that warp).  The band (128 pairs) bounds the spread of the
//      delays inside a warp: rows 8 apart share a 16-byte bank group and are replayed when they meet in one wavefront;
//   4. the 16 pairs of a warp are put in distance order, so that each half-warp (one wavefront of the fast path) and each
//      quarter-warp (one wavefront of the slow path) spans only a few slots.
// Any order gives the same sums; this table only decides how fast.  One CTA of 512 threads per offset, once at create.
template <class G>
__global__ void __launch_bounds__(OBCELLS) k_build_perm(int ndx, int ndy, int ntx, int nty, int ntz, jefi_geom g, int band,
                                                        unsigned short* __restrict__ perm) {
  __shared__ float keys[OBCELLS];
  __shared__ unsigned short order[OBCELLS];
  __shared__ unsigned long long mask[G::CX][OBCELLS / 2];
  __shared__ unsigned short picked[OBCELLS / 2];
  __shared__ unsigned red[2][OBCELLS / 32];
  __shared__ unsigned short pairU[OBCELLS];  // units of lane pair p: pairU[2p], pairU[2p+1]
  __shared__ unsigned char usedr[OBCELLS];   // by position in the distance order
  __shared__ int cand[8];
  const int c = threadIdx.x;  // unit (G::CX cells along x) in home order
  const int ix = blockIdx.x % ndx, iy = (blockIdx.x / ndx) % ndy, iz = blockIdx.x / (ndx * ndy);
  const int Dxi = G::TSX * (ix - (ntx - 1)), Dyi = G::TSY * (iy - (nty - 1)), Dzi = G::TSZ * (iz - (ntz - 1));
  const int cx = G::CX * (c % G::UX), cy = (c / G::UX) % G::OBY, cz = c / (G::UX * G::OBY);
  const float rx = g.kx * ((float)Dxi + (float)cx + 0.5f * (float)(G::CX - 1) - 0.5f * (float)(G::TSX - 1)),
              ry = g.ky * ((float)Dyi + (float)cy - 0.5f * (float)(G::TSY - 1)), rz = g.kz * ((float)Dzi + (float)cz - 0.5f * (float)(G::TSZ - 1));
  const float key = rx * rx + ry * ry + rz * rz;
  keys[c] = key;
  __syncthreads();
  int pos = 0;
  for (int j = 0; j < OBCELLS; j++) {
    float kj = keys[j];
    pos += (kj < key) || (kj == key && j < c);
  }
  order[pos] = (unsigned short)c;
  __syncthreads();
  // 1b. lane pairs.  Unit `a` = the first free unit of the distance order; its partner = the one of the next 8 free units whose
  // delays agree with a's on the most source cells (ties: the nearer in the order).  Equal distance to the tile's centre makes
  // the delays to the centre agree; how they vary over the 64 source cells depends on how far apart the two units are, which the
  // distance order alone does not see.  8 groups of 64 threads: group = candidate, thread = source cell.
  {
    const int grp = c >> 6, sc = c & 63;
    const int lx = sc % G::TSX, ly = (sc / G::TSX) % G::TSY, lz = sc / (G::TSX * G::TSY);
    usedr[c] = 0;
    __syncthreads();
    int head = 0;
    for (int p = 0; p < OBCELLS / 2; p++) {
      while (usedr[head]) head++;  // the same in every thread (shared flags, read after the barrier below)
      int found = -1;
      for (int j = head + 1, cnt = -1; j < OBCELLS; j++)
        if (!usedr[j] && ++cnt == grp) { found = j; break; }
      unsigned bits = 0;
      if (found >= 0) {
        const int a = order[head], b = order[found];
        const int axc = G::CX * (a % G::UX), ayc = (a / G::UX) % G::OBY, azc = a / (G::UX * G::OBY);
        const int bxc = G::CX * (b % G::UX), byc = (b / G::UX) % G::OBY, bzc = b / (G::UX * G::OBY);
#pragma unroll
        for (int i = 0; i < G::CX; i++) {
          const float qa = jefi_q_fp32(g.kx, g.ky, g.kz, (float)(Dxi + axc + i - lx), (float)(Dyi + ayc - ly), (float)(Dzi + azc - lz));
          const float qb = jefi_q_fp32(g.kx, g.ky, g.kz, (float)(Dxi + bxc + i - lx), (float)(Dyi + byc - ly), (float)(Dzi + bzc - lz));
          const int ma = qa > 0.f ? jefi_delay_fp32(qa) : 0, mb = qb > 0.f ? jefi_delay_fp32(qb) : 0;
          bits += (ma != mb) ? 1u : 0u;
        }
      }
      const unsigned tot = __reduce_add_sync(0xffffffffu, bits);
      if ((c & 31) == 0) red[0][c >> 5] = tot;
      if (sc == 0) cand[grp] = found;
      __syncthreads();
      unsigned best = 0xffffffffu;
#pragma unroll
      for (int q = 0; q < 8; q++)
        if (cand[q] >= 0) best = min(best, ((red[0][2 * q] + red[0][2 * q + 1]) << 16) | (unsigned)cand[q]);
      const int partner = (int)(best & 0xffffu);
      __syncthreads();  // everyone has read red / cand / usedr of this step
      if (c == 0) {
        pairU[2 * p] = order[head];
        pairU[2 * p + 1] = order[partner];
        usedr[head] = 1;
        usedr[partner] = 1;
      }
      __syncthreads();
    }
  }
  // 2. pair c = units pairU[2c], pairU[2c+1]: source cells whose delay differs between the two, per cell of the unit
  unsigned long long mine[G::CX];
#pragma unroll
  for (int i = 0; i < G::CX; i++) mine[i] = 0;
  bool avail = c < OBCELLS / 2;
  if (avail) {
    const int a = pairU[2 * c], b = pairU[2 * c + 1];
    const int axc = G::CX * (a % G::UX), ayc = (a / G::UX) % G::OBY, azc = a / (G::UX * G::OBY);
    const int bxc = G::CX * (b % G::UX), byc = (b / G::UX) % G::OBY, bzc = b / (G::UX * G::OBY);
    for (int sc = 0; sc < JEFI_TCELLS; sc++) {
      const int lx = sc % G::TSX, ly = (sc / G::TSX) % G::TSY, lz = sc / (G::TSX * G::TSY);
#pragma unroll
      for (int i = 0; i < G::CX; i++) {
        const float qa = jefi_q_fp32(g.kx, g.ky, g.kz, (float)(Dxi + axc + i - lx), (float)(Dyi + ayc - ly), (float)(Dzi + azc - lz));
        const float qb = jefi_q_fp32(g.kx, g.ky, g.kz, (float)(Dxi + bxc + i - lx), (float)(Dyi + byc - ly), (float)(Dzi + bzc - lz));
        const int ma = qa > 0.f ? jefi_delay_fp32(qa) : 0, mb = qb > 0.f ? jefi_delay_fp32(qb) : 0;
        mine[i] |= (unsigned long long)(ma != mb) << sc;
      }
    }
#pragma unroll
    for (int i = 0; i < G::CX; i++) mask[i][c] = mine[i];
  }
  __syncthreads();
  // 3. greedy deal of the pairs to the warps (block-wide argmin per pick; keys are (cost << 16) | pair, pairs in distance order)
  const unsigned lane = c & 31, warp = c >> 5;
  int pick = 0;
  for (int w = 0; w < OBCELLS / 32; w++) {
    unsigned long long uni[G::CX];
#pragma unroll
    for (int i = 0; i < G::CX; i++) uni[i] = 0;
    int lo = 0;  // the warp's first pair = the lowest free pair; the others come from the `band` pairs that follow it
    for (int i = 0; i < 16; i++, pick++) {
      unsigned k = 0xffffffffu;
      if (avail) {
        unsigned cost = 0u;
        if (i != 0) {
          if (c < lo + band) {
#pragma unroll
            for (int q = 0; q < G::CX; q++) cost += (unsigned)__popcll(uni[q] | mine[q]);
          } else {
            cost = 0x7fffu;
          }
        }
        k = (cost << 16) | (unsigned)c;
      }
      k = __reduce_min_sync(0xffffffffu, k);
      if (lane == 0) red[pick & 1][warp] = k;
      __syncthreads();
      unsigned best = 0xffffffffu;
#pragma unroll
      for (int q = 0; q < OBCELLS / 32; q++) best = min(best, red[pick & 1][q]);
      const int sel = (int)(best & 0xffffu);
      if (i == 0) lo = sel;
      if (c == sel) avail = false;
      if (c == 0) picked[pick] = (unsigned short)sel;
#pragma unroll
      for (int q = 0; q < G::CX; q++) uni[q] |= mask[q][sel];
    }
  }
  __syncthreads();
  if (c < OBCELLS / 32) {  // the 16 pairs of warp c in distance order: every half- and quarter-warp then spans few slots
    unsigned short* q = picked + 16 * c;
    for (int i = 1; i < 16; i++) {
      const unsigned short v = q[i];
      int j = i - 1;
      for (; j >= 0 && q[j] > v; j--) q[j + 1] = q[j];
      q[j + 1] = v;
    }
  }
  __syncthreads();
  perm[(size_t)blockIdx.x * OBCELLS + c] = pairU[2 * picked[c >> 1] + (c & 1)];
}

// window pitches the kernel is compiled for (ring rows per stage); a wider window is served in several passes
static const int kPitches[] = {36, 48};
typedef void (*tiled_fn)(tiled_params);
template <class G>
static tiled_fn tiled_kernel_of(int wp, bool linear, bool multi) {
  if (multi) return linear ? k_field_tiled<G, 48, true, true> : k_field_tiled<G, 48, false, true>;  // several passes: largest pitch
  if constexpr (G::CX == 1) {
    if (wp == 36) return linear ? k_field_tiled<G, 36, true, false> : k_field_tiled<G, 36, false, false>;
  }
  if (wp == 48) return linear ? k_field_tiled<G, 48, true, false> : k_field_tiled<G, 48, false, false>;
  return nullptr;
}
static tiled_fn tiled_kernel_for(const jefi_ctx* c) {
  const bool linear = c->cfg.delay_rule == JEFI_DELAY_LINEAR, multi = c->wmax > c->wpitch;
  switch (c->tile_geom) {
    case JEFI_GEOM_SLABX: return tiled_kernel_of<jefi_geom_slabx>(c->wpitch, linear, multi);
    case JEFI_GEOM_DYAD: return tiled_kernel_of<jefi_geom_dyad>(c->wpitch, linear, multi);
  }
  return tiled_kernel_of<jefi_geom_cube>(c->wpitch, linear, multi);
}
static size_t tiled_smem_for(int wp, int cells) {
  if (cells == 1024) return stage_layout<48, 1024>::TOTAL;
  return wp == 36 ? stage_layout<36, 512>::TOTAL : stage_layout<48, 512>::TOTAL;
}

// How the source range is split over blockIdx.y.  Grids with at least four waves of observation tiles use 32 pieces (L2
// locality, below).  Smaller grids split the source tiles so that the CTAs fill whole waves of the GPU: cost model = waves x (tiles per CTA + c0), c0 = 1.5 tiles of fixed cost per CTA
// (accumulator zeroing, barrier set-up, first copy latency, epilogue).
static void choose_split(int nobs, int ntiles, int nsm, int request, int& chunk, int& nsplit) {
  if (request == -1) {
    chunk = ntiles;
  } else if (request == 0 && nobs >= 4 * nsm) {
    // Large grids: 32 pieces.  CTAs are scheduled blockIdx.y-major, so all observation tiles work through the same 1/32 of the
    // ring before any moves on, and the windows they fetch overlap in L2 (96^3: 1 / 8 / 32 / 128 pieces = 670.8 / 656.8 / 653.2 /
    // 652.6 ms including k_reduce_partials; the partial sums take 24 N bytes per piece).
    chunk = (ntiles + 31) / 32;
  } else if (request > 0) {
    chunk = request < ntiles ? request : ntiles;
  } else {
    double best = 1e300;
    chunk = ntiles;
    for (int ns = 1; ns <= ntiles && ns <= 256; ns++) {
      const int ch = (ntiles + ns - 1) / ns;
      const int pieces = (ntiles + ch - 1) / ch;
      const long ctas = (long)nobs * pieces;
      const long waves = (ctas + nsm - 1) / nsm;
      const double cost = (double)waves * ((double)ch + 1.5);
      if (cost < best * 0.999) { best = cost; chunk = ch; }
    }
  }
  if (chunk < 1) chunk = 1;
  if ((ntiles + chunk - 1) / chunk > 65535) chunk = (ntiles + 65534) / 65535;
  nsplit = (ntiles + chunk - 1) / chunk;
}

// Largest slot window over all relative placements of an observation tile and a source tile (host, fp64),
// shared-memory opt-in, and the evaluation-order table.
int jefi_tiled_prepare(jefi_ctx* c) {
  const jefi_dims& d = c->dims;
  const double L0 = c->c * c->cfg.dt;
  const int nobx = (d.nx + d.obx - 1) / d.obx, noby = (d.ny + d.oby - 1) / d.oby, nobz = (d.nz + d.obz - 1) / d.obz;
  int wmax = 1;
  // the window depends only on the per-axis difference D = ox0 - sx0 (a multiple of the source tile edge)
  for (int Dz = -(d.ntz - 1) * d.tsz; Dz <= (nobz - 1) * d.obz; Dz += d.tsz)
    for (int Dy = -(d.nty - 1) * d.tsy; Dy <= (noby - 1) * d.oby; Dy += d.tsy)
      for (int Dx = -(d.ntx - 1) * d.tsx; Dx <= (nobx - 1) * d.obx; Dx += d.tsx) {
        int mnx, mxx, mny, mxy, mnz, mxz;
        abs_range(Dx - (d.tsx - 1), Dx + d.obx - 1, mnx, mxx);
        abs_range(Dy - (d.tsy - 1), Dy + d.oby - 1, mny, mxy);
        abs_range(Dz - (d.tsz - 1), Dz + d.obz - 1, mnz, mxz);
        double rlo = sqrt(pow(mnx * c->cfg.dx, 2) + pow(mny * c->cfg.dy, 2) + pow(mnz * c->cfg.dz, 2));
        double rhi = sqrt(pow(mxx * c->cfg.dx, 2) + pow(mxy * c->cfg.dy, 2) + pow(mxz * c->cfg.dz, 2));
        int w = (int)floor(rhi / L0 + 0.5) - (int)floor(rlo / L0 + 0.5) + 1;
        if (w > wmax) wmax = w;
      }
  c->wmax = wmax;
  int wp = kPitches[sizeof(kPitches) / sizeof(int) - 1];  // wider windows: several passes through the largest pitch
  for (int cand : kPitches)
    if (cand >= wmax) { wp = cand; break; }
  if (c->tile_geom == JEFI_GEOM_DYAD) wp = 48;  // compiled for the large pitch only (its windows reach 47 slots at dx = 2 c dt)
  c->wpitch = wp;
  c->tiled_smem = tiled_smem_for(wp, d.obx * d.oby * d.obz);
  int dev = c->cfg.device, max_optin = 0;
  cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
  if (c->tiled_smem > (size_t)max_optin) {
    char buf[160];
    snprintf(buf, sizeof buf, "tiled kernel needs %zu B of shared memory (window %d slots), device allows %d", c->tiled_smem, wmax, max_optin);
    c->err = buf;
    return JEFI_ESTATE;
  }
  cudaError_t e = cudaFuncSetAttribute(tiled_kernel_for(c), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->tiled_smem);
  if (e != cudaSuccess) { c->err = std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
  int nsm = 148;
  cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev);
  const int nobs = nobx * noby * nobz, ntiles = d.ntx * d.nty * d.ntz;
  choose_split(nobs, ntiles, nsm, c->cfg.field_chunk, c->chunk, c->nsplit);
  // Partial sums of a split launch: 24 N bytes per piece (680 MB for 32 pieces at 96^3, 1.6 GB at 128^3).  When the ring already
  // fills most of the device that allocation can fail; the split only buys L2 locality (0.5-2.6 % at 96^3, choose_split) or whole
  // waves on small grids, so fall back to a quarter of the pieces each time and finally to one piece, which needs no buffer,
  // rather than give up the tiled kernel.  jefi_get_tile_info reports the split that is in use.
  while (c->nsplit > 1) {
    const size_t bytes = (size_t)c->nsplit * 6 * (size_t)d.N * sizeof(float);
    if ((e = cudaMalloc(&c->partial, bytes)) == cudaSuccess) break;
    c->partial = nullptr;
    (void)cudaGetLastError();  // the failed allocation must not surface as the next launch's error
    const int fewer = c->nsplit / 4;
    choose_split(nobs, ntiles, nsm, fewer > 1 ? (ntiles + fewer - 1) / fewer : -1, c->chunk, c->nsplit);
  }
  // evaluation-order table over all relative tile offsets
  c->ndx = d.ntx + (d.obx / d.tsx) * (nobx - 1); c->ndy = d.nty + (d.oby / d.tsy) * (noby - 1); c->ndz = d.ntz + (d.obz / d.tsz) * (nobz - 1);
  size_t rows = (size_t)c->ndx * c->ndy * c->ndz;
  if ((e = cudaMalloc(&c->perm, rows * OBCELLS * sizeof(unsigned short))) != cudaSuccess) {
    c->perm = nullptr;
    c->err = std::string("permutation table allocation: ") + cudaGetErrorString(e);
    return JEFI_ENOMEM;
  }
  // pairs a warp may draw from, counted from its first pair in the distance order: wide enough to find pairs that differ on
  // the same source cells, narrow enough that the delays of one warp stay within 8 slots (rows 8 apart share a bank group)
  const int band = 128;  // measured on cfg4 96^3: band 64 unsorted 741.3 ms, 64 / 96 / 128 / 256 with step 4: 741.2 / 739.7 / 738.9 / 738.7 ms
  if (c->tile_geom == JEFI_GEOM_SLABX)
    k_build_perm<jefi_geom_slabx><<<(unsigned)rows, OBCELLS, 0, c->stream>>>(c->ndx, c->ndy, d.ntx, d.nty, d.ntz, c->geom, band, c->perm);
  else if (c->tile_geom == JEFI_GEOM_DYAD)
    k_build_perm<jefi_geom_dyad><<<(unsigned)rows, OBCELLS, 0, c->stream>>>(c->ndx, c->ndy, d.ntx, d.nty, d.ntz, c->geom, band, c->perm);
  else
    k_build_perm<jefi_geom_cube><<<(unsigned)rows, OBCELLS, 0, c->stream>>>(c->ndx, c->ndy, d.ntx, d.nty, d.ntz, c->geom, band, c->perm);
  if ((e = cudaGetLastError()) != cudaSuccess) { c->err = std::string("k_build_perm: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
  c->launches++;
  return JEFI_OK;
}

int jefi_launch_field_tiled(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz,
                            float* eb_packed) {
  const jefi_dims& d = c->dims;
  tiled_params P;
  P.d = d; P.g = c->geom; P.n = (int)c->step; P.nslot = (int)(c->step % d.H);
  P.nobx = (d.nx + d.obx - 1) / d.obx; P.noby = (d.ny + d.oby - 1) / d.oby;
  P.ndx = c->ndx; P.ndy = c->ndy;
  P.chunk = c->chunk;
  P.to_partial = c->nsplit > 1 ? 1 : 0;
  P.step_dev = c->capturing ? c->step_dev : nullptr;
  P.ring = c->ring; P.perm = c->perm;
  P.tile_first = c->tile_first; P.tile_last = c->tile_last;
  P.ex = ex; P.ey = ey; P.ez = ez; P.bx = bx; P.by = by; P.bz = bz;
  P.pack = reinterpret_cast<float4*>(eb_packed);
  P.partial = c->partial;
  P.obz0 = k0 / d.obz; P.k1 = k1;
  const int nlayers = (k1 - k0 + d.obz - 1) / d.obz;
  dim3 grid((unsigned)(P.nobx * P.noby * nlayers), (unsigned)c->nsplit);
  tiled_kernel_for(c)<<<grid, TILED_THREADS, c->tiled_smem, c->stream>>>(P);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  if (c->nsplit > 1) {
    const long c0 = (long)k0 * d.nx * d.ny, c1 = (long)k1 * d.nx * d.ny;
    k_reduce_partials<<<(unsigned)((c1 - c0 + 255) / 256), 256, 0, c->stream>>>(d.N, c->nsplit, c0, c1, c->partial, ex, ey, ez, bx, by, bz, P.pack);
    JEFI_CUDA_TRY(c, cudaGetLastError());
    c->launches++;
  }
  return JEFI_OK;
}
