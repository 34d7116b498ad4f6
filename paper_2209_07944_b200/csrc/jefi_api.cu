// libjefi: context, history ring buffer and debug exports.  Boundary: include/jefi.h.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "jefi_ctx.h"

static thread_local std::string g_create_err;  // jefi_last_error(NULL): per calling thread

static int fail_create(jefi_ctx* c, int code, const std::string& msg) {
  g_create_err = msg;
  if (c) {
    c->err = msg;
    jefi_destroy(c);
  }
  return code;
}

extern "C" int jefi_config_init(jefi_config* cfg, unsigned long sizeof_cfg) {
  if (!cfg || sizeof_cfg != sizeof(jefi_config)) {
    g_create_err = !cfg ? "jefi_config_init: cfg is NULL"
                        : "jefi_config_init: the caller's jefi_config has " + std::to_string(sizeof_cfg) + " bytes, this library's has " +
                              std::to_string(sizeof(jefi_config)) + ": rebuild against this library's include/jefi.h";
    return JEFI_EINVAL;
  }
  memset(cfg, 0, sizeof *cfg);
  return JEFI_OK;
}

extern "C" const char* jefi_last_error(const jefi_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" long jefi_launch_count(const jefi_ctx* ctx) { return ctx ? ctx->launches : 0; }

extern "C" int jefi_get_info(const jefi_ctx* ctx, int* H, int* ndt, int* field_impl, long* step, long* ring_bytes) {
  if (!ctx) return JEFI_EINVAL;
  if (H) *H = ctx->dims.H;
  if (ndt) *ndt = ctx->ndt;
  if (field_impl) *field_impl = ctx->field_impl;
  if (step) *step = ctx->step;
  if (ring_bytes) *ring_bytes = ctx->ring_bytes;
  return JEFI_OK;
}

extern "C" const char* jefi_field_impl_reason(const jefi_ctx* ctx) { return ctx ? ctx->impl_reason.c_str() : ""; }

extern "C" int jefi_get_tile_info(const jefi_ctx* ctx, int obs_tile[3], int src_tile[3], int* window_slots, int* window_pitch,
                                  int* source_split) {
  if (!ctx) return JEFI_EINVAL;
  const jefi_dims& d = ctx->dims;
  if (obs_tile) { obs_tile[0] = d.obx; obs_tile[1] = d.oby; obs_tile[2] = d.obz; }
  if (src_tile) { src_tile[0] = d.tsx; src_tile[1] = d.tsy; src_tile[2] = d.tsz; }
  if (window_slots) *window_slots = ctx->wmax;
  if (window_pitch) *window_pitch = ctx->wpitch;
  if (source_split) *source_split = ctx->nsplit;
  return JEFI_OK;
}


extern "C" int jefi_create(const jefi_config* cfg, jefi_ctx** out) {
  if (out) *out = nullptr;
  if (!cfg || !out) return fail_create(nullptr, JEFI_EINVAL, "jefi_create: NULL argument");
  if (cfg->nx < 1 || cfg->ny < 1 || cfg->nz < 1 || !(cfg->dx > 0) || !(cfg->dy > 0) || !(cfg->dz > 0) || !(cfg->dt > 0) ||
      cfg->c < 0 || cfg->eps0 < 0 || cfg->H < 0 || cfg->hist_cap < 0 || cfg->deposit_mode < 0 || cfg->deposit_mode > 3 || cfg->delay_rule < 0 || cfg->delay_rule > 1 ||
      cfg->shape_order < 0 || cfg->shape_order > 2 || cfg->field_chunk < -1 || cfg->field_tile < 0 || cfg->field_tile > 2 || cfg->field_impl < 0 || cfg->field_impl > 2)
    return fail_create(nullptr, JEFI_EINVAL, "jefi_create: grid sizes, spacings and dt must be positive, switches in range");
  if ((long)cfg->nx * cfg->ny * cfg->nz > (1L << 30)) return fail_create(nullptr, JEFI_EINVAL, "jefi_create: grid too large");
  jefi_ctx* c = new (std::nothrow) jefi_ctx();
  if (!c) return fail_create(nullptr, JEFI_ENOMEM, "jefi_create: host allocation failed");
  c->cfg = *cfg;
  c->ring = nullptr;
  c->mtab_dev = nullptr;
  c->mtab_host = nullptr;
  c->src_stage = c->eb_stage = nullptr;
  c->perm = nullptr;
  c->tile_first = c->tile_last = nullptr;
  c->partial = nullptr;
  c->step_dev = nullptr;
  c->step_dev_value = -2;
  c->capturing = false;
  c->pic_exec = nullptr;
  c->sort_gen = 0;
  c->pic_launches = 0;
  c->wmax = c->wpitch = 0;
  c->chunk = 0;
  c->nsplit = 1;
  c->tiled_smem = 0;
  c->shape_order = cfg->shape_order == 2 ? 2 : 1;
  c->sort_count = c->sort_offset = c->sort_sums = nullptr;
  c->sort_key = c->sort_rank = c->sort_order = nullptr;
  c->sort_cap = 0;
  c->sorted_np = -1;
  c->deposits_since_sort = 0;
  c->sort_buf = nullptr;
  c->eb_pack = nullptr;
  for (int i = 0; i < JEFI_NEVENTS; i++) c->ev0[i] = c->ev1[i] = nullptr;
  c->field_calls = 0;
  c->launches = 0;
  c->step = -1;
  c->stream = (cudaStream_t)cfg->stream;
  c->c = cfg->c > 0 ? cfg->c : 299792458.0;
  c->eps0 = cfg->eps0 > 0 ? cfg->eps0 : 8.8541878128e-12;
  c->mu0 = 1.0 / (c->eps0 * c->c * c->c);

  // the caller's current device is restored on return (every later entry point does the same, jefi_device_guard)
  struct restore_dev { int prev = -1; ~restore_dev() { if (prev >= 0) cudaSetDevice(prev); } } rd;
  cudaGetDevice(&rd.prev);
  cudaError_t e = cudaSetDevice(cfg->device);
  if (e != cudaSuccess) return fail_create(c, JEFI_ECUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e));

  // ---- history depth ----
  const double L0 = c->c * cfg->dt;  // light-step length
  double lx = cfg->nx * cfg->dx, ly = cfg->ny * cfg->dy, lz = cfg->nz * cfg->dz;
  double lmax = sqrt(lx * lx + ly * ly + lz * lz);
  long cap = cfg->hist_cap > 0 ? cfg->hist_cap : 10000;
  long ndt = (long)ceil(lmax / L0);
  if (ndt > cap) ndt = cap;
  c->ndt = (int)ndt;
  int H = cfg->H > 0 ? cfg->H : (int)ndt + 2;
  if (H < 2) return fail_create(c, JEFI_EINVAL, "jefi_create: H must be >= 2 (value and backward difference)");

  jefi_dims& d = c->dims;
  d.nx = cfg->nx; d.ny = cfg->ny; d.nz = cfg->nz;
  // tile geometry: cubes, or x-thin tiles for the paper's 1 x ny x nz slabs
  // (field_tile): two x-neighbour cells per thread once the grid has 32 tiles of 16x8x8 and x does not pad much worse than with
  // 8-wide tiles (measured on B200, kernel ms of one step, 8x8x8 / 16x8x8 tiles: 32^3 1.056 / 1.035, 48^3 11.33 / 10.99,
  // 64^3 63.1 / 59.8, 80^3 248.1 / 223.4, 96^3 741 / 675)
  const long ndyad = (long)((cfg->nx + 15) / 16) * ((cfg->ny + 7) / 8) * ((cfg->nz + 7) / 8);
  const bool xpad_ok = ((cfg->nx + 15) / 16) * 16 == ((cfg->nx + 7) / 8) * 8 || cfg->nx >= 64;
  const bool dyad = cfg->nx >= 16 && (cfg->field_tile == JEFI_TILE_DYAD || (cfg->field_tile == JEFI_TILE_AUTO && ndyad >= 32 && xpad_ok));
  c->tile_geom = cfg->nx <= 3 ? JEFI_GEOM_SLABX : (dyad ? JEFI_GEOM_DYAD : JEFI_GEOM_CUBE);
  if (c->tile_geom == JEFI_GEOM_SLABX) {
    d.tsx = jefi_geom_slabx::TSX; d.tsy = jefi_geom_slabx::TSY; d.tsz = jefi_geom_slabx::TSZ;
    d.obx = jefi_geom_slabx::OBX; d.oby = jefi_geom_slabx::OBY; d.obz = jefi_geom_slabx::OBZ;
  } else if (c->tile_geom == JEFI_GEOM_DYAD) {
    d.tsx = jefi_geom_dyad::TSX; d.tsy = jefi_geom_dyad::TSY; d.tsz = jefi_geom_dyad::TSZ;
    d.obx = jefi_geom_dyad::OBX; d.oby = jefi_geom_dyad::OBY; d.obz = jefi_geom_dyad::OBZ;
  } else {
    d.tsx = jefi_geom_cube::TSX; d.tsy = jefi_geom_cube::TSY; d.tsz = jefi_geom_cube::TSZ;
    d.obx = jefi_geom_cube::OBX; d.oby = jefi_geom_cube::OBY; d.obz = jefi_geom_cube::OBZ;
  }
  d.ntx = (cfg->nx + d.tsx - 1) / d.tsx; d.nty = (cfg->ny + d.tsy - 1) / d.tsy; d.ntz = (cfg->nz + d.tsz - 1) / d.tsz;
  d.H = H;
  d.N = (long)cfg->nx * cfg->ny * cfg->nz;
  d.ncell_pad = (long)d.ntx * d.nty * d.ntz * JEFI_TCELLS;

  // ---- scaled geometry: d' = d/(c dt), J stored as J/c ----
  const double dV = cfg->dx * cfg->dy * cfg->dz;
  const double PI = 3.14159265358979323846;
  c->geom.kx = (float)(cfg->dx / L0);
  c->geom.ky = (float)(cfg->dy / L0);
  c->geom.kz = (float)(cfg->dz / L0);
  c->geom.prefE = (float)(dV / (4.0 * PI * c->eps0) / (L0 * L0));
  c->geom.prefB = (float)(-c->mu0 * dV / (4.0 * PI) * c->c / (L0 * L0));

  // ---- ring: zero-initialised = "J and rho are simply set to zero" before t0 ----
  size_t ring_quads = (size_t)d.ntx * d.nty * d.ntz * H * JEFI_ROW_QUADS;
  c->ring_bytes = (long)(ring_quads * sizeof(float4));
  if ((e = cudaMalloc(&c->ring, ring_quads * sizeof(float4))) != cudaSuccess)
    return fail_create(c, JEFI_ENOMEM, std::string("ring allocation (") + std::to_string(c->ring_bytes) + " B): " + cudaGetErrorString(e));
  if ((e = cudaMemsetAsync(c->ring, 0, ring_quads * sizeof(float4), c->stream)) != cudaSuccess)
    return fail_create(c, JEFI_ECUDA, std::string("ring zero fill: ") + cudaGetErrorString(e));
  // per source tile, the span of steps whose ring row holds anything but zeros (k_push_sources keeps it; the tiled kernel skips
  // tile pairs whose window lies outside it): first = 0x7f7f7f7f, last = -1 mean "never"
  const size_t ntile_all = (size_t)d.ntx * d.nty * d.ntz;
  if ((e = cudaMalloc(&c->tile_first, ntile_all * sizeof(int))) != cudaSuccess || (e = cudaMalloc(&c->tile_last, ntile_all * sizeof(int))) != cudaSuccess)
    return fail_create(c, JEFI_ENOMEM, std::string("tile occupancy allocation: ") + cudaGetErrorString(e));
  if ((e = cudaMemsetAsync(c->tile_first, 0x7f, ntile_all * sizeof(int), c->stream)) != cudaSuccess ||
      (e = cudaMemsetAsync(c->tile_last, 0xff, ntile_all * sizeof(int), c->stream)) != cudaSuccess)
    return fail_create(c, JEFI_ECUDA, std::string("tile occupancy fill: ") + cudaGetErrorString(e));

  // ---- delay table, fp64 on the host: m = floor(R/(c dt) + 1/2) (Eq. 2.6, reading A1) ----
  const int ex = jefi_table_extent(d.nx, d.obx), ey = jefi_table_extent(d.ny, d.oby), ez = jefi_table_extent(d.nz, d.obz);
  c->tex = ex; c->tey = ey; c->tez = ez;
  size_t tn = (size_t)ex * ey * ez;
  c->mtab_host = (int*)malloc(tn * sizeof(int));
  if (!c->mtab_host) return fail_create(c, JEFI_ENOMEM, "delay table host allocation failed");
  for (int kc = 0; kc < ez; kc++)
    for (int jb = 0; jb < ey; jb++)
      for (int ia = 0; ia < ex; ia++) {
        double ddx = ia * cfg->dx, ddy = jb * cfg->dy, ddz = kc * cfg->dz;
        double R = sqrt(ddx * ddx + ddy * ddy + ddz * ddz);
        c->mtab_host[ia + (size_t)ex * (jb + (size_t)ey * kc)] = (int)floor(R / L0 + 0.5);
      }
  if ((e = cudaMalloc(&c->step_dev, 4 * sizeof(int))) != cudaSuccess)
    return fail_create(c, JEFI_ENOMEM, std::string("step state allocation: ") + cudaGetErrorString(e));
  if ((e = cudaMalloc(&c->mtab_dev, tn * sizeof(int))) != cudaSuccess)
    return fail_create(c, JEFI_ENOMEM, std::string("delay table device allocation: ") + cudaGetErrorString(e));
  if ((e = cudaMemcpyAsync(c->mtab_dev, c->mtab_host, tn * sizeof(int), cudaMemcpyHostToDevice, c->stream)) != cudaSuccess)
    return fail_create(c, JEFI_ECUDA, std::string("delay table upload: ") + cudaGetErrorString(e));

  for (int i = 0; i < JEFI_NEVENTS; i++)
    if ((e = cudaEventCreate(&c->ev0[i])) != cudaSuccess || (e = cudaEventCreate(&c->ev1[i])) != cudaSuccess)
      return fail_create(c, JEFI_ECUDA, std::string("cudaEventCreate: ") + cudaGetErrorString(e));

  // ---- choose the field kernel ----
  c->field_impl = JEFI_FIELD_REFERENCE;
  c->impl_reason = "reference: requested (JEFI_FIELD_REFERENCE)";
  if (cfg->field_impl != JEFI_FIELD_REFERENCE) {
    // Proof that the tiled kernel's fp32 delay arithmetic equals the fp64 table on every offset.  An offset whose s = R/(c dt)
    // lies within fp32 rounding of a half-integer (a near-tie of the nearest-step rule) can come out one step off; the scaled
    // spacings kx, ky, kz are then moved by a few units in the last place (|eps| <= 8 * 2^-23: the field values change by
    // <= 3e-6 relative, the delays are the TABLE's or the proof fails) until all offsets agree.  Exact ties (s = m + 1/2 in exact
    // arithmetic, e.g. kappa = 1.5) survive every such move: the reference kernel then runs and says so.
    const jefi_geom g0 = c->geom;
    long mism = -1, noff = 0, mism0 = -1;
    int moved = 0;
    for (int trial = 0; trial <= 16 && mism != 0; trial++) {
      moved = (trial + 1) / 2 * ((trial & 1) ? 1 : -1);  // 0, +1, -1, +2, -2, ..
      const double f = 1.0 + moved * 1.1920928955078125e-07;
      c->geom.kx = (float)((double)g0.kx * f); c->geom.ky = (float)((double)g0.ky * f); c->geom.kz = (float)((double)g0.kz * f);
      int rc = jefi_verify_delay_fp32(c, &mism, &noff);
      if (rc != JEFI_OK) return fail_create(c, rc, c->err);
      if (trial == 0) mism0 = mism;
    }
    if (mism != 0) { c->geom = g0; moved = 0; mism = mism0; }
    int prep = (mism == 0) ? jefi_tiled_prepare(c) : JEFI_ESTATE;
    char buf[400];
    if (mism == 0 && prep == JEFI_OK) {
      c->field_impl = JEFI_FIELD_TILED;
      char mv[96] = "";
      if (moved != 0) snprintf(mv, sizeof mv, " (scaled spacings moved by %+d ulp to clear %ld near-ties)", moved, mism0);
      snprintf(buf, sizeof buf, "tiled: fp32 delays proven equal to the fp64 table on %ld offsets%s; tiles %dx%dx%d / %dx%dx%d, window %d slots "
               "in pitch %d (%d pass%s), source range in %d piece%s", noff, mv, d.obx, d.oby, d.obz, d.tsx, d.tsy, d.tsz, c->wmax, c->wpitch,
               (c->wmax + c->wpitch - 1) / c->wpitch, c->wmax > c->wpitch ? "es" : "", c->nsplit, c->nsplit > 1 ? "s" : "");
      c->impl_reason = buf;
    } else {
      if (mism != 0)
        snprintf(buf, sizeof buf, "reference: %ld of %ld fp32 delays differ from the fp64 table, also with the spacings moved by up to 8 ulp "
                 "(exact ties s = m + 1/2 of the nearest-step rule): the tiled kernel cannot be proven", mism, noff);
      else
        snprintf(buf, sizeof buf, "reference: tiled kernel could not be prepared (rc=%d: %s)", prep, c->err.c_str());
      c->impl_reason = buf;
      if (cfg->field_impl == JEFI_FIELD_TILED) return fail_create(c, JEFI_ESTATE, std::string("tiled field kernel not usable; ") + buf);
    }
  }
  if ((e = cudaStreamSynchronize(c->stream)) != cudaSuccess)
    return fail_create(c, JEFI_ECUDA, std::string("create sync: ") + cudaGetErrorString(e));
  c->err.clear();
  *out = c;
  return JEFI_OK;
}

extern "C" void jefi_destroy(jefi_ctx* c) {
  if (!c) return;
  jefi_device_guard guard(c);
  cudaStreamSynchronize(c->stream);
  if (c->ring) cudaFree(c->ring);
  if (c->mtab_dev) cudaFree(c->mtab_dev);
  if (c->perm) cudaFree(c->perm);
  if (c->tile_first) cudaFree(c->tile_first);
  if (c->tile_last) cudaFree(c->tile_last);
  if (c->partial) cudaFree(c->partial);
  if (c->step_dev) cudaFree(c->step_dev);
  if (c->pic_exec) cudaGraphExecDestroy(c->pic_exec);
  if (c->src_stage) cudaFree(c->src_stage);
  if (c->eb_stage) cudaFree(c->eb_stage);
  if (c->sort_count) cudaFree(c->sort_count);
  if (c->sort_offset) cudaFree(c->sort_offset);
  if (c->sort_sums) cudaFree(c->sort_sums);
  if (c->sort_key) cudaFree(c->sort_key);
  if (c->sort_rank) cudaFree(c->sort_rank);
  if (c->sort_order) cudaFree(c->sort_order);
  if (c->sort_buf) cudaFree(c->sort_buf);
  if (c->eb_pack) cudaFree(c->eb_pack);
  if (c->mtab_host) free(c->mtab_host);
  for (int i = 0; i < JEFI_NEVENTS; i++) {
    if (c->ev0[i]) cudaEventDestroy(c->ev0[i]);
    if (c->ev1[i]) cudaEventDestroy(c->ev1[i]);
  }
  delete c;
}

// ------------------------------------------------------------------------------------------------------------
// Row a1: history push.  One thread per padded ring cell, in ring order (tile, cell): the 16-byte writes of a tile
// row are contiguous.  Reads the previous slot, writes value and backward difference.
// Traffic: 16 B in (4 SoA floats) + 16 B read (previous) + 32 B written per cell.
// ------------------------------------------------------------------------------------------------------------
// step_dev != NULL (jefi_pic_step's graph): slot and previous slot come from the device-side step state.
__global__ void __launch_bounds__(256) k_push_sources(jefi_dims d, float inv_c, int n, int slot, int prev_slot, const int* __restrict__ step_dev,
                                                      const float* __restrict__ rho, const float* __restrict__ jx,
                                                      const float* __restrict__ jy, const float* __restrict__ jz,
                                                      float4* __restrict__ ring, int* __restrict__ tile_first, int* __restrict__ tile_last) {
  const long r = (long)blockIdx.x * blockDim.x + threadIdx.x;  // a warp's 32 cells belong to one tile (64 cells per tile)
  if (step_dev) { n = step_dev[0]; slot = step_dev[1]; prev_slot = step_dev[2]; }
  const long tile = r / JEFI_TCELLS;
  const int cell = (int)(r - tile * JEFI_TCELLS);
  const int tx = (int)(tile % d.ntx), ty = (int)((tile / d.ntx) % d.nty), tz = (int)(tile / ((long)d.ntx * d.nty));
  const int i = tx * d.tsx + cell % d.tsx, j = ty * d.tsy + (cell / d.tsx) % d.tsy, k = tz * d.tsz + cell / (d.tsx * d.tsy);
  bool nz = false;
  if (r < d.ncell_pad && i < d.nx && j < d.ny && k < d.nz) {  // padded cells stay zero
    const size_t cidx = (size_t)i + (size_t)d.nx * ((size_t)j + (size_t)d.ny * k);
    const size_t q = jefi_ring_quad(d, tile, slot, cell);
    const float4 s = make_float4(jx[cidx] * inv_c, jz[cidx] * inv_c, rho[cidx], jy[cidx] * inv_c);
    const float4 p = prev_slot >= 0 ? ring[jefi_ring_quad(d, tile, prev_slot, cell)] : make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 dd = make_float4(s.x - p.x, s.y - p.y, s.z - p.z, s.w - p.w);
    ring[q] = s;
    ring[q + JEFI_TCELLS] = dd;
    nz = !(s.x == 0.f && s.y == 0.f && s.z == 0.f && s.w == 0.f && dd.x == 0.f && dd.y == 0.f && dd.z == 0.f && dd.w == 0.f);  // NaN counts
  }
  // the span of steps in which this tile's row is not all zero (read by the tiled field kernel to skip empty source tiles)
  if (__any_sync(0xffffffffu, nz) && (threadIdx.x & 31) == 0) {
    atomicMin(tile_first + tile, n);
    atomicMax(tile_last + tile, n);
  }
}

__global__ void k_advance_step(int* __restrict__ st, int H) {  // n += 1 on the device (first kernel of the PIC-step graph)
  const int n = st[0] + 1;
  st[0] = n;
  st[1] = n % H;
  st[2] = n >= 1 ? (n - 1) % H : -1;
}

int jefi_launch_push_sources(jefi_ctx* c, const float* rho, const float* jx, const float* jy, const float* jz) {
  const jefi_dims& d = c->dims;
  unsigned blocks = (unsigned)((d.ncell_pad + 255) / 256);
  if (c->capturing) {  // recorded once, replayed every step: the step lives on the device, the host counter is advanced per replay
    k_advance_step<<<1, 1, 0, c->stream>>>(c->step_dev, d.H);
    k_push_sources<<<blocks, 256, 0, c->stream>>>(d, (float)(1.0 / c->c), 0, 0, -1, c->step_dev, rho, jx, jy, jz, c->ring, c->tile_first, c->tile_last);
    JEFI_CUDA_TRY(c, cudaGetLastError());
    c->launches += 2;
    return JEFI_OK;
  }
  long n = c->step + 1;
  int slot = (int)(n % d.H);
  int prev = n >= 1 ? (int)((n - 1) % d.H) : -1;
  k_push_sources<<<blocks, 256, 0, c->stream>>>(d, (float)(1.0 / c->c), (int)n, slot, prev, nullptr, rho, jx, jy, jz, c->ring, c->tile_first, c->tile_last);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  c->launches++;
  c->step = n;
  return JEFI_OK;
}

extern "C" int jefi_push_sources(jefi_ctx* c, const float* rho, const float* jx, const float* jy, const float* jz) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (!rho || !jx || !jy || !jz) { c->err = "jefi_push_sources: NULL array"; return JEFI_EINVAL; }
  return jefi_launch_push_sources(c, rho, jx, jy, jz);
}

int jefi_field_step_impl(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz,
                         float* eb_packed) {
  if (!ex || !ey || !ez || !bx || !by || !bz) { c->err = "jefi_field_step: NULL array"; return JEFI_EINVAL; }
  if (k0 < 0 || k1 > c->dims.nz || k0 > k1 || (k0 % c->dims.obz) != 0) {
    c->err = "jefi_field_step_slab: need 0 <= k0 <= k1 <= nz with k0 a multiple of the observation tile's z edge (jefi_get_tile_info)";
    return JEFI_EINVAL;
  }
  if (c->capturing) {  // inside jefi_pic_step's graph: the push of this step precedes it; no event records in a graph
    return c->field_impl == JEFI_FIELD_TILED ? jefi_launch_field_tiled(c, k0, k1, ex, ey, ez, bx, by, bz, eb_packed)
                                             : jefi_launch_field_reference(c, k0, k1, ex, ey, ez, bx, by, bz, eb_packed);
  }
  if (c->step < 0) { c->err = "jefi_field_step before any jefi_push_sources"; return JEFI_ESTATE; }
  if (k0 == k1) return JEFI_OK;
  const int evi = (int)(c->field_calls % JEFI_NEVENTS);
  JEFI_CUDA_TRY(c, cudaEventRecord(c->ev0[evi], c->stream));
  int rc = c->field_impl == JEFI_FIELD_TILED ? jefi_launch_field_tiled(c, k0, k1, ex, ey, ez, bx, by, bz, eb_packed)
                                             : jefi_launch_field_reference(c, k0, k1, ex, ey, ez, bx, by, bz, eb_packed);
  if (rc != JEFI_OK) return rc;
  JEFI_CUDA_TRY(c, cudaEventRecord(c->ev1[evi], c->stream));
  c->field_calls++;
  return JEFI_OK;
}

extern "C" int jefi_field_step_slab(jefi_ctx* c, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  return jefi_field_step_impl(c, k0, k1, ex, ey, ez, bx, by, bz, nullptr);
}

extern "C" int jefi_field_step(jefi_ctx* c, float* ex, float* ey, float* ez, float* bx, float* by, float* bz) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  return jefi_field_step_impl(c, 0, c->dims.nz, ex, ey, ez, bx, by, bz, nullptr);
}

extern "C" int jefi_field_step_packed(jefi_ctx* c, float* ex, float* ey, float* ez, float* bx, float* by, float* bz, float* eb_packed) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (!eb_packed || ((uintptr_t)eb_packed & 15u)) { c->err = "jefi_field_step_packed: eb_packed must be a 16-byte aligned device array of 8 N floats"; return JEFI_EINVAL; }
  return jefi_field_step_impl(c, 0, c->dims.nz, ex, ey, ez, bx, by, bz, eb_packed);
}

extern "C" float jefi_field_kernel_ms(jefi_ctx* c, int calls_back) {
  if (!c || calls_back < 0 || calls_back >= JEFI_NEVENTS || calls_back >= c->field_calls) return -1.f;
  jefi_device_guard guard(c);
  const int evi = (int)((c->field_calls - 1 - calls_back) % JEFI_NEVENTS);
  if (cudaEventSynchronize(c->ev1[evi]) != cudaSuccess) return -1.f;
  float ms = -1.f;
  if (cudaEventElapsedTime(&ms, c->ev0[evi], c->ev1[evi]) != cudaSuccess) return -1.f;
  return ms;
}

extern "C" float jefi_last_field_kernel_ms(jefi_ctx* c) { return jefi_field_kernel_ms(c, 0); }

// ------------------------------------------------------------------------------------------------------------
// One whole PIC step: deposit -> push_sources -> field_step_packed -> push_particles_packed, as ONE CUDA
// graph launch.  On 16^3 .. 32^3 grids the kernels of a step take tens of microseconds and the 6-8 launches + memset nodes
// cost as much again; the graph is captured on the first call (and again whenever an argument changes) and replayed after.
// ------------------------------------------------------------------------------------------------------------
extern "C" int jefi_pic_step(jefi_ctx* c, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz, const float* qw,
                             const float* q_over_m, unsigned char* alive, float* rho, float* jx, float* jy, float* jz, float* ex,
                             float* ey, float* ez, float* bx, float* by, float* bz, float* eb_packed) {
  if (!c) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  if (np < 0 || np > 0x7fffffffL || !rho || !jx || !jy || !jz || !ex || !ey || !ez || !bx || !by || !bz || !eb_packed || ((uintptr_t)eb_packed & 15u) ||
      (np > 0 && (!x || !y || !z || !ux || !uy || !uz || !qw || !q_over_m || !alive))) {
    c->err = "jefi_pic_step: NULL or misaligned array, or np out of range";
    return JEFI_EINVAL;
  }
  auto direct = [&]() -> int {
    int rc = jefi_deposit_impl(c, np, x, y, z, ux, uy, uz, qw, alive, rho, jx, jy, jz);
    if (rc == JEFI_OK) rc = jefi_launch_push_sources(c, rho, jx, jy, jz);
    if (rc == JEFI_OK) rc = jefi_field_step_impl(c, 0, c->dims.nz, ex, ey, ez, bx, by, bz, eb_packed);
    if (rc == JEFI_OK) rc = jefi_push_packed_impl(c, np, x, y, z, ux, uy, uz, q_over_m, alive, eb_packed);
    return rc;
  };
  if (c->stream == nullptr || c->stream == cudaStreamLegacy) return direct();  // the legacy default stream cannot be captured
  const void* ptrs[] = {x, y, z, ux, uy, uz, qw, q_over_m, alive, rho, jx, jy, jz, ex, ey, ez, bx, by, bz, eb_packed};
  unsigned long long key[24] = {0};
  key[0] = (unsigned long long)np;
  for (int i = 0; i < 20; i++) key[1 + i] = (unsigned long long)(uintptr_t)ptrs[i];
  // Context state the captured graph bakes in besides the caller's pointers: the sort scratch it scatters into (reallocated by
  // any call that arrives with a longer list) and the run-deposit kernel, which jefi_deposit_impl picks from how long ago the
  // caller's list was cell-sorted.  Either changing makes the key differ, so the step is captured afresh instead of replaying
  // a graph that writes freed memory or keeps the kernel of the first step for ever.
  key[21] = (unsigned long long)c->sort_gen;
  key[22] = (c->sorted_np == np && c->deposits_since_sort < 64) ? 1ull : 0ull;
  const bool replay = c->pic_exec && memcmp(key, c->pic_key, sizeof key) == 0;
  if (replay && c->deposits_since_sort < (1 << 30)) c->deposits_since_sort++;  // a replay is a deposit too (capturing counts its own)
  if (!c->pic_exec || memcmp(key, c->pic_key, sizeof key) != 0) {
    if (c->pic_exec) { cudaGraphExecDestroy(c->pic_exec); c->pic_exec = nullptr; }
    int rc = jefi_prepare_deposit_scratch(c, np);
    if (rc != JEFI_OK) return rc;
    key[21] = (unsigned long long)c->sort_gen;  // the scratch as it is now
    JEFI_CUDA_TRY(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
    const long l0 = c->launches;
    c->capturing = true;
    rc = direct();
    c->capturing = false;
    c->pic_launches = c->launches - l0;
    c->launches = l0;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
    if (rc != JEFI_OK || e != cudaSuccess) {
      if (graph) cudaGraphDestroy(graph);
      if (rc == JEFI_OK) { c->err = std::string("jefi_pic_step: graph capture: ") + cudaGetErrorString(e); rc = JEFI_ECUDA; }
      return rc;
    }
    e = cudaGraphInstantiate(&c->pic_exec, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { c->pic_exec = nullptr; c->err = std::string("jefi_pic_step: cudaGraphInstantiate: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
    memcpy(c->pic_key, key, sizeof key);
  }
  if (c->step_dev_value != c->step) {  // other calls advanced the step since the last replay: bring the device copy up to date
    const jefi_dims& d = c->dims;
    const int h[4] = {(int)c->step, c->step >= 0 ? (int)(c->step % d.H) : -1, c->step >= 1 ? (int)((c->step - 1) % d.H) : -1, 0};
    JEFI_CUDA_TRY(c, cudaMemcpyAsync(c->step_dev, h, sizeof h, cudaMemcpyHostToDevice, c->stream));
  }
  JEFI_CUDA_TRY(c, cudaGraphLaunch(c->pic_exec, c->stream));
  c->step += 1;
  c->step_dev_value = c->step;
  c->launches += c->pic_launches;
  return JEFI_OK;
}

extern "C" int jefi_field_step_host(jefi_ctx* c, const float* src_host, float* eb_host) {
  if (!c) return JEFI_EINVAL;
  if (!src_host || !eb_host) { c->err = "jefi_field_step_host: NULL array"; return JEFI_EINVAL; }
  jefi_device_guard guard(c);
  const long N = c->dims.N;
  // the two staging buffers are allocated independently, so that a failed second allocation is retried by the next call
  if (!c->src_stage && cudaMalloc(&c->src_stage, 4 * N * sizeof(float)) != cudaSuccess) {
    c->src_stage = nullptr;
    c->err = "jefi_field_step_host: staging allocation (sources) failed";
    return JEFI_ENOMEM;
  }
  if (!c->eb_stage && cudaMalloc(&c->eb_stage, 6 * N * sizeof(float)) != cudaSuccess) {
    c->eb_stage = nullptr;
    c->err = "jefi_field_step_host: staging allocation (fields) failed";
    return JEFI_ENOMEM;
  }
  JEFI_CUDA_TRY(c, cudaMemcpyAsync(c->src_stage, src_host, 4 * N * sizeof(float), cudaMemcpyHostToDevice, c->stream));
  float* s = c->src_stage;
  int rc = jefi_launch_push_sources(c, s, s + N, s + 2 * N, s + 3 * N);
  if (rc != JEFI_OK) return rc;
  float* o = c->eb_stage;
  rc = jefi_field_step_impl(c, 0, c->dims.nz, o, o + N, o + 2 * N, o + 3 * N, o + 4 * N, o + 5 * N, nullptr);
  if (rc != JEFI_OK) return rc;
  JEFI_CUDA_TRY(c, cudaMemcpyAsync(eb_host, o, 6 * N * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
  JEFI_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// debug exports
// ------------------------------------------------------------------------------------------------------------
extern "C" int jefi_debug_check_errors(jefi_ctx* c, long errors_host[4]) {
  if (!c || !errors_host) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  unsigned long long h[4] = {0, 0, 0, 0};
  JEFI_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  JEFI_CUDA_TRY(c, jefi_field_check_errors(h));      // [0] address outside the staged rows, [1] item sequence
  JEFI_CUDA_TRY(c, jefi_particle_check_errors(h + 2));  // [2] sort scatter index outside the list
  for (int i = 0; i < 4; i++) errors_host[i] = (long)h[i];
#ifdef JEFI_CHECKED
  return 1;  // a checked build: the counters are live
#else
  return JEFI_OK;
#endif
}

extern "C" int jefi_debug_delay_table(jefi_ctx* c, int* m_out_host) {
  if (!c || !m_out_host) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  const jefi_dims& d = c->dims;
  const int ex = c->tex, ey = c->tey;
  // read the DEVICE copy back so the export shows what the kernels actually index
  size_t tn = (size_t)ex * ey * c->tez;
  int* tmp = (int*)malloc(tn * sizeof(int));
  if (!tmp) return JEFI_ENOMEM;
  cudaError_t e = cudaMemcpyAsync(tmp, c->mtab_dev, tn * sizeof(int), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) { free(tmp); c->err = cudaGetErrorString(e); return JEFI_ECUDA; }
  for (int kc = 0; kc < d.nz; kc++)
    for (int jb = 0; jb < d.ny; jb++)
      for (int ia = 0; ia < d.nx; ia++)
        m_out_host[ia + (size_t)d.nx * (jb + (size_t)d.ny * kc)] = tmp[ia + (size_t)ex * (jb + (size_t)ey * kc)];
  free(tmp);
  return JEFI_OK;
}

__global__ void __launch_bounds__(256) k_history_slot(jefi_dims d, float cc, int slot, const float4* __restrict__ ring,
                                                      float* __restrict__ out) {
  long cidx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (cidx >= d.N) return;
  int i = (int)(cidx % d.nx), j = (int)((cidx / d.nx) % d.ny), k = (int)(cidx / ((long)d.nx * d.ny));
  long tile; int cell;
  jefi_tile_cell(d, i, j, k, tile, cell);
  float4 s = ring[jefi_ring_quad(d, tile, slot, cell)];  // (Jx/c, Jz/c, rho, Jy/c)
  out[cidx] = s.z;
  out[d.N + cidx] = s.x * cc;
  out[2 * d.N + cidx] = s.w * cc;
  out[3 * d.N + cidx] = s.y * cc;
}

extern "C" int jefi_debug_history_slot(jefi_ctx* c, int steps_back, float* out4N) {
  if (!c || !out4N) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  const jefi_dims& d = c->dims;
  long t = c->step - steps_back;
  if (steps_back < 0 || steps_back > d.H - 1 || t < 0) { c->err = "jefi_debug_history_slot: step not in the ring"; return JEFI_EINVAL; }
  k_history_slot<<<(unsigned)((d.N + 255) / 256), 256, 0, c->stream>>>(d, (float)c->c, (int)(t % d.H), c->ring, out4N);
  JEFI_CUDA_TRY(c, cudaGetLastError());
  JEFI_CUDA_TRY(c, cudaStreamSynchronize(c->stream));
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Row a2: proof that the tiled kernel's fp32 delay arithmetic equals the fp64 table on every offset it can form.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_verify_delay(int ex, int ey, int ez, jefi_geom g, const int* __restrict__ mtab,
                                                      unsigned long long* __restrict__ mismatches) {
  long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
  long tn = (long)ex * ey * ez;
  if (idx >= tn || idx == 0) return;  // offset (0,0,0) is the self cell: never evaluated
  int ia = (int)(idx % ex), jb = (int)((idx / ex) % ey), kc = (int)(idx / ((long)ex * ey));
  float q = jefi_q_fp32(g.kx, g.ky, g.kz, (float)ia, (float)jb, (float)kc);
  if (jefi_delay_fp32(q) != mtab[idx]) atomicAdd(mismatches, 1ull);
}

int jefi_verify_delay_fp32(jefi_ctx* c, long* mismatches, long* offsets) {
  const int ex = c->tex, ey = c->tey, ez = c->tez;
  unsigned long long* cnt = nullptr;
  JEFI_CUDA_TRY(c, cudaMalloc(&cnt, sizeof(unsigned long long)));
  cudaMemsetAsync(cnt, 0, sizeof(unsigned long long), c->stream);
  long tn = (long)ex * ey * ez;
  k_verify_delay<<<(unsigned)((tn + 255) / 256), 256, 0, c->stream>>>(ex, ey, ez, c->geom, c->mtab_dev, cnt);
  cudaError_t e = cudaGetLastError();
  unsigned long long h = 0;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, cnt, sizeof h, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(cnt);
  if (e != cudaSuccess) { c->err = std::string("delay verification: ") + cudaGetErrorString(e); return JEFI_ECUDA; }
  c->launches++;
  *mismatches = (long)h;
  *offsets = tn - 1;
  return JEFI_OK;
}
