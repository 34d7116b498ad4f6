// libjefi: FP32 roofline probe (not on the hot path).  MEASURED_PEAKS.json carries HBM and BF16 figures but no FP32 one, and
// the field kernel is bound by the plain FP32 pipe ("bound": "alu"), so the library measures the pipe itself: every SM runs
// independent register-resident FMA chains, timed with CUDA events on the context's stream.
#include "jefi_ctx.h"

template <int MODE>
__global__ void __launch_bounds__(512) k_fp32_peak(int iters, float x, float* __restrict__ out) {
  float a[16];
  unsigned long long p[8];
#pragma unroll
  for (int i = 0; i < 16; i++) a[i] = x + (float)i + (float)threadIdx.x;
#pragma unroll
  for (int i = 0; i < 8; i++) p[i] = ((unsigned long long)__float_as_uint(a[2 * i]) << 32) | __float_as_uint(a[2 * i + 1]);
  const float b = x * 1.0001f, c = x * 0.5f;
  const unsigned long long pb = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
  const unsigned long long pc = ((unsigned long long)__float_as_uint(c) << 32) | __float_as_uint(c);
  // MODE 2, 3: every chain has its own multiplier and addend registers, so that each FMA reads three registers no
  // neighbouring instruction reads (nothing for the operand reuse cache to serve): the register-file side of the pipe
  float bb[16], cb[16];
  unsigned long long pbb[8], pcb[8];
#pragma unroll
  for (int i = 0; i < 16; i++) { bb[i] = 1.0f + 1e-6f * (float)(i + 1) * x; cb[i] = 1e-3f * (float)(i + 1) * x; }
#pragma unroll
  for (int i = 0; i < 8; i++) {
    pbb[i] = ((unsigned long long)__float_as_uint(bb[2 * i]) << 32) | __float_as_uint(bb[2 * i + 1]);
    pcb[i] = ((unsigned long long)__float_as_uint(cb[2 * i]) << 32) | __float_as_uint(cb[2 * i + 1]);
  }
  for (int it = 0; it < iters; it++) {
    if (MODE == 0) {  // 16 independent scalar FFMA chains per thread: a = a*b + c, b and c shared by all chains
#pragma unroll
      for (int i = 0; i < 16; i++) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(b), "f"(c));
    } else if (MODE == 1) {  // 8 independent packed chains (fma.rn.f32x2 = SASS FFMA2), the same 16 FMA per thread and iteration
#pragma unroll
      for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(pb), "l"(pc));
    } else if (MODE == 2) {  // scalar, three distinct register operands per FMA
#pragma unroll
      for (int i = 0; i < 16; i++) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(bb[i]), "f"(cb[i]));
    } else {                 // packed, three distinct register pairs per FFMA2
#pragma unroll
      for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(pbb[i]), "l"(pcb[i]));
    }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; i++) s += a[i];
#pragma unroll
  for (int i = 0; i < 8; i++) s += __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32));
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int jefi_debug_fp32_peak(jefi_ctx* c, int mode, double* tflops_out, int* sm_count_out) {
  if (!c || !tflops_out || mode < 0 || mode > 3) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  int nsm = 0;
  JEFI_CUDA_TRY(c, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->cfg.device));
  const int blocks = nsm * 4, threads = 512, iters = 40000;  // 2048 resident threads per SM
  float* out = nullptr;
  JEFI_CUDA_TRY(c, cudaMalloc(&out, (size_t)blocks * threads * sizeof(float)));
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  cudaError_t err = cudaSuccess;
  for (int rep = 0; rep < 4 && err == cudaSuccess; rep++) {  // first repetition warms up; best of the rest
    cudaEventRecord(e0, c->stream);
    switch (mode) {
      case 0: k_fp32_peak<0><<<blocks, threads, 0, c->stream>>>(iters, 1.0f, out); break;
      case 1: k_fp32_peak<1><<<blocks, threads, 0, c->stream>>>(iters, 1.0f, out); break;
      case 2: k_fp32_peak<2><<<blocks, threads, 0, c->stream>>>(iters, 1.0f, out); break;
      default: k_fp32_peak<3><<<blocks, threads, 0, c->stream>>>(iters, 1.0f, out); break;
    }
    cudaEventRecord(e1, c->stream);
    err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
    c->launches++;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (err != cudaSuccess) { c->err = std::string("fp32 peak probe: ") + cudaGetErrorString(err); return JEFI_ECUDA; }
  const double fma = 16.0 * iters * (double)blocks * threads;
  *tflops_out = 2.0 * fma / (best * 1e-3) / 1e12;
  if (sm_count_out) *sm_count_out = nsm;
  return JEFI_OK;
}

// ------------------------------------------------------------------------------------------------------------
// Shared-memory delivery probe: what one LDS.128 costs the SM's data pipe, by address pattern.  The field kernel reads two
// quads per pair from ring rows of JEFI_ROW_BYTES with a per-lane row (the lane's delay); this kernel issues the same
// instruction (ld.shared.v2.b64, volatile so that ptxas keeps every load) from 16 warps per SM with the rows given per lane.
// ------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) k_lds128_cost(const int* __restrict__ rows, int iters, float* __restrict__ out) {
  extern __shared__ __align__(128) unsigned char sm[];
  for (int i = threadIdx.x; i < 48 * JEFI_ROW_BYTES / 4; i += blockDim.x) reinterpret_cast<float*>(sm)[i] = (float)i;
  __syncthreads();
  const unsigned addr = (unsigned)__cvta_generic_to_shared(sm) + (unsigned)rows[threadIdx.x & 31] * JEFI_ROW_BYTES;
  unsigned long long a0 = 0, a1 = 0;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int c = 0; c < 32; c++) {
      unsigned long long x, y;
      asm volatile("ld.volatile.shared.v2.b64 {%0, %1}, [%2];" : "=l"(x), "=l"(y) : "r"(addr + c * 16));
      a0 ^= x; a1 ^= y;
    }
  }
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = (float)(a0 ^ a1);
}

extern "C" int jefi_debug_lds128_cycles(jefi_ctx* c, int pattern, double* cycles_out) {
  if (!c || !cycles_out || pattern < 0 || pattern > 4) return JEFI_EINVAL;
  jefi_device_guard guard(c);
  int nsm = 0, khz = 0;
  JEFI_CUDA_TRY(c, cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->cfg.device));
  JEFI_CUDA_TRY(c, cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, c->cfg.device));
  int rows[32];
  for (int l = 0; l < 32; l++) {
    switch (pattern) {
      case 0: rows[l] = 3; break;                                  // every lane the same quad
      case 1: rows[l] = l / 2; break;                              // lane pairs (2k, 2k+1) share a quad: 16 rows
      case 2: rows[l] = l; break;                                  // 32 rows
      case 3: rows[l] = l == 1 ? 20 : l / 2; break;                // as 1, but ONE pair (lanes 0, 1) differs
      default: rows[l] = ((l / 4) % 4) * 8 + ((l / 2) % 2) + 2 * (l / 16); break;  // as 1, rows 8 apart inside a half-warp
    }
  }
  int* drows = nullptr;
  float* out = nullptr;
  const int iters = 4000;
  const size_t smem = 48 * JEFI_ROW_BYTES;
  JEFI_CUDA_TRY(c, cudaFuncSetAttribute(k_lds128_cost, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  JEFI_CUDA_TRY(c, cudaMalloc(&drows, sizeof rows));
  cudaError_t err = cudaMalloc(&out, (size_t)nsm * 512 * sizeof(float));
  if (err == cudaSuccess) err = cudaMemcpyAsync(drows, rows, sizeof rows, cudaMemcpyHostToDevice, c->stream);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4 && err == cudaSuccess; rep++) {
    cudaEventRecord(e0, c->stream);
    k_lds128_cost<<<nsm, 512, smem, c->stream>>>(drows, iters, out);  // one CTA of 16 warps per SM
    cudaEventRecord(e1, c->stream);
    err = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (err == cudaSuccess) err = cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
    c->launches++;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(drows);
  if (out) cudaFree(out);
  if (err != cudaSuccess) { c->err = std::string("LDS.128 probe: ") + cudaGetErrorString(err); return JEFI_ECUDA; }
  *cycles_out = (double)best * 1e-3 * (double)khz * 1e3 / ((double)iters * 32.0 * 16.0);  // SM cycles (at the maximum clock) per warp-wide LDS.128
  return JEFI_OK;
}
