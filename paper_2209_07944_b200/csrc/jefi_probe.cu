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
  for (int it = 0; it < iters; it++) {
    if (MODE == 0) {  // 16 independent scalar FFMA chains per thread: a = a*b + c
#pragma unroll
      for (int i = 0; i < 16; i++) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[i]) : "f"(b), "f"(c));
    } else {          // 8 independent packed chains (fma.rn.f32x2 = SASS FFMA2), the same 16 FMA per thread and iteration
#pragma unroll
      for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(pb), "l"(pc));
    }
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; i++) s += a[i];
#pragma unroll
  for (int i = 0; i < 8; i++) s += __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32));
  out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

extern "C" int jefi_debug_fp32_peak(jefi_ctx* c, int packed, double* tflops_out, int* sm_count_out) {
  if (!c || !tflops_out) return JEFI_EINVAL;
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
    if (packed) k_fp32_peak<1><<<blocks, threads, 0, c->stream>>>(iters, 1.0f, out);
    else k_fp32_peak<0><<<blocks, threads, 0, c->stream>>>(iters, 1.0f, out);
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
