// Register-only FMA microbenchmark behind dg_measure_fma (include/dgrtm.h): the plain-ALU ceilings that
// SURVEY.md 8(d) / BASELINE.md 2 ask for before any kernel is called ALU-bound.  Every thread keeps NACC
// independent accumulator chains in registers and issues fused multiply-adds on them: FFMA (fp32), FFMA2
// (packed fp32x2, sm_100) or DFMA (fp64).  Nothing touches memory inside the loop; one predicated store
// keeps the chains alive.
#include <cuda_runtime.h>

#include "../../include/dgrtm.h"

namespace {

constexpr int NACC = 16;

template <int KIND>
__global__ void __launch_bounds__(256) k_fma(float* sink, int iters, float a0, float b0) {
  if constexpr (KIND == 0) {
    float acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = (float)(threadIdx.x + i);
    const float a = a0, b = b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = fmaf(acc[i], a, b);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    if (s == 12345.678f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
  } else if constexpr (KIND == 1) {
    float2 acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = make_float2((float)(threadIdx.x + i), (float)i);
    const float2 a = make_float2(a0, a0), b = make_float2(b0, b0);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = __ffma2_rn(acc[i], a, b);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i].x + acc[i].y;
    if (s == 12345.678f) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;
  } else {
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = (double)(threadIdx.x + i);
    const double a = (double)a0, b = (double)b0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    if (s == 12345.678) sink[blockIdx.x * blockDim.x + threadIdx.x] = (float)s;
  }
}

}  // namespace

extern "C" int dg_measure_fma(int kind, void* dscratch, size_t scratch_bytes, void* cuda_stream, double* tflops) {
  if (!tflops || !dscratch || kind < 0 || kind > 2) return DG_ERR_ARG;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return DG_ERR_CUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return DG_ERR_CUDA;
  const int threads = 256, grid = sms * 8;
  if (scratch_bytes < (size_t)grid * threads * sizeof(float)) return DG_ERR_NOMEM;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int iters = kind == 2 ? 2000 : 8000;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return DG_ERR_CUDA;
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {      // first pass = warm-up; best of the rest
    cudaEventRecord(e0, s);
    if (kind == 0) k_fma<0><<<grid, threads, 0, s>>>((float*)dscratch, iters, 0.999f, 0.001f);
    else if (kind == 1) k_fma<1><<<grid, threads, 0, s>>>((float*)dscratch, iters, 0.999f, 0.001f);
    else k_fma<2><<<grid, threads, 0, s>>>((float*)dscratch, iters, 0.999f, 0.001f);
    cudaEventRecord(e1, s);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return DG_ERR_CUDA; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (cudaGetLastError() != cudaSuccess) return DG_ERR_CUDA;
  const double fma_per_thread = (double)iters * 8 * NACC * (kind == 1 ? 2 : 1);
  *tflops = 2.0 * fma_per_thread * (double)grid * threads / (best * 1e-3) * 1e-12;
  return DG_OK;
}
