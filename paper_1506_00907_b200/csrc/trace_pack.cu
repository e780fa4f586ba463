// Packing of boundary-trace records for the host copy of a spilled history (rtm_set_spill_packing, include/dgrtm.h): every
// value in half the bytes - fp64 -> fp32, fp32 -> bf16 (same exponent range, 8 significant bits: relative rounding 2^-8).
// The paper names compression of the boundary data as future work; this is the simplest lossy variant,
// applied only on the way to and from host memory: the device ring and every kernel of the hot path keep full precision.
#include <cuda_bf16.h>
#include <cuda_runtime.h>

#include <cstddef>

namespace dgrtm {
namespace {

__global__ void k_pack_f64(const double* __restrict__ src, float* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = (float)src[i];
}
__global__ void k_unpack_f64(const float* __restrict__ src, double* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = (double)src[i];
}
__global__ void k_pack_f32(const float* __restrict__ src, __nv_bfloat16* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = __float2bfloat16_rn(src[i]);
}
__global__ void k_unpack_f32(const __nv_bfloat16* __restrict__ src, float* __restrict__ dst, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) dst[i] = __bfloat162float(src[i]);
}

inline unsigned grid_for(size_t n) {
  const size_t b = (n + 255) / 256;
  return (unsigned)(b < 1 ? 1 : (b > 1184 ? 1184 : b));       // 8 CTAs per SM at most: these run beside the step kernels
}

}  // namespace

// n values of the device precision (64 or 32) at src -> n values of half the size at dst, and back
void launch_trace_pack(const void* src, void* dst, size_t n, int precision, cudaStream_t s) {
  if (!n) return;
  if (precision == 64) k_pack_f64<<<grid_for(n), 256, 0, s>>>(static_cast<const double*>(src), static_cast<float*>(dst), n);
  else k_pack_f32<<<grid_for(n), 256, 0, s>>>(static_cast<const float*>(src), static_cast<__nv_bfloat16*>(dst), n);
}
void launch_trace_unpack(const void* src, void* dst, size_t n, int precision, cudaStream_t s) {
  if (!n) return;
  if (precision == 64) k_unpack_f64<<<grid_for(n), 256, 0, s>>>(static_cast<const float*>(src), static_cast<double*>(dst), n);
  else k_unpack_f32<<<grid_for(n), 256, 0, s>>>(static_cast<const __nv_bfloat16*>(src), static_cast<float*>(dst), n);
}

}  // namespace dgrtm
