// dg_step_lserk4_static (include/dgrtm.h): the LSERK4 time loop of dg_step with the 2N-storage residual of the stage
// kernel (k_update<real, N, 1>, `res` of RkArgs) in a file-scope device array instead of the bound workspace, for callers
// that cannot or may not allocate: this entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//
// The array costs kStaticScratchBytes on every GPU that loads the library, until the process exits.  It is SHARED by every
// call of every context on that GPU and keeps the last call's contents: each call clears the part it uses first, and two
// calls whose kernels overlap on the GPU (different streams) race on it - serialise them.
//
// In host code the array's name is a host-side stand-in, not a device address: the address comes from
// cudaGetSymbolAddress, once per device, with that device current, and is handed to the kernel as an argument.
#include <mutex>

#include "ctx.h"
#include "kernels.cuh"

namespace dgrtm {
namespace {

constexpr size_t kStaticScratchBytes = (size_t)8 << 20;          // 8 MiB: one [nslots][4 Np] field array of the state
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
void* g_scratch_ptr[kMaxDevices] = {};
int g_sms[kMaxDevices] = {};

template <typename real, int N> cudaError_t prepare_kernel() {
  return cudaFuncSetAttribute(k_update<real, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)UpdSmem<N>::template bytes<real>(1));
}

// once per device, with that device current: device address of the array, shared-memory limits of the stage kernels
void* scratch_of_current_device(int* sms) {
  int dev = 0;
  cuda_check(cudaGetDevice(&dev), "cudaGetDevice");
  if (dev < 0 || dev >= kMaxDevices) throw ApiError(DG_ERR_UNSUPPORTED, "device ordinal beyond the static-scratch table");
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_ptr[dev]) {
    void* p = nullptr;
    cuda_check(cudaGetSymbolAddress(&p, g_static_scratch), "cudaGetSymbolAddress(static scratch)");
    if (!p || ((uintptr_t)p & 255) != 0) throw ApiError(DG_ERR_CUDA, "static scratch has no 256-byte aligned device address");
    cuda_check(cudaDeviceGetAttribute(&g_sms[dev], cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute");
    cudaError_t e = cudaSuccess;
    auto acc = [&](cudaError_t x) { if (e == cudaSuccess) e = x; };
    acc(prepare_kernel<float, 1>()); acc(prepare_kernel<float, 2>()); acc(prepare_kernel<float, 3>());
    acc(prepare_kernel<float, 4>()); acc(prepare_kernel<float, 5>()); acc(prepare_kernel<float, 6>());
    acc(prepare_kernel<double, 1>()); acc(prepare_kernel<double, 2>()); acc(prepare_kernel<double, 3>());
    acc(prepare_kernel<double, 4>()); acc(prepare_kernel<double, 5>()); acc(prepare_kernel<double, 6>());
    cuda_check(e, "cudaFuncSetAttribute(LSERK4 stage kernel)");
    g_scratch_ptr[dev] = p;
  }
  *sms = g_sms[dev];
  return g_scratch_ptr[dev];
}

template <typename real, int N> void launch_stage(const RkArgs& a, int sms, cudaStream_t s) {
  const int cap = sms * 4, grid = a.nblk < cap ? a.nblk : cap;
  k_update<real, N, 1><<<grid, 32 * Tiling<N>::T, UpdSmem<N>::template bytes<real>(1), s>>>(UpdateArgs(), a);
}

template <typename real> void launch_stage_order(int N, const RkArgs& a, int sms, cudaStream_t s) {
  switch (N) {
    case 1: launch_stage<real, 1>(a, sms, s); break;
    case 2: launch_stage<real, 2>(a, sms, s); break;
    case 3: launch_stage<real, 3>(a, sms, s); break;
    case 4: launch_stage<real, 4>(a, sms, s); break;
    case 5: launch_stage<real, 5>(a, sms, s); break;
    case 6: launch_stage<real, 6>(a, sms, s); break;
    default: throw ApiError(DG_ERR_UNSUPPORTED, "order must be in 1..6");
  }
}

}  // namespace
}  // namespace dgrtm

using namespace dgrtm;

extern "C" int dg_step_lserk4_static(dg_ctx* ctx, int nsteps) {
  // five-stage LSERK4 of Carpenter & Kennedy (reading Q8), the coefficients of run_lserk4 (api_step.cpp)
  static const double A[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                              -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
  static const double B[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                              1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                              2277821191437.0 / 14882151754819.0};
  static const double C[5] = {0.0, 1432997174477.0 / 9575080441755.0, 2526269341429.0 / 6820363962896.0,
                              2006345519317.0 / 3224310063776.0, 2802321613138.0 / 2924317926251.0};
  DG_TRY(ctx)
  require_bound(ctx);
  if (nsteps < 0) throw ApiError(DG_ERR_ARG, "nsteps must be >= 0");
  if (ctx->integrator != DG_INTEGRATOR_LSERK4) throw ApiError(DG_ERR_STATE, "dg_set_integrator(DG_INTEGRATOR_LSERK4) first");
  const Model& md = ctx->model;
  if (md.nlevels != 1) throw ApiError(DG_ERR_UNSUPPORTED, "LSERK4 is single-rate only");
  if (ctx->has_prescribed && !ctx->has_ext) throw ApiError(DG_ERR_STATE, "prescribed-exterior faces need dg_set_exterior");
  if (ctx->prof) throw ApiError(DG_ERR_STATE, "dg_set_profiling creates an event pair per launch: switch it off for the allocation-free call");
  const size_t need = field_bytes(ctx);
  if (need > kStaticScratchBytes)
    throw ApiError(DG_ERR_NOMEM, "dg_step_lserk4_static: the state needs " + std::to_string(need) + " bytes of scratch, the static array holds " +
                                     std::to_string(kStaticScratchBytes) + " (8 MiB): use dg_step");
  int sms = 0;
  char* res = static_cast<char*>(scratch_of_current_device(&sms));
  // the array keeps whatever the last call (of any context) left: the residual must start finite (A_1 = 0 multiplies it)
  cuda_check(cudaMemsetAsync(res, 0, need, ctx->stream), "cudaMemsetAsync(static scratch)");
  Field& F = ctx->F;
  normalize_traces(ctx, F);
  const double dt = ctx->dt_local;
  for (int n = 0; n < nsteps; ++n) {
    const double t = ctx->t0 + (double)(ctx->fine + n) * dt;
    for (int st = 0; st < 5; ++st) {
      char* r = F.hist[0];
      launch_rhs(ctx, F, r, 0, 1, RHS_VOL | RHS_SURF, 1.0, nullptr, nullptr);
      if (ctx->has_src) {
        PointArgs p;
        std::memset(&p, 0, sizeof(p));
        p.rhs = r; p.src_slot = (int)md.slot_of[ctx->src_k]; p.src_w = ctx->d_src_w;
        p.amp_now = ricker(t + C[st] * dt, ctx->f0, ctx->tp, ctx->amp);
        DG_LAUNCH(ctx, KC_SOURCE, ctx->kt->source(p, ctx->stream));
      }
      RkArgs k;
      std::memset(&k, 0, sizeof(k));
      k.q = F.q; k.qf = F.qf; k.res = res; k.r = r; k.geo = ctx->geo; k.wperm = ctx->wperm;
      k.blk0 = 0; k.nblk = (int)md.nblocks; k.A = A[st]; k.B = B[st]; k.dt = dt; k.ops = ctx->ops;
      DG_LAUNCH(ctx, KC_RK, ctx->precision == 64 ? launch_stage_order<double>(ctx->N, k, sms, ctx->stream)
                                                 : launch_stage_order<float>(ctx->N, k, sms, ctx->stream));
    }
  }
  ctx->fine += nsteps;
  check_launches(ctx);
  DG_CATCH(ctx)
}

extern "C" int dg_static_scratch_bytes(size_t* n) {
  if (!n) return DG_ERR_ARG;
  *n = dgrtm::kStaticScratchBytes;
  return DG_OK;
}
