// One translation unit per order: compiled six times with -DDG_ORDER=1..6 (float and double each).
#include "tc_kernel.cuh"

#ifndef DG_ORDER
#error "compile with -DDG_ORDER=<1..6>"
#endif

namespace dgrtm {
namespace {

constexpr int N = DG_ORDER;
int g_sms = 148;            // B200; replaced by the current device's SM count in Launch::init()
cudaError_t g_launch_error = cudaSuccess;   // first failed cudaLaunchKernelEx (reported by Launch::take_error)

template <typename F> int blocks_per_sm(F kernel, int threads, size_t smem) {
  int n = 0;
  cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, kernel, threads, smem);
  return n < 1 ? 1 : n;
}

inline int persistent_grid(int nblk, int per_sm) {
  const int cap = g_sms * per_sm;
  return nblk < cap ? nblk : cap;
}

// launch with programmatic stream serialization: the kernel's prologue may overlap the previous kernel's
// tail; the kernel itself waits (griddepcontrol.wait) before touching data the previous launch wrote
template <typename K>
void launch_pdl(K kernel, int grid, int threads, size_t smem, cudaStream_t s, const StepArgs& a) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)grid); cfg.blockDim = dim3((unsigned)threads);
  cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  const cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, a);
  if (e != cudaSuccess && g_launch_error == cudaSuccess) g_launch_error = e;
}

template <typename real> struct Launch {
  static int occ_rhs, occ_upd, occ_rk, occ_img;

  static int take_error() { const int e = (int)g_launch_error; g_launch_error = cudaSuccess; return e; }
  static int init() {
    cudaError_t e;
    int dev = 0, sms = 0;
    e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return (int)e;
    if (sms > 0) g_sms = sms;
    e = cudaFuncSetAttribute(k_rhs<real, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RhsSmem<real, N>::bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_update<real, N, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)UpdSmem<N>::template bytes<real>(1));
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_update<real, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)UpdSmem<N>::template bytes<real>(1));
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_image_update<real, N>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)UpdSmem<N>::template bytes<real>(2));
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_step<real, N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)StepSmem<real, N, false>::bytes);
    if (e != cudaSuccess) return (int)e;
    e = cudaFuncSetAttribute(k_step<real, N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)StepSmem<real, N, true>::bytes);
    if (e != cudaSuccess) return (int)e;
    if constexpr (PipeCfg<real, N>::enabled && PipeSmem<real, N>::fits) {
      const int pb = (int)PipeSmem<real, N>::bytes;
      e = cudaFuncSetAttribute(k_pipe<real, N, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, pb);
      if (e != cudaSuccess) return (int)e;
      e = cudaFuncSetAttribute(k_pipe<real, N, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, pb);
      if (e != cudaSuccess) return (int)e;
      e = cudaFuncSetAttribute(k_pipe<real, N, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, pb);
      if (e != cudaSuccess) return (int)e;
      e = cudaFuncSetAttribute(k_pipe<real, N, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, pb);
      if (e != cudaSuccess) return (int)e;
    }
    if constexpr (sizeof(real) == 4 && TcCfg<N>::enabled) {
      e = cudaFuncSetAttribute(k_tc<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TcSmem<N>::bytes);
      if (e != cudaSuccess) return (int)e;
    }
    const int th = 32 * Tiling<N>::T;
    occ_rhs = blocks_per_sm(k_rhs<real, N>, th, RhsSmem<real, N>::bytes);
    occ_upd = blocks_per_sm(k_update<real, N, 0>, th, UpdSmem<N>::template bytes<real>(1));
    occ_rk = blocks_per_sm(k_update<real, N, 1>, th, UpdSmem<N>::template bytes<real>(1));
    occ_img = blocks_per_sm(k_image_update<real, N>, th, UpdSmem<N>::template bytes<real>(2));
    return 0;
  }
  static void rhs(const RhsArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    k_rhs<real, N><<<persistent_grid(a.nblk, occ_rhs), 32 * Tiling<N>::T, RhsSmem<real, N>::bytes, s>>>(a);
  }
  static void update(const UpdateArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    k_update<real, N, 0><<<persistent_grid(a.nblk, occ_upd), 32 * Tiling<N>::T, UpdSmem<N>::template bytes<real>(1), s>>>(a, RkArgs());
  }
  static void rk(const RkArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    k_update<real, N, 1><<<persistent_grid(a.nblk, occ_rk), 32 * Tiling<N>::T, UpdSmem<N>::template bytes<real>(1), s>>>(UpdateArgs(), a);
  }
  static void image_update(const ImageArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    k_image_update<real, N><<<persistent_grid(a.nblk, occ_img), 32 * Tiling<N>::T, UpdSmem<N>::template bytes<real>(2), s>>>(a);
  }
  static void step(const StepArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    using SM = StepSmem<real, N, false>;
    k_step<real, N, false><<<a.nblk < g_sms ? a.nblk : g_sms, SM::G * StepCfg<real, N>::NT * 32, SM::bytes, s>>>(a);
  }
  static void step2(const StepArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    using SM = StepSmem<real, N, true>;
    k_step<real, N, true><<<a.nblk < g_sms ? a.nblk : g_sms, SM::G * StepCfg<real, N>::NT * 32, SM::bytes, s>>>(a);
  }
  static void pipe(const StepArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    using C = PipeCfg<real, N>;
    const int grid = a.nblk < g_sms ? a.nblk : g_sms;
    if (a.sched_mode) launch_pdl(k_pipe<real, N, false, true>, grid, C::G * C::NT * 32, PipeSmem<real, N>::bytes, s, a);
    else launch_pdl(k_pipe<real, N, false, false>, grid, C::G * C::NT * 32, PipeSmem<real, N>::bytes, s, a);
  }
  static void pipe2(const StepArgs& a, cudaStream_t s) {
    if (a.nblk <= 0) return;
    using C = PipeCfg<real, N>;
    const int grid = a.nblk < g_sms ? a.nblk : g_sms;
    if (a.sched_mode) launch_pdl(k_pipe<real, N, true, true>, grid, C::G * C::NT * 32, PipeSmem<real, N>::bytes, s, a);
    else launch_pdl(k_pipe<real, N, true, false>, grid, C::G * C::NT * 32, PipeSmem<real, N>::bytes, s, a);
  }
  static void tc(const StepArgs& a, cudaStream_t s) {
    if constexpr (sizeof(real) == 4 && TcCfg<N>::enabled) {
      if (a.nblk <= 0) return;
      launch_pdl(k_tc<N>, a.nblk < g_sms ? a.nblk : g_sms, TcCfg<N>::G * 128, TcSmem<N>::bytes, s, a);
    }
  }
  static void source(const PointArgs& a, cudaStream_t s) { k_source<real, N><<<1, 96, 0, s>>>(a); }
  static void record(const PointArgs& a, cudaStream_t s) {
    if (a.nr <= 0) return;
    k_record<real, N><<<(a.nr + 127) / 128, 128, 0, s>>>(a);
  }
  static void inject(const PointArgs& a, cudaStream_t s) {
    if (a.ng <= 0) return;
    const long n = (long)a.ng * Order<N>::Np;
    k_inject<real, N><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(a);
  }
  static void halo(const HaloArgs& a, cudaStream_t s) {
    if (a.nh <= 0) return;
    const long n = (long)a.nh * Order<N>::Nfp;
    k_halo<real, N><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(a);
  }
  static void capture(const CaptureArgs& a, cudaStream_t s) {
    if (a.nfaces <= 0) return;
    const long n = (long)a.nfaces * Order<N>::Nfp;
    k_capture<real, N><<<(unsigned)((n + 127) / 128), 128, 0, s>>>(a);
  }
};
template <typename real> int Launch<real>::occ_rhs = 1;
template <typename real> int Launch<real>::occ_upd = 1;
template <typename real> int Launch<real>::occ_rk = 1;
template <typename real> int Launch<real>::occ_img = 1;

template <typename real> KernelTable make_table(int precision) {
  KernelTable t;
  t.N = N; t.precision = precision; t.Np = Order<N>::Np; t.Nfp = Order<N>::Nfp;
  t.rhs = Launch<real>::rhs; t.update = Launch<real>::update; t.rk = Launch<real>::rk;
  t.image_update = Launch<real>::image_update;
  t.source = Launch<real>::source; t.record = Launch<real>::record; t.inject = Launch<real>::inject;
  t.capture = Launch<real>::capture; t.halo = Launch<real>::halo; t.init = Launch<real>::init; t.take_error = Launch<real>::take_error;
  t.pipe = nullptr; t.pipe2 = nullptr; t.pipe_TO = t.pipe_NT = t.pipe_RL = t.pipe_LL = 0; t.pipe_blob_bytes = 0;
  t.tc = nullptr; t.tc_K1 = t.tc_K2 = t.tc_NN = 0; t.tc_blob_bytes = 0;
  if constexpr (sizeof(real) == 4 && TcCfg<N>::enabled && TcSmem<N>::fits) {
    t.tc = Launch<real>::tc; t.tc_K1 = TcSmem<N>::K1; t.tc_K2 = TcSmem<N>::K2; t.tc_NN = TcSmem<N>::NN;
    t.tc_blob_bytes = TcSmem<N>::ops_bytes;
  }
  static_assert(!PipeCfg<real, N>::enabled || PipeSmem<real, N>::fits, "an enabled pipelined configuration must fit the 227 KB of shared memory");
  if constexpr (PipeCfg<real, N>::enabled && PipeSmem<real, N>::fits) {
    t.pipe = Launch<real>::pipe; t.pipe2 = Launch<real>::pipe2;
    t.pipe_TO = PipeCfg<real, N>::TO; t.pipe_NT = PipeCfg<real, N>::NT;
    t.pipe_RL = PipeSmem<real, N>::RL; t.pipe_LL = PipeSmem<real, N>::LL;
    t.pipe_blob_bytes = PipeSmem<real, N>::ops_bytes;
  }
  t.step = Launch<real>::step; t.step2 = Launch<real>::step2; t.step_npad = StepSmem<real, N, false>::NPAD;
  return t;
}

}  // namespace

#define DG_CAT2(a, b) a##b
#define DG_CAT(a, b) DG_CAT2(a, b)
const KernelTable* DG_CAT(dg_kernel_table_order, DG_ORDER)(int precision) {
  static const KernelTable t32 = make_table<float>(32);
  static const KernelTable t64 = make_table<double>(64);
  return precision == 32 ? &t32 : &t64;
}

}  // namespace dgrtm
