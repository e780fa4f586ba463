// k_step: the fused hot path of one fine time step for every level that sits at the step start
// (Alg. 1): volume (Alg. 2) + surface (Alg. 3) right-hand side, point terms (eq (15)),
// AB update (18), exposed traces and half-step traces (19) (Alg. 4), boundary-trace capture / replay
// and - with two wavefields - the imaging contribution (24).
//
// Why fused (differs from the paper's three kernels): the update of an element needs only
// its own right-hand side, so it is applied while that right-hand side is still in registers; q is
// rewritten in place (nobody else reads it) and the traces are double-buffered per level, the reader
// picking, per neighbour level, the buffer that holds the traces at the step-start time (or the half-step
// buffer for a coarser neighbour in mid-step).  Algorithmic traffic per element: q in 4Np, neighbour
// traces in 8Nfp, two older right-hand sides in 8Np, new right-hand side out 4Np, q out 4Np, traces out
// 8Nfp, factors ~31  =  20Np + 16Nfp + 31 scalars (SURVEY.md 8(d) "fused floor").
//
// Mapping: lane = element, a GROUP of NT warps owns one 32-element block at a time; warp w of the group
// produces the TO output nodes n0 = w*TO .. with 5*TO register accumulators; a CTA holds G independent
// groups that share the operator matrices in shared memory.  The block's nodal values are fetched by one
// cp.async.bulk (TMA, 1-D) per block into shared memory columns [value][lane] (conflict-free); operator
// entries are warp-uniform and fetched VW at a time (LDS.128 / LDS.64 broadcast).
#pragma once
#include "kernels.cuh"

namespace dgrtm {

template <typename real, int N> struct StepCfg;
//                                            TO = outputs per warp, NT = warps per block, G = groups per CTA,
//                                            PK = older right-hand sides parked in tensor memory (N = 5 fp32: the
//                                            96-register budget of its 21 warps has no room for the chunk in flight)
template <> struct StepCfg<float, 1> { static constexpr int TO = 4, NT = 1, G = 16, PK = 1; };
template <> struct StepCfg<float, 2> { static constexpr int TO = 12, NT = 1, G = 12, PK = 1; };
template <> struct StepCfg<float, 3> { static constexpr int TO = 10, NT = 2, G = 10, PK = 1; };
template <> struct StepCfg<float, 4> { static constexpr int TO = 12, NT = 3, G = 5, PK = 1; };
template <> struct StepCfg<float, 5> { static constexpr int TO = 8, NT = 7, G = 3, PK = 0; };
template <> struct StepCfg<float, 6> { static constexpr int TO = 12, NT = 7, G = 2, PK = 1; };
template <> struct StepCfg<double, 1> { static constexpr int TO = 4, NT = 1, G = 12, PK = 1; };
template <> struct StepCfg<double, 2> { static constexpr int TO = 10, NT = 1, G = 8, PK = 1; };
template <> struct StepCfg<double, 3> { static constexpr int TO = 10, NT = 2, G = 5, PK = 1; };
template <> struct StepCfg<double, 4> { static constexpr int TO = 6, NT = 6, G = 2, PK = 1; };
template <> struct StepCfg<double, 5> { static constexpr int TO = 8, NT = 7, G = 1, PK = 1; };
template <> struct StepCfg<double, 6> { static constexpr int TO = 12, NT = 7, G = 1, PK = 1; };

template <typename real, int N, bool DUAL> struct StepSmem {
  using O = Order<N>;
  using C = StepCfg<real, N>;
  static constexpr int NPAD = C::TO * C::NT;                       // padded output count (>= Np)
  static constexpr size_t ops_reals = (size_t)3 * O::Np * NPAD + (size_t)O::NF * NPAD;
  static constexpr size_t tab_ints = O::NF + 3 * O::Np + UpdSmem<N>::kMaxPerm * O::Nfp;
  // imaging scalars of the source field between the two field passes: shared memory if one group with
  // them fits, else a global scratch array (N = 6 in fp64 only)
  static constexpr bool img_in_smem = DUAL && (size_t)(8 * O::Np + 2 * O::NF + DG_NGEO + 4) * 32 * sizeof(real) + 4096 <= 227 * 1024;
  // per group: q [4Np][32], penalties / trace staging [2NF][32], factors [DG_NGEO][32], (imaging scalars),
  // neighbour codes [4][32] int
  static constexpr size_t group_reals = (size_t)(4 * O::Np + 2 * O::NF + DG_NGEO + (img_in_smem ? 4 * O::Np : 0)) * 32 +
                                        4 * 32 * sizeof(int) / sizeof(real);
  static constexpr size_t group_bytes = group_reals * sizeof(real);
  // operators in shared memory if they fit next to one group; otherwise read from global (L1-resident)
  static constexpr bool ops_in_smem =
      ops_reals * sizeof(real) + tab_ints * sizeof(int) + 128 + 128 + 1024 + group_bytes <= 227 * 1024;
  static constexpr size_t raw = (ops_in_smem ? ops_reals * sizeof(real) : 0) + tab_ints * sizeof(int);
  static constexpr size_t ops_bytes = (raw + 127) / 128 * 128;
  static constexpr int Gfit = (int)((227 * 1024 - 1024 - 256 - ops_bytes) / group_bytes);
  static constexpr int G = Gfit < 1 ? 1 : (Gfit < C::G ? Gfit : C::G);
  static constexpr size_t bytes = ops_bytes + 256 + (size_t)G * group_bytes;   // + mbarriers, tensor-memory slot
  static_assert(NPAD >= O::Np, "tiles must cover Np");
};

// ---- small PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n .reg .pred p;\n WAIT_%=:\n"
      " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      " @p bra DONE_%=;\n bra WAIT_%=;\n DONE_%=:\n}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_prefetch_l2(const void* src, unsigned bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// barrier among the NT warps of one group (ids 1..15; id 0 is __syncthreads)
template <int NT> __device__ __forceinline__ void group_sync(int g) {
  if (NT == 1) __syncwarp();
  else asm volatile("bar.sync %0, %1;" ::"r"(g + 1), "r"(NT * 32) : "memory");
}

// VW consecutive warp-uniform reals from shared memory in one instruction
template <typename real, int VW> struct VecT;
template <> struct VecT<float, 4> { using T = float4; };
template <> struct VecT<float, 2> { using T = float2; };
template <> struct VecT<float, 1> { using T = float; };
template <> struct VecT<double, 2> { using T = double2; };
template <> struct VecT<double, 1> { using T = double; };
template <typename real, int TO> struct OpVec {
  static constexpr int MAXW = 16 / (int)sizeof(real);
  static constexpr int VW = (TO % MAXW == 0) ? MAXW : ((TO % 2 == 0 && MAXW >= 2) ? 2 : 1);
};
template <typename real, int TO>
__device__ __forceinline__ void load_row(const real* __restrict__ p, real (&out)[TO]) {
  constexpr int VW = OpVec<real, TO>::VW;
  using V = typename VecT<real, VW>::T;
#pragma unroll
  for (int v = 0; v < TO / VW; ++v) {
    const V x = reinterpret_cast<const V*>(p)[v];
    const real* xs = reinterpret_cast<const real*>(&x);
#pragma unroll
    for (int e = 0; e < VW; ++e) out[v * VW + e] = xs[e];
  }
}

// one trace record (REC consecutive reals at a REC-aligned offset) with the widest aligned vector loads
template <typename real, int REC>
__device__ __forceinline__ void load_record(const real* __restrict__ p, real (&out)[REC]) {
  constexpr int B = REC * (int)sizeof(real);
  constexpr int VW = (B % 16 == 0) ? 16 / (int)sizeof(real) : ((B % 8 == 0) ? 8 / (int)sizeof(real) : 1);
  using V = typename VecT<real, VW>::T;
#pragma unroll
  for (int v = 0; v < REC / VW; ++v) {
    const V x = __ldg(reinterpret_cast<const V*>(p) + v);
    const real* xs = reinterpret_cast<const real*>(&x);
#pragma unroll
    for (int e = 0; e < VW; ++e) out[v * VW + e] = xs[e];
  }
}

// tensor memory as a parking lot for per-lane values (32x32b shape: thread i of the warp <-> lane base + i, NW
// consecutive 32-bit columns per thread)
template <int NW> __device__ __forceinline__ void tmem_st(unsigned taddr, const unsigned (&r)[NW]) {
  static_assert(NW == 4 || NW == 8 || NW == 16, "4, 8 or 16 columns");
  if constexpr (NW == 4)
    asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
  else if constexpr (NW == 8)
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
                 "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
  else
    asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
                 "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
                 "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]) : "memory");
}
template <int NW> __device__ __forceinline__ void tmem_ld(unsigned taddr, unsigned (&r)[NW]) {
  static_assert(NW == 4 || NW == 8 || NW == 16, "4, 8 or 16 columns");
  if constexpr (NW == 4)
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
  else if constexpr (NW == 8)
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]),
                 "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr) : "memory");
  else
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                   "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
// eight reals <-> 8 (float) or 16 (double) 32-bit words
template <typename real> struct Words8;
template <> struct Words8<float> {
  static constexpr int NW = 8;
  static __device__ __forceinline__ void pack(const float (&v)[8], unsigned (&r)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) r[i] = __float_as_uint(v[i]);
  }
  static __device__ __forceinline__ void unpack(const unsigned (&r)[8], float (&v)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
  }
};
template <> struct Words8<double> {
  static constexpr int NW = 16;
  static __device__ __forceinline__ void pack(const double (&v)[8], unsigned (&r)[16]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) { r[2 * i] = (unsigned)__double2loint(v[i]); r[2 * i + 1] = (unsigned)__double2hiint(v[i]); }
  }
  static __device__ __forceinline__ void unpack(const unsigned (&r)[16], double (&v)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = __hiloint2double((int)r[2 * i + 1], (int)r[2 * i]);
  }
};

template <typename real> struct Words4;
template <> struct Words4<float> {
  static constexpr int NW = 4;
  static __device__ __forceinline__ void pack(const float (&v)[4], unsigned (&r)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) r[i] = __float_as_uint(v[i]);
  }
  static __device__ __forceinline__ void unpack(const unsigned (&r)[4], float (&v)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = __uint_as_float(r[i]);
  }
};
template <> struct Words4<double> {
  static constexpr int NW = 8;
  static __device__ __forceinline__ void pack(const double (&v)[4], unsigned (&r)[8]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) { r[2 * i] = (unsigned)__double2loint(v[i]); r[2 * i + 1] = (unsigned)__double2hiint(v[i]); }
  }
  static __device__ __forceinline__ void unpack(const unsigned (&r)[8], double (&v)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) v[i] = __hiloint2double((int)r[2 * i + 1], (int)r[2 * i]);
  }
};

// ---- the kernel ---------------------------------------------------------------------------------------
template <typename real, int N, bool DUAL>
__global__ void __launch_bounds__(StepSmem<real, N, DUAL>::G * StepCfg<real, N>::NT * 32, 1)
k_step(const __grid_constant__ StepArgs a) {
  using O = Order<N>;
  using Cfg = StepCfg<real, N>;
  using SM = StepSmem<real, N, DUAL>;
  constexpr int Np = O::Np, Nfp = O::Nfp, NF = O::NF, REC = O::REC;
  constexpr int TO = Cfg::TO, NT = Cfg::NT, G = SM::G, NPAD = SM::NPAD;
  constexpr bool INPLACE = NT > 1;
  constexpr int NTHREADS = G * NT * 32;
  constexpr unsigned QBYTES = 4 * Np * 32 * sizeof(real);

  extern __shared__ __align__(128) unsigned char smem_raw[];
  constexpr bool OPS_SMEM = SM::ops_in_smem;
  real* sDs = reinterpret_cast<real*>(smem_raw);                  // [Np(m)][3][NPAD(n)]
  real* sLs = sDs + (OPS_SMEM ? 3 * Np * NPAD : 0);               // [NF(j)][NPAD(n)]
  int* sF = reinterpret_cast<int*>(sLs + (OPS_SMEM ? NF * NPAD : 0));   // [NF]
  int* sInv = sF + NF;                                            // [Np][3]
  int* sP = sInv + 3 * Np;                                        // [kMaxPerm][Nfp]
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_raw + SM::ops_bytes);
  real* gbase = reinterpret_cast<real*>(smem_raw + SM::ops_bytes + 256);

  const int tid = threadIdx.x, lane = tid & 31, wg = tid >> 5, g = wg / NT, w = wg - g * NT;
  real* qs = gbase + (size_t)g * SM::group_reals;                 // [4Np][32]
  real* pen = qs + 4 * Np * 32;                                   // [2NF][32], later trace staging [4REC][32]
  real* sgeo = pen + 2 * NF * 32;                                 // [DG_NGEO][32]
  real* simg = sgeo + DG_NGEO * 32;                               // DUAL: [4][Np][32] (or global scratch)
  int* snbr = reinterpret_cast<int*>(simg + (SM::img_in_smem ? 4 * Np * 32 : 0));   // [4][32]
  // the two older right-hand sides of the warp's own output nodes are loaded from L2 in chunks during the lift loop
  // and PARKED in tensor memory (lane = element, columns = values; idle otherwise), where the update finds them
  // without a global-load latency: per warp 8 TO reals, warps of one lane quarter side by side
  constexpr bool PARK = Cfg::PK != 0;
  constexpr int PW = Words8<real>::NW;                            // 32-bit columns per node
  constexpr int PCOLS_NEED = (G * NT + 3) / 4 * TO * PW;
  constexpr int PCOLS = PCOLS_NEED <= 32 ? 32 : (PCOLS_NEED <= 64 ? 64 : (PCOLS_NEED <= 128 ? 128 : (PCOLS_NEED <= 256 ? 256 : 512)));
  static_assert(PCOLS_NEED <= 512, "tensor memory has 512 columns");
  constexpr int PCN = (TO + 3) / 4;                               // nodes per chunk: one chunk per face of the lift loop
  unsigned* tmem_slot = reinterpret_cast<unsigned*>(bars + G);
  constexpr unsigned GBYTES = DG_NGEO * 32 * sizeof(real), NBYTES = 4 * 32 * sizeof(int);

  {
    const real* gD = static_cast<const real*>(a.ops.D3T);
    const real* gL = static_cast<const real*>(a.ops.LIFTT);
    if (OPS_SMEM) {
      for (int i = tid; i < 3 * Np * NPAD; i += NTHREADS) sDs[i] = gD[i];
      for (int i = tid; i < NF * NPAD; i += NTHREADS) sLs[i] = gL[i];
    }
    for (int i = tid; i < NF; i += NTHREADS) sF[i] = a.ops.Fmask[i];
    if (w == 0 && lane == 0) mbar_init(&bars[g], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if constexpr (PARK) {
      if (wg == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(PCOLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    load_face_tables<N>(a.ops, sInv, sP, NTHREADS);               // ends with __syncthreads
    if constexpr (PARK) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }
  const unsigned tpark = PARK ? *tmem_slot + ((unsigned)((wg & 3) * 32) << 16) + (unsigned)((wg >> 2) * TO * PW) : 0u;

  const real* sD = OPS_SMEM ? sDs : static_cast<const real*>(a.ops.D3T);
  const real* sL = OPS_SMEM ? sLs : static_cast<const real*>(a.ops.LIFTT);
  // contiguous chunk of blocks per CTA (even per-SM load, neighbour reads stay L2-local)
  const int lo = a.blk0 + (int)(((long long)a.nblk * blockIdx.x) / gridDim.x);
  const int hi = a.blk0 + (int)(((long long)a.nblk * (blockIdx.x + 1)) / gridDim.x);
  const real dir = (real)a.dir;
  unsigned phase = 0;

  for (int b = lo + g; b < hi; b += G) {
    int l = 0;
    while (b >= a.lv[l].blk_end) ++l;
    const StepLevel& L = a.lv[l];
    const int slot_lo = (l > 0 ? a.lv[l - 1].blk_end : 0) * 32, slot_hi = L.blk_end * 32;
    const int lm = l > 0 ? l - 1 : 0, lp = l + 1 < a.nlevels ? l + 1 : l;
    const real* geo = sgeo + lane;
    const size_t base = (size_t)b * (4 * Np * 32) + lane;
    if (DUAL && !SM::img_in_smem) simg = static_cast<real*>(a.img_scratch) + (size_t)b * (4 * Np * 32);
    const real c0 = (real)L.c[0], c1 = (real)L.c[1], c2 = (real)L.c[2];
    const int n0 = w * TO;

#pragma unroll 1
    for (int fi = 0; fi < (DUAL ? 2 : 1); ++fi) {
      real* qg = static_cast<real*>(a.q[fi]);
      group_sync<NT>(g);                       // previous pass is done with qs / pen
      if (w == 0 && lane == 0) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&bars[g], QBYTES + (fi == 0 ? GBYTES + NBYTES : 0));
        bulk_g2s(qs, qg + (size_t)b * (4 * Np * 32), QBYTES, &bars[g]);
        if (fi == 0) {
          bulk_g2s(sgeo, static_cast<const real*>(a.geo) + (size_t)b * DG_NGEO * 32, GBYTES, &bars[g]);
          bulk_g2s(snbr, a.nbr + (size_t)b * 4 * 32, NBYTES, &bars[g]);
        }
        // the two older right-hand sides are read at the end of the block: pull them into L2 now
        bulk_prefetch_l2(static_cast<const real*>(L.r1[fi]) + (size_t)b * (4 * Np * 32), QBYTES);
        bulk_prefetch_l2(static_cast<const real*>(L.r2[fi]) + (size_t)b * (4 * Np * 32), QBYTES);
      }
      mbar_wait(&bars[g], phase);
      phase ^= 1;
      const real rc2 = geo[GEO_RC2 * 32], irho = geo[GEO_IRHO * 32];

      // ---- penalties at the face nodes (Alg. 3, first half; eqs (11)-(12), readings Q2, Q4, Q6)
      {
        const real* qfm = static_cast<const real*>(a.lv[lm].qf_read[fi]);
        const real* qf0 = static_cast<const real*>(L.qf_read[fi]);
        const real* qfp = static_cast<const real*>(a.lv[lp].qf_read[fi]);
        real* capt = fi == 0 ? static_cast<real*>(L.capture) : nullptr;
        const real* repl = fi == 0 ? static_cast<const real*>(L.replay) : nullptr;
#pragma unroll 1
        for (int f = w; f < 4; f += NT) {
          const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32],
                     nz = geo[(GEO_FACE + 5 * f + 2) * 32], gs = geo[(GEO_FACE + 5 * f + 3) * 32],
                     Zf = geo[(GEO_FACE + 5 * f + 4) * 32];
          const int code = snbr[f * 32 + lane];
          int bc = 0, bpos = 0;
          real rv[REC];                          // the neighbour's record, all loads issued before any use
          if (code >= 0) {
            const int s2 = code >> 2;
            const real* qfn = s2 >= slot_hi ? qfp : (s2 < slot_lo ? qfm : qf0);
            load_record<real, REC>(qfn + (size_t)code * REC, rv);
          } else {
#pragma unroll
            for (int i = 0; i < REC; ++i) rv[i] = 0;
            bc = (-1 - code) & 7;
            bpos = (-1 - code) >> 3;
          }
          const real half_gs = (real)0.5 * gs, iZ = (real)1 / Zf;
#pragma unroll
          for (int i = 0; i < Nfp; ++i) {
            const int j = f * Nfp + i, n = sF[j];
            const real pm = qs[n * 32 + lane];
            const real nvm = nx * qs[(Np + n) * 32 + lane] + ny * qs[(2 * Np + n) * 32 + lane] +
                             nz * qs[(3 * Np + n) * 32 + lane];
            real dp, dnv;
            if (code >= 0) {
              dp = rv[i] - pm;
              dnv = -rv[Nfp + i] - nvm;                                // reading Q6b
            } else if (bc == 1) { dp = -2 * pm; dnv = 0;               // free surface
            } else if (bc == 3) { dp = 0; dnv = -2 * nvm;              // rigid wall
            } else if (bc == 2) {                                      // absorbing, eq (3)
              if (capt) { capt[(size_t)bpos * REC + i] = pm; capt[(size_t)bpos * REC + Nfp + i] = nvm; }
              if (repl) { dp = repl[(size_t)bpos * REC + i] - pm; dnv = repl[(size_t)bpos * REC + Nfp + i] - nvm; }
              else { dp = -pm; dnv = -nvm; }
            } else if (bc == 4) {
              const long long hr = a.halo_rec ? a.halo_rec[bpos] : -1;
              if (hr >= 0) {       // halo face: the neighbouring sub-domain's exposed trace (see StepArgs)
                const real* r = static_cast<const real*>((fi == 0 ? a.halo_src : a.halo_src2)[a.halo_set[bpos]]) + (size_t)hr * REC;
                const int jn = a.halo_pos[(size_t)bpos * Nfp + i];
                dp = r[jn] - pm; dnv = -r[Nfp + jn] - nvm;
              } else {
                const real* ex = static_cast<const real*>(a.ext) + ((size_t)bpos * Nfp + i) * 2;
                dp = ex[0] - pm; dnv = ex[1] - nvm;
              }
            } else { dp = 0; dnv = 0; }
            pen[j * 32 + lane] = rc2 * half_gs * (dnv - dir * dp * iZ);
            pen[(NF + j) * 32 + lane] = irho * half_gs * (dp - dir * Zf * dnv);
          }
        }
      }
      const real g00 = geo[0 * 32], g01 = geo[1 * 32], g02 = geo[2 * 32], g10 = geo[3 * 32], g11 = geo[4 * 32],
                 g12 = geo[5 * 32], g20 = geo[6 * 32], g21 = geo[7 * 32], g22 = geo[8 * 32];
      if (INPLACE) {                            // v -> (U.Gr, U.Gs, U.Gt) once per block (Alg. 2)
        group_sync<NT>(g);                      // penalties read the velocities
        for (int m = w; m < Np; m += NT) {
          const real vx = qs[(Np + m) * 32 + lane], vy = qs[(2 * Np + m) * 32 + lane], vz = qs[(3 * Np + m) * 32 + lane];
          qs[(Np + m) * 32 + lane] = g00 * vx + g10 * vy + g20 * vz;
          qs[(2 * Np + m) * 32 + lane] = g01 * vx + g11 * vy + g21 * vz;
          qs[(3 * Np + m) * 32 + lane] = g02 * vx + g12 * vy + g22 * vz;
        }
      }
      group_sync<NT>(g);

      // ---- volume (eqs (13)-(14), Alg. 2): this warp's TO output nodes, all four fields
      real rp[TO], rx[TO], ry[TO], rz[TO];
      {
        real aD[TO], aR[TO], aS[TO], aT[TO];
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) { aD[nn] = 0; aR[nn] = 0; aS[nn] = 0; aT[nn] = 0; }
        const real* dbase = sD + n0;
#pragma unroll 2
        for (int m = 0; m < Np; ++m) {
          const real p = qs[m * 32 + lane];
          real ur, us, ut;
          if (INPLACE) {
            ur = qs[(Np + m) * 32 + lane]; us = qs[(2 * Np + m) * 32 + lane]; ut = qs[(3 * Np + m) * 32 + lane];
          } else {
            const real vx = qs[(Np + m) * 32 + lane], vy = qs[(2 * Np + m) * 32 + lane], vz = qs[(3 * Np + m) * 32 + lane];
            ur = g00 * vx + g10 * vy + g20 * vz;
            us = g01 * vx + g11 * vy + g21 * vz;
            ut = g02 * vx + g12 * vy + g22 * vz;
          }
          real dr[TO], ds[TO], dt[TO];
          load_row<real, TO>(dbase + (m * 3 + 0) * NPAD, dr);
          load_row<real, TO>(dbase + (m * 3 + 1) * NPAD, ds);
          load_row<real, TO>(dbase + (m * 3 + 2) * NPAD, dt);
#pragma unroll
          for (int nn = 0; nn < TO; ++nn) {
            aD[nn] += dr[nn] * ur + ds[nn] * us + dt[nn] * ut;
            aR[nn] += dr[nn] * p; aS[nn] += ds[nn] * p; aT[nn] += dt[nn] * p;
          }
        }
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) {
          rp[nn] = -rc2 * aD[nn];
          rx[nn] = -irho * (g00 * aR[nn] + g01 * aS[nn] + g02 * aT[nn]);
          ry[nn] = -irho * (g10 * aR[nn] + g11 * aS[nn] + g12 * aT[nn]);
          rz[nn] = -irho * (g20 * aR[nn] + g21 * aS[nn] + g22 * aT[nn]);
        }
      }
      // ---- surface (Alg. 3, second half): lift of the penalties; P^{v_i} = n_i * (scalar) per face.  Chunk f of the
      // older right-hand sides is in flight from L2 during the lift of face f and parked in tensor memory after it
      const real* h1g = static_cast<const real*>(L.r1[fi]) + base + (size_t)n0 * 32;
      const real* h2g = static_cast<const real*>(L.r2[fi]) + base + (size_t)n0 * 32;
      real hc[PARK ? PCN : 1][8];
      auto load_chunk = [&](int c) {
#pragma unroll
        for (int j = 0; j < PCN; ++j) {
          const int nn = c * PCN + j;
          if (nn < TO && n0 + nn < Np) {
#pragma unroll
            for (int fld = 0; fld < 4; ++fld) {
              hc[j][fld] = __ldg(h1g + (fld * Np + nn) * 32);
              hc[j][4 + fld] = __ldg(h2g + (fld * Np + nn) * 32);
            }
          }
        }
      };
      auto park_chunk = [&](int c) {
#pragma unroll
        for (int j = 0; j < PCN; ++j) {
          const int nn = c * PCN + j;
          if (nn < TO) {                                           // warp-uniform: tcgen05.st is .aligned
            unsigned wd[PW];
            Words8<real>::pack(hc[j], wd);
            tmem_st<PW>(tpark + (unsigned)(nn * PW), wd);
          }
        }
      };
      if constexpr (PARK) load_chunk(0);
#pragma unroll 1
      for (int f = 0; f < 4; ++f) {
        real av[TO];
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) av[nn] = 0;
#pragma unroll 2
        for (int i = 0; i < Nfp; ++i) {
          const int j = f * Nfp + i;
          const real Pp = pen[j * 32 + lane], Pv = pen[(NF + j) * 32 + lane];
          real lv[TO];
          load_row<real, TO>(sL + j * NPAD + n0, lv);
#pragma unroll
          for (int nn = 0; nn < TO; ++nn) { rp[nn] -= lv[nn] * Pp; av[nn] += lv[nn] * Pv; }
        }
        const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32],
                   nz = geo[(GEO_FACE + 5 * f + 2) * 32];
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) { rx[nn] -= nx * av[nn]; ry[nn] -= ny * av[nn]; rz[nn] -= nz * av[nn]; }
        if constexpr (PARK) {
          park_chunk(f);
          if (f + 1 < 4) load_chunk(f + 1);
        }
      }
      if constexpr (PARK) tmem_wait_st();

      // ---- point terms (eq (15)), update (18), imaging (24); new values stay in rp/rx/ry/rz
      {
        real* r0g = static_cast<real*>(L.r0[fi]);
        const real* r1g = static_cast<const real*>(L.r1[fi]);
        const real* r2g = static_cast<const real*>(L.r2[fi]);
        const int pi = a.pt_index[fi] ? a.pt_index[fi][(size_t)b * 32 + lane] : -1;
        const real* ptv = static_cast<const real*>(a.pt_val[fi]) + (size_t)(pi < 0 ? 0 : pi) * Np;
        const real pts = (real)a.pt_scale[fi];
        const bool imaging = DUAL && L.image_on;
        const real Z = (imaging && a.characteristic) ? geo[GEO_Z * 32] : (real)0;
        const real ex = (real)a.e[0], ey = (real)a.e[1], ez = (real)a.e[2];
        const real sgn = fi == 0 ? (real)-1 : (real)1;      // q_S^- = p - Z e.v ; q_R^+ = p + Z e.v  (eq (8))
        const real dts = (real)L.dts, adts = dts < 0 ? -dts : dts;
        real* img = static_cast<real*>(a.image);
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) {
          const int n = n0 + nn;
          if (n < Np) {
            real r0v[4] = {rp[nn], rx[nn], ry[nn], rz[nn]}, qo[4], h1[4], h2[4], v[4];
            if (pi >= 0) r0v[0] += pts * ptv[n];
            if constexpr (PARK) {
              unsigned wd[PW];
              real hv[8];
              tmem_ld<PW>(tpark + (unsigned)(nn * PW), wd);
              tmem_wait_ld();
              Words8<real>::unpack(wd, hv);
#pragma unroll
              for (int fld = 0; fld < 4; ++fld) { h1[fld] = hv[fld]; h2[fld] = hv[4 + fld]; }
            }
#pragma unroll
            for (int fld = 0; fld < 4; ++fld) {
              const size_t o = base + (size_t)(fld * Np + n) * 32;
              qo[fld] = (INPLACE && fld > 0) ? qg[o] : qs[(fld * Np + n) * 32 + lane];
              if constexpr (!PARK) { h1[fld] = r1g[o]; h2[fld] = r2g[o]; }
            }
#pragma unroll
            for (int fld = 0; fld < 4; ++fld) {
              const size_t o = base + (size_t)(fld * Np + n) * 32;
              v[fld] = qo[fld] + (c0 * r0v[fld] + c1 * h1[fld] + c2 * h2[fld]);
              r0g[o] = r0v[fld];
              qg[o] = v[fld];
            }
            if (imaging) {
              const real A0 = qo[0] + sgn * Z * (ex * qo[1] + ey * qo[2] + ez * qo[3]);
              const real A1 = r0v[0] + sgn * Z * (ex * r0v[1] + ey * r0v[2] + ez * r0v[3]);
              const real A2 = h1[0] + sgn * Z * (ex * h1[1] + ey * h1[2] + ez * h1[3]);
              const real A3 = h2[0] + sgn * Z * (ex * h2[1] + ey * h2[2] + ez * h2[3]);
              if (fi == 0) {
                simg[(0 * Np + n) * 32 + lane] = A0; simg[(1 * Np + n) * 32 + lane] = A1;
                simg[(2 * Np + n) * 32 + lane] = A2; simg[(3 * Np + n) * 32 + lane] = A3;
              } else {
                const real S0 = simg[(0 * Np + n) * 32 + lane];
                const real rA[3] = {simg[(1 * Np + n) * 32 + lane], simg[(2 * Np + n) * 32 + lane],
                                    simg[(3 * Np + n) * 32 + lane]};
                const real rB[3] = {A1, A2, A3};
                real acc = S0 * A0;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                  acc += dts * (real)L.abar[k] * (S0 * rB[k] + A0 * rA[k]);
#pragma unroll
                  for (int k2 = 0; k2 < 3; ++k2) acc += dts * dts * (real)L.C[3 * k + k2] * rA[k] * rB[k2];
                }
                if (a.trapezoid)                  // (21): mean of the integrand at the step ends; the new values are q + sum_s c_s r_s
                  acc = (real)0.5 * (S0 * A0 + (S0 + (c0 * rA[0] + c1 * rA[1] + c2 * rA[2])) * (A0 + (c0 * rB[0] + c1 * rB[1] + c2 * rB[2])));
                const size_t oi = ((size_t)b * Np + n) * 32 + lane;
                img[oi] += adts * acc;
              }
            }
            rp[nn] = v[0]; rx[nn] = v[1]; ry[nn] = v[2]; rz[nn] = v[3];
          }
        }
      }

      // ---- exposed traces of the new values (Alg. 4), then half-step traces (19)
      const int wp = a.wperm[(size_t)b * 32 + lane];
      const bool need_half = L.qf_half[fi] != nullptr && (a.blkflag[b] & 1);
#pragma unroll 1
      for (int pass = 0; pass < (need_half ? 2 : 1); ++pass) {
        if (pass == 1) {                        // value at the half step = new value + sum_s d_s r_s
          const real d0 = (real)L.d[0], d1 = (real)L.d[1], d2 = (real)L.d[2];
          const real* r0g = static_cast<const real*>(L.r0[fi]);
          const real* r1g = static_cast<const real*>(L.r1[fi]);
          const real* r2g = static_cast<const real*>(L.r2[fi]);
#pragma unroll
          for (int nn = 0; nn < TO; ++nn) {
            const int n = n0 + nn;
            if (n < Np) {
              const size_t o = base + (size_t)n * 32;
              rp[nn] += d0 * r0g[o] + d1 * r1g[o] + d2 * r2g[o];
              rx[nn] += d0 * r0g[o + (size_t)Np * 32] + d1 * r1g[o + (size_t)Np * 32] + d2 * r2g[o + (size_t)Np * 32];
              ry[nn] += d0 * r0g[o + (size_t)2 * Np * 32] + d1 * r1g[o + (size_t)2 * Np * 32] + d2 * r2g[o + (size_t)2 * Np * 32];
              rz[nn] += d0 * r0g[o + (size_t)3 * Np * 32] + d1 * r1g[o + (size_t)3 * Np * 32] + d2 * r2g[o + (size_t)3 * Np * 32];
            }
          }
        }
        group_sync<NT>(g);                      // pen (pass 0) / previous staging (pass 1) is consumed
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) {
          const int n = n0 + nn;
          if (n < Np) {
#pragma unroll
            for (int e = 0; e < 3; ++e) {
              const int j = sInv[n * 3 + e];
              if (j >= 0) {
                const int f = j / Nfp, i = j - f * Nfp;
                const int pos = sP[((wp >> (8 * f)) & 255) * Nfp + i];
                const real fnx = geo[(GEO_FACE + 5 * f + 0) * 32], fny = geo[(GEO_FACE + 5 * f + 1) * 32],
                           fnz = geo[(GEO_FACE + 5 * f + 2) * 32];
                // staging [row][lane] with the lane rotated by row / VS (conflict-free piece-wise reads below)
                constexpr int VSt = 16 / (int)sizeof(real);
                const int rwp = f * REC + pos, rwv = rwp + Nfp;
                pen[rwp * 32 + ((lane + rwp / VSt) & 31)] = rp[nn];
                pen[rwv * 32 + ((lane + rwv / VSt) & 31)] = fnx * rx[nn] + fny * ry[nn] + fnz * rz[nn];
              }
            }
          }
        }
        group_sync<NT>(g);
        // cooperative write-out: the block's 32 x 4 records are one contiguous run; consecutive lanes store
        // consecutive 16-byte pieces (piece P = element-lane P / NV, rows VS (P % NV) ..)
        {
          constexpr int VS = 16 / (int)sizeof(real), ROWS = 4 * REC, NV = ROWS / VS;
          using V = typename VecT<real, VS>::T;
          V* dst = reinterpret_cast<V*>(static_cast<real*>(pass == 0 ? L.qf_write[fi] : L.qf_half[fi]) + (size_t)b * 32 * ROWS);
          for (int it = w; it < NV; it += NT) {
            const int P = it * 32 + lane, el = P / NV, o4 = P - el * NV;
            V x;
            real* xs = reinterpret_cast<real*>(&x);
#pragma unroll
            for (int e = 0; e < VS; ++e) xs[e] = pen[(o4 * VS + e) * 32 + ((el + o4) & 31)];
            dst[P] = x;
          }
        }
      }
    }
  }
  if constexpr (PARK) {
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();                              // every warp is done with its columns: release the tensor memory
    if (wg == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_slot), "r"(PCOLS));
  }
}

}  // namespace dgrtm
