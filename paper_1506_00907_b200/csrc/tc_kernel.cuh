// k_tc: the fused step of pipe_kernel.cuh with both contractions on the 5th-generation tensor cores
// (tcgen05.mma, kind::tf32, A operand and accumulator in tensor memory), fp32, one wavefield.
//
// The whole right-hand side of a 32-element block is ONE accumulator tile  C[(field f, element e)][node n]
// (M = 4 x 32 = 128 rows, N = Np padded to a multiple of 16), the sum of two GEMMs that share nothing but C:
//   volume   C += A1 . B1,  K = 3 Np:  B1[(j,m)][n] = D_j[n][m]  (D_r, D_s, D_t stacked, eqs (13)-(14)),
//            row (p, e)   : A1 = -rho c^2 (U.G)_j(m)            (Alg. 2: velocities combined with the factors)
//            row (v_i, e) : A1 = -(1/rho) g_ij p(m)
//   surface  C += A2 . B2,  K = 4 Nfp: B2[j][n] = LIFT[n][j]     (Alg. 3)
//            row (p, e)   : A2 = -P^p_j ;   row (v_i, e) : A2 = -n_i(face of j) P^v_j
// Warp w of a group owns field w = tensor-memory lanes 32w..32w+31, lane = element: it writes its rows of A with
// tcgen05.st, one elected thread issues the MMAs, and tcgen05.ld hands every thread the right-hand side of its
// (field, element) at all nodes, ready for the AB update.  B1, B2 are constants in shared memory (K-major, no
// swizzle, built on the host).  TF32 keeps 10 mantissa bits, the tolerance needs fp32: every product is
// split 3 x TF32:  a b ~ a_hi b_hi + a_lo b_hi + a_hi b_lo  (a_hi = rn_tf32(a), a_lo = rn_tf32(a - a_hi) on the
// device, b_hi, b_lo likewise on the host) - error ~2^-21 relative per product, fp32 accumulation in the tensor core.
// Everything else (operand ring, penalties, traces, update) is pipe_kernel.cuh's.
#pragma once
#include "pipe_kernel.cuh"

namespace dgrtm {

template <int N> struct TcCfg { static constexpr bool enabled = false; static constexpr int G = 1; };
template <> struct TcCfg<3> { static constexpr bool enabled = true; static constexpr int G = 3; };
// N = 4: the 3xTF32 split of A needs 2 x 112 + 48 = 272 of the 512 tensor-memory columns per group: one group per SM
// (N >= 5 does not fit at all: 2 x 184 + 64 columns at N = 5 leave no second group, N = 6 needs 608)
template <> struct TcCfg<4> { static constexpr bool enabled = true; static constexpr int G = 1; };

template <int N> struct TcSmem {
  using O = Order<N>;
  static constexpr int K1 = (3 * O::Np + 7) / 8 * 8;             // volume contraction length (padded)
  static constexpr int K2 = (O::NF + 7) / 8 * 8;                 // surface contraction length
  static constexpr int NN = (O::Np + 15) / 16 * 16;              // accumulator columns
  static constexpr int KA = K1 > K2 ? K1 : K2;                   // tensor-memory columns of one A half
  static constexpr int TCOLS = 2 * KA + NN;                      // per group: A_hi | A_lo | C
  // B tables: per k-step of 8 one 8 x NN core-matrix slab of NN * 32 bytes
  static constexpr size_t b1_floats = (size_t)K1 * NN, b2_floats = (size_t)K2 * NN;
  static constexpr size_t tab_ints = O::NF + UpdSmem<N>::kMaxPerm * O::Nfp;
  static constexpr size_t ops_bytes = ((2 * b1_floats + 2 * b2_floats) * 4 + tab_ints * 4 + 127) / 128 * 128;
  static constexpr int PV = (O::Nfp + 3) / 4;
  static constexpr size_t pen_floats = (size_t)(8 * PV * 4 > 2 * O::NF ? 8 * PV * 4 : 2 * O::NF) * 32;
  static constexpr size_t stage_floats = (size_t)(4 * O::Np + DG_NGEO) * 32;
  static constexpr size_t group_floats = 2 * stage_floats + (size_t)(4 * O::REC) * 32 + pen_floats;
  static constexpr size_t bytes = ops_bytes + 256 + (size_t)TcCfg<N>::G * group_floats * 4;
  static constexpr bool fits = bytes <= 227 * 1024 && TcCfg<N>::G * TCOLS <= 512;
};

__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// 8 consecutive tensor-memory columns of this thread's lane <- v (hi part) and v - hi (lo part, KA columns on)
template <int KA>
__device__ __forceinline__ void tc_store8_split(unsigned taddr, const float (&v)[8]) {
  unsigned h[8], l[8];
#pragma unroll
  for (int e = 0; e < 8; ++e) {
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(h[e]) : "f"(v[e]));                    // hi = a rounded to TF32
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(l[e]) : "f"(v[e] - __uint_as_float(h[e])));   // lo = (a - hi) rounded to TF32
  }
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(h[0]), "r"(h[1]),
               "r"(h[2]), "r"(h[3]), "r"(h[4]), "r"(h[5]), "r"(h[6]), "r"(h[7]) : "memory");
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr + KA), "r"(l[0]), "r"(l[1]),
               "r"(l[2]), "r"(l[3]), "r"(l[4]), "r"(l[5]), "r"(l[6]), "r"(l[7]) : "memory");
}
// one 128 x NN x 8 TF32 MMA: C[tmem] (+)= A[tmem] . B[smem descriptor]
__device__ __forceinline__ void tc_mma(unsigned tmem_c, unsigned tmem_a, unsigned long long desc_b, unsigned idesc, unsigned acc) {
  asm volatile(
      "{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n"
      " tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, {%5, %6, %7, %8}, p;\n}" ::"r"(tmem_c), "r"(tmem_a), "l"(desc_b),
      "r"(idesc), "r"(acc), "r"(0), "r"(0), "r"(0), "r"(0) : "memory");
}
// K-major, no swizzle: ((8,n),2):((1,SBO),LBO) in 16-byte units; one k-step of 8 = [chunk(2)][n/8][8 rows][16 B]
template <int NN> __device__ __forceinline__ unsigned long long tc_desc(unsigned smem_addr) {
  unsigned long long d = (unsigned long long)((smem_addr >> 4) & 0x3FFF);
  d |= (unsigned long long)(NN & 0x3FFF) << 16;       // LBO: NN rows x 16 B between the two K chunks
  d |= (unsigned long long)8 << 32;                   // SBO: 8 rows x 16 B between 8-row groups
  d |= 1ull << 46;                                    // descriptor version 1 (Blackwell)
  return d;
}

template <int N>
__global__ void __launch_bounds__(TcCfg<N>::G * 128, 1) k_tc(const __grid_constant__ StepArgs a) {
  using real = float;
  using O = Order<N>;
  using SM = TcSmem<N>;
  constexpr int Np = O::Np, Nfp = O::Nfp, NF = O::NF, REC = O::REC, G = TcCfg<N>::G, NT = 4;
  constexpr int K1 = SM::K1, K2 = SM::K2, NN = SM::NN, KA = SM::KA, PV = SM::PV, VW = 4;
  constexpr unsigned QBYTES = 4 * Np * 32 * sizeof(real), GBYTES = DG_NGEO * 32 * sizeof(real);
  constexpr int RB = REC * (int)sizeof(real), CPB = RB % 16 == 0 ? 16 : (RB % 8 == 0 ? 8 : 4), CPW = CPB / 4;
  constexpr unsigned IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((unsigned)(NN >> 3) << 17) | ((unsigned)(128 >> 4) << 24);

  extern __shared__ __align__(128) unsigned char smem_raw[];
  const real* sB1h = reinterpret_cast<const real*>(smem_raw);     // [K1/8][2][NN][4] canonical K-major
  const real* sB1l = sB1h + SM::b1_floats;
  const real* sB2h = sB1l + SM::b1_floats;
  const real* sB2l = sB2h + SM::b2_floats;
  const int* sF = reinterpret_cast<const int*>(sB2l + SM::b2_floats);   // [NF]
  const int* sP = sF + NF;                                        // [kMaxPerm][Nfp]
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_raw + SM::ops_bytes);   // [G][3], tables; then tmem base
  unsigned* tmem_slot = reinterpret_cast<unsigned*>(bars + 3 * G + 1);
  real* gbase = reinterpret_cast<real*>(smem_raw + SM::ops_bytes + 256);

  const int tid = threadIdx.x, lane = tid & 31, wg = tid >> 5, g = wg >> 2, w = wg & 3;
  real* grp = gbase + (size_t)g * SM::group_floats;
  real* TR = grp + 2 * SM::stage_floats;                          // [4][32][REC]
  real* pen = TR + 4 * REC * 32;                                  // penalties, later trace staging [4REC][32]
  unsigned long long* full = bars + 3 * g;                        // [0], [1]: q stages; [2]: MMA completion
  unsigned long long* tabbar = bars + 3 * G;

  if (tid == 0) {
    mbar_init(tabbar, 1);
    for (int x = 0; x < 3 * G; ++x) mbar_init(&bars[x], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    mbar_expect_tx(tabbar, (unsigned)SM::ops_bytes);
    bulk_g2s(smem_raw, a.ops2_LTQ, (unsigned)SM::ops_bytes, tabbar);
  }
  if (wg == 0) {                                                  // tensor memory: 512 columns for the CTA
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tbase = *tmem_slot + (unsigned)g * SM::TCOLS;    // this group's columns: A_hi | A_lo | C
  const unsigned trow = tbase + ((unsigned)(w * 32) << 16);       // this warp's lanes
  const unsigned tC = tbase + 2 * KA;

  const int lo = a.blk0 + (int)(((long long)a.nblk * blockIdx.x) / gridDim.x);
  const int hi = a.blk0 + (int)(((long long)a.nblk * (blockIdx.x + 1)) / gridDim.x);
  const int nmine = (hi - lo - g + G - 1) / G;
  const int nitems = nmine > 0 ? nmine : 0;
  const real dir = (real)a.dir;

  auto item_block = [&](int i) { return lo + g + i * G; };
  auto level_of = [&](int b) { int l = 0; while (b >= a.lv[l].blk_end) ++l; return l; };
  auto load_code = [&](int i) { return i < nitems ? a.nbr[((size_t)item_block(i) * 4 + w) * 32 + lane] : -1; };
  auto issue_q = [&](int i, int s) {
    if (w == 0 && lane == 0) {
      const int b = item_block(i);
      real* Q = grp + (size_t)s * SM::stage_floats;
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&full[s], QBYTES + GBYTES);
      bulk_g2s(Q, static_cast<const real*>(a.q[0]) + (size_t)b * (4 * Np * 32), QBYTES, &full[s]);
      bulk_g2s(Q + 4 * Np * 32, static_cast<const real*>(a.geo) + (size_t)b * DG_NGEO * 32, GBYTES, &full[s]);
      const StepLevel& L = a.lv[level_of(b)];                     // the older right-hand sides: into L2
      bulk_prefetch_l2(static_cast<const real*>(L.r1[0]) + (size_t)b * (4 * Np * 32), QBYTES);
      bulk_prefetch_l2(static_cast<const real*>(L.r2[0]) + (size_t)b * (4 * Np * 32), QBYTES);
    }
  };
  auto issue_tr = [&](int i, int code) {                          // face w of item i: the neighbour's record
    if (code >= 0) {
      const int b = item_block(i), l = level_of(b);
      const StepLevel& L = a.lv[l];
      const int slot_lo = (l > 0 ? a.lv[l - 1].blk_end : 0) * 32, slot_hi = L.blk_end * 32;
      const int lm = l > 0 ? l - 1 : 0, lp = l + 1 < a.nlevels ? l + 1 : l;
      const int s2 = code >> 2;
      const real* qf = static_cast<const real*>(s2 >= slot_hi ? a.lv[lp].qf_read[0] : (s2 < slot_lo ? a.lv[lm].qf_read[0] : L.qf_read[0]));
      const real* src = qf + (size_t)code * REC;
      real* dst = TR + ((size_t)w * (REC / CPW) * 32 + lane) * CPW;     // [face][piece][lane][CPW]: a warp's pieces are contiguous
#pragma unroll
      for (int v = 0; v < REC / CPW; ++v) cp_async<CPB>(dst + v * 32 * CPW, src + v * CPW);
    }
  };

  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
  int codeA = load_code(0);
  if (nitems > 0) { issue_q(0, 0); issue_tr(0, codeA); }
  int codeB = load_code(1);
  mbar_wait(tabbar, 0);
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  int fofs[Nfp];                                                  // own-trace offsets of face w in Q
#pragma unroll
  for (int i2 = 0; i2 < Nfp; ++i2) fofs[i2] = sF[w * Nfp + i2] * 32 + lane;
  const unsigned long long dB1h = tc_desc<NN>(smem_u32(sB1h)), dB1l = tc_desc<NN>(smem_u32(sB1l));
  const unsigned long long dB2h = tc_desc<NN>(smem_u32(sB2h)), dB2l = tc_desc<NN>(smem_u32(sB2l));

#pragma unroll 1
  for (int i = 0; i < nitems; ++i) {
    const int s = i & 1, b = item_block(i), l = level_of(b);
    const StepLevel& L = a.lv[l];
    real* Q = grp + (size_t)s * SM::stage_floats;                 // [4Np][32]
    const real* geo = Q + 4 * Np * 32 + lane;
    const size_t base = (size_t)b * (4 * Np * 32) + lane;
    const real c0 = (real)L.c[0], c1 = (real)L.c[1], c2 = (real)L.c[2];

    group_sync<NT>(g);                          // the group has left the previous item
    mbar_wait(&full[s], (unsigned)(i >> 1) & 1u);
    cp_async_wait_all();
    const real rc2 = geo[GEO_RC2 * 32], irho = geo[GEO_IRHO * 32];

    // ---- penalties of face w (Alg. 3, first half; same arithmetic as k_pipe)
    {
      const int f = w;
      real* capt = static_cast<real*>(L.capture);
      const real* repl = static_cast<const real*>(L.replay);
      const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32],
                 nz = geo[(GEO_FACE + 5 * f + 2) * 32], gs = geo[(GEO_FACE + 5 * f + 3) * 32], Zf = geo[(GEO_FACE + 5 * f + 4) * 32];
      const int code = codeA;
      const int bc = code >= 0 ? 0 : ((-1 - code) & 7), bpos = code >= 0 ? 0 : ((-1 - code) >> 3);
      real ep[Nfp], ev[Nfp];
      {
        real rv[REC];
        const real* src = TR + ((size_t)f * (REC / CPW) * 32 + lane) * CPW;
        using V = typename VecT<real, CPW>::T;
#pragma unroll
        for (int v = 0; v < REC / CPW; ++v) {
          const V x = reinterpret_cast<const V*>(src)[v * 32];
          const real* xs = reinterpret_cast<const real*>(&x);
#pragma unroll
          for (int e = 0; e < CPW; ++e) rv[v * CPW + e] = xs[e];
        }
#pragma unroll
        for (int i2 = 0; i2 < Nfp; ++i2) { ep[i2] = code >= 0 ? rv[i2] : (real)0; ev[i2] = code >= 0 ? -rv[Nfp + i2] : (real)0; }
      }
      const real ap = (code >= 0 || bc == 2 || bc == 4) ? (real)-1 : (bc == 1 ? (real)-2 : (real)0);
      const real av = (code >= 0 || bc == 2 || bc == 4) ? (real)-1 : (bc == 3 ? (real)-2 : (real)0);
      const bool rep_lane = bc == 2 && repl != nullptr, ext_lane = bc == 4;
      if (__any_sync(0xffffffffu, rep_lane || ext_lane)) {
        if (rep_lane) {
#pragma unroll
          for (int i2 = 0; i2 < Nfp; ++i2) { ep[i2] = repl[(size_t)bpos * REC + i2]; ev[i2] = repl[(size_t)bpos * REC + Nfp + i2]; }
        } else if (ext_lane) {
          const real* ex = static_cast<const real*>(a.ext) + (size_t)bpos * Nfp * 2;
#pragma unroll
          for (int i2 = 0; i2 < Nfp; ++i2) { ep[i2] = ex[2 * i2]; ev[i2] = ex[2 * i2 + 1]; }
        }
      }
      const bool cap_lane = bc == 2 && capt != nullptr;
      const bool cap_any = __any_sync(0xffffffffu, cap_lane);
      const real kp = rc2 * (real)0.5 * gs, kv = irho * (real)0.5 * gs, diZ = dir / Zf, dZ = dir * Zf;
      real Pp[PV * VW], Pv[PV * VW];
#pragma unroll
      for (int i2 = Nfp; i2 < PV * VW; ++i2) { Pp[i2] = 0; Pv[i2] = 0; }
#pragma unroll
      for (int i2 = 0; i2 < Nfp; ++i2) {
        const int o = fofs[i2];
        const real pm = Q[o];
        const real nvm = nx * Q[Np * 32 + o] + ny * Q[2 * Np * 32 + o] + nz * Q[3 * Np * 32 + o];
        if (cap_any && cap_lane) { capt[(size_t)bpos * REC + i2] = pm; capt[(size_t)bpos * REC + Nfp + i2] = nvm; }
        const real dp = ap * pm + ep[i2], dnv = av * nvm + ev[i2];
        Pp[i2] = kp * (dnv - diZ * dp);
        Pv[i2] = kv * (dp - dZ * dnv);
      }
      float4* dstp = reinterpret_cast<float4*>(pen) + ((size_t)(f * 2 + 0) * PV) * 32 + lane;
      float4* dstv = reinterpret_cast<float4*>(pen) + ((size_t)(f * 2 + 1) * PV) * 32 + lane;
#pragma unroll
      for (int v = 0; v < PV; ++v) {
        dstp[v * 32] = *reinterpret_cast<const float4*>(&Pp[v * VW]);
        dstv[v * 32] = *reinterpret_cast<const float4*>(&Pv[v * VW]);
      }
    }

    // ---- A1: this warp's rows (field w, element lane) of the volume GEMM -> tensor memory (hi | lo)
    if (w == 0) {                               // row (p, e): -rho c^2 (U.G)_j(m), j = r, s, t
      real vx[Np], vy[Np], vz[Np], cg[3][3];
#pragma unroll
      for (int m = 0; m < Np; ++m) { vx[m] = Q[(Np + m) * 32 + lane]; vy[m] = Q[(2 * Np + m) * 32 + lane]; vz[m] = Q[(3 * Np + m) * 32 + lane]; }
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int d = 0; d < 3; ++d) cg[j][d] = -rc2 * geo[(d * 3 + j) * 32];
#pragma unroll
      for (int c = 0; c < K1 / 8; ++c) {
        real v8[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          const int kap = c * 8 + e, j = kap / Np, m = kap - j * Np;
          v8[e] = kap < 3 * Np ? cg[j < 3 ? j : 0][0] * vx[m < Np ? m : 0] + cg[j < 3 ? j : 0][1] * vy[m < Np ? m : 0] + cg[j < 3 ? j : 0][2] * vz[m < Np ? m : 0] : (real)0;
        }
        tc_store8_split<KA>(trow + c * 8, v8);
      }
    } else {                                    // row (v_i, e): -(1/rho) g_ij p(m)
      real pv[Np], cj[3];
#pragma unroll
      for (int m = 0; m < Np; ++m) pv[m] = Q[m * 32 + lane];
#pragma unroll
      for (int j = 0; j < 3; ++j) cj[j] = -irho * geo[((w - 1) * 3 + j) * 32];
#pragma unroll
      for (int c = 0; c < K1 / 8; ++c) {
        real v8[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) {
          const int kap = c * 8 + e, j = kap / Np, m = kap - j * Np;
          v8[e] = kap < 3 * Np ? cj[j < 3 ? j : 0] * pv[m < Np ? m : 0] : (real)0;
        }
        tc_store8_split<KA>(trow + c * 8, v8);
      }
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    tc_fence_before();
    group_sync<NT>(g);                          // penalties are in shared memory, A1 is in tensor memory
    if (w == 0 && lane == 0) {                  // one thread issues the volume GEMM: K1/8 k-steps x 3 (3xTF32)
      tc_fence_after();
#pragma unroll
      for (int ks = 0; ks < K1 / 8; ++ks) {
        const unsigned long long off = (unsigned long long)(ks * 2 * NN);          // 32 NN bytes per k-step, in 16 B units
        tc_mma(tC, tbase + ks * 8, dB1h + off, IDESC, ks > 0);
        tc_mma(tC, tbase + KA + ks * 8, dB1h + off, IDESC, 1);
        tc_mma(tC, tbase + ks * 8, dB1l + off, IDESC, 1);
#ifdef DG_TC_4TERM
        tc_mma(tC, tbase + KA + ks * 8, dB1l + off, IDESC, 1);
#endif
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&full[2])) : "memory");
    }
    // ---- the other q stage and the trace ring are free: fetch the next item; code two items ahead
    if (i + 1 < nitems) { issue_q(i + 1, s ^ 1); issue_tr(i + 1, codeB); }
    const int codeC = load_code(i + 2);
    const int wp = a.wperm[(size_t)b * 32 + lane];
    const int pi = (w == 0 && a.pt_index[0]) ? a.pt_index[0][(size_t)b * 32 + lane] : -1;
    // the two older right-hand sides of this thread's field, from L2 (prefetched one item ahead)
    real h1[Np], h2[Np];
    {
      const real* r1p = static_cast<const real*>(L.r1[0]) + base + (size_t)w * Np * 32;
      const real* r2p = static_cast<const real*>(L.r2[0]) + base + (size_t)w * Np * 32;
#pragma unroll
      for (int n = 0; n < Np; ++n) { h1[n] = r1p[n * 32]; h2[n] = r2p[n * 32]; }
    }
    // ---- A2: rows of the surface GEMM: -P^p_j (field p), -n_i(face of j) P^v_j (field v_i)
    real a2[K2];
    {
#pragma unroll
      for (int f = 0; f < 4; ++f) {
        const float4* src = reinterpret_cast<const float4*>(pen) + ((size_t)(f * 2 + (w == 0 ? 0 : 1)) * PV) * 32 + lane;
        const real sc = w == 0 ? (real)-1 : -geo[(GEO_FACE + 5 * f + (w - 1)) * 32];
        real pv4[PV * 4];
#pragma unroll
        for (int v = 0; v < PV; ++v) *reinterpret_cast<float4*>(&pv4[v * 4]) = src[v * 32];
#pragma unroll
        for (int i2 = 0; i2 < Nfp; ++i2) a2[f * Nfp + i2] = sc * pv4[i2];
      }
#pragma unroll
      for (int j = NF; j < K2; ++j) a2[j] = 0;
    }
    mbar_wait(&full[2], 0);                     // volume GEMM done: the A columns are free
    tc_fence_after();
#pragma unroll
    for (int c = 0; c < K2 / 8; ++c) {
      real v8[8];
#pragma unroll
      for (int e = 0; e < 8; ++e) v8[e] = a2[c * 8 + e];
      tc_store8_split<KA>(trow + c * 8, v8);
    }
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    tc_fence_before();
    group_sync<NT>(g);                          // A2 is in tensor memory; everybody has read Q (A1) and pen (A2)
    if (w == 0 && lane == 0) {
      tc_fence_after();
#pragma unroll
      for (int ks = 0; ks < K2 / 8; ++ks) {
        const unsigned long long off = (unsigned long long)(ks * 2 * NN);
        tc_mma(tC, tbase + ks * 8, dB2h + off, IDESC, 1);
        tc_mma(tC, tbase + KA + ks * 8, dB2h + off, IDESC, 1);
        tc_mma(tC, tbase + ks * 8, dB2l + off, IDESC, 1);
#ifdef DG_TC_4TERM
        tc_mma(tC, tbase + KA + ks * 8, dB2l + off, IDESC, 1);
#endif
      }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&full[2])) : "memory");
    }
    mbar_wait(&full[2], 1);                     // right-hand side complete in C
    tc_fence_after();
    // ---- right-hand side of (field w, element lane) at all nodes: tensor memory -> registers
    real r0[NN];
#pragma unroll
    for (int c = 0; c < NN / 16; ++c) {
      unsigned u[16];
      asm volatile(
          "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
          : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]), "=r"(u[8]), "=r"(u[9]),
            "=r"(u[10]), "=r"(u[11]), "=r"(u[12]), "=r"(u[13]), "=r"(u[14]), "=r"(u[15])
          : "r"(trow + 2 * KA + c * 16));
#pragma unroll
      for (int e = 0; e < 16; ++e) r0[c * 16 + e] = __uint_as_float(u[e]);
    }
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    tc_fence_before();                          // the next item's MMAs overwrite C after the next barriers

    // ---- point terms (eq (15)), update (18): this thread's field at every node; new values into Q
    const bool need_half = L.qf_half[0] != nullptr && (a.blkflag[b] & 1);
    real vh[Np];
    {
      real* r0p = static_cast<real*>(L.r0[0]) + base + (size_t)w * Np * 32;
      real* qp = static_cast<real*>(a.q[0]) + base + (size_t)w * Np * 32;
      real* Qt = Q + w * Np * 32 + lane;
      const real* ptv = static_cast<const real*>(a.pt_val[0]) + (size_t)(pi < 0 ? 0 : pi) * Np;
      const real pts = (real)a.pt_scale[0];
      const real d0 = (real)L.d[0], d1 = (real)L.d[1], d2 = (real)L.d[2];
#pragma unroll
      for (int n = 0; n < Np; ++n) {
        real r = r0[n];
        if (pi >= 0) r += pts * ptv[n];
        const real v = Qt[n * 32] + (c0 * r + c1 * h1[n] + c2 * h2[n]);
        r0p[n * 32] = r;
        qp[n * 32] = v;
        Qt[n * 32] = v;
        vh[n] = need_half ? v + (d0 * r + d1 * h1[n] + d2 * h2[n]) : v;
      }
    }
    // ---- exposed traces (Alg. 4) of the new values, then of the half-step values (19), face w per warp
#pragma unroll 1
    for (int pass = 0; pass < (need_half ? 2 : 1); ++pass) {
      if (pass == 1) {
        group_sync<NT>(g);                      // pass 0 has gathered from Q
        real* Qt = Q + w * Np * 32 + lane;
#pragma unroll
        for (int n = 0; n < Np; ++n) Qt[n * 32] = vh[n];
      }
      group_sync<NT>(g);                        // Q holds the values of this pass; pen is free
      {
        const int f = w;
        const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32], nz = geo[(GEO_FACE + 5 * f + 2) * 32];
        const int* prow = sP + ((wp >> (8 * f)) & 255) * Nfp;
        real* st = pen + f * REC * 32 + lane;
#pragma unroll
        for (int i2 = 0; i2 < Nfp; ++i2) {
          const int o = fofs[i2], pos = prow[i2];
          st[pos * 32] = Q[o];
          st[(Nfp + pos) * 32] = nx * Q[Np * 32 + o] + ny * Q[2 * Np * 32 + o] + nz * Q[3 * Np * 32 + o];
        }
      }
      group_sync<NT>(g);
      {
        constexpr int ROWS = 4 * REC, NV = ROWS / 4;
        real* dst = static_cast<real*>(pass == 0 ? L.qf_write[0] : L.qf_half[0]) + ((size_t)b * 32 + lane) * ROWS;
        for (int v = w; v < NV; v += NT) {
          float4 x;
          x.x = pen[(v * 4 + 0) * 32 + lane]; x.y = pen[(v * 4 + 1) * 32 + lane];
          x.z = pen[(v * 4 + 2) * 32 + lane]; x.w = pen[(v * 4 + 3) * 32 + lane];
          reinterpret_cast<float4*>(dst)[v] = x;
        }
      }
    }
    codeA = codeB;
    codeB = codeC;
  }
  tc_fence_before();
  __syncthreads();
  if (wg == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_slot), "r"(512));
}

}  // namespace dgrtm
