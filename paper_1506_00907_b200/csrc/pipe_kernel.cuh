// k_pipe: the fused step of step_kernel.cuh as a software pipeline.  Same arithmetic, same StepArgs;
// what changes is how operands reach the SM:
//   * every contiguous input of a work item (one 32-element block of one wavefield) - q, the two older
//     right-hand sides, the geometric factors - arrives by cp.async.bulk (TMA, 1-D) in a two-stage shared
//     memory ring, issued one item ahead and completed on an mbarrier;
//   * the neighbours' trace records (an indirect gather, one record per lane and face) arrive by per-lane
//     cp.async (LDGSTS) one item ahead, issued and consumed by the same lane;
//   * the consumer warps therefore never wait on a global load: they read shared memory, issue FMAs and
//     fire-and-forget stores (new right-hand side, new q, new traces).
// Operator tables are packed per output tile: D3Q[tile][m][RL] = Dr[n0..][m], Ds[..][m], Dt[..][m] (RL =
// 3 TO rounded up to the vector width), LTQ[tile][j][LL], so every operator fetch is a full-width LDS.
#pragma once
#include "step_kernel.cuh"

namespace dgrtm {

// Tiling and staging of one (precision, order); the values are the winners of the sweeps in profiles/r1b, r2_experiments:
//   TO outputs per warp, NT warps per block, G groups per CTA;
//   QS = stages of the q ring (2: fetched one item ahead; 1: requested during the previous item's trace write-out, from
//        L2, where a prefetch issued one item ahead has put it);
//   RS = 1: the two older right-hand sides go through shared memory (bulk copy); 0: no room for them there;
//   TP (with RS = 0): they are loaded from L2 in chunks during the lift loop and PARKED in tensor memory (tcgen05.st; lane =
//        element, columns = values), from where the update reads them back (tcgen05.ld) - shared memory and the register
//        file are full, the 256 KB of tensor memory are idle.  1: one chunk buffer, 2: two alternating (one-field kernel);
//   UG = 1: velocities -> U.G once per block, in place in shared memory; 0: every warp forms U.G on the fly (9 more FMAs
//        per input node and warp, two shared-memory passes and one barrier fewer);
//   F2 = 1: the volume contraction uses packed fp32x2 FMAs (__ffma2_rn, sm_100): half the FMA instructions for twice the
//        accumulators (N = 3: 395 -> 387 us on the config-4 mesh; N = 4: slower, 857 -> 911 us).
template <typename real, int N> struct PipeCfg { static constexpr bool enabled = false; static constexpr int TO = 1, NT = 1, G = 1, QS = 1, RS = 1, UG = 1, F2 = 0, TP = 0; };
template <> struct PipeCfg<float, 2> { static constexpr bool enabled = true; static constexpr int TO = 5, NT = 2, G = 6, QS = 1, RS = 1, UG = 0, F2 = 1, TP = 0; };
template <> struct PipeCfg<double, 2> { static constexpr bool enabled = true; static constexpr int TO = 5, NT = 2, G = 3, QS = 1, RS = 1, UG = 0, F2 = 0, TP = 0; };
template <> struct PipeCfg<float, 3> { static constexpr bool enabled = true; static constexpr int TO = 5, NT = 4, G = 3, QS = 2, RS = 1, UG = 0, F2 = 1, TP = 0; };
template <> struct PipeCfg<float, 4> { static constexpr bool enabled = true; static constexpr int TO = 9, NT = 4, G = 3, QS = 1, RS = 0, UG = 0, F2 = 0, TP = 1; };
template <> struct PipeCfg<float, 5> { static constexpr bool enabled = true; static constexpr int TO = 7, NT = 8, G = 2, QS = 1, RS = 0, UG = 0, F2 = 0, TP = 1; };
template <> struct PipeCfg<float, 6> { static constexpr bool enabled = true; static constexpr int TO = 12, NT = 7, G = 1, QS = 1, RS = 0, UG = 0, F2 = 1, TP = 1; };
template <> struct PipeCfg<double, 3> { static constexpr bool enabled = true; static constexpr int TO = 5, NT = 4, G = 3, QS = 1, RS = 0, UG = 0, F2 = 0, TP = 2; };

template <> struct PipeCfg<double, 4> { static constexpr bool enabled = true; static constexpr int TO = 5, NT = 7, G = 1, QS = 1, RS = 0, UG = 0, F2 = 0, TP = 2; };

template <typename real, int N> struct PipeSmem {
  using O = Order<N>;
  using C = PipeCfg<real, N>;
  static constexpr int VW = 16 / (int)sizeof(real);
  static constexpr int RL = (3 * C::TO + VW - 1) / VW * VW;        // packed derivative row
  static constexpr int LL = (C::TO + VW - 1) / VW * VW;            // packed lift row
  static constexpr size_t ops_reals = (size_t)C::NT * O::Np * RL + (size_t)C::NT * O::NF * LL;
  static constexpr size_t tab_ints = O::NF + UpdSmem<N>::kMaxPerm * O::Nfp;     // Fmask, permutation table
  static constexpr size_t ops_bytes = (ops_reals * sizeof(real) + tab_ints * sizeof(int) + 127) / 128 * 128;
  // two stages of q [4Np][32] + factors [DG_NGEO][32]; single buffers: r1, r2 [4Np][32] each (fetched after
  // the previous item's update), neighbour records [4][32][REC] (fetched after the previous item's
  // penalties), penalties / trace staging [2NF][32]
  static constexpr size_t stage_reals = (size_t)(4 * O::Np + DG_NGEO) * 32;
  // penalties: [face][Pp | Pv][ceil(Nfp / VW)][lane][VW] (one vector load = VW face nodes of my element)
  static constexpr int PV = (O::Nfp + VW - 1) / VW;               // vectors per face and penalty kind
  // trace staging (after the update the penalties are dead): [element-lane][4 REC reals] = the block's records exactly as
  // they lie in global memory, the element stride padded to an ODD number SU of 16-byte units (vector stores of 8
  // consecutive lanes then cover all banks once)
  static constexpr int UE = 4 * O::REC * (int)sizeof(real) / 16;  // 16-byte units of one element's four records
  static constexpr int SU = UE | 1;
  static constexpr size_t stg_reals = (size_t)32 * SU * 16 / sizeof(real);
  static constexpr size_t pen0_reals = (size_t)(8 * PV * VW > 2 * O::NF ? 8 * PV * VW : 2 * O::NF) * 32;
  static constexpr size_t pen_reals = pen0_reals > stg_reals ? pen0_reals : stg_reals;
  static constexpr size_t group_reals = C::QS * stage_reals + (size_t)(C::RS * 8 * O::Np + 4 * O::REC) * 32 + pen_reals;
  static constexpr size_t group_bytes = group_reals * sizeof(real);
  // control region behind the tables: mbarriers [G][3] + table barrier, tensor-memory slot, ticket rings [G][4]
  static constexpr size_t ring_off = ((size_t)(3 * C::G + 1) * 8 + 16 + 15) / 16 * 16;
  // the gather table of the trace phase, qtab[perm][face][pos] = offset in q of the own face node whose value goes to
  // position pos of the record the neighbour reads, is built in the prologue OVER the permutation table of the blob
  // (kMaxPerm x Nfp ints = kPerm x 4 x Nfp: a triangle's node set has at most 6 such permutations)
  static constexpr int kPerm = UpdSmem<N>::kMaxPerm / 4;
  static constexpr size_t ctl_bytes = (ring_off + (size_t)C::G * 16 + 127) / 128 * 128;
  static constexpr size_t bytes = ops_bytes + ctl_bytes + (size_t)C::G * group_bytes;
  static constexpr bool fits = bytes <= 227 * 1024;
};

__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
template <int BYTES>
__device__ __forceinline__ void cp_async(void* dst, const void* src) {
  if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
  else if (BYTES == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
  else asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
// full-width vector loads of a packed operator row
template <typename real, int LEN>
__device__ __forceinline__ void load_packed(const real* __restrict__ p, real (&out)[LEN]) {
  constexpr int VW = 16 / (int)sizeof(real);
  using V = typename VecT<real, VW>::T;
#pragma unroll
  for (int v = 0; v < LEN / VW; ++v) {
    const V x = reinterpret_cast<const V*>(p)[v];
    const real* xs = reinterpret_cast<const real*>(&x);
#pragma unroll
    for (int e = 0; e < VW; ++e) out[v * VW + e] = xs[e];
  }
}


template <typename real, int N, bool DUAL, bool TICKETS>
__global__ void __launch_bounds__(PipeCfg<real, N>::G * PipeCfg<real, N>::NT * 32, 1)
k_pipe(const __grid_constant__ StepArgs a) {
  using O = Order<N>;
  using Cfg = PipeCfg<real, N>;
  using SM = PipeSmem<real, N>;
  constexpr int Np = O::Np, Nfp = O::Nfp, NF = O::NF, REC = O::REC;
  constexpr int TO = Cfg::TO, NT = Cfg::NT, G = Cfg::G, RL = SM::RL, LL = SM::LL, VW = SM::VW, PV = SM::PV;
  constexpr bool INPLACE = NT > 1 && Cfg::UG;
  constexpr int QS = Cfg::QS, RS = Cfg::RS;
  constexpr int NTHREADS = G * NT * 32, NFLD = DUAL ? 2 : 1;
  constexpr unsigned QBYTES = 4 * Np * 32 * sizeof(real), GBYTES = DG_NGEO * 32 * sizeof(real);
  constexpr int RB = REC * (int)sizeof(real), CPB = RB % 16 == 0 ? 16 : (RB % 8 == 0 ? 8 : 4);
  constexpr int CPW = CPB / (int)sizeof(real);
  constexpr int FPW = (4 + NT - 1) / NT;                          // faces per warp

  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* sD = reinterpret_cast<real*>(smem_raw);                   // [NT][Np][RL]
  real* sL = sD + NT * Np * RL;                                   // [NT][NF][LL]
  int* sF = reinterpret_cast<int*>(sL + NT * NF * LL);            // [NF]
  int* sP = sF + NF;                                              // [kMaxPerm][Nfp]
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_raw + SM::ops_bytes);   // [G][3], tables
  real* gbase = reinterpret_cast<real*>(smem_raw + SM::ops_bytes + SM::ctl_bytes);

  const int tid = threadIdx.x, lane = tid & 31, wg = tid >> 5, g = wg / NT, w = wg - g * NT;
  real* grp = gbase + (size_t)g * SM::group_reals;
  real* R1 = grp + QS * SM::stage_reals;                          // [4Np][32]
  real* R2 = R1 + RS * 4 * Np * 32;                               // [4Np][32]
  real* TR = R2 + RS * 4 * Np * 32;                               // [4][32][REC]
  real* pen = TR + 4 * REC * 32;                                  // [2NF][32], later trace staging [4REC][32]
  unsigned long long* full = bars + 3 * g;                        // [0], [1]: q stages; [2]: r1, r2
  unsigned long long* tabbar = bars + 3 * G;
  // tensor-memory parking: per warp 8 TO reals (h1, h2 of its TO nodes, 4 fields); warps of one lane quarter side by side
  constexpr bool PARK = Cfg::TP && !RS;
  constexpr bool IPARK = DUAL;                                    // imaging scalars of the source field wait in tensor memory
  constexpr int PW = Words8<real>::NW;                            // 32-bit columns per node
  constexpr int IW = Words4<real>::NW;                            // 32-bit columns per node of the imaging scalars
  constexpr int WCOLS = (PARK ? TO * PW : 0) + (IPARK ? TO * IW : 0);   // columns of one warp
  constexpr int PCOLS_NEED = (G * NT + 3) / 4 * WCOLS;
  constexpr int PCOLS = PCOLS_NEED <= 32 ? 32 : (PCOLS_NEED <= 64 ? 64 : (PCOLS_NEED <= 128 ? 128 : (PCOLS_NEED <= 256 ? 256 : 512)));
  static_assert(PCOLS_NEED <= 512, "tensor memory has 512 columns");
  constexpr bool TMEM = PARK || IPARK;
  // two register buffers alternating (five chunks, two faces of latency each) or one (four chunks, one face each)
  constexpr bool PARK2 = PARK && Cfg::TP == 2 && !DUAL;
  constexpr int PCN = PARK2 ? (TO + 4) / 5 : (TO + 3) / 4;        // nodes per chunk
  unsigned* tmem_slot = reinterpret_cast<unsigned*>(bars + 3 * G + 1);

  {  // operator tables + Fmask + permutation table: one blob, laid out on the host exactly as here
    if (tid == 0) {
      mbar_init(tabbar, 1);
      for (int x = 0; x < 3 * G; ++x) mbar_init(&bars[x], 1);
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      mbar_expect_tx(tabbar, (unsigned)SM::ops_bytes);
      bulk_g2s(smem_raw, a.ops2_D3Q, (unsigned)SM::ops_bytes, tabbar);
    }
    if constexpr (TMEM) {
      if (wg == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(PCOLS));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    }
    __syncthreads();
    if constexpr (TMEM) asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  }
  // this warp's parking columns: lanes of quarter wg % 4, columns of its rank wg / 4 within the quarter
  const unsigned tpark = TMEM ? (*tmem_slot + ((unsigned)((wg & 3) * 32) << 16) + (unsigned)((wg >> 2) * WCOLS)) : 0u;
  const unsigned timg = tpark + (unsigned)(PARK ? TO * PW : 0);
  const real* myD = sD + (size_t)w * Np * RL;
  const real* myL = sL + (size_t)w * NF * LL;

  // work distribution.  TICKETS = false (single-rate launches): fixed contiguous chunks per CTA, the groups of a CTA
  // taking every G-th block of its chunk - the streams stay sequential and every block costs the same.  TICKETS = true
  // (multi-rate launches): the first three turns of a group interleaved over all groups, then blocks by ticket from
  // a global counter (one atomic per block, taken three turns ahead) - blocks differ in cost (levels, half-step
  // traces) and sit sorted by level, so fixed chunks would load the SMs unevenly, and a launch of a few hundred blocks
  // spreads over all SMs.  ring[j & 3] = block of the group's j-th turn (TICKETS only); bend = no block
  int* ring = reinterpret_cast<int*>(smem_raw + SM::ops_bytes + SM::ring_off) + 4 * g;
  const int bend = a.blk0 + a.nblk, ngroups = (int)gridDim.x * G;
  const int lo = a.blk0 + (int)(((long long)a.nblk * blockIdx.x) / gridDim.x);
  const int hi = a.blk0 + (int)(((long long)a.nblk * (blockIdx.x + 1)) / gridDim.x);
  const int base0 = a.blk0 + g * (int)gridDim.x + (int)blockIdx.x;
  const long long dyn0 = (long long)a.blk0 + 3LL * ngroups;
  const int limit = dyn0 < bend ? (int)dyn0 : bend;
  unsigned* const ticket = a.sched + a.sched_sel;
  const real dir = (real)a.dir;
  const int n0 = w * TO;

  const int nmine = (hi - lo - g + G - 1) / G;                    // fixed chunks: blocks of this group
  const int nitems = nmine > 0 ? nmine * NFLD : 0;
  auto item_block = [&](int i) {
    if constexpr (TICKETS) return ring[(i / NFLD) & 3];
    else return a.reverse ? hi - 1 - g - (i / NFLD) * G : lo + g + (i / NFLD) * G;
  };
  auto has_item = [&](int i) {                                    // the group has an i-th item
    if constexpr (TICKETS) return ring[(i / NFLD) & 3] < bend;
    else return i < nitems;
  };
  auto level_of = [&](int b) { int l = 0; while (b >= a.lv[l].blk_end) ++l; return l; };
  auto load_codes = [&](int i, int (&code)[FPW]) {
    const int b = item_block(i);
#pragma unroll
    for (int k = 0; k < FPW; ++k) {
      const int f = w + k * NT;
      code[k] = (f < 4 && has_item(i)) ? a.nbr[((size_t)b * 4 + f) * 32 + lane] : -1;
    }
  };
  // everything item i needs, into stage s: bulk copies by one lane, trace records by their consumer lanes
  // the two older right-hand sides of item i (single buffer: call after the previous item's update)
  auto issue_r = [&](int i) {
    if (w == 0 && lane == 0) {
      const int b = item_block(i), fi = i % NFLD;
      const StepLevel& L = a.lv[level_of(b)];
      const size_t off = (size_t)b * (4 * Np * 32);
      if (RS) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        mbar_expect_tx(&full[2], 2 * QBYTES);
        bulk_g2s(R1, static_cast<const real*>(L.r1[fi]) + off, QBYTES, &full[2]);
        bulk_g2s(R2, static_cast<const real*>(L.r2[fi]) + off, QBYTES, &full[2]);
      } else {
        bulk_prefetch_l2(static_cast<const real*>(L.r1[fi]) + off, QBYTES);
        bulk_prefetch_l2(static_cast<const real*>(L.r2[fi]) + off, QBYTES);
      }
    }
  };
  // q and the factors of item i into stage s (bulk copies by one lane)
  auto issue_q = [&](int i, int s) {
    if (w == 0 && lane == 0) {
      const int b = item_block(i), fi = i % NFLD;
      real* Q = grp + (size_t)s * SM::stage_reals;
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      mbar_expect_tx(&full[s], QBYTES + GBYTES);
      bulk_g2s(Q, static_cast<const real*>(a.q[fi]) + (size_t)b * (4 * Np * 32), QBYTES, &full[s]);
      bulk_g2s(Q + 4 * Np * 32, static_cast<const real*>(a.geo) + (size_t)b * DG_NGEO * 32, GBYTES, &full[s]);
    }
  };
  auto prefetch_q = [&](int i) {
    if (w == 0 && lane == 0) {
      const int b = item_block(i), fi = i % NFLD;
      bulk_prefetch_l2(static_cast<const real*>(a.q[fi]) + (size_t)b * (4 * Np * 32), QBYTES);
      bulk_prefetch_l2(static_cast<const real*>(a.geo) + (size_t)b * DG_NGEO * 32, GBYTES);
    }
  };
  // write-out pieces of this warp (it = w + k NT): staging offset of piece P = it*32 + lane (rows VS (P % NV) .. of
  // element-lane P / NV, column rotated by the piece index)
  constexpr int WO_NV = SM::UE, WOK = (WO_NV + NT - 1) / NT;
  int wo_src[WOK];                                                // byte offset of the piece in the staging
#pragma unroll
  for (int k = 0; k < WOK; ++k) {
    const int P = (w + k * NT) * 32 + lane, el = P / WO_NV, o4 = P - el * WO_NV;
    wo_src[k] = (el * SM::SU + o4) * 16;
  }
  // piece P = it*32 + lane of a face's 32 records belongs to element-lane P / NP, offset (P % NP) CPW in its record
  int gth_r[REC / CPW], gth_v[REC / CPW];
#pragma unroll
  for (int it = 0; it < REC / CPW; ++it) { const int P = it * 32 + lane; gth_r[it] = P / (REC / CPW); gth_v[it] = (P - gth_r[it] * (REC / CPW)) * CPW; }
  // the neighbours' trace records of item i (per-lane cp.async by their consumer lanes)
  auto issue_tr = [&](int i, const int (&code)[FPW]) {
    const int b = item_block(i), fi = i % NFLD, l = level_of(b);
    const StepLevel& L = a.lv[l];
    const int slot_lo = (l > 0 ? a.lv[l - 1].blk_end : 0) * 32, slot_hi = L.blk_end * 32;
    const int lm = l > 0 ? l - 1 : 0, lp = l + 1 < a.nlevels ? l + 1 : l;
    const real* qfm = static_cast<const real*>(a.lv[lm].qf_read[fi]);
    const real* qf0 = static_cast<const real*>(L.qf_read[fi]);
    const real* qfp = static_cast<const real*>(a.lv[lp].qf_read[fi]);
    // cooperative gather: consecutive lanes fetch consecutive 16-byte pieces of the SAME neighbour record (a
    // record is one contiguous line or two), so an instruction touches ~NP times fewer lines than one record per
    // lane would; piece P = it*32 + lane belongs to element-lane r = P / NP, whose code comes by shuffle
    constexpr int NP = REC / CPW;
#pragma unroll
    for (int k = 0; k < FPW; ++k) {
      const int f = w + k * NT;
      if (f < 4) {
#pragma unroll
        for (int it = 0; it < NP; ++it) {
          const int gr = gth_r[it], gv = gth_v[it];
          const int c = __shfl_sync(0xffffffffu, code[k], gr);
          if (c >= 0) {
            const int s2 = c >> 2;
            const real* src = (s2 >= slot_hi ? qfp : (s2 < slot_lo ? qfm : qf0)) + (size_t)c * REC + gv;
            // [face][element-lane][REC] = [face][piece P]: a warp writes 512 contiguous bytes
            cp_async<CPB>(TR + (size_t)f * 32 * REC + (it * 32 + lane) * CPW, src);
          }
        }
      }
    }
  };

  int codeA[FPW], codeB[FPW], codeC[FPW];
  // programmatic dependent launch: everything down to griddepcontrol.wait overlaps the tail of the previous launch
  // on the stream and touches only what no launch writes (tables, neighbour codes); after it the previous launch's
  // results (q, right-hand sides, traces, ticket counter) are read
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  if constexpr (TICKETS) {
    if (w == 0 && lane < 3) {                   // the first three turns
      const int bs = base0 + lane * ngroups;
      ring[lane] = bs < limit ? bs : bend;
    }
    group_sync<NT>(g);
  }
  load_codes(0, codeA);
  load_codes(1, codeB);
  mbar_wait(tabbar, 0);
  int* sQT = sP;                                                  // [kPerm][4][Nfp], built in place over the permutation table
  {
    constexpr int EPT = (SM::kPerm * 4 * Nfp + NTHREADS - 1) / NTHREADS;   // entries per thread
    const int np = a.ops.nperm < SM::kPerm ? a.ops.nperm : SM::kPerm;
    int dst_i[EPT], val[EPT];
#pragma unroll
    for (int e = 0; e < EPT; ++e) {
      const int x = tid + e * NTHREADS;
      dst_i[e] = -1;
      if (x < np * 4 * Nfp) {
        const int pf = x / Nfp, i2 = x - pf * Nfp, pid = pf >> 2, f = pf & 3;
        dst_i[e] = pf * Nfp + sP[pid * Nfp + i2];
        val[e] = sF[f * Nfp + i2] * 32;
      }
    }
    __syncthreads();                                              // every entry of the permutation table has been read
#pragma unroll
    for (int e = 0; e < EPT; ++e) if (dst_i[e] >= 0) sQT[dst_i[e]] = val[e];
    __syncthreads();
  }
  int fofs[FPW][Nfp];                                             // own-trace offsets of this warp's faces in Q
#pragma unroll
  for (int k = 0; k < FPW; ++k)
#pragma unroll
    for (int i2 = 0; i2 < Nfp; ++i2) fofs[k][i2] = (w + k * NT < 4 ? sF[(w + k * NT) * Nfp + i2] : 0) * 32 + lane;
  asm volatile("griddepcontrol.wait;" ::: "memory");
  if (TICKETS && blockIdx.x == 0 && tid == 0) a.sched[a.sched_sel ^ 1] = 0u;   // the next launch's counter (this launch's predecessor is done with it)
  if (has_item(0)) { issue_q(0, 0); issue_tr(0, codeA); issue_r(0); }

  unsigned tk = 0;
#pragma unroll 1
  for (int i = 0; has_item(i); ++i) {
    const int s = QS == 2 ? (i & 1) : 0, b = item_block(i), fi = i % NFLD, l = level_of(b);
    const bool more = has_item(i + 1);                            // another item follows
    // ticket of the block three turns ahead: taken now, stored at the end of this block's last item
    if (TICKETS && w == 0 && lane == 0 && fi == 0) tk = atomicAdd(ticket, 1u);
    const StepLevel& L = a.lv[l];
    real* Q = grp + (size_t)s * SM::stage_reals;                  // [4Np][32]
    const real* geo = Q + 4 * Np * 32 + lane;
    real* qg = static_cast<real*>(a.q[fi]);
    const size_t base = (size_t)b * (4 * Np * 32) + lane;
    const real c0 = (real)L.c[0], c1 = (real)L.c[1], c2 = (real)L.c[2];

    group_sync<NT>(g);                          // the group has left the previous item (pen is free)
    mbar_wait(&full[s], (unsigned)(QS == 2 ? (i >> 1) : i) & 1u);
    cp_async_wait_all();
    __syncwarp();                               // the pieces of my record were fetched by other lanes of this warp
    const real rc2 = geo[GEO_RC2 * 32], irho = geo[GEO_IRHO * 32];
    real vold[3][TO];                                             // this tile's velocities before the in-place transform
    if (INPLACE) {
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) {
        const int n = n0 + nn < Np ? n0 + nn : Np - 1;
        vold[0][nn] = Q[(Np + n) * 32 + lane]; vold[1][nn] = Q[(2 * Np + n) * 32 + lane]; vold[2][nn] = Q[(3 * Np + n) * 32 + lane];
      }
    }

    // ---- penalties at the face nodes (Alg. 3, first half; eqs (11)-(12), readings Q2, Q4, Q6).  Branch-free
    // inner loop: [[p]] = ap p- + ep_i, n.[[v]] = av (n.v)- + ev_i with per-face (ap, av) and exterior arrays
    {
      real* capt = fi == 0 ? static_cast<real*>(L.capture) : nullptr;
      const real* repl = fi == 0 ? static_cast<const real*>(L.replay) : nullptr;
#pragma unroll
      for (int k = 0; k < FPW; ++k) {
        const int f = w + k * NT;
        if (f < 4) {
          const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32],
                     nz = geo[(GEO_FACE + 5 * f + 2) * 32], gs = geo[(GEO_FACE + 5 * f + 3) * 32],
                     Zf = geo[(GEO_FACE + 5 * f + 4) * 32];
          const int code = codeA[k];
          const int bc = code >= 0 ? 0 : ((-1 - code) & 7), bpos = code >= 0 ? 0 : ((-1 - code) >> 3);
          real ep[Nfp], ev[Nfp];
          {
            real rv[REC];
            const real* src = TR + ((size_t)f * 32 + lane) * REC;
            using V = typename VecT<real, CPW>::T;
#pragma unroll
            for (int v = 0; v < REC / CPW; ++v) {
              const V x = reinterpret_cast<const V*>(src)[v];
              const real* xs = reinterpret_cast<const real*>(&x);
#pragma unroll
              for (int e = 0; e < CPW; ++e) rv[v * CPW + e] = xs[e];
            }
#pragma unroll
            for (int i2 = 0; i2 < Nfp; ++i2) {                       // interior: p+, n-.v+ = -(n+.v+) (reading Q6b)
              ep[i2] = code >= 0 ? rv[i2] : (real)0;
              ev[i2] = code >= 0 ? -rv[Nfp + i2] : (real)0;
            }
          }
          // interior, absorbing, prescribed: -1, -1; free surface: -2, 0; rigid wall: 0, -2; padding slot: 0, 0
          const real ap = (code >= 0 || bc == 2 || bc == 4) ? (real)-1 : (bc == 1 ? (real)-2 : (real)0);
          const real av = (code >= 0 || bc == 2 || bc == 4) ? (real)-1 : (bc == 3 ? (real)-2 : (real)0);
          const bool rep_lane = bc == 2 && repl != nullptr, ext_lane = bc == 4;
          if (__any_sync(0xffffffffu, rep_lane || ext_lane)) {       // rare: exterior state from memory
            if (rep_lane) {
#pragma unroll
              for (int i2 = 0; i2 < Nfp; ++i2) { ep[i2] = repl[(size_t)bpos * REC + i2]; ev[i2] = repl[(size_t)bpos * REC + Nfp + i2]; }
            } else if (ext_lane) {
              const long long hr = a.halo_rec ? a.halo_rec[bpos] : -1;
              if (hr >= 0) {       // halo face: the neighbouring sub-domain's exposed trace, n-.v+ = -(n+.v+) (reading Q6b)
                const real* r = static_cast<const real*>((fi == 0 ? a.halo_src : a.halo_src2)[a.halo_set[bpos]]) + (size_t)hr * REC;
                const int* hp = a.halo_pos + (size_t)bpos * Nfp;
#pragma unroll
                for (int i2 = 0; i2 < Nfp; ++i2) { const int j = hp[i2]; ep[i2] = r[j]; ev[i2] = -r[Nfp + j]; }
              } else {
                const real* ex = static_cast<const real*>(a.ext) + (size_t)bpos * Nfp * 2;
#pragma unroll
                for (int i2 = 0; i2 < Nfp; ++i2) { ep[i2] = ex[2 * i2]; ev[i2] = ex[2 * i2 + 1]; }
              }
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
            const int o = fofs[k][i2];
            const real pm = Q[o];
            const real nvm = nx * Q[Np * 32 + o] + ny * Q[2 * Np * 32 + o] + nz * Q[3 * Np * 32 + o];
            if (cap_any && cap_lane) { capt[(size_t)bpos * REC + i2] = pm; capt[(size_t)bpos * REC + Nfp + i2] = nvm; }
            const real dp = ap * pm + ep[i2], dnv = av * nvm + ev[i2];
            Pp[i2] = kp * (dnv - diZ * dp);
            Pv[i2] = kv * (dp - dZ * dnv);
          }
          {
            using V = typename VecT<real, VW>::T;
            V* dstp = reinterpret_cast<V*>(pen) + ((size_t)(f * 2 + 0) * PV) * 32 + lane;
            V* dstv = reinterpret_cast<V*>(pen) + ((size_t)(f * 2 + 1) * PV) * 32 + lane;
#pragma unroll
            for (int v = 0; v < PV; ++v) {
              dstp[v * 32] = *reinterpret_cast<const V*>(&Pp[v * VW]);
              dstv[v * 32] = *reinterpret_cast<const V*>(&Pv[v * VW]);
            }
          }
        }
      }
    }
    const real g00 = geo[0 * 32], g01 = geo[1 * 32], g02 = geo[2 * 32], g10 = geo[3 * 32], g11 = geo[4 * 32],
               g12 = geo[5 * 32], g20 = geo[6 * 32], g21 = geo[7 * 32], g22 = geo[8 * 32];
    group_sync<NT>(g);                          // penalties done; every warp has left the previous item
    // ---- the other stage is free now: fetch the next item; codes two items ahead
    if (more) {
      if (QS == 2) issue_q(i + 1, s ^ 1); else prefetch_q(i + 1);
      issue_tr(i + 1, codeB);
    }
    load_codes(i + 2, codeC);
    const int wp = a.wperm[(size_t)b * 32 + lane];
    const int pi = a.pt_index[fi] ? a.pt_index[fi][(size_t)b * 32 + lane] : -1;
    real imgv[TO];                              // image values of this tile, fetched long before their update
    if (DUAL && fi == 1 && L.image_on) {
      const real* ip = static_cast<const real*>(a.image) + ((size_t)b * Np + n0) * 32 + lane;
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) imgv[nn] = (TO * NT == Np || n0 + nn < Np) ? ip[nn * 32] : (real)0;
    }
    if (INPLACE) {                              // v -> (U.Gr, U.Gs, U.Gt) once per block (Alg. 2)
      for (int m = w; m < Np; m += NT) {
        const real vx = Q[(Np + m) * 32 + lane], vy = Q[(2 * Np + m) * 32 + lane], vz = Q[(3 * Np + m) * 32 + lane];
        Q[(Np + m) * 32 + lane] = g00 * vx + g10 * vy + g20 * vz;
        Q[(2 * Np + m) * 32 + lane] = g01 * vx + g11 * vy + g21 * vz;
        Q[(3 * Np + m) * 32 + lane] = g02 * vx + g12 * vy + g22 * vz;
      }
      group_sync<NT>(g);
    }

    // ---- volume (eqs (13)-(14), Alg. 2)
    real rp[TO], rx[TO], ry[TO], rz[TO];
    if constexpr (sizeof(real) == 4 && Cfg::F2) {  // packed fp32x2 FMAs (sm_100): one instruction per pair of row entries
                                                 // (the two-field kernel is register-bound and keeps scalar FMAs)
      float2 aG2[RL / 2], aD2[RL / 2];
#pragma unroll
      for (int k = 0; k < RL / 2; ++k) { aG2[k] = make_float2(0.f, 0.f); aD2[k] = make_float2(0.f, 0.f); }
      constexpr int UM2 = 5;
#pragma unroll UM2
      for (int m = 0; m < Np; ++m) {
        const float p = Q[m * 32 + lane];
        const float vx = Q[(Np + m) * 32 + lane], vy = Q[(2 * Np + m) * 32 + lane], vz = Q[(3 * Np + m) * 32 + lane];
        float ur, us, ut;
        if (INPLACE) { ur = vx; us = vy; ut = vz; }
        else { ur = g00 * vx + g10 * vy + g20 * vz; us = g01 * vx + g11 * vy + g21 * vz; ut = g02 * vx + g12 * vy + g22 * vz; }
        float d[RL];
        load_packed<float, RL>(reinterpret_cast<const float*>(myD) + m * RL, d);
        const float2 pp = make_float2(p, p);
#pragma unroll
        for (int k = 0; k < RL / 2; ++k) {
          const int e0 = 2 * k, e1 = 2 * k + 1;
          const float u0 = e0 < TO ? ur : (e0 < 2 * TO ? us : (e0 < 3 * TO ? ut : 0.f));
          const float u1 = e1 < TO ? ur : (e1 < 2 * TO ? us : (e1 < 3 * TO ? ut : 0.f));
          const float2 dk = make_float2(d[e0], d[e1]);
          aG2[k] = __ffma2_rn(dk, pp, aG2[k]);
          aD2[k] = __ffma2_rn(dk, make_float2(u0, u1), aD2[k]);
        }
      }
      const float* fG = reinterpret_cast<const float*>(aG2);
      const float* fD = reinterpret_cast<const float*>(aD2);
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) {
        const float aDn = fD[nn] + fD[TO + nn] + fD[2 * TO + nn], aRn = fG[nn], aSn = fG[TO + nn], aTn = fG[2 * TO + nn];
        rp[nn] = -rc2 * aDn;
        rx[nn] = -irho * (g00 * aRn + g01 * aSn + g02 * aTn);
        ry[nn] = -irho * (g10 * aRn + g11 * aSn + g12 * aTn);
        rz[nn] = -irho * (g20 * aRn + g21 * aSn + g22 * aTn);
      }
    } else
    {
      real aD[TO], aR[TO], aS[TO], aT[TO];
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) { aD[nn] = 0; aR[nn] = 0; aS[nn] = 0; aT[nn] = 0; }
      constexpr int UM = 5;
#pragma unroll UM
      for (int m = 0; m < Np; ++m) {
        const real p = Q[m * 32 + lane];
        real ur, us, ut;
        if (INPLACE) {
          ur = Q[(Np + m) * 32 + lane]; us = Q[(2 * Np + m) * 32 + lane]; ut = Q[(3 * Np + m) * 32 + lane];
        } else {
          const real vx = Q[(Np + m) * 32 + lane], vy = Q[(2 * Np + m) * 32 + lane], vz = Q[(3 * Np + m) * 32 + lane];
          ur = g00 * vx + g10 * vy + g20 * vz; us = g01 * vx + g11 * vy + g21 * vz; ut = g02 * vx + g12 * vy + g22 * vz;
        }
        real d[RL];
        load_packed<real, RL>(myD + m * RL, d);
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) {
          aD[nn] = fma(d[nn], ur, aD[nn]); aD[nn] = fma(d[TO + nn], us, aD[nn]); aD[nn] = fma(d[2 * TO + nn], ut, aD[nn]);
          aR[nn] = fma(d[nn], p, aR[nn]); aS[nn] = fma(d[TO + nn], p, aS[nn]); aT[nn] = fma(d[2 * TO + nn], p, aT[nn]);
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
    group_sync<NT>(g);                          // every warp has read Q: the update may overwrite its tile's nodes
    // ---- surface (Alg. 3, second half).  With PARK the older right-hand sides (h1, h2 of this warp's nodes, 4 fields)
    // come from L2 in chunks of PCN nodes and are parked in tensor memory.  One buffer (TP = 1): chunk f is in flight
    // during the lift of face f.  Two alternating buffers (TP = 2, fp64 N = 3 where one face is shorter than the L2 round
    // trip): chunk 0 is requested before the loop into A, chunk f + 1 at the start of face f (into B for even f, A for
    // odd f), and a buffer is parked just before it is reused or after the loop - two faces to land
    const real* h1g = static_cast<const real*>(L.r1[fi]) + base + (size_t)n0 * 32;
    const real* h2g = static_cast<const real*>(L.r2[fi]) + base + (size_t)n0 * 32;
    real hA[PARK ? PCN : 1][8], hB[PARK2 ? PCN : 1][8];
    auto load_chunk = [&](int c, real (&hc)[PARK ? PCN : 1][8]) {
#pragma unroll
      for (int j = 0; j < PCN; ++j) {
        const int nn = c * PCN + j;
        if (nn < TO && (TO * NT == Np || n0 + nn < Np)) {
#pragma unroll
          for (int fld = 0; fld < 4; ++fld) {
            hc[j][fld] = __ldg(h1g + (fld * Np + nn) * 32);
            hc[j][4 + fld] = __ldg(h2g + (fld * Np + nn) * 32);
          }
        }
      }
    };
    auto park_chunk = [&](int c, const real (&hc)[PARK ? PCN : 1][8]) {   // (hB has this extent only with PARK2, its only user)
#pragma unroll
      for (int j = 0; j < PCN; ++j) {
        const int nn = c * PCN + j;
        if (nn < TO) {                                             // warp-uniform: tcgen05.st is .aligned
          unsigned wd[PW];
          Words8<real>::pack(hc[j], wd);
          tmem_st<PW>(tpark + (unsigned)(nn * PW), wd);
        }
      }
    };
    auto lift_face = [&](int f) {
      real av[TO];
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) av[nn] = 0;
      real Ppv[PV * VW], Pvv[PV * VW];
      {
        using V = typename VecT<real, VW>::T;
        const V* srcp = reinterpret_cast<const V*>(pen) + ((size_t)(f * 2 + 0) * PV) * 32 + lane;
        const V* srcv = reinterpret_cast<const V*>(pen) + ((size_t)(f * 2 + 1) * PV) * 32 + lane;
#pragma unroll
        for (int v = 0; v < PV; ++v) {
          *reinterpret_cast<V*>(&Ppv[v * VW]) = srcp[v * 32];
          *reinterpret_cast<V*>(&Pvv[v * VW]) = srcv[v * 32];
        }
      }
#pragma unroll
      for (int i2 = 0; i2 < Nfp; ++i2) {
        const int j = f * Nfp + i2;
        const real Pp = Ppv[i2], Pv = Pvv[i2];
        real lv[LL];
        load_packed<real, LL>(myL + j * LL, lv);
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) { rp[nn] -= lv[nn] * Pp; av[nn] += lv[nn] * Pv; }
      }
      const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32], nz = geo[(GEO_FACE + 5 * f + 2) * 32];
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) { rx[nn] -= nx * av[nn]; ry[nn] -= ny * av[nn]; rz[nn] -= nz * av[nn]; }
    };
    if constexpr (PARK && !PARK2) {               // one buffer: chunk f in flight during the lift of face f
      load_chunk(0, hA);
#pragma unroll 1
      for (int f = 0; f < 4; ++f) {
        lift_face(f);
        park_chunk(f, hA);
        if (f + 1 < 4) load_chunk(f + 1, hA);
      }
    } else if constexpr (PARK2) {
      load_chunk(0, hA);
#pragma unroll 1
      for (int fp = 0; fp < 2; ++fp) {
        const int f = 2 * fp;
        if (fp > 0) park_chunk(f - 1, hB);        // chunk f - 1, requested at the start of face f - 2
        load_chunk(f + 1, hB);
        lift_face(f);
        park_chunk(f, hA);                        // chunk f, requested at the start of face f - 1 (chunk 0: before the loop)
        load_chunk(f + 2, hA);
        lift_face(f + 1);
      }
      park_chunk(3, hB);
      park_chunk(4, hA);
    } else {
#pragma unroll 1
      for (int f = 0; f < 4; ++f) lift_face(f);
    }
    if constexpr (PARK) tmem_wait_st();

    // ---- point terms (eq (15)), update (18), imaging (24); the new values replace the tile's nodes in Q
    const bool need_half = L.qf_half[fi] != nullptr && (a.blkflag[b] & 1);
    if (RS) mbar_wait(&full[2], (unsigned)i & 1u);
    {
      constexpr bool FULL = TO * NT == Np;                          // no padded outputs: no guards
      real* r0p = static_cast<real*>(L.r0[fi]) + base + (size_t)n0 * 32;
      real* qp = qg + base + (size_t)n0 * 32;
      const real* ptv = static_cast<const real*>(a.pt_val[fi]) + (size_t)(pi < 0 ? 0 : pi) * Np;
      const real pts = (real)a.pt_scale[fi];
      const bool imaging = DUAL && L.image_on;
      const real Z = (imaging && a.characteristic) ? geo[GEO_Z * 32] : (real)0;
      const real ex = (real)a.e[0], ey = (real)a.e[1], ez = (real)a.e[2];
      const real sgn = fi == 0 ? (real)-1 : (real)1;      // q_S^- = p - Z e.v ; q_R^+ = p + Z e.v  (eq (8))
      const real dts = (real)L.dts, adts = dts < 0 ? -dts : dts;
      real* imgp = static_cast<real*>(a.image) + ((size_t)b * Np + n0) * 32 + lane;
      const real d0 = (real)L.d[0], d1 = (real)L.d[1], d2 = (real)L.d[2];
      real* Qt = Q + n0 * 32 + lane;
      const real* R1t = RS ? R1 + n0 * 32 + lane : static_cast<const real*>(L.r1[fi]) + base + (size_t)n0 * 32;
      const real* R2t = RS ? R2 + n0 * 32 + lane : static_cast<const real*>(L.r2[fi]) + base + (size_t)n0 * 32;
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) {
        {
          if (FULL || n0 + nn < Np) {
            real h1[4], h2[4];
            if constexpr (PARK) {                                    // parked in tensor memory during the lift loop
              unsigned wd[PW];
              real hv[8];
              tmem_ld<PW>(tpark + (unsigned)(nn * PW), wd);
              tmem_wait_ld();
              Words8<real>::unpack(wd, hv);
#pragma unroll
              for (int fld = 0; fld < 4; ++fld) { h1[fld] = hv[fld]; h2[fld] = hv[4 + fld]; }
            } else {
#pragma unroll
              for (int fld = 0; fld < 4; ++fld) { h1[fld] = R1t[(fld * Np + nn) * 32]; h2[fld] = R2t[(fld * Np + nn) * 32]; }
            }
            real r0v[4] = {rp[nn], rx[nn], ry[nn], rz[nn]}, qo[4], v[4];
            if (pi >= 0) r0v[0] += pts * ptv[n0 + nn];
            qo[0] = Qt[nn * 32];
#pragma unroll
            for (int fld = 1; fld < 4; ++fld) qo[fld] = INPLACE ? vold[fld - 1][nn] : Qt[(fld * Np + nn) * 32];
#pragma unroll
            for (int fld = 0; fld < 4; ++fld) {
              v[fld] = qo[fld] + (c0 * r0v[fld] + c1 * h1[fld] + c2 * h2[fld]);
              r0p[(fld * Np + nn) * 32] = r0v[fld];
              qp[(fld * Np + nn) * 32] = v[fld];
              Qt[(fld * Np + nn) * 32] = v[fld];
            }
            if (imaging) {
              const real A0 = qo[0] + sgn * Z * (ex * qo[1] + ey * qo[2] + ez * qo[3]);
              const real A1 = r0v[0] + sgn * Z * (ex * r0v[1] + ey * r0v[2] + ez * r0v[3]);
              const real A2 = h1[0] + sgn * Z * (ex * h1[1] + ey * h1[2] + ez * h1[3]);
              const real A3 = h2[0] + sgn * Z * (ex * h2[1] + ey * h2[2] + ez * h2[3]);
              if (fi == 0) {                    // parked until the receiver field of this block is updated
                const real sv[4] = {A0, A1, A2, A3};
                unsigned wd[IW];
                Words4<real>::pack(sv, wd);
                tmem_st<IW>(timg + (unsigned)(nn * IW), wd);
              } else {
                real sv[4];
                {
                  unsigned wd[IW];
                  tmem_ld<IW>(timg + (unsigned)(nn * IW), wd);
                  tmem_wait_ld();
                  Words4<real>::unpack(wd, sv);
                }
                const real S0 = sv[0];
                const real rA[3] = {sv[1], sv[2], sv[3]};
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
                imgp[nn * 32] = imgv[nn] + adts * acc;
              }
            }
            // value at the half step (19) = new value + sum_s d_s r_s; kept for the second trace pass
            if (need_half) {
#pragma unroll
              for (int fld = 0; fld < 4; ++fld) v[fld] += d0 * r0v[fld] + d1 * h1[fld] + d2 * h2[fld];
            }
            rp[nn] = v[0]; rx[nn] = v[1]; ry[nn] = v[2]; rz[nn] = v[3];
          }
        }
      }
    }

    if constexpr (IPARK) { if (fi == 0) tmem_wait_st(); }
    group_sync<NT>(g);                          // Q holds the new values; r1, r2 are consumed
    if (more) issue_r(i + 1);
    // ---- exposed traces (Alg. 4) of the new values, then of the half-step values (19): gathered
    // per face from Q, placed at the reader's positions (permutation table), staged in pen as [row][lane]
#pragma unroll 1
    for (int pass = 0; pass < (need_half ? 2 : 1); ++pass) {
      if (pass == 1) {
        group_sync<NT>(g);                      // pass 0 has gathered from Q
        constexpr bool FULL = TO * NT == Np;
        real* Qt = Q + n0 * 32 + lane;
#pragma unroll
        for (int nn = 0; nn < TO; ++nn)
          if (FULL || n0 + nn < Np) {
            Qt[nn * 32] = rp[nn]; Qt[(Np + nn) * 32] = rx[nn]; Qt[(2 * Np + nn) * 32] = ry[nn]; Qt[(3 * Np + nn) * 32] = rz[nn];
          }
      }
      if (pass == 1) group_sync<NT>(g);         // Q holds the values of this pass; pen is free
      // gather formulation: position r of the record (the READER's node order) takes the own face node qtab[perm][f][r];
      // the record is built in registers in its final order and stored with vector stores into the staging, which has
      // the block's global layout [element-lane][face][p | n.v] (element stride padded, PipeSmem)
      char* stg = reinterpret_cast<char*>(pen);
#pragma unroll
      for (int k = 0; k < FPW; ++k) {
        const int f = w + k * NT;
        if (f < 4) {
          const real nx = geo[(GEO_FACE + 5 * f + 0) * 32], ny = geo[(GEO_FACE + 5 * f + 1) * 32], nz = geo[(GEO_FACE + 5 * f + 2) * 32];
          const int* qrow = sQT + (((wp >> (8 * f)) & 255) * 4 + f) * Nfp;
          const real* Ql = Q + lane;
          constexpr int SWB = (REC * (int)sizeof(real)) % 16 == 0 ? 16 : 8, SW = SWB / (int)sizeof(real);   // store width
          using VS_t = typename VecT<real, SW>::T;
          VS_t* out = reinterpret_cast<VS_t*>(stg + (size_t)lane * (SM::SU * 16) + (size_t)f * (REC * sizeof(real)));
          constexpr bool QREG = Nfp >= 10;                         // keep the offsets in registers (each is used for p and for n.v)
          int qo[QREG ? Nfp : 1];                                   // offsets of the record's nodes, in the reader's order
          if constexpr (QREG) {
#pragma unroll
            for (int r = 0; r < Nfp; ++r) qo[r] = qrow[r];
          }
#pragma unroll
          for (int c = 0; c < REC / SW; ++c) {
            VS_t x;
            real* xs = reinterpret_cast<real*>(&x);
#pragma unroll
            for (int e = 0; e < SW; ++e) {
              const int r = c * SW + e;                             // compile-time: p at position r, or n.v at position r - Nfp
              const int o = QREG ? qo[QREG ? (r < Nfp ? r : r - Nfp) : 0] : qrow[r < Nfp ? r : r - Nfp];
              if (r < Nfp) xs[e] = Ql[o];
              else xs[e] = nx * Ql[Np * 32 + o] + ny * Ql[2 * Np * 32 + o] + nz * Ql[3 * Np * 32 + o];
            }
            out[c] = x;
          }
        }
      }
      group_sync<NT>(g);
      // single-stage q ring: the last pass has gathered from Q, so the next item's q may land during the write-out
      if (QS == 1 && pass == (need_half ? 1 : 0) && more) issue_q(i + 1, 0);
      {  // cooperative write-out: the block's 32 x 4 records are one contiguous run; consecutive lanes store
         // consecutive 16-byte pieces (piece P = unit P % UE of element-lane P / UE): one vector load, one vector store
        constexpr int VS = 16 / (int)sizeof(real), ROWS = 4 * REC, NV = SM::UE;
        using V = typename VecT<real, VS>::T;
        V* dst = reinterpret_cast<V*>(static_cast<real*>(pass == 0 ? L.qf_write[fi] : L.qf_half[fi]) + (size_t)b * 32 * ROWS);
        if constexpr (DUAL) {                   // register-bound: a rolled loop that recomputes the piece offsets
          for (int it = w; it < NV; it += NT) {
            const int P = it * 32 + lane, el = P / NV, o4 = P - el * NV;
            dst[P] = *reinterpret_cast<const V*>(stg + (el * SM::SU + o4) * 16);
          }
        } else {
#pragma unroll
          for (int k = 0; k < WOK; ++k) {
            const int it = w + k * NT;
            if (it < NV) dst[it * 32 + lane] = *reinterpret_cast<const V*>(stg + wo_src[k]);
          }
        }
      }
    }
#pragma unroll
    for (int k = 0; k < FPW; ++k) { codeA[k] = codeB[k]; codeB[k] = codeC[k]; }
    if (TICKETS && w == 0 && lane == 0 && fi == NFLD - 1) {       // slot of the finished turn <- block three turns ahead
      const long long nb = dyn0 + (long long)tk;
      ring[(i / NFLD + 3) & 3] = nb < bend ? (int)nb : bend;
    }
  }
  if constexpr (TMEM) {                         // every warp is done with its columns: release the tensor memory
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (wg == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(*tmem_slot), "r"(PCOLS));
  }
}

}  // namespace dgrtm
