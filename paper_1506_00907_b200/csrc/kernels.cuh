// CUDA kernels of the DGTD hot path for sm_100a.  One lane = one element; a CTA of T warps owns one
// 32-element block at a time (persistent loop over blocks); element data live in shared memory as
// [value][lane] columns (conflict-free, a register-file extension); each warp produces tiles of TO
// output nodes with 5*TO register accumulators, so every staged value feeds TO..6*TO FMAs.
//
//   k_rhs          volume (eqs (13)-(14) PAPER.md:113-118, Alg. 2) and/or surface
//                  (penalties (11)-(12) PAPER.md:100-111, App. A, Alg. 3)
//                  incl. boundary-trace capture / replay
//   k_update       AB update (18) + exposed traces (Alg. 4)
//   k_rk           LSERK4 stage (reading Q8)
//   k_image_update backward update of source + receiver fields fused with the image contribution
//                  (eqs (7)-(8) PAPER.md:61-65, (20)-(24) PAPER.md:174-204, readings Q1, Q1b)
//   k_source / k_record / k_inject   point terms (eq (15))
//   k_capture      traces of the stored boundary faces at the final time (reading Q12)
#pragma once
#include "kernels.h"

namespace dgrtm {

template <int N> struct Order {
  static constexpr int Np = (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int Nfp = (N + 1) * (N + 2) / 2;
  static constexpr int NF = 4 * Nfp;
  static constexpr int REC = 2 * Nfp;          // one face record of qf: p[Nfp], n.v[Nfp]
};
// tile of output nodes per warp pass / warps per CTA
template <int N> struct Tiling;
template <> struct Tiling<1> { static constexpr int TO = 4, T = 1; };
template <> struct Tiling<2> { static constexpr int TO = 5, T = 2; };
template <> struct Tiling<3> { static constexpr int TO = 5, T = 4; };
template <> struct Tiling<4> { static constexpr int TO = 7, T = 5; };
template <> struct Tiling<5> { static constexpr int TO = 7, T = 8; };
template <> struct Tiling<6> { static constexpr int TO = 7, T = 12; };

template <typename real, int N> struct RhsSmem {
  using O = Order<N>;
  static constexpr size_t ops_reals = 3 * O::Np * O::Np + O::NF * O::Np;
  static constexpr size_t data_bytes = (size_t)(4 * O::Np + 2 * O::NF + DG_NGEO) * 32 * sizeof(real) +
                                       (size_t)(4 * 32 + O::NF) * sizeof(int);
  static constexpr bool ops_in_smem = data_bytes + ops_reals * sizeof(real) <= 225 * 1024;
  static constexpr size_t bytes = data_bytes + (ops_in_smem ? ops_reals * sizeof(real) : 0);
};

template <typename real> __device__ __forceinline__ real ldg(const real* p) { return __ldg(p); }

// -------------------------------------------------------------------------------------------------
template <typename real, int N>
__global__ void __launch_bounds__(32 * Tiling<N>::T) k_rhs(RhsArgs a) {
  using O = Order<N>;
  constexpr int Np = O::Np, Nfp = O::Nfp, NF = O::NF, REC = O::REC;
  constexpr int TO = Tiling<N>::TO, T = Tiling<N>::T, NT = Np / TO;
  static_assert(Np % TO == 0, "tile must divide Np");
  constexpr bool OPS_SMEM = RhsSmem<real, N>::ops_in_smem;

  extern __shared__ __align__(16) unsigned char smem_raw[];
  real* qs = reinterpret_cast<real*>(smem_raw);      // [4Np][32]
  real* pen = qs + 4 * Np * 32;                        // [2NF][32]: Pp, then Pv
  real* sg = pen + 2 * NF * 32;                        // [DG_NGEO][32]
  real* sops = sg + DG_NGEO * 32;                      // D3T, LIFTT (if OPS_SMEM)
  int* snbr = reinterpret_cast<int*>(sops + (OPS_SMEM ? RhsSmem<real, N>::ops_reals : 0));  // [4][32]
  int* sF = snbr + 4 * 32;                             // [NF]

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const real* gD = static_cast<const real*>(a.ops.D3T);
  const real* gL = static_cast<const real*>(a.ops.LIFTT);
  if (OPS_SMEM) {
    for (int i = threadIdx.x; i < 3 * Np * Np; i += 32 * T) sops[i] = gD[i];
    for (int i = threadIdx.x; i < NF * Np; i += 32 * T) sops[3 * Np * Np + i] = gL[i];
  }
  for (int i = threadIdx.x; i < NF; i += 32 * T) sF[i] = a.ops.Fmask[i];
  const real* D3 = OPS_SMEM ? sops : gD;
  const real* LT = OPS_SMEM ? sops + 3 * Np * Np : gL;

  const real* q = static_cast<const real*>(a.q);
  const real* qf = static_cast<const real*>(a.qf);
  real* rhs = static_cast<real*>(a.rhs);
  const real* geo = static_cast<const real*>(a.geo);
  const real dir = (real)a.dir;
  const bool do_vol = a.mode & RHS_VOL, do_surf = a.mode & RHS_SURF;

  for (int b = a.blk0 + blockIdx.x; b < a.blk0 + a.nblk; b += gridDim.x) {
    __syncthreads();
    const real* qb = q + (size_t)b * (4 * Np * 32);
    for (int idx = w; idx < 4 * Np; idx += T) qs[idx * 32 + lane] = qb[idx * 32 + lane];
    for (int idx = w; idx < DG_NGEO; idx += T) sg[idx * 32 + lane] = geo[((size_t)b * DG_NGEO + idx) * 32 + lane];
    if (w == 0) {
#pragma unroll
      for (int f = 0; f < 4; ++f) snbr[f * 32 + lane] = a.nbr[((size_t)b * 4 + f) * 32 + lane];
    }
    __syncthreads();

    // ---- penalties at the face nodes (Alg. 3, first half)
    if (do_surf) {
      const real rc2 = sg[GEO_RC2 * 32 + lane], irho = sg[GEO_IRHO * 32 + lane];
      for (int j = w; j < NF; j += T) {
        const int f = j / Nfp, i = j - f * Nfp, n = sF[j];
        const real nx = sg[(GEO_FACE + 5 * f + 0) * 32 + lane], ny = sg[(GEO_FACE + 5 * f + 1) * 32 + lane],
                   nz = sg[(GEO_FACE + 5 * f + 2) * 32 + lane], gs = sg[(GEO_FACE + 5 * f + 3) * 32 + lane],
                   Zf = sg[(GEO_FACE + 5 * f + 4) * 32 + lane];
        const real pm = qs[n * 32 + lane];
        const real nvm = nx * qs[(Np + n) * 32 + lane] + ny * qs[(2 * Np + n) * 32 + lane] +
                         nz * qs[(3 * Np + n) * 32 + lane];
        const int code = snbr[f * 32 + lane];
        real dp, dnv;
        if (code >= 0) {                       // interior face: neighbour's exposed traces, my order
          const real* rec = qf + (size_t)code * REC;
          dp = rec[i] - pm;
          dnv = -rec[Nfp + i] - nvm;           // n- . v+ = -(n+ . v+)   (reading Q6b)
        } else {
          const int bc = (-1 - code) & 7, bpos = (-1 - code) >> 3;
          if (bc == 1) { dp = -2 * pm; dnv = 0; }                 // free surface  (reading Q6)
          else if (bc == 3) { dp = 0; dnv = -2 * nvm; }           // rigid wall
          else if (bc == 2) {                                     // absorbing / transparent, eq (3)
            if (a.capture) {
              real* cap = static_cast<real*>(a.capture) + (size_t)bpos * REC;
              cap[i] = pm; cap[Nfp + i] = nvm;
            }
            if (a.replay) {
              const real* rep = static_cast<const real*>(a.replay) + (size_t)bpos * REC;
              dp = rep[i] - pm; dnv = rep[Nfp + i] - nvm;
            } else { dp = -pm; dnv = -nvm; }
          } else if (bc == 4) {                                   // prescribed exterior
            const real* ex = static_cast<const real*>(a.ext) + ((size_t)bpos * Nfp + i) * 2;
            dp = ex[0] - pm; dnv = ex[1] - nvm;
          } else { dp = 0; dnv = 0; }                             // padding slot
        }
        const real half_gs = (real)0.5 * gs;
        pen[j * 32 + lane] = rc2 * half_gs * (dnv - dir * dp / Zf);
        pen[(NF + j) * 32 + lane] = irho * half_gs * (dp - dir * Zf * dnv);
      }
    }
    __syncthreads();
    // ---- v -> (U.Gr, U.Gs, U.Gt) in place (Alg. 2: combine velocities with geometric factors)
    if (do_vol) {
      const real g00 = sg[0 * 32 + lane], g01 = sg[1 * 32 + lane], g02 = sg[2 * 32 + lane],
                 g10 = sg[3 * 32 + lane], g11 = sg[4 * 32 + lane], g12 = sg[5 * 32 + lane],
                 g20 = sg[6 * 32 + lane], g21 = sg[7 * 32 + lane], g22 = sg[8 * 32 + lane];
      for (int m = w; m < Np; m += T) {
        const real vx = qs[(Np + m) * 32 + lane], vy = qs[(2 * Np + m) * 32 + lane], vz = qs[(3 * Np + m) * 32 + lane];
        qs[(Np + m) * 32 + lane] = g00 * vx + g10 * vy + g20 * vz;
        qs[(2 * Np + m) * 32 + lane] = g01 * vx + g11 * vy + g21 * vz;
        qs[(3 * Np + m) * 32 + lane] = g02 * vx + g12 * vy + g22 * vz;
      }
    }
    __syncthreads();
    // ---- output tiles
    real* rb = rhs + (size_t)b * (4 * Np * 32);
    for (int tl = w; tl < NT; tl += T) {
      const int n0 = tl * TO;
      real rp[TO], rx[TO], ry[TO], rz[TO];
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) { rp[nn] = 0; rx[nn] = 0; ry[nn] = 0; rz[nn] = 0; }
      if (do_vol) {
        real aD[TO], aR[TO], aS[TO], aT[TO];
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) { aD[nn] = 0; aR[nn] = 0; aS[nn] = 0; aT[nn] = 0; }
#pragma unroll 2
        for (int m = 0; m < Np; ++m) {
          const real p = qs[m * 32 + lane], ur = qs[(Np + m) * 32 + lane], us = qs[(2 * Np + m) * 32 + lane],
                     ut = qs[(3 * Np + m) * 32 + lane];
          const real* d3 = D3 + (m * Np + n0) * 3;
#pragma unroll
          for (int nn = 0; nn < TO; ++nn) {
            const real dr = OPS_SMEM ? d3[3 * nn] : ldg(d3 + 3 * nn), ds = OPS_SMEM ? d3[3 * nn + 1] : ldg(d3 + 3 * nn + 1),
                       dt = OPS_SMEM ? d3[3 * nn + 2] : ldg(d3 + 3 * nn + 2);
            aD[nn] += dr * ur + ds * us + dt * ut;
            aR[nn] += dr * p; aS[nn] += ds * p; aT[nn] += dt * p;
          }
        }
        const real rc2 = sg[GEO_RC2 * 32 + lane], irho = sg[GEO_IRHO * 32 + lane];
        const real g00 = sg[0 * 32 + lane], g01 = sg[1 * 32 + lane], g02 = sg[2 * 32 + lane],
                   g10 = sg[3 * 32 + lane], g11 = sg[4 * 32 + lane], g12 = sg[5 * 32 + lane],
                   g20 = sg[6 * 32 + lane], g21 = sg[7 * 32 + lane], g22 = sg[8 * 32 + lane];
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) {
          rp[nn] = -rc2 * aD[nn];
          rx[nn] = -irho * (g00 * aR[nn] + g01 * aS[nn] + g02 * aT[nn]);
          ry[nn] = -irho * (g10 * aR[nn] + g11 * aS[nn] + g12 * aT[nn]);
          rz[nn] = -irho * (g20 * aR[nn] + g21 * aS[nn] + g22 * aT[nn]);
        }
      } else {                                  // surface-only pass accumulates into rhs (Alg. 3)
#pragma unroll
        for (int nn = 0; nn < TO; ++nn) {
          rp[nn] = rb[(n0 + nn) * 32 + lane]; rx[nn] = rb[(Np + n0 + nn) * 32 + lane];
          ry[nn] = rb[(2 * Np + n0 + nn) * 32 + lane]; rz[nn] = rb[(3 * Np + n0 + nn) * 32 + lane];
        }
      }
      if (do_surf) {
#pragma unroll
        for (int f = 0; f < 4; ++f) {
          real av[TO];
#pragma unroll
          for (int nn = 0; nn < TO; ++nn) av[nn] = 0;
#pragma unroll 2
          for (int i = 0; i < Nfp; ++i) {
            const int j = f * Nfp + i;
            const real Pp = pen[j * 32 + lane], Pv = pen[(NF + j) * 32 + lane];
            const real* l = LT + j * Np + n0;
#pragma unroll
            for (int nn = 0; nn < TO; ++nn) {
              const real lv = OPS_SMEM ? l[nn] : ldg(l + nn);
              rp[nn] -= lv * Pp; av[nn] += lv * Pv;
            }
          }
          const real nx = sg[(GEO_FACE + 5 * f + 0) * 32 + lane], ny = sg[(GEO_FACE + 5 * f + 1) * 32 + lane],
                     nz = sg[(GEO_FACE + 5 * f + 2) * 32 + lane];
#pragma unroll
          for (int nn = 0; nn < TO; ++nn) { rx[nn] -= nx * av[nn]; ry[nn] -= ny * av[nn]; rz[nn] -= nz * av[nn]; }
        }
      }
#pragma unroll
      for (int nn = 0; nn < TO; ++nn) {
        rb[(n0 + nn) * 32 + lane] = rp[nn]; rb[(Np + n0 + nn) * 32 + lane] = rx[nn];
        rb[(2 * Np + n0 + nn) * 32 + lane] = ry[nn]; rb[(3 * Np + n0 + nn) * 32 + lane] = rz[nn];
      }
    }
  }
}

// -------------------------------------------------------------------------------------------------
// exposed traces of one node's new values -> staging buffer (writer-permuted positions)
template <typename real, int N>
__device__ __forceinline__ void stage_traces(real* st, int STR, int lane, int n, real p, real vx, real vy, real vz,
                                             const real* nrm, const int* sInv, const int* sP, int wp) {
  constexpr int Nfp = Order<N>::Nfp, REC = Order<N>::REC;
#pragma unroll
  for (int e = 0; e < 3; ++e) {
    const int j = sInv[n * 3 + e];
    if (j < 0) continue;
    const int f = j / Nfp, i = j - f * Nfp;
    const int pos = sP[((wp >> (8 * f)) & 255) * Nfp + i];
    st[lane * STR + f * REC + pos] = p;
    st[lane * STR + f * REC + Nfp + pos] = nrm[3 * f] * vx + nrm[3 * f + 1] * vy + nrm[3 * f + 2] * vz;
  }
}

// tables shared by the update-type kernels: inverse face mask [Np][3] and the permutation table
template <int N>
__device__ __forceinline__ void load_face_tables(const OpsDev& ops, int* sInv, int* sP, int nthreads) {
  constexpr int Np = Order<N>::Np, Nfp = Order<N>::Nfp, NF = Order<N>::NF;
  for (int i = threadIdx.x; i < 3 * Np; i += nthreads) sInv[i] = -1;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int j = 0; j < NF; ++j) {
      const int n = ops.Fmask[j];
      int e = 0;
      while (sInv[n * 3 + e] >= 0) ++e;
      sInv[n * 3 + e] = j;
    }
  }
  for (int i = threadIdx.x; i < ops.nperm * Nfp; i += nthreads) sP[i] = ops.ptab[i];
  __syncthreads();
}

template <int N> struct UpdSmem {
  static constexpr int STR = 4 * Order<N>::REC + 1;
  static constexpr int kMaxPerm = 32;
  template <typename real> static constexpr size_t bytes(int nfields) {
    return (size_t)nfields * 32 * STR * sizeof(real) + (size_t)(3 * Order<N>::Np + kMaxPerm * Order<N>::Nfp) * sizeof(int);
  }
};

template <typename real, int N>
__device__ __forceinline__ void write_traces(real* qf, const real* st, int b, int nthreads) {
  constexpr int REC4 = 4 * Order<N>::REC, STR = UpdSmem<N>::STR;
  real* out = qf + (size_t)b * 32 * REC4;
  for (int x = threadIdx.x; x < 32 * REC4; x += nthreads) {
    const int l = x / REC4, o = x - l * REC4;
    out[x] = st[l * STR + o];
  }
}

template <typename real>
__device__ __forceinline__ void load_normals(const real* geo, int b, int lane, real* nrm) {
#pragma unroll
  for (int f = 0; f < 4; ++f)
#pragma unroll
    for (int d = 0; d < 3; ++d) nrm[3 * f + d] = geo[((size_t)b * DG_NGEO + GEO_FACE + 5 * f + d) * 32 + lane];
}

// MODE 0: AB update (18).  MODE 1: LSERK4 stage.
template <typename real, int N, int MODE>
__global__ void __launch_bounds__(32 * Tiling<N>::T) k_update(UpdateArgs a, RkArgs rk) {
  using O = Order<N>;
  constexpr int Np = O::Np, T = Tiling<N>::T, STR = UpdSmem<N>::STR;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  real* st = reinterpret_cast<real*>(smem_raw);
  int* sInv = reinterpret_cast<int*>(st + 32 * STR);
  int* sP = sInv + 3 * Np;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const OpsDev& ops = MODE == 0 ? a.ops : rk.ops;
  load_face_tables<N>(ops, sInv, sP, 32 * T);
  real* q = static_cast<real*>(MODE == 0 ? a.q : rk.q);
  real* qf = static_cast<real*>(MODE == 0 ? a.qf : rk.qf);
  const real* geo = static_cast<const real*>(MODE == 0 ? a.geo : rk.geo);
  const int* wperm = MODE == 0 ? a.wperm : rk.wperm;
  const int blk0 = MODE == 0 ? a.blk0 : rk.blk0, nblk = MODE == 0 ? a.nblk : rk.nblk;
  const real* h0 = static_cast<const real*>(a.h0);
  const real* h1 = static_cast<const real*>(a.h1);
  const real* h2 = static_cast<const real*>(a.h2);
  const real c0 = (real)a.c0, c1 = (real)a.c1, c2 = (real)a.c2;
  real* res = static_cast<real*>(rk.res);
  const real* rr = static_cast<const real*>(rk.r);
  const real rA = (real)rk.A, rB = (real)rk.B, rdt = (real)rk.dt;

  for (int b = blk0 + blockIdx.x; b < blk0 + nblk; b += gridDim.x) {
    real nrm[12];
    load_normals(geo, b, lane, nrm);
    const int wp = wperm[b * 32 + lane];
    const size_t base = (size_t)b * (4 * Np * 32) + lane;
    for (int n = w; n < Np; n += T) {
      real v[4];
#pragma unroll
      for (int fld = 0; fld < 4; ++fld) {
        const size_t o = base + (size_t)(fld * Np + n) * 32;
        if (MODE == 0) {
          v[fld] = q[o] + (c0 * h0[o] + c1 * h1[o] + c2 * h2[o]);
        } else {
          const real rs = rA * res[o] + rdt * rr[o];
          res[o] = rs;
          v[fld] = q[o] + rB * rs;
        }
        q[o] = v[fld];
      }
      stage_traces<real, N>(st, STR, lane, n, v[0], v[1], v[2], v[3], nrm, sInv, sP, wp);
    }
    __syncthreads();
    write_traces<real, N>(qf, st, b, 32 * T);
    __syncthreads();
  }
}

// -------------------------------------------------------------------------------------------------
template <typename real, int N>
__global__ void __launch_bounds__(32 * Tiling<N>::T) k_image_update(ImageArgs a) {
  using O = Order<N>;
  constexpr int Np = O::Np, T = Tiling<N>::T, STR = UpdSmem<N>::STR;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  real* stS = reinterpret_cast<real*>(smem_raw);
  real* stR = stS + 32 * STR;
  int* sInv = reinterpret_cast<int*>(stR + 32 * STR);
  int* sP = sInv + 3 * Np;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  load_face_tables<N>(a.ops, sInv, sP, 32 * T);
  real* qS = static_cast<real*>(a.qS);
  real* qR = static_cast<real*>(a.qR);
  const real* hS[3] = {static_cast<const real*>(a.hS0), static_cast<const real*>(a.hS1), static_cast<const real*>(a.hS2)};
  const real* hR[3] = {static_cast<const real*>(a.hR0), static_cast<const real*>(a.hR1), static_cast<const real*>(a.hR2)};
  real* img = static_cast<real*>(a.image);
  const real* geo = static_cast<const real*>(a.geo);
  const real dts = (real)a.dts, adts = dts < 0 ? -dts : dts;
  const real ex = (real)a.e[0], ey = (real)a.e[1], ez = (real)a.e[2];

  for (int b = a.blk0 + blockIdx.x; b < a.blk0 + a.nblk; b += gridDim.x) {
    real nrm[12];
    load_normals(geo, b, lane, nrm);
    const int wp = a.wperm[b * 32 + lane];
    const real Z = a.characteristic ? geo[((size_t)b * DG_NGEO + GEO_Z) * 32 + lane] : (real)0;
    const size_t base = (size_t)b * (4 * Np * 32) + lane;
    for (int n = w; n < Np; n += T) {
      real s[4], r[4], sh[3][4], rh[3][4];
#pragma unroll
      for (int fld = 0; fld < 4; ++fld) {
        const size_t o = base + (size_t)(fld * Np + n) * 32;
        s[fld] = qS[o]; r[fld] = qR[o];
#pragma unroll
        for (int k = 0; k < 3; ++k) { sh[k][fld] = hS[k][o]; rh[k][fld] = hR[k][o]; }
      }
      // q_S^- = p - c rho e.v (source), q_R^+ = p + c rho e.v (receivers), eq (8) PAPER.md:65;
      // the classical condition (4) is Z = 0
      const real A = s[0] - Z * (ex * s[1] + ey * s[2] + ez * s[3]);
      const real B = r[0] + Z * (ex * r[1] + ey * r[2] + ez * r[3]);
      real rA[3], rB[3];
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        rA[k] = sh[k][0] - Z * (ex * sh[k][1] + ey * sh[k][2] + ez * sh[k][3]);
        rB[k] = rh[k][0] + Z * (ex * rh[k][1] + ey * rh[k][2] + ez * rh[k][3]);
      }
      real acc = A * B;
#pragma unroll
      for (int k = 0; k < 3; ++k) {
        acc += dts * (real)a.abar[k] * (A * rB[k] + B * rA[k]);
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2) acc += dts * dts * (real)a.C[3 * k + k2] * rA[k] * rB[k2];
      }
      const size_t oi = ((size_t)b * Np + n) * 32 + lane;
      img[oi] += adts * acc;
      // update (18) of both wavefields
#pragma unroll
      for (int fld = 0; fld < 4; ++fld) {
        const size_t o = base + (size_t)(fld * Np + n) * 32;
        s[fld] += dts * ((real)a.a[0] * sh[0][fld] + (real)a.a[1] * sh[1][fld] + (real)a.a[2] * sh[2][fld]);
        r[fld] += dts * ((real)a.a[0] * rh[0][fld] + (real)a.a[1] * rh[1][fld] + (real)a.a[2] * rh[2][fld]);
        qS[o] = s[fld]; qR[o] = r[fld];
      }
      stage_traces<real, N>(stS, STR, lane, n, s[0], s[1], s[2], s[3], nrm, sInv, sP, wp);
      stage_traces<real, N>(stR, STR, lane, n, r[0], r[1], r[2], r[3], nrm, sInv, sP, wp);
    }
    __syncthreads();
    write_traces<real, N>(static_cast<real*>(a.qfS), stS, b, 32 * T);
    write_traces<real, N>(static_cast<real*>(a.qfR), stR, b, 32 * T);
    __syncthreads();
  }
}

// own traces of listed boundary faces -> history record (final time, reading Q12)
template <typename real, int N>
__global__ void k_capture(CaptureArgs a) {
  using O = Order<N>;
  constexpr int Np = O::Np, Nfp = O::Nfp, REC = O::REC;
  const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long)a.nfaces * Nfp) return;
  const int e = (int)(tid / Nfp), i = (int)(tid - (long)e * Nfp);
  const int sf = a.faces[e], slot = sf >> 2, f = sf & 3, b = slot >> 5, lane = slot & 31;
  const int n = a.ops.Fmask[f * Nfp + i];
  const real* q = static_cast<const real*>(a.q);
  const real* geo = static_cast<const real*>(a.geo);
  const size_t o = (size_t)b * (4 * Np * 32) + (size_t)n * 32 + lane;
  const real* gf = geo + ((size_t)b * DG_NGEO + GEO_FACE + 5 * f) * 32 + lane;
  real* rec = static_cast<real*>(a.record) + (size_t)e * REC;
  rec[i] = q[o];
  rec[Nfp + i] = gf[0] * q[o + (size_t)Np * 32] + gf[32] * q[o + (size_t)2 * Np * 32] + gf[64] * q[o + (size_t)3 * Np * 32];
}

// halo exchange of a domain decomposition ("transfer the traces of fields situated at the interface
// between two sub-domains"): the cut faces are prescribed-exterior faces here; their exterior state (p+, n-.v+) is the
// neighbouring sub-domain's exposed trace at the coinciding node, with n-.v+ = -(n+.v+) (reading Q6b).  src_qf may be
// a peer pointer: the loads then cross NVLink, nothing is staged on the host
template <typename real, int N>
__global__ void k_halo(HaloArgs a) {
  constexpr int Nfp = Order<N>::Nfp, REC = Order<N>::REC;
  const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long)a.nh * Nfp) return;
  const int h = (int)(tid / Nfp), i = (int)(tid - (long)h * Nfp);
  const real* r = static_cast<const real*>(a.src_qf) + (size_t)a.rec[h] * REC;
  const int j = a.pos[tid];
  real* e = static_cast<real*>(a.ext) + ((size_t)a.bnd[h] * Nfp + i) * 2;
  e[0] = r[j];
  e[1] = -r[Nfp + j];
}

// -------------------------------------------------------------------------------------------------
// point terms (eq (15))
template <typename real, int N>
__global__ void k_source(PointArgs a) {
  constexpr int Np = Order<N>::Np;
  const int n = threadIdx.x;
  if (n >= Np) return;
  const int b = a.src_slot >> 5, lane = a.src_slot & 31;
  real* rhs = static_cast<real*>(a.rhs);
  rhs[(size_t)b * (4 * Np * 32) + (size_t)n * 32 + lane] += (real)a.amp_now * static_cast<const real*>(a.src_w)[n];
}

template <typename real, int N>
__global__ void k_record(PointArgs a) {
  constexpr int Np = Order<N>::Np;
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= a.nr) return;
  const int slot = a.rcv_slot[r], b = slot >> 5, lane = slot & 31, lev = a.rcv_level[r];
  const real w0 = (real)a.lw[lev][0], w1 = (real)a.lw[lev][1], w2 = (real)a.lw[lev][2];
  const bool mid = (a.lw[lev][0] != 0.0) || (a.lw[lev][1] != 0.0) || (a.lw[lev][2] != 0.0);
  const real* q = static_cast<const real*>(a.q);
  const int cur = a.cur[lev];
  const real* h0 = static_cast<const real*>(a.hist[cur]);
  const real* h1 = static_cast<const real*>(a.hist[(cur + 2) % 3]);
  const real* h2 = static_cast<const real*>(a.hist[(cur + 1) % 3]);
  const real* row = static_cast<const real*>(a.rcv_row) + (size_t)r * Np;
  real acc = 0;
  for (int n = 0; n < Np; ++n) {
    const size_t o = (size_t)b * (4 * Np * 32) + (size_t)n * 32 + lane;
    real p = q[o];
    if (mid) p += w0 * h0[o] + w1 * h1[o] + w2 * h2[o];
    acc += row[n] * p;
  }
  static_cast<real*>(a.data)[(size_t)r * a.nsamp + a.sample] = acc;
}

// thread = (group g, node n): rhs^p[slot_g][n] += sum_{r in g} d_r(sample) w_r[n]
template <typename real, int N>
__global__ void k_inject(PointArgs a) {
  constexpr int Np = Order<N>::Np;
  const long tid = (long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long)a.ng * Np) return;
  const int g = a.g0 + (int)(tid / Np), n = (int)(tid % Np);
  const int slot = a.grp_slot[g], b = slot >> 5, lane = slot & 31;
  const real* data = static_cast<const real*>(a.data);
  const real* w = static_cast<const real*>(a.rcv_w);
  real acc = 0;
  for (int x = a.grp_off[g]; x < a.grp_off[g + 1]; ++x) {
    const int r = a.grp_rcv[x];
    acc += data[(size_t)r * a.nsamp + a.sample] * w[(size_t)r * Np + n];
  }
  if (a.pt_out) static_cast<real*>(a.pt_out)[(size_t)g * Np + n] = acc;       // fused step kernel adds it
  else static_cast<real*>(a.rhs)[(size_t)b * (4 * Np * 32) + (size_t)n * 32 + lane] += acc;
}

}  // namespace dgrtm
