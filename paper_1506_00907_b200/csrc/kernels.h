// Launch interface between the host runtime (dgrtm_api.cpp) and the per-(N, precision) kernel
// instantiations (kernels_inst.cu).  Device layout (all "blocked by 32 elements", one lane = one
// element, consecutive lanes = consecutive addresses):
//   q, rhs history, res : [block][4*Np][32]          field-major, then node, then lane
//   image               : [block][Np][32]
//   geo                 : [block][DG_NGEO][32]       (see GeoIndex)
//   nbr                 : [block][4][32] int32        >=0: trace record (slot'*4+f'); <0: -1-(bpos*8+bc)
//   wperm               : [block][32] int32           4 x 8-bit ids into the face-permutation table
//   qf (exposed traces) : [slot][4][2][Nfp]           ELEMENT-major: record (slot,f) holds p then n.v of
//                         the owner's face nodes, stored at the positions of the READER's face nodes
//                         (each interior face has exactly one reader).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace dgrtm {

enum GeoIndex {
  GEO_G = 0,        // 9: g[i*3+j] = d r_j / d x_i  (App. A, reading Q3)
  GEO_RC2 = 9,      // rho c^2
  GEO_IRHO = 10,    // 1/rho
  GEO_Z = 11,       // rho c (imaging, eq (8))
  GEO_FACE = 12,    // 4 x {nx, ny, nz, gsur = J_f/J, Zf (single-valued face impedance, reading Q4)}
  DG_NGEO = 32
};

enum { RHS_VOL = 1, RHS_SURF = 2 };

struct OpsDev {            // device pointers, element type = real of the instantiation
  const void* D3T;         // [Np(m)][Np(n)][3]  = Dr[n][m], Ds[n][m], Dt[n][m]
  const void* LIFTT;       // [4Nfp(j)][Np(n)]   = LIFT[n][j]
  const int* Fmask;        // [4Nfp]
  const int* ptab;         // [nperm][Nfp] face-permutation table (writer position of face node i)
  int nperm;
};

struct RhsArgs {
  const void* q; const void* qf; void* rhs;
  const void* geo; const int* nbr;
  int blk0, nblk, mode;
  double dir;              // +1 forward, -1 backward (sign of tau_p, tau_v)
  void* capture;           // record to write own traces of stored boundary faces into, or null
  const void* replay;      // record to read exterior states of stored boundary faces from, or null
  const void* ext;         // [nbnd][Nfp][2] prescribed exterior states, or null
  OpsDev ops;
};

struct UpdateArgs {        // q += c0 h0 + c1 h1 + c2 h2 (eq (18)); traces refreshed
  void* q; void* qf; const void* h0; const void* h1; const void* h2;
  const void* geo; const int* wperm;
  int blk0, nblk;
  double c0, c1, c2;
  OpsDev ops;
};

struct RkArgs {            // res = A res + dt r; q += B res (LSERK4, reading Q8)
  void* q; void* qf; void* res; const void* r;
  const void* geo; const int* wperm;
  int blk0, nblk;
  double A, B, dt;
  OpsDev ops;
};

struct HalfArgs {          // traces of q + c0 h0 + c1 h1 + c2 h2 (eq (19)) for a list of slots
  const void* q; void* qf; const void* h0; const void* h1; const void* h2;
  const void* geo; const int* wperm; const int* list; int nlist;
  double c0, c1, c2;
  OpsDev ops;
};

struct ImageArgs {         // backward update of two wavefields with the imaging contribution (24)
  void* qS; void* qfS; const void* hS0; const void* hS1; const void* hS2;
  void* qR; void* qfR; const void* hR0; const void* hR1; const void* hR2;
  void* image;
  const void* geo; const int* wperm;
  int blk0, nblk;
  double dts;              // signed local step
  double a[3], abar[3], C[9];
  double e[3];             // updir
  int characteristic;
  OpsDev ops;
};

struct PointArgs {         // source term / receiver sampling / receiver injection
  void* rhs; const void* q;
  const void* hist[3]; int cur[8];   // rotating right-hand-side buffers and the newest one per level
  // source
  int src_slot; const void* src_w; double amp_now;
  // receivers
  int nr; const int* rcv_slot; const void* rcv_row; const void* rcv_w; const int* rcv_level;
  void* data; int64_t nsamp; int64_t sample;
  double lw[8][3];         // per level: signed-step-scaled partial AB weights (reading Q13)
  // injection groups
  int g0, ng; const int* grp_slot; const int* grp_off; const int* grp_rcv;
};

struct CaptureArgs {       // own traces of a list of (slot*4+f) faces -> record
  const void* q; const void* geo; const int* faces; int nfaces; void* record; OpsDev ops;
};

struct KernelTable {
  int N, precision, Np, Nfp;
  void (*rhs)(const RhsArgs&, cudaStream_t);
  void (*update)(const UpdateArgs&, cudaStream_t);
  void (*rk)(const RkArgs&, cudaStream_t);
  void (*half)(const HalfArgs&, cudaStream_t);
  void (*image_update)(const ImageArgs&, cudaStream_t);
  void (*source)(const PointArgs&, cudaStream_t);
  void (*record)(const PointArgs&, cudaStream_t);
  void (*inject)(const PointArgs&, cudaStream_t);
  void (*capture)(const CaptureArgs&, cudaStream_t);
  int (*init)();           // sets shared-memory attributes; returns cudaError
};

const KernelTable* get_kernel_table(int N, int precision);

}  // namespace dgrtm
