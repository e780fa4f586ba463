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
  void* pt_out;            // if set: injection amounts go to pt_out[group][Np] instead of into rhs
};

struct CaptureArgs {       // own traces of a list of (slot*4+f) faces -> record
  const void* q; const void* geo; const int* faces; int nfaces; void* record; OpsDev ops;
};

struct HaloArgs {          // exterior states of halo faces <- exposed traces of the neighbouring sub-domain
  const void* src_qf;        // the neighbour's trace buffer [slot][4][2][Nfp] (a peer pointer over NVLink, or local)
  void* ext;                 // this sub-domain's prescribed-exterior array [nbnd][Nfp][2]
  const int* bnd;            // [nh] boundary-face-list index of the halo face here
  const long long* rec;      // [nh] record (slot * 4 + f) of the same face in the neighbour's buffer
  const int* pos;            // [nh][Nfp] position in that record of the node that coincides with my face node i
  int nh;
};

// ---- fused step kernel (step_kernel.cuh) ---------------------------------------------------------
// One launch advances every level that sits at the start of the fine step.  Per level (contiguous block
// range): where its right-hand sides rotate, where its traces are read / written, its AB weights.
struct StepLevel {
  int blk_end;               // first block past this level
  int active;                // evaluated and updated by this launch
  int image_on;              // this step contributes to the image (two-field launches)
  int pad_;
  void* r0[2];               // per field: newest right-hand side (written)
  const void* r1[2];         // per field: the two older ones (read)
  const void* r2[2];
  const void* qf_read[2];    // per field: traces of this level's elements AT THE STEP START, as seen by readers
  void* qf_write[2];         // per field: traces at the end of this level's step
  void* qf_half[2];          // per field: half-step traces (19) for finer neighbours (null: none needed)
  void* capture;             // field 0: boundary-trace record written at this evaluation, or null
  const void* replay;        // field 0: record read as exterior state of the stored faces, or null
  double c[3];               // dts * a_s   (eq (18))
  double d[3];               // dts * (b_s - a_s): half-step value = updated value + sum d_s r_s  (eq (19))
  double dts;                // signed local step
  double abar[3], C[9];      // image weights of the AB order in use (eqs (22)-(24), reading Q1)
};

struct StepArgs {
  void* q[2];                // nodal values of field 0 (source / forward) and field 1 (receivers)
  int nfields;
  int blk0, nblk;            // block range covered by the launch (levels l_min .. L-1)
  int nlevels;
  const void* geo; const int* nbr; const int* wperm;
  const unsigned char* blkflag;   // per block: bit 0 = some element has a finer face neighbour
  unsigned* sched; int sched_sel;   // two ticket counters of the pipelined kernel's work distribution; this launch uses [sched_sel]
  int sched_mode;                   // 0: fixed contiguous chunks per CTA; 1: interleaved start, then blocks by ticket
  int reverse;                      // fixed chunks walked from their end: alternates from launch to launch, so a step starts
                                    // with the blocks the previous step left in L2 (matters when the mesh nearly fits it)
  const void* ext;           // prescribed exterior states or null
  // fused halo exchange of a domain decomposition (dg_halo_sources): a prescribed face b with halo_rec[b] >= 0 takes its
  // exterior state straight from the neighbouring sub-domain's trace buffer halo_src[halo_set[b]] (a peer pointer over
  // NVLink, or local), record halo_rec[b], node i at position halo_pos[b][i]; NULL halo_rec: every prescribed face reads ext
  const long long* halo_rec; const int* halo_set; const int* halo_pos;
  const void* halo_src[32];
  const void* halo_src2[32];   // the same for field 1 (backward phase: the receiver wavefield of the neighbouring sub-domain)
  double dir;
  // point terms (eq (15)): per field a per-slot row index (-1: none) into pt_val[row][Np], times pt_scale
  const int* pt_index[2]; const void* pt_val[2]; double pt_scale[2];
  void* image; double e[3]; int characteristic;
  int trapezoid;             // image integral by the trapezoid rule (21) instead of the AB-consistent (24)
  void* img_scratch;         // [block][4Np][32] scratch for the imaging scalars when they do not fit in shared memory
  OpsDev ops;                // D3T / LIFTT here are the PADDED tables: D3P [m][3][NPAD], LTP [j][NPAD]
  const void* ops2_D3Q;      // pipelined kernel: tile-packed tables D3Q [tile][m][RL], LTQ [tile][j][LL]
  const void* ops2_LTQ;
  StepLevel lv[8];
};

struct KernelTable {
  int N, precision, Np, Nfp;
  void (*rhs)(const RhsArgs&, cudaStream_t);
  void (*update)(const UpdateArgs&, cudaStream_t);
  void (*rk)(const RkArgs&, cudaStream_t);
  void (*image_update)(const ImageArgs&, cudaStream_t);
  void (*source)(const PointArgs&, cudaStream_t);
  void (*record)(const PointArgs&, cudaStream_t);
  void (*inject)(const PointArgs&, cudaStream_t);
  void (*capture)(const CaptureArgs&, cudaStream_t);
  void (*halo)(const HaloArgs&, cudaStream_t);
  void (*step)(const StepArgs&, cudaStream_t);        // one wavefield
  void (*step2)(const StepArgs&, cudaStream_t);       // two wavefields + imaging
  int step_npad;                                       // padded output count of the step kernel's tables
  // software-pipelined variant (pipe_kernel.cuh); pipe == nullptr if not instantiated for this (N, precision)
  void (*pipe)(const StepArgs&, cudaStream_t);
  void (*pipe2)(const StepArgs&, cudaStream_t);
  int pipe_TO, pipe_NT, pipe_RL, pipe_LL;
  size_t pipe_blob_bytes;                              // [D3Q | LTQ | Fmask | perm table], the kernel's table image
  // tensor-core variant (tc_kernel.cuh; fp32, one wavefield); tc == nullptr if not instantiated
  void (*tc)(const StepArgs&, cudaStream_t);
  int tc_K1, tc_K2, tc_NN;
  size_t tc_blob_bytes;                                // [B1 hi | B1 lo | B2 hi | B2 lo | Fmask | perm table]
  int (*init)();           // sets shared-memory attributes, reads the device's SM count; returns cudaError
  int (*take_error)();     // first error of a programmatic-dependent launch since the last call (cudaError), then cleared
};

const KernelTable* get_kernel_table(int N, int precision);

}  // namespace dgrtm
