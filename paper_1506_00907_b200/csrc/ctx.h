// Host runtime state behind the opaque dg_ctx handle of include/dgrtm.h.
#pragma once
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstring>
#include <stdexcept>
#include <string>
#include <thread>
#include <vector>

#include "../../include/dgrtm.h"
#include "kernels.h"
#include "mesh_setup.h"
#include "refelem.h"

namespace dgrtm {

constexpr int kMaxLevels = 8;
constexpr int kMaxHaloSets = 32;   // (neighbouring sub-domain, level of the elements behind the cut) pairs of one sub-domain

// kernel classes of the launch counter / per-kernel timing (dg_get_kernel_times)
enum KernelClass { KC_RHS = 0, KC_UPDATE, KC_HALO, KC_IMAGE, KC_SOURCE, KC_RECORD, KC_INJECT, KC_CAPTURE, KC_RK, KC_STEP, KC_STEP_IMAGE, KC_COUNT };
struct ProfEvent { cudaEvent_t a, b; int cls; };

struct ApiError : std::runtime_error {
  int code;
  ApiError(int c, const std::string& m) : std::runtime_error(m), code(c) {}
};

inline void cuda_check(cudaError_t e, const char* what) {
  if (e != cudaSuccess) throw ApiError(DG_ERR_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// One wavefield on the device: nodal values, the three most recent own right-hand sides (rotating
// buffers, never the physical shift of PAPER.md:344) and the exposed traces.
struct Field {
  char* q = nullptr;
  char* hist[3] = {nullptr, nullptr, nullptr};
  char* qf = nullptr;      // = qfb[0]: the array the unfused kernels (k_rhs, k_update, k_half) use
  // fused step kernel: traces double-buffered per level + half-step traces of coarse neighbours
  char* qfb[2] = {nullptr, nullptr};
  char* qfh = nullptr;
  int par[kMaxLevels];     // per level: which of qfb[] holds the level's current traces
  int cur[kMaxLevels];     // per level: which of hist[] holds the newest right-hand side
  int nhist[kMaxLevels];   // per level: number of valid history entries (start-up order, reading Q7)
  void reset_history() {
    for (int l = 0; l < kMaxLevels; ++l) { cur[l] = 0; nhist[l] = 0; par[l] = 0; }
  }
  const char* h(int l, int s) const { return hist[(cur[l] + 3 - s) % 3]; }   // s = 0 newest
};

// carves 256-byte aligned regions out of a caller-owned device buffer
struct Carver {
  char* base = nullptr;
  size_t used = 0;
  char* take(size_t bytes) {
    char* p = base ? base + used : nullptr;
    used += (bytes + 255) & ~(size_t)255;
    return p;
  }
};

// Adams-Bashforth weights of order 1..3 (eqs (18), (19), (22)-(24); readings Q1, Q7)
struct AbCoef {
  double a[3], b[3], abar[3], C[9];
};
const AbCoef& ab_coef(int order);
// I_s(theta) = int_0^theta l_s for the order-`order` interpolant (22)
void ab_partial(int order, double theta, double w[3]);
double ricker(double t, double f0, double tp, double amp);

}  // namespace dgrtm

#define DG_TRY(ctx) \
  if (!(ctx)) return DG_ERR_ARG; \
  try {
#define DG_CATCH(ctx) \
  } catch (const dgrtm::ApiError& e) { (ctx)->err = e.what(); return e.code; \
  } catch (const std::bad_alloc&) { (ctx)->err = "out of host memory"; return DG_ERR_NOMEM; \
  } catch (const std::exception& e) { (ctx)->err = e.what(); return DG_ERR_ARG; } \
  return DG_OK;

struct dg_ctx {
  std::string err;
  int N = 0, precision = 0, Np = 0, Nfp = 0, NF = 0, REC = 0;
  size_t rs = 4;                            // sizeof(real)
  dgrtm::RefElem re;
  dgrtm::Mesh mesh;
  dgrtm::Model model;
  dgrtm::Locator locator;
  const dgrtm::KernelTable* kt = nullptr;
  bool has_model = false;
  int integrator = DG_INTEGRATOR_AB3;
  double dt_local = 0;
  int nlocal = 1;                           // fine steps per global step
  bool has_prescribed = false;

  // point source (eq (15))
  bool has_src = false;
  int64_t src_k = -1;
  std::vector<double> src_w;
  double f0 = 0, tp = 0, amp = 0;
  // receivers
  int64_t nr = 0;
  int64_t nr_reserve = 0;                   // rtm_set_receiver_capacity
  int64_t nr_cap = 0;                       // receiver capacity of the bound RTM region
  bool data_valid = false;                  // d_data holds signals of the current receiver set
  std::vector<int32_t> rcv_k;
  std::vector<double> rcv_row, rcv_w;
  std::vector<int32_t> grp_slot, grp_off, grp_rcv;   // receivers grouped by element, groups by level
  int grp_lvl0[dgrtm::kMaxLevels + 1];

  // ---- forward workspace
  bool bound = false;
  char* ws = nullptr;
  size_t ws_bytes = 0;
  cudaStream_t stream = nullptr;
  dgrtm::OpsDev ops;
  char* geo = nullptr;
  int* nbr = nullptr;
  int* wperm = nullptr;
  dgrtm::Field F;
  char* scratch = nullptr;                  // LSERK4 residual / dg_get_rhs output
  char* ext = nullptr;                      // prescribed exterior states [nbnd][Nfp][2]
  bool has_ext = false;
  char* d_src_w = nullptr;
  char* d_D3P = nullptr;                    // step kernel's padded operator tables [m][3][NPAD], [j][NPAD]
  char* d_LTP = nullptr;
  char* d_D3Q = nullptr;                    // pipelined kernel's tile-packed tables
  char* d_LTQ = nullptr;
  bool use_pipe = true;                     // DGRTM_KERNEL=step selects the non-pipelined fused kernel
  bool use_tc = false;                      // DGRTM_KERNEL=tc selects the tensor-core kernel (fp32, one wavefield)
  unsigned char* d_blkflag = nullptr;       // per block: bit 0 = some element has a finer face neighbour; then the ticket counters
  int sched_sel = 0;                        // ticket counter the next pipelined launch uses (the kernel zeroes the other one)
  int* d_pt_src = nullptr;                  // per slot: 0 at the source element, else -1
  // ---- halo faces of a domain decomposition (dg_set_halo): tables [bnd | rec | pos] in one carved region
  char* d_halo = nullptr;
  int64_t halo_off[dgrtm::kMaxHaloSets + 1] = {};   // faces of halo set s (one set per neighbouring sub-domain): [halo_off[s], halo_off[s+1])
  // the same tables by boundary face for the fused exchange (dg_halo_sources): host mirrors, device [hrec | hset | hpos]
  char* d_halo_face = nullptr;
  std::vector<long long> h_hrec; std::vector<int32_t> h_hset, h_hpos;
  const void* halo_src[dgrtm::kMaxHaloSets] = {};   // source buffers of the next step's launches
  bool halo_src_valid = false;              // set by dg_halo_sources, consumed by the next dg_step / dg_step_fine
  const void* halo_src2[dgrtm::kMaxHaloSets] = {};  // the same for the receiver wavefield (rtm_halo_sources)
  bool halo_src2_valid = false;
  bool part_fresh = false;                  // the phase is initialised and no fine step of it has run
  int part_phase = 0, part_nsteps = 0;      // rtm_forward_part / rtm_backward_part: phase in progress (1 forward, 2 backward), its global steps
  std::vector<double> bnd_Zext;             // exterior impedance per boundary face (> 0: Z_f = (Z- + Zext) / 2), dg_set_exterior_impedance
  int* d_stored[dgrtm::kMaxLevels];         // per level: slot*4+f of the stored boundary faces
  double t0 = 0;
  int64_t fine = 0;                         // time = t0 + fine * dt_local

  // ---- RTM region
  bool hist_bound = false;
  int hist_nsteps = 0;
  char* hs = nullptr;
  size_t hs_bytes = 0;
  char* rec[dgrtm::kMaxLevels];             // per level: trace records [nrec][nfaces][2][Nfp]
  char* d_data = nullptr;                   // [nr][nfine+1] recorded / injected signals
  int* d_rcv_slot = nullptr;
  int* d_rcv_level = nullptr;
  char* d_rcv_row = nullptr;
  char* d_rcv_w = nullptr;
  int* d_grp_slot = nullptr;
  int* d_grp_off = nullptr;
  int* d_grp_rcv = nullptr;
  int* d_pt_rcv = nullptr;                  // per slot: receiver group of the element or -1
  char* d_pt_val = nullptr;                 // [ngroups][Np] injection amounts of the current fine step
  dgrtm::Field R;                           // receiver wavefield of the backward phase
  char* image = nullptr;
  char* qfinal = nullptr;
  bool have_final = false, have_backward = false;
  int final_nsteps = 0;
  // ---- boundary-trace spill to host memory (off by default): the device
  // keeps a ring of spill_window << level records per level, the whole history lives in caller-owned pinned host memory
  char* spill_host = nullptr;
  size_t spill_bytes = 0;
  int spill_window = 0;                     // records of the coarsest level on the device; 0 = no spill
  bool spill_packed = false;                // the host copy keeps every value in half the bytes (rtm_set_spill_packing)
  char* pack_stage = nullptr;               // device staging of one packed record (carved from the RTM region)
  char* hrec[dgrtm::kMaxLevels];            // per level: the host copy [nrec][nfaces][2][Nfp]
  cudaStream_t copy_stream = nullptr;
  std::vector<int64_t> slot_rec[dgrtm::kMaxLevels];   // record held (or being loaded) by every ring slot, -1 = none
  std::vector<cudaEvent_t> ev_step[dgrtm::kMaxLevels];   // bound stream: the launch that wrote / read the slot
  std::vector<cudaEvent_t> ev_copy[dgrtm::kMaxLevels];   // copy stream: the slot's last transfer

  // pinned host staging for the field transfers of dg_set_state / dg_get_fields / rtm_get_fields (grown on demand)
  char* stage_host = nullptr;
  size_t stage_bytes = 0;
  int64_t launches = 0;
  // per-kernel timing (dg_set_profiling): one CUDA event pair per launch on the bound stream
  bool prof = false;
  std::vector<dgrtm::ProfEvent> prof_ev;
  ~dg_ctx();
};

namespace dgrtm {

// ---- helpers shared by the api_*.cpp files
size_t field_bytes(const dg_ctx* c);        // one [nslots][4Np] array
// the two ticket counters of the pipelined kernel: 16-byte aligned behind the block flags (zeroed with them)
inline unsigned* sched_counters(const dg_ctx* c) {
  return reinterpret_cast<unsigned*>(((uintptr_t)c->d_blkflag + (size_t)c->model.nblocks + 15) & ~(uintptr_t)15);
}
size_t trace_bytes(const dg_ctx* c);        // one qf array
void upload_real(dg_ctx* c, void* dst, const double* src, size_t n);
void download_real(dg_ctx* c, double* dst, const void* src, size_t n);
void upload_raw(dg_ctx* c, void* dst, const void* src, size_t bytes);
void sync_stream(dg_ctx* c);
// user order q[K][4][Np]  <->  device [block][4Np][32]
void fields_to_device(dg_ctx* c, char* dq, const double* q);
void fields_from_device(dg_ctx* c, double* q, const char* dq);
// [0, n) split over host threads (conversions between the caller's doubles and the device precision)
template <typename F> void parallel_range(size_t n, F body) {
  unsigned nt = std::thread::hardware_concurrency();
  nt = nt == 0 ? 1 : (nt > 16 ? 16 : nt);
  if (n < (size_t)1 << 16) nt = 1;
  if (nt == 1) { body((size_t)0, n); return; }
  std::vector<std::thread> th;
  const size_t per = (n + nt - 1) / nt;
  for (unsigned t = 0; t < nt; ++t) {
    const size_t a = t * per, b = std::min(n, a + per);
    if (a >= b) break;
    th.emplace_back([=] { body(a, b); });
  }
  for (auto& x : th) x.join();
}
char* host_stage(dg_ctx* c, size_t bytes);   // the ctx's pinned staging buffer, at least `bytes` large
void image_from_device(dg_ctx* c, double* I, const char* dimg);   // user order I[K][Np] <- device [block][Np][32]
void refresh_traces(dg_ctx* c, Field& F);   // qf := traces of q, all levels
void normalize_traces(dg_ctx* c, Field& F);
void upload_point_source(dg_ctx* c);        // per-slot point-term index of the forward field // current traces of every level -> qfb[0] (= qf)
void clear_field(dg_ctx* c, Field& F);
void upload_receiver_tables(dg_ctx* c);     // receiver rows / weights / groups -> the bound RTM region
// trace records: device address of record j of level l (a ring slot when the history spills to the host), and the
// stream choreography around the launch that captures (forward) or replays (backward) it
char* record_ptr(dg_ctx* c, int l, int64_t j);
void spill_before_capture(dg_ctx* c, int l, int64_t j);
void spill_after_capture(dg_ctx* c, int l, int64_t j);
void spill_before_replay(dg_ctx* c, int l, int64_t j);
void spill_after_replay(dg_ctx* c, int l, int64_t j);
// trace_pack.cu: n values of the device precision <-> n values of half the size (fp64 <-> fp32, fp32 <-> bf16)
void launch_trace_pack(const void* src, void* dst, size_t n, int precision, cudaStream_t s);
void launch_trace_unpack(const void* src, void* dst, size_t n, int precision, cudaStream_t s);
void restart_history(dg_ctx* c);            // after dg_set_integrator / dg_set_dt

struct RunOpts {
  int direction = 1;
  Field* fields[2] = {nullptr, nullptr};
  int nfields = 1;
  bool source_on[2] = {false, false};
  bool capture = false, replay = false, record = false;
  int inject_field = -1;
  bool finish = true;                        // the run reaches the end of the phase: final capture / final receiver sample
  int64_t fine_phase = 0, nfine = -1;        // dg_step_fine: fine index within the cycle at the start, fine steps to run (-1: whole global steps)
  bool image = false;
  int imaging = DG_IMAGING_CHARACTERISTIC;
  double updir[3] = {0, 0, -1};
  int64_t image_min_fine = 0;               // steps whose end index (forward numbering) is below do not image
  int64_t first_fine = 0;                   // absolute fine index of the start time, forward numbering
  double t0 = 0;                            // start time
};
void run_mrab(dg_ctx* c, int nglobal, const RunOpts& o);
void run_lserk4(dg_ctx* c, int nsteps);
void launch_rhs(dg_ctx* c, Field& F, char* out, int l0, int l1, int mode, double dir, char* capture,
                const char* replay);
void carve_workspace(dg_ctx* c, Carver& cv);
void require_bound(dg_ctx* c);
void check_launches(dg_ctx* c);             // cudaGetLastError + the first failed dependent launch, as DG_ERR_CUDA

// counts a launch and, in profiling mode, brackets it with an event pair on the bound stream
struct LaunchScope {
  dg_ctx* c; bool on;
  ProfEvent e;
  LaunchScope(dg_ctx* ctx, int cls) : c(ctx), on(ctx->prof) {
    c->launches++;
    if (on) {
      e.cls = cls;
      cuda_check(cudaEventCreate(&e.a), "cudaEventCreate");
      cuda_check(cudaEventCreate(&e.b), "cudaEventCreate");
      cudaEventRecord(e.a, c->stream);
    }
  }
  ~LaunchScope() {
    if (on) { cudaEventRecord(e.b, c->stream); c->prof_ev.push_back(e); }
  }
};

}  // namespace dgrtm

#define DG_LAUNCH(ctx_, cls_, call_) do { dgrtm::LaunchScope ls_((ctx_), (cls_)); call_; } while (0)
